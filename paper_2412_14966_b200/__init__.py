"""B200-native primary-vertex finder hot path of arXiv:2412.14966.

The product is the C-ABI shared library `libpvfinder.so` (include/pv_finder.h) built from csrc/ for sm_100a;
this package is its thin Python binding.
"""
from .binding import (DeviceBatch, HostPipeline, Params, Debug, PvError, default_params, multivertex_params, find, lib, nbins,  # noqa: F401
                      workspace_bytes, last_launch_info, EXPORTS, FIELDS)
from . import shard  # noqa: F401,E402
