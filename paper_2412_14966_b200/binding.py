"""Thin ctypes binding of the C ABI in include/pv_finder.h (argument marshalling only; every step of the
hot path runs in the CUDA kernels of csrc/).  PyTorch is used for device memory and streams only.

There is no CPU fallback: if libpvfinder.so is missing or no CUDA device is present, the calls raise.
"""
from __future__ import annotations

import ctypes as C
import os
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libpvfinder.so")

FIXED_ONE = 1 << 20
MAX_BINS = 4096
MAX_VTX = 32
MAX_TRACKS_PER_EVENT = 2047
EVT_TOO_MANY_TRACKS = 1
EVT_VTX_OVERFLOW = 2
EVT_SINGULAR_FIT = 4
EVT_RECORD_OVERFLOW = 8
STATIC_WORKSPACE_BYTES = 16 << 20
E_STATIC_LIMIT = -6
FLAVOUR_EXPLICIT = 0
FLAVOUR_MULTIVERTEX = 1
FILL_POLYNOMIAL = 0
FILL_TEMPLATE = 1

FIELDS = ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")

EXPORTS = (
    "pv_params_default", "pv_nbins", "pv_workspace_bytes", "pv_find", "pv_find_debug", "pv_find_ext", "pv_find_static", "pv_track_ip",
    "pv_host_ctx_create", "pv_host_ctx_destroy", "pv_find_host", "pv_find_host_compact", "pv_host_register", "pv_host_unregister",
    "pv_last_launch_info", "pv_kernel_timing", "pv_kernel_time_ms", "pv_kernel_times_ms", "pv_error_string", "pv_last_cuda_error",
)


class Params(C.Structure):
    """struct pv_params (include/pv_finder.h)."""
    _fields_ = [
        ("z_min", C.c_float), ("z_max", C.c_float), ("dz", C.c_float), ("z_split", C.c_float),
        ("beam_x", C.c_float), ("beam_y", C.c_float), ("beam_tx", C.c_float), ("beam_ty", C.c_float),
        ("max_sigma_poca", C.c_float * 2), ("min_bin_content", C.c_float), ("min_dip", C.c_float),
        ("min_cluster_integral", C.c_float * 2), ("min_tracks_seed", C.c_int32 * 2),
        ("min_tracks_pv", C.c_int32 * 2), ("chi2_max", C.c_float), ("max_iter", C.c_int32),
        ("conv_dchi2", C.c_float), ("conv_dz", C.c_float), ("merge_ratio", C.c_float),
        ("max_beam_dist", C.c_float), ("max_vtx_per_event", C.c_int32),
        ("flavour", C.c_int32), ("chi2_window", C.c_float), ("split_mode", C.c_int32), ("fill_mode", C.c_int32),
    ]


class Debug(C.Structure):
    """struct pv_debug (include/pv_finder.h)."""
    _fields_ = [
        ("hist", C.c_void_p), ("n_hist_events", C.c_int32),
        ("z_poca", C.c_void_p), ("sigma_poca", C.c_void_p), ("trk_bin", C.c_void_p),
        ("n_seeds_raw", C.c_void_p), ("n_seeds", C.c_void_p), ("seed_z", C.c_void_p), ("seed_bins", C.c_void_p),
        ("trk_seed", C.c_void_p), ("seed_pos", C.c_void_p), ("seed_cov", C.c_void_p), ("seed_chi2", C.c_void_p),
        ("seed_ntrk", C.c_void_p), ("seed_niter", C.c_void_p), ("seed_fate", C.c_void_p),
    ]


class TrackCov(C.Structure):
    """struct pv_track_cov (include/pv_finder.h): optional x-tx / y-ty covariance elements, DEVICE pointers."""
    _fields_ = [("cov_xtx", C.c_void_p), ("cov_yty", C.c_void_p)]


# struct pv_vertex (include/pv_finder.h): one PV as pv_find_host_compact returns it
VERTEX_DTYPE = np.dtype([("pos", np.float32, 3), ("cov", np.float32, 6), ("chi2", np.float32),
                         ("ntracks", np.int32), ("niter", np.int32)])
assert VERTEX_DTYPE.itemsize == 48


class PvError(RuntimeError):
    pass


_lib = None


def lib():
    """Load libpvfinder.so (built by paper_2412_14966_b200.build).  Fails loudly if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise PvError(f"{_SO} not found: run `python -m paper_2412_14966_b200.build` (there is no CPU fallback)")
        L = C.CDLL(_SO)
        vp, i32, i64 = C.c_void_p, C.c_int, C.c_longlong
        L.pv_params_default.argtypes = [C.POINTER(Params)]
        L.pv_nbins.argtypes = [C.POINTER(Params)]
        L.pv_workspace_bytes.argtypes = [i32, i64, C.POINTER(Params), C.POINTER(C.c_size_t)]
        find_args = [vp] * 9 + [vp, i32, i64, C.POINTER(Params)] + [vp] * 9 + [vp, C.c_size_t, vp]
        L.pv_find.argtypes = find_args
        L.pv_find_debug.argtypes = find_args + [C.POINTER(Debug)]
        L.pv_find_ext.argtypes = find_args + [C.POINTER(TrackCov), C.POINTER(Debug)]
        L.pv_find_static.argtypes = find_args[:-3] + [vp]
        L.pv_track_ip.argtypes = [vp] * 9 + [vp, i32, i64, C.POINTER(Params)] + [vp] * 3 + [vp] * 3 + [C.POINTER(TrackCov), vp]
        L.pv_host_ctx_create.argtypes = [C.POINTER(vp), i32, i64, C.POINTER(Params), i32]
        L.pv_host_ctx_destroy.argtypes = [vp]
        L.pv_find_host.argtypes = [vp] + [vp] * 9 + [vp, i32, C.POINTER(Params)] + [vp] * 9 + [i32]
        L.pv_find_host_compact.argtypes = [vp] + [vp] * 9 + [vp, i32, C.POINTER(Params)] + [vp, i64, vp, vp, vp, vp, vp, i32]
        L.pv_host_register.argtypes = [vp, C.c_size_t]
        L.pv_host_unregister.argtypes = [vp]
        L.pv_last_launch_info.argtypes = [C.POINTER(i32)] * 4
        L.pv_kernel_timing.argtypes = [i32]
        L.pv_kernel_time_ms.restype = C.c_float
        L.pv_kernel_times_ms.argtypes = [C.POINTER(C.c_float), i32]
        L.pv_error_string.argtypes = [i32]
        L.pv_error_string.restype = C.c_char_p
        L.pv_last_cuda_error.restype = C.c_char_p
        _lib = L
    return _lib


def _check(rc: int, what: str):
    if rc != 0:
        L = lib()
        msg = L.pv_error_string(rc).decode()
        cerr = L.pv_last_cuda_error().decode()
        raise PvError(f"{what} failed: {rc} ({msg}){': ' + cerr if cerr and rc == -4 else ''}")


def default_params(**over) -> Params:
    p = Params()
    _check(lib().pv_params_default(C.byref(p)), "pv_params_default")
    for k, v in over.items():
        cur = getattr(p, k)
        if hasattr(cur, "__len__"):
            for i, vi in enumerate(v):
                cur[i] = vi
        else:
            setattr(p, k, v)
    return p


def multivertex_params(**over) -> Params:
    """The paper's GPU flavour: implicit association, Eq. 19 weights, convergence on
    |dz| < 0.5 um alone (conv_dchi2 = inf)."""
    kw = dict(flavour=FLAVOUR_MULTIVERTEX, conv_dchi2=float("inf"), conv_dz=5e-4)
    kw.update(over)
    return default_params(**kw)


def nbins(p: Params) -> int:
    n = lib().pv_nbins(C.byref(p))
    if n < 0:
        _check(n, "pv_nbins")
    return n


def workspace_bytes(n_events: int, n_tracks: int, p: Params) -> int:
    out = C.c_size_t(0)
    _check(lib().pv_workspace_bytes(n_events, n_tracks, C.byref(p), C.byref(out)), "pv_workspace_bytes")
    return out.value


def last_launch_info() -> Dict[str, int]:
    a, b, c, d = C.c_int(0), C.c_int(0), C.c_int(0), C.c_int(0)
    lib().pv_last_launch_info(C.byref(a), C.byref(b), C.byref(c), C.byref(d))
    return dict(n_kernels=a.value, grid=b.value, block=c.value, smem_bytes=d.value)


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise PvError("no CUDA device: the PV finder has no CPU fallback")
    return torch


class DeviceBatch:
    """Track SoA + offsets resident in HBM, plus caller-owned output buffers and workspace (torch tensors)."""

    def __init__(self, data: Dict[str, np.ndarray], p: Params, device: str = "cuda:0", debug: bool = False,
                 n_hist_events: int = 0):
        torch = _torch()
        self.device = torch.device(device)
        self.p = p
        off = np.ascontiguousarray(data["offsets"], dtype=np.int32)
        self.E = int(off.size - 1)
        self.T = int(off[-1]) if off.size else 0
        dev = self.device
        self.inp = {k: torch.from_numpy(np.ascontiguousarray(data[k], dtype=np.float32)).to(dev) for k in FIELDS}
        self.offsets = torch.from_numpy(off).to(dev)
        self.cov = None                                    # optional covariance cross terms (Eq. 2)
        if "cov_xtx" in data or "cov_yty" in data:
            zero = np.zeros(self.T, np.float32)
            self.cov_t = [torch.from_numpy(np.ascontiguousarray(data.get(k, zero), dtype=np.float32)).to(dev)
                          for k in ("cov_xtx", "cov_yty")]
            self.cov = TrackCov(self.cov_t[0].data_ptr(), self.cov_t[1].data_ptr())
        mv = p.max_vtx_per_event
        E, T = self.E, self.T
        z = lambda shape, dt: torch.zeros(shape, dtype=dt, device=dev)
        self.out = dict(
            vtx_pos=z((E, mv, 3), torch.float32), vtx_cov=z((E, mv, 6), torch.float32), vtx_chi2=z((E, mv), torch.float32),
            vtx_ntracks=z((E, mv), torch.int32), vtx_niter=z((E, mv), torch.int32), n_vtx=z((E,), torch.int32),
            trk_weight=z((T,), torch.float32), trk_vertex=torch.full((T,), -1, dtype=torch.int32, device=dev),
            event_status=z((E,), torch.int32))
        self.workspace = torch.zeros(max(workspace_bytes(E, T, p), 256), dtype=torch.uint8, device=dev)
        self.dbg = None
        self.dbg_struct = None
        if debug:
            nb = nbins(p)
            nh = min(int(n_hist_events), E)
            self.dbg = dict(
                hist=z((max(nh, 1), nb), torch.int32), z_poca=z((T,), torch.float32), sigma_poca=z((T,), torch.float32),
                trk_bin=torch.full((T,), -1, dtype=torch.int32, device=dev),
                n_seeds_raw=z((E,), torch.int32), n_seeds=z((E,), torch.int32), seed_z=z((E, mv), torch.float32),
                seed_bins=z((E, mv, 3), torch.int32), trk_seed=torch.full((T,), -1, dtype=torch.int32, device=dev),
                seed_pos=z((E, mv, 3), torch.float32), seed_cov=z((E, mv, 6), torch.float32),
                seed_chi2=z((E, mv), torch.float32), seed_ntrk=z((E, mv), torch.int32),
                seed_niter=z((E, mv), torch.int32), seed_fate=torch.full((E, mv), -9, dtype=torch.int32, device=dev))
            d = Debug()
            for name, _t in Debug._fields_:
                if name == "n_hist_events":
                    d.n_hist_events = nh
                else:
                    setattr(d, name, self.dbg[name].data_ptr())
            if nh == 0:
                d.hist = None
            self.dbg_struct = d

    def bytes_in(self) -> int:
        return self.T * 36 + (self.E + 1) * 4

    def find(self, stream=None) -> None:
        """Enqueue pv_find (or pv_find_debug) on `stream` (torch.cuda.Stream; default: current stream)."""
        torch = _torch()
        L = lib()
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        i, o = self.inp, self.out
        args = [i[k].data_ptr() for k in FIELDS] + [self.offsets.data_ptr(), self.E, self.T, C.byref(self.p)] + [
            o["vtx_pos"].data_ptr(), o["vtx_cov"].data_ptr(), o["vtx_chi2"].data_ptr(), o["vtx_ntracks"].data_ptr(),
            o["vtx_niter"].data_ptr(), o["n_vtx"].data_ptr(), o["trk_weight"].data_ptr(), o["trk_vertex"].data_ptr(),
            o["event_status"].data_ptr(), self.workspace.data_ptr(), self.workspace.numel(), s.cuda_stream]
        with torch.cuda.device(self.device):
            if self.cov is not None:
                _check(L.pv_find_ext(*args, C.byref(self.cov), C.byref(self.dbg_struct) if self.dbg_struct is not None else None),
                       "pv_find_ext")
            elif self.dbg_struct is not None:
                _check(L.pv_find_debug(*args, C.byref(self.dbg_struct)), "pv_find_debug")
            else:
                _check(L.pv_find(*args), "pv_find")

    def find_static(self, stream=None) -> None:
        """Enqueue pv_find_static on `stream`: pv_find for callers that may not allocate device memory (a plug-in of a
        framework that owns the GPU's memory, a loop in which cudaMalloc is forbidden).  Its scratch is the 16 MiB
        array built into the library instead of self.workspace, so the batch must need no more than
        STATIC_WORKSPACE_BYTES (PvError with code -6 otherwise), and calls that may overlap on the GPU must not be
        issued.  No taps, no covariance cross terms."""
        torch = _torch()
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        i, o = self.inp, self.out
        args = [i[k].data_ptr() for k in FIELDS] + [self.offsets.data_ptr(), self.E, self.T, C.byref(self.p)] + [
            o["vtx_pos"].data_ptr(), o["vtx_cov"].data_ptr(), o["vtx_chi2"].data_ptr(), o["vtx_ntracks"].data_ptr(),
            o["vtx_niter"].data_ptr(), o["n_vtx"].data_ptr(), o["trk_weight"].data_ptr(), o["trk_vertex"].data_ptr(),
            o["event_status"].data_ptr(), s.cuda_stream]
        with torch.cuda.device(self.device):
            _check(lib().pv_find_static(*args), "pv_find_static")

    def track_ip(self, stream=None) -> None:
        """Enqueue pv_track_ip on the vertices of the last find(); results in self.ip (ip, ip_chi2, ip_vertex)."""
        torch = _torch()
        s = stream if stream is not None else torch.cuda.current_stream(self.device)
        if not hasattr(self, "ip"):
            self.ip = dict(ip=torch.zeros(self.T, dtype=torch.float32, device=self.device),
                           ip_chi2=torch.zeros(self.T, dtype=torch.float32, device=self.device),
                           ip_vertex=torch.zeros(self.T, dtype=torch.int32, device=self.device))
        i, o = self.inp, self.out
        args = [i[k].data_ptr() for k in FIELDS] + [self.offsets.data_ptr(), self.E, self.T, C.byref(self.p)] + [
            o["vtx_pos"].data_ptr(), o["vtx_cov"].data_ptr(), o["n_vtx"].data_ptr(),
            self.ip["ip"].data_ptr(), self.ip["ip_chi2"].data_ptr(), self.ip["ip_vertex"].data_ptr(),
            C.byref(self.cov) if self.cov is not None else None, s.cuda_stream]
        with torch.cuda.device(self.device):
            _check(lib().pv_track_ip(*args), "pv_track_ip")

    def ip_results(self) -> Dict[str, np.ndarray]:
        _torch().cuda.synchronize(self.device)
        return {k: v.cpu().numpy() for k, v in self.ip.items()}

    def results(self) -> Dict[str, np.ndarray]:
        torch = _torch()
        torch.cuda.synchronize(self.device)
        r = {k: v.cpu().numpy() for k, v in self.out.items()}
        r["event_status"] = r["event_status"].view(np.uint32)
        if self.dbg is not None:
            r["debug"] = {k: v.cpu().numpy() for k, v in self.dbg.items()}
        return r


def find(data: Dict[str, np.ndarray], p: Optional[Params] = None, device: str = "cuda:0", debug: bool = False,
         n_hist_events: int = 0) -> Dict[str, np.ndarray]:
    """Convenience: upload a synth.events batch, run the hot path once, download the results."""
    if p is None:
        p = default_params()
    b = DeviceBatch(data, p, device=device, debug=debug, n_hist_events=n_hist_events)
    b.find()
    return b.results()


class HostPipeline:
    """pv_find_host: HOST numpy buffers in, HOST numpy buffers out; H2D / kernel / D2H are pipelined over the
    context's streams inside the library."""

    def __init__(self, max_events: int, max_tracks: int, p: Params, n_streams: int = 4, device: str = "cuda:0"):
        torch = _torch()
        self.device = torch.device(device)
        self.p = p
        self.ctx = C.c_void_p(None)
        with torch.cuda.device(self.device):
            _check(lib().pv_host_ctx_create(C.byref(self.ctx), max_events, max_tracks, C.byref(p), n_streams),
                   "pv_host_ctx_create")
        self.max_events, self.max_tracks = max_events, max_tracks
        self._pinned = []

    def alloc_outputs(self, E: int, T: int, pinned: bool = True, compact: bool = True) -> Dict[str, np.ndarray]:
        """Pinned host output buffers.  compact (pv_find_host_compact): `vertices` (pv_vertex records, capacity
        E * max_vtx), `vtx_begin` [E + 1], int8 `trk_vertex`; else the fixed-stride arrays of pv_find_host."""
        torch = _torch()
        mv = self.p.max_vtx_per_event
        if compact:
            spec = dict(vertices=((E * mv * 48,), torch.uint8), vtx_begin=((E + 1,), torch.int32), n_vtx=((E,), torch.int32),
                        trk_weight=((T,), torch.float32), trk_vertex=((T,), torch.int8), event_status=((E,), torch.int32))
        else:
            spec = dict(vtx_pos=((E, mv, 3), torch.float32), vtx_cov=((E, mv, 6), torch.float32), vtx_chi2=((E, mv), torch.float32),
                        vtx_ntracks=((E, mv), torch.int32), vtx_niter=((E, mv), torch.int32), n_vtx=((E,), torch.int32),
                        trk_weight=((T,), torch.float32), trk_vertex=((T,), torch.int32), event_status=((E,), torch.int32))
        out = {}
        for k, (shape, dt) in spec.items():
            t = torch.zeros(shape, dtype=dt, pin_memory=pinned)
            self._pinned.append(t)
            out[k] = t.numpy().view(VERTEX_DTYPE) if k == "vertices" else t.numpy()
        return out

    def pin_inputs(self, data: Dict[str, np.ndarray]) -> Dict[str, np.ndarray]:
        """Copy a batch into pinned host memory (once, outside any timed region)."""
        torch = _torch()
        out = {}
        for k in FIELDS + ("offsets",):
            dt = np.int32 if k == "offsets" else np.float32
            t = torch.from_numpy(np.ascontiguousarray(data[k], dtype=dt)).pin_memory()
            self._pinned.append(t)
            out[k] = t.numpy()
        return out

    def find(self, data: Dict[str, np.ndarray], out: Dict[str, np.ndarray], n_chunks: int = 8) -> None:
        """pv_find_host_compact when `out` holds `vertices` (alloc_outputs(compact=True)), else pv_find_host."""
        torch = _torch()
        E = int(data["offsets"].size - 1)
        ptr = lambda a: a.ctypes.data
        with torch.cuda.device(self.device):
            if "vertices" in out:
                rc = lib().pv_find_host_compact(
                    self.ctx, *[ptr(data[k]) for k in FIELDS], ptr(data["offsets"]), E, C.byref(self.p),
                    ptr(out["vertices"]), out["vertices"].size, ptr(out["vtx_begin"]), ptr(out["n_vtx"]),
                    ptr(out["trk_weight"]), ptr(out["trk_vertex"]), ptr(out["event_status"]), n_chunks)
                _check(rc, "pv_find_host_compact")
            else:
                rc = lib().pv_find_host(
                    self.ctx, *[ptr(data[k]) for k in FIELDS], ptr(data["offsets"]), E, C.byref(self.p),
                    ptr(out["vtx_pos"]), ptr(out["vtx_cov"]), ptr(out["vtx_chi2"]), ptr(out["vtx_ntracks"]),
                    ptr(out["vtx_niter"]), ptr(out["n_vtx"]), ptr(out["trk_weight"]), ptr(out["trk_vertex"]),
                    ptr(out["event_status"]), n_chunks)
                _check(rc, "pv_find_host")

    def bytes_per_call(self, data: Dict[str, np.ndarray], out: Dict[str, np.ndarray]):
        """(host->device, device->host) bytes the last find() moved, counted from the buffers it copies."""
        E = int(data["offsets"].size - 1)
        T = int(data["offsets"][-1])
        h2d = T * 36 + (E + 1) * 4
        if "vertices" in out:
            nv = int(out["vtx_begin"][E])
            d2h = nv * 48 + E * 8 + T * 5 + 4 * min(E, 256)
        else:
            d2h = E * self.p.max_vtx_per_event * 48 + E * 8 + T * 8
        return h2d, d2h

    def matches(self, out: Dict[str, np.ndarray], dev: Dict[str, np.ndarray]) -> bool:
        """Bit-for-bit equality of a host-pipeline result with DeviceBatch.results() of the same batch."""
        mv = self.p.max_vtx_per_event
        nv = dev["n_vtx"]
        m = np.arange(mv)[None, :] < nv[:, None]
        ok = np.array_equal(out["n_vtx"], nv) and np.array_equal(out["event_status"].view(np.uint32), dev["event_status"])
        ok = ok and np.array_equal(out["trk_weight"], dev["trk_weight"]) and np.array_equal(out["trk_vertex"].astype(np.int32), dev["trk_vertex"])
        if not ok:
            return False
        if "vertices" in out:
            v = out["vertices"][:int(nv.sum())]
            return bool(np.array_equal(out["vtx_begin"], np.concatenate([[0], np.cumsum(nv)]).astype(np.int32))
                        and np.array_equal(v["pos"], dev["vtx_pos"][m]) and np.array_equal(v["cov"], dev["vtx_cov"][m])
                        and np.array_equal(v["chi2"], dev["vtx_chi2"][m]) and np.array_equal(v["ntracks"], dev["vtx_ntracks"][m])
                        and np.array_equal(v["niter"], dev["vtx_niter"][m]))
        return all(np.array_equal(out[k][m], dev[k][m]) for k in ("vtx_pos", "vtx_cov", "vtx_chi2", "vtx_ntracks", "vtx_niter"))

    def close(self):
        if self.ctx:
            lib().pv_host_ctx_destroy(self.ctx)
            self.ctx = C.c_void_p(None)

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass
