"""ctypes wrapper of the CPU ORACLE (oracle/pv_oracle.c).

TEST INFRASTRUCTURE ONLY: imported by tests/, __graft_entry__.smoke() and the cpu_baseline /
--impl reference legs of bench.py.  Never imported by paper_2412_14966_b200 (the product).
Argument marshalling only; every number comes out of pv_oracle.c.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from typing import Dict, Optional

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "libpvoracle.so")
_SRC = [os.path.join(_HERE, "pv_oracle.c"), os.path.join(_HERE, "pv_oracle.h")]

S = 1 << 20
TRACE_ITERS = 16
TRACE_STRIDE = 11
TRK_ASSIGNABLE = 1
TRK_HISTOGRAMMED = 2
EVT_TOO_MANY_TRACKS = 1
EVT_VTX_OVERFLOW = 2
EVT_SINGULAR_FIT = 4


class Params(C.Structure):
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
    _fields_ = [
        ("hist", C.c_void_p), ("n_hist_events", C.c_int32),
        ("z_poca", C.c_void_p), ("sigma_poca", C.c_void_p), ("trk_bin", C.c_void_p), ("trk_flags", C.c_void_p),
        ("n_seeds", C.c_void_p), ("n_seeds_raw", C.c_void_p), ("seed_z", C.c_void_p), ("seed_bins", C.c_void_p),
        ("trk_seed", C.c_void_p), ("seed_pos", C.c_void_p), ("seed_cov", C.c_void_p), ("seed_chi2", C.c_void_p),
        ("seed_ntrk", C.c_void_p), ("seed_niter", C.c_void_p), ("seed_fate", C.c_void_p), ("trace", C.c_void_p),
        ("seed_edge_last", C.c_void_p), ("seed_edge_any", C.c_void_p), ("seed_pivot_min", C.c_void_p),
        ("seed_nact_min", C.c_void_p), ("trk_w2", C.c_void_p), ("trk_w1", C.c_void_p),
    ]


def build(force: bool = False) -> str:
    """Compile pv_oracle.c with gcc (no fast-math, no FP contraction: the fp32 contract needs each
    operation rounded on its own)."""
    if not force and os.path.exists(_SO) and all(os.path.getmtime(_SO) >= os.path.getmtime(s) for s in _SRC):
        return _SO
    cmd = ["gcc", "-O2", "-std=gnu11", "-fPIC", "-shared", "-fopenmp", "-ffp-contract=off", "-fno-fast-math",
           "-Wall", "-Wextra", "-o", _SO, _SRC[0], "-lm"]
    subprocess.run(cmd, check=True)
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_SO)
        L.pvo_params_default.argtypes = [C.POINTER(Params)]
        L.pvo_nbins.argtypes = [C.POINTER(Params)]
        L.pvo_nbins.restype = C.c_int
        L.pvo_edge_q.argtypes = [C.c_int, C.c_float, C.c_float, C.POINTER(Params)]
        L.pvo_edge_q.restype = C.c_int32
        L.pvo_seed_z.argtypes = [C.c_void_p, C.c_int, C.POINTER(Params)]
        L.pvo_seed_z.restype = C.c_float
        L.pvo_peaks.restype = C.c_int
        L.pvo_assign.restype = C.c_int
        L.pvo_fit.restype = C.c_int
        L.pvo_find.restype = C.c_int
        L.pvo_fit_mv.restype = C.c_int
        L.pvo_tmpl_class.argtypes = [C.c_float, C.POINTER(Params)]
        L.pvo_tmpl_class.restype = C.c_int
        L.pvo_tmpl_halfwidth.argtypes = [C.c_int]
        L.pvo_tmpl_halfwidth.restype = C.c_int
        L.pvo_tmpl_bin.argtypes = [C.c_int, C.c_int, C.c_int]
        L.pvo_tmpl_bin.restype = C.c_int32
        L.pvo_mv_weight.restype = C.c_double
        L.pvo_mv_weight.argtypes = [C.c_double, C.c_double, C.c_void_p, C.c_int]
        L.pvo_track_chi2.restype = C.c_double
        L.pvo_ip_one.restype = C.c_int
        L.pvo_track_ip.restype = C.c_int
        _lib = L
    return _lib


class Cross(C.Structure):
    """struct pvo_cross: optional x-tx / y-ty covariance elements (Eq. 2)."""
    _fields_ = [("xtx", C.c_void_p), ("yty", C.c_void_p)]


def _cross(tracks):
    """(ctypes argument, keep-alive list) for the optional "cov_xtx" / "cov_yty" arrays of a track dict."""
    if "cov_xtx" not in tracks and "cov_yty" not in tracks:
        return None, []
    n = np.asarray(tracks["x"]).size
    a = _f32(tracks.get("cov_xtx", np.zeros(n, np.float32)))
    b = _f32(tracks.get("cov_yty", np.zeros(n, np.float32)))
    cx = Cross(a.ctypes.data, b.ctypes.data)
    return C.byref(cx), [a, b, cx]


def default_params(**over) -> Params:
    p = Params()
    lib().pvo_params_default(C.byref(p))
    for k, v in over.items():
        cur = getattr(p, k)
        if hasattr(cur, "__len__"):
            for i, vi in enumerate(v):
                cur[i] = vi
        else:
            setattr(p, k, v)
    return p


def nbins(p: Params) -> int:
    return lib().pvo_nbins(C.byref(p))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _ptr(a):
    return a.ctypes.data_as(C.c_void_p)


def project(x, y, z, tx, ty, var_x, p: Params):
    x, y, z, tx, ty, var_x = map(_f32, (x, y, z, tx, ty, var_x))
    n = x.size
    zp = np.empty(n, np.float32); sp = np.empty(n, np.float32)
    b = np.empty(n, np.int32); fl = np.empty(n, np.int32)
    lib().pvo_project(C.c_int(n), _ptr(x), _ptr(y), _ptr(z), _ptr(tx), _ptr(ty), _ptr(var_x), C.byref(p),
                      _ptr(zp), _ptr(sp), _ptr(b), _ptr(fl))
    return zp, sp, b, fl


def edge_q(k: int, zp: float, sp: float, p: Params) -> int:
    return int(lib().pvo_edge_q(int(k), C.c_float(zp), C.c_float(sp), C.byref(p)))


def fill(zp, sp, flags, p: Params, full_range: bool = False) -> np.ndarray:
    zp, sp, flags = _f32(zp), _f32(sp), _i32(flags)
    H = np.zeros(nbins(p), np.int32)
    lib().pvo_fill(C.c_int(zp.size), _ptr(zp), _ptr(sp), _ptr(flags), C.byref(p), _ptr(H), C.c_int(int(full_range)))
    return H


def tmpl_class(sigma_poca: float, p: Params) -> int:
    return int(lib().pvo_tmpl_class(C.c_float(sigma_poca), C.byref(p)))


def tmpl_halfwidth(k: int) -> int:
    return int(lib().pvo_tmpl_halfwidth(int(k)))


def tmpl(k: int, j: int) -> np.ndarray:
    """Template histogram (k, j): contents of the relative bins -W_k .. W_k."""
    W = tmpl_halfwidth(k)
    return np.array([lib().pvo_tmpl_bin(int(k), int(j), i) for i in range(-W, W + 1)], np.int64)


def fill_template(zp, sp, bins, flags, p: Params) -> np.ndarray:
    zp, sp, bins, flags = _f32(zp), _f32(sp), _i32(bins), _i32(flags)
    H = np.zeros(nbins(p), np.int32)
    lib().pvo_fill_template(C.c_int(zp.size), _ptr(zp), _ptr(sp), _ptr(bins), _ptr(flags), C.byref(p), _ptr(H))
    return H


def fill_exact(zp, sp, flags, p: Params) -> np.ndarray:
    zp, sp, flags = _f32(zp), _f32(sp), _i32(flags)
    H = np.zeros(nbins(p), np.float64)
    lib().pvo_fill_exact(C.c_int(zp.size), _ptr(zp), _ptr(sp), _ptr(flags), C.byref(p), _ptr(H))
    return H


def peaks(H, p: Params, cap: int = 4096):
    H = _i32(H)
    assert H.size == nbins(p)
    b = np.empty(cap, np.int32); e = np.empty(cap, np.int32); k = np.empty(cap, np.int32)
    n = lib().pvo_peaks(_ptr(H), C.byref(p), C.c_int(cap), _ptr(b), _ptr(e), _ptr(k))
    m = min(n, cap)
    return b[:m].copy(), e[:m].copy(), k[:m].copy(), n


def seed_z(H, peak: int, p: Params) -> float:
    H = _i32(H)
    return float(lib().pvo_seed_z(_ptr(H), int(peak), C.byref(p)))


def assign(bins, flags, begin, end, peak, z_seed, p: Params):
    bins, flags = _i32(bins), _i32(flags)
    begin, end, peak = _i32(begin).copy(), _i32(end).copy(), _i32(peak).copy()
    z_seed = _f32(z_seed).copy()
    ts = np.empty(bins.size, np.int32)
    n = lib().pvo_assign(C.c_int(bins.size), _ptr(bins), _ptr(flags), C.c_int(begin.size), _ptr(begin), _ptr(end),
                         _ptr(peak), _ptr(z_seed), C.byref(p), _ptr(ts))
    return ts, begin[:n], end[:n], peak[:n], z_seed[:n]


def fit(tracks: Dict[str, np.ndarray], idx, seed, p: Params):
    """Fit one vertex over tracks[idx]; returns dict(pos, cov, chi2, ntrk, niter, w, trace, rc)."""
    a = {k: _f32(tracks[k]) for k in ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")}
    idx = _i32(idx)
    seed = np.ascontiguousarray(seed, dtype=np.float64)
    pos = np.zeros(3); cov = np.zeros(6); chi2 = C.c_double(0); ntrk = C.c_int32(0); niter = C.c_int32(0)
    w = np.zeros(max(idx.size, 1)); trace = np.zeros((TRACE_ITERS, TRACE_STRIDE))
    cx, _keep = _cross(tracks)
    rc = lib().pvo_fit(C.c_int(idx.size), _ptr(idx), _ptr(a["x"]), _ptr(a["y"]), _ptr(a["z"]), _ptr(a["tx"]),
                       _ptr(a["ty"]), _ptr(a["var_x"]), _ptr(a["var_y"]), _ptr(a["var_tx"]), _ptr(a["var_ty"]),
                       _ptr(seed), C.byref(p), cx, _ptr(pos), _ptr(cov), C.byref(chi2), C.byref(ntrk), C.byref(niter),
                       _ptr(w), _ptr(trace))
    return dict(pos=pos, cov=cov, chi2=chi2.value, ntrk=ntrk.value, niter=niter.value, w=w[:idx.size], trace=trace, rc=rc)


def mv_params(**over) -> Params:
    """Parameters of the paper's GPU flavour: implicit association, Eq. 19 weights,
    convergence on |dz| < 0.5 um alone."""
    kw = dict(flavour=1, conv_dchi2=float("inf"), conv_dz=5e-4)
    kw.update(over)
    return default_params(**kw)


def mv_weight(chi2_own: float, chi2_max: float, chi2_others=()) -> float:
    o = np.ascontiguousarray(chi2_others, dtype=np.float64)
    return float(lib().pvo_mv_weight(float(chi2_own), float(chi2_max), _ptr(o) if o.size else None, int(o.size)))


def track_chi2(tracks: Dict[str, np.ndarray], i: int, pos) -> float:
    a = {k: _f32(tracks[k]) for k in ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")}
    pos = np.ascontiguousarray(pos, dtype=np.float64)
    cx, _keep = _cross(tracks)
    return float(lib().pvo_track_chi2(C.c_int(i), _ptr(a["x"]), _ptr(a["y"]), _ptr(a["z"]), _ptr(a["tx"]), _ptr(a["ty"]),
                                      _ptr(a["var_x"]), _ptr(a["var_y"]), _ptr(a["var_tx"]), _ptr(a["var_ty"]), cx, _ptr(pos)))


def fit_mv(tracks: Dict[str, np.ndarray], idx, seed, other, p: Params):
    """Multi-vertex fit of one vertex over tracks[idx] with other[j] as in pv_oracle.h."""
    a = {k: _f32(tracks[k]) for k in ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")}
    idx = _i32(idx)
    seed = np.ascontiguousarray(seed, dtype=np.float64)
    other = np.ascontiguousarray(other, dtype=np.float64)
    assert other.size == idx.size
    cx, _keep = _cross(tracks)
    pos = np.zeros(3); cov = np.zeros(6); chi2 = C.c_double(0); ntrk = C.c_int32(0); niter = C.c_int32(0)
    w = np.zeros(max(idx.size, 1)); trace = np.zeros((TRACE_ITERS, TRACE_STRIDE))
    rc = lib().pvo_fit_mv(C.c_int(idx.size), _ptr(idx), _ptr(a["x"]), _ptr(a["y"]), _ptr(a["z"]), _ptr(a["tx"]),
                          _ptr(a["ty"]), _ptr(a["var_x"]), _ptr(a["var_y"]), _ptr(a["var_tx"]), _ptr(a["var_ty"]),
                          _ptr(seed), C.byref(p), _ptr(other), cx, _ptr(pos), _ptr(cov), C.byref(chi2), C.byref(ntrk),
                          C.byref(niter), _ptr(w), _ptr(trace))
    return dict(pos=pos, cov=cov, chi2=chi2.value, ntrk=ntrk.value, niter=niter.value, w=w[:idx.size], trace=trace, rc=rc)


def ip_one(tracks: Dict[str, np.ndarray], i: int, pos, cov):
    """(rc, ip, ip_chi2) of track i to one vertex."""
    a = {k: _f32(tracks[k]) for k in ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")}
    pos = np.ascontiguousarray(pos, dtype=np.float64); cov = np.ascontiguousarray(cov, dtype=np.float64)
    d = C.c_double(0); c2 = C.c_double(0)
    cx, _keep = _cross(tracks)
    rc = lib().pvo_ip_one(C.c_int(i), _ptr(a["x"]), _ptr(a["y"]), _ptr(a["z"]), _ptr(a["tx"]), _ptr(a["ty"]), _ptr(a["var_x"]),
                          _ptr(a["var_y"]), _ptr(a["var_tx"]), _ptr(a["var_ty"]), cx, _ptr(pos), _ptr(cov), C.byref(d), C.byref(c2))
    return rc, d.value, c2.value


def track_ip(data: Dict[str, np.ndarray], vtx_pos, vtx_cov, n_vtx) -> Dict[str, np.ndarray]:
    """Per track: the vertex of its event with the smallest IP chi2, that chi2 and the IP to it."""
    a = {k: _f32(data[k]) for k in ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")}
    off = _i32(data["offsets"])
    E, T = off.size - 1, a["x"].size
    vp = np.ascontiguousarray(vtx_pos, dtype=np.float64); vc = np.ascontiguousarray(vtx_cov, dtype=np.float64)
    nv = _i32(n_vtx)
    mv = vp.shape[1] if vp.ndim == 3 else 1
    out = dict(ip=np.zeros(T), ip_chi2=np.zeros(T), ip_vertex=np.zeros(T, np.int32))
    cx, _keep = _cross(data)
    rc = lib().pvo_track_ip(_ptr(a["x"]), _ptr(a["y"]), _ptr(a["z"]), _ptr(a["tx"]), _ptr(a["ty"]), _ptr(a["var_x"]),
                            _ptr(a["var_y"]), _ptr(a["var_tx"]), _ptr(a["var_ty"]), cx, _ptr(off), C.c_int(E), C.c_int(mv),
                            _ptr(vp), _ptr(vc), _ptr(nv), _ptr(out["ip"]), _ptr(out["ip_chi2"]), _ptr(out["ip_vertex"]))
    if rc != 0:
        raise RuntimeError(f"pvo_track_ip failed: {rc}")
    return out


def find(data: Dict[str, np.ndarray], p: Optional[Params] = None, debug: bool = False, n_hist_events: int = 0,
         trace: bool = False, n_threads: int = 1) -> Dict[str, np.ndarray]:
    """Run the whole hot path on a batch from synth.events (host numpy arrays)."""
    if p is None:
        p = default_params()
    a = {k: _f32(data[k]) for k in ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")}
    off = _i32(data["offsets"])
    E = off.size - 1
    T = a["x"].size
    mv = p.max_vtx_per_event
    out = dict(
        vtx_pos=np.zeros((E, mv, 3)), vtx_cov=np.zeros((E, mv, 6)), vtx_chi2=np.zeros((E, mv)),
        vtx_ntracks=np.zeros((E, mv), np.int32), vtx_niter=np.zeros((E, mv), np.int32),
        n_vtx=np.zeros(E, np.int32), trk_weight=np.zeros(T), trk_vertex=np.full(T, -1, np.int32),
        event_status=np.zeros(E, np.uint32))
    dbg = None
    if debug:
        nb = nbins(p)
        n_hist_events = min(n_hist_events, E)
        d = dict(
            hist=np.zeros((max(n_hist_events, 1), nb), np.int32),
            z_poca=np.zeros(T, np.float32), sigma_poca=np.zeros(T, np.float32),
            trk_bin=np.zeros(T, np.int32), trk_flags=np.zeros(T, np.int32),
            n_seeds=np.zeros(E, np.int32), n_seeds_raw=np.zeros(E, np.int32),
            seed_z=np.zeros((E, mv), np.float32), seed_bins=np.zeros((E, mv, 3), np.int32),
            trk_seed=np.full(T, -1, np.int32), seed_pos=np.zeros((E, mv, 3)), seed_cov=np.zeros((E, mv, 6)),
            seed_chi2=np.zeros((E, mv)), seed_ntrk=np.zeros((E, mv), np.int32),
            seed_niter=np.zeros((E, mv), np.int32), seed_fate=np.zeros((E, mv), np.int32),
            seed_edge_last=np.full((E, mv), np.inf), seed_edge_any=np.full((E, mv), np.inf),
            seed_pivot_min=np.full((E, mv), np.inf), seed_nact_min=np.zeros((E, mv), np.int32), trk_w2=np.zeros(T), trk_w1=np.zeros(T))
        if trace:
            d["trace"] = np.zeros((E, mv, TRACE_ITERS, TRACE_STRIDE))
        dbg = Debug()
        for k, _t in Debug._fields_:
            if k == "n_hist_events":
                dbg.n_hist_events = n_hist_events
            elif k in d:
                setattr(dbg, k, d[k].ctypes.data)
            else:
                setattr(dbg, k, None)
        out["debug"] = d
        if n_hist_events == 0:
            dbg.hist = None
    cx, _keep = _cross(data)
    rc = lib().pvo_find(_ptr(a["x"]), _ptr(a["y"]), _ptr(a["z"]), _ptr(a["tx"]), _ptr(a["ty"]), _ptr(a["var_x"]),
                        _ptr(a["var_y"]), _ptr(a["var_tx"]), _ptr(a["var_ty"]), cx, _ptr(off), C.c_int(E), C.byref(p),
                        _ptr(out["vtx_pos"]), _ptr(out["vtx_cov"]), _ptr(out["vtx_chi2"]), _ptr(out["vtx_ntracks"]),
                        _ptr(out["vtx_niter"]), _ptr(out["n_vtx"]), _ptr(out["trk_weight"]), _ptr(out["trk_vertex"]),
                        _ptr(out["event_status"]), C.byref(dbg) if dbg is not None else None, C.c_int(n_threads))
    if rc != 0:
        raise RuntimeError(f"pvo_find failed: {rc}")
    return out
