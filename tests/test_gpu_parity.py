"""Parity of the CUDA path (through the C ABI) against the CPU oracle on the same seeded inputs.
All tests here need a B200 (`-m gpu`)."""
import dataclasses
import json
import os

import numpy as np
import pytest

from synth import events

NTHREADS = os.cpu_count() or 1

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def pv():
    import torch
    assert torch.cuda.is_available(), "these tests need a CUDA device"
    from paper_2412_14966_b200 import build as pvbuild
    pvbuild.build()
    import paper_2412_14966_b200 as pv
    return pv


def _both(pv, oracle, data, n_hist=None, **over):
    from oracle import compare
    p = pv.default_params(**over)
    po = oracle.default_params(**over)
    E = data["offsets"].size - 1
    nh = E if n_hist is None else min(n_hist, E)
    got = pv.find(data, p, debug=True, n_hist_events=nh)
    ref = oracle.find(data, po, debug=True, n_hist_events=nh, trace=True, n_threads=NTHREADS)
    rep = compare.compare(got, ref, np.asarray(data["offsets"]), p)
    return got, ref, rep


def _log_rules(rep, **extra):
    """One JSON line per comparison: how often each near-tie rule of the comparator fired (also appended to the file
    named by PV_PARITY_LOG, so that a run can be summarised in DESIGN.md section 6)."""
    test = os.environ.get("PYTEST_CURRENT_TEST", "").split("::")[-1].replace(" (call)", "")
    line = json.dumps(dict(test=test, fitted_seeds=rep.get("n_fitted_seeds"), vertices=rep.get("n_vertices"),
                           near_ties=rep.get("n_near_ties"), rules=rep.get("rules"), failures=len(rep["failures"]), **extra))
    print("PARITY_RULES", line)
    if os.environ.get("PV_PARITY_LOG"):
        with open(os.environ["PV_PARITY_LOG"], "a") as f:
            f.write(line + "\n")


def _assert_parity(rep, allow_ties_frac=5e-4):
    """No failure, and no more logged near-ties than twice the largest rate measured on B200 (2e-4 of the fitted
    seeds, multi-vertex flavour on high pile-up; 1e-5 on configs[1] at full size; 0 on most cases)."""
    _log_rules(rep)
    assert not rep["failures"], "\n".join(rep["failures"][:10])
    for t in rep["near_ties"][:10]:
        print("LOGGED", t)
    nfit = max(rep.get("n_fitted_seeds", 1), 1)
    assert rep["n_near_ties"] <= max(2, allow_ties_frac * nfit), (rep["n_near_ties"], nfit)


def test_config0_every_tap(pv, oracle, cfg0):
    """configs[0]: 1000 events; bit-exact projection, histograms (all 1000), seeds, assignment; fit within
    1e-3 mm / 1e-3 rel; identical vertex counts."""
    got, ref, rep = _both(pv, oracle, cfg0)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    assert rep["hist_mismatch"] == 0 and rep["seed_z_mismatch"] == 0 and rep["trk_seed_mismatch"] == 0
    assert rep["n_vertices"] > 4000
    assert rep["assign_agreement"] >= 0.999


@pytest.mark.parametrize("idx,n", [(1, 3000), (2, None), (3, None), (4, 100_000)])
def test_configs_at_their_stated_sizes(pv, oracle, idx, n):
    """BASELINE.json configs[2] (50 000 high pile-up events: multi-chunk events, > 256 tracks, many seeds, the
    4 / 8 / 32-lane fit paths), configs[3] (20 000 close pairs) and configs[4] at 100 000 events, every tap against
    the oracle (histograms of the first 300 events); configs[1] as a 3000-event slice here and at full size in
    test_full_size_throughput_config."""
    data = events.generate(events.config(idx, n))
    got, ref, rep = _both(pv, oracle, data, n_hist=300)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    assert rep["assign_agreement"] >= 0.999
    if idx == 1:
        assert (ref["vtx_pos"][..., 2][np.arange(32)[None, :] < ref["n_vtx"][:, None]] < -300).sum() > 100   # p-gas PVs present
    if idx == 2:
        assert np.diff(data["offsets"]).max() > 600 and ref["n_vtx"].max() >= 18


@pytest.mark.parametrize("mv", [False, True])
def test_anisotropic_covariances(pv, oracle, mv):
    """Per-track var_y = k var_x with k in [1/4, 4], var_tx != var_ty, and (through a transport of every state by up to
    40 mm) cov_xtx != cov_yty: a slip that used the x variance for y (Eq. 2 / Eq. 7) anywhere in the
    record build, the chi2 of the multi-vertex association or the IP chi2 fails here.  Both flavours + pv_track_ip."""
    from oracle import compare
    d = events.generate(dataclasses.replace(events.config(1, 2500), aniso=True))
    assert np.abs(d["var_y"] / d["var_x"] - 1).mean() > 0.3 and np.abs(d["var_ty"] / d["var_tx"] - 1).mean() > 0.2
    rng = np.random.default_rng(21)
    L = rng.uniform(-40, 40, d["x"].size)
    t = {k: np.asarray(d[k], np.float64) for k in events.FIELDS}
    m = dict(d)
    m["x"] = (t["x"] + L * t["tx"]).astype(np.float32); m["y"] = (t["y"] + L * t["ty"]).astype(np.float32)
    m["z"] = (t["z"] + L).astype(np.float32)
    m["var_x"] = (t["var_x"] + L * L * t["var_tx"]).astype(np.float32); m["cov_xtx"] = (L * t["var_tx"]).astype(np.float32)
    m["var_y"] = (t["var_y"] + L * L * t["var_ty"]).astype(np.float32); m["cov_yty"] = (L * t["var_ty"]).astype(np.float32)
    for data in (d, m):                                        # diagonal anisotropic, then with distinct cross terms
        p, po = (pv.multivertex_params(), oracle.mv_params()) if mv else (pv.default_params(), oracle.default_params())
        b = pv.DeviceBatch(data, p, debug=True, n_hist_events=50)
        b.find()
        b.track_ip()
        got, gip = b.results(), b.ip_results()
        ref = oracle.find(data, po, debug=True, n_hist_events=50, trace=True, n_threads=NTHREADS)
        rep = compare.compare(got, ref, np.asarray(data["offsets"]), p)
        print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
        _assert_parity(rep)
        assert rep["n_vertices"] > 8000
        rip = oracle.track_ip(data, got["vtx_pos"], got["vtx_cov"], got["n_vtx"])
        same = gip["ip_vertex"] == rip["ip_vertex"]
        assert same.mean() >= 0.999
        ok = same & (rip["ip_vertex"] >= 0)
        assert np.all(np.abs(gip["ip_chi2"][ok] - rip["ip_chi2"][ok]) <= 3e-3 * np.maximum(rip["ip_chi2"][ok], 1.0))
        assert np.abs(gip["ip"][ok] - rip["ip"][ok]).max() <= 1e-3


def test_empty_and_degenerate_events(pv, oracle):
    """Empty batch, events without tracks, single-track events, tracks parallel to the beamline, NaN / zero
    variances, tracks outside the histogram range."""
    got = pv.find(dict(events.from_lists([])))
    assert got["n_vtx"].size == 0
    rng = np.random.default_rng(5)
    base = events.generate(events.config(0, 6))
    evs = []
    off = base["offsets"]
    for e in range(6):
        evs.append({k: base[k][off[e]:off[e + 1]].copy() for k in events.FIELDS})
    empty = {k: np.zeros(0, np.float32) for k in events.FIELDS}
    one = {k: v[:1] for k, v in evs[0].items()}
    par = {k: v.copy() for k, v in evs[1].items()}
    par["tx"][:5] = 0.0; par["ty"][:5] = 0.0                     # parallel to the beamline: invalid
    par["var_x"][5:8] = 0.0                                      # sigma_poca = 0: not histogrammed
    par["var_x"][8:10] = np.nan
    par["var_y"][10:12] = -1.0                                   # unusable in the fit
    far = {k: v.copy() for k, v in evs[2].items()}
    far["z"][:10] += 5000.0                                      # out of the histogram range
    far["x"][10:14] = 50.0                                       # far from the beamline
    lst = [empty, evs[0], empty, one, par, far, evs[3], empty]
    data = events.from_lists(lst)
    got, ref, rep = _both(pv, oracle, data)
    _assert_parity(rep)
    assert list(got["n_vtx"][[0, 2, 3, 7]]) == [0, 0, 0, 0]


def test_wide_tracks_many_fill_units(pv, oracle):
    """Events whose tracks have sigma_poca of several mm in the p-gas region (window of up to ~240 bins = 30 fill
    units each): the flat unit list of a chunk overflows its capacity and is processed in several rounds; a
    second event mixes such tracks with narrow ones across the two-chunk boundary."""
    rng = np.random.default_rng(11)

    def gas_event(n, sig_lo, sig_hi, slope):
        z0 = -450.0
        tx = rng.normal(0, slope, n).astype(np.float32)
        ty = rng.normal(0, slope, n).astype(np.float32)
        sig = rng.uniform(sig_lo, sig_hi, n).astype(np.float32)
        ev = dict(x=(sig * rng.normal(0, 1, n)).astype(np.float32), y=(sig * rng.normal(0, 1, n)).astype(np.float32),
                  z=np.full(n, z0, np.float32), tx=tx, ty=ty, var_x=sig * sig, var_y=sig * sig,
                  var_tx=np.full(n, 1e-6, np.float32), var_ty=np.full(n, 1e-6, np.float32))
        return ev
    wide = gas_event(200, 0.3, 0.6, 0.08)          # sigma_poca ~ 4..10 mm: most pass the 10 mm gas cut
    mixed = gas_event(150, 0.01, 0.5, 0.1)
    data = events.from_lists([wide, mixed, gas_event(40, 0.02, 0.05, 0.15)])
    got, ref, rep = _both(pv, oracle, data)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    sp = ref["debug"]["sigma_poca"][:200]
    assert (sp > 5.0).sum() > 30 and rep["hist_mismatch"] == 0      # units per chunk well above the list capacity
    assert ref["debug"]["hist"][0].sum() > 100 * (1 << 20)


def test_many_proto_clusters_slow_path(pv, oracle):
    """Combs of isolated narrow tracks (one proto-cluster each, none with the integral of a seed) plus a few real
    vertices.  Event 0 and 2: 580 tracks 1 mm apart (8 runs per histogram word).  Event 3: 400 tracks 0.5 mm apart, each
    in the middle of its bin (16 runs per word, the most a word can start): more than 256 proto-cluster starts in one
    pass of 32 words, so the peak search falls back to passes of 16 words; seeds must still come out z-ordered and
    bit-exact."""
    rng = np.random.default_rng(7)
    pv_z = np.array([-250.3, -100.1, 10.2, 150.4, 280.6])

    def comb(zc):
        z = np.concatenate([zc, np.repeat(pv_z, 8)]).astype(np.float32)
        n = z.size
        phi = rng.uniform(0, 2 * np.pi, n)
        sl = 0.3
        ev = dict(x=rng.normal(0, 0.01, n).astype(np.float32), y=rng.normal(0, 0.01, n).astype(np.float32), z=z,
                  tx=(sl * np.cos(phi)).astype(np.float32), ty=(sl * np.sin(phi)).astype(np.float32),
                  var_x=np.full(n, 1e-4, np.float32), var_y=np.full(n, 1e-4, np.float32),
                  var_tx=np.full(n, 1e-6, np.float32), var_ty=np.full(n, 1e-6, np.float32))
        perm = rng.permutation(n)
        return {k: v[perm] for k, v in ev.items()}
    ev = comb(np.arange(-290.0, 290.0, 1.0))
    dense = comb(-80.0 + 0.125 + 0.5 * np.arange(400))
    # exact positions for the dense comb: on the beamline, so that z_poca is the state's z and stays inside its bin
    dense["x"][:] = 0.0
    dense["y"][:] = 0.0
    small = events.generate(events.config(0, 2))
    so = small["offsets"]
    data = events.from_lists([ev, {k: small[k][so[0]:so[1]] for k in events.FIELDS}, ev, dense])
    got, ref, rep = _both(pv, oracle, data)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)

    def most_starts_in_32_words(H):
        above = H > int(0.25 * (1 << 20))
        starts = above & ~np.concatenate([[False], above[:-1]])
        per_word = starts[: (H.size // 32) * 32].reshape(-1, 32).sum(axis=1)
        touched = np.flatnonzero(H[: (H.size // 32) * 32].reshape(-1, 32).any(axis=1))
        return max(per_word[touched[i:i + 32]].sum() for i in range(0, len(touched), 32))
    assert most_starts_in_32_words(ref["debug"]["hist"][0]) >= 250
    assert most_starts_in_32_words(ref["debug"]["hist"][3]) > 256      # the list of one pass overflows
    assert ref["n_vtx"][0] == 5 and got["n_vtx"][0] == 5 and got["n_vtx"][2] == 5 and got["n_vtx"][3] == ref["n_vtx"][3]


def test_histogram_pool_runs_dry(pv, oracle):
    """The seed kernel takes the histogram words an event touches from a pool shared by the 32 warps of an SM (1333
    words).  Here every event spreads 136 isolated tracks over the whole z range (about 100 of its 107 words touched; 32 such
    events want twice the pool), in a batch large enough to keep every warp of the GPU busy: warps wait for words, and
    warps that hold words while the pool is dry give them back and start their event again.  The results must not
    show any of it: bit-exact against the oracle, and bit-identical from run to run."""
    rng = np.random.default_rng(23)
    E, n = 6000, 160
    # 136 isolated tracks on a jittered grid of 6.17 mm (one proto-cluster each, none a seed) + two real vertices
    z = (-545.0 + 6.17 * np.arange(n)[None, :] + rng.uniform(-1.0, 1.0, (E, n))).astype(np.float32)
    z[:, :24] = np.repeat(rng.uniform(-100.0, 100.0, (E, 2)), 12, axis=1)
    z = rng.permuted(z, axis=1)
    phi = rng.uniform(0, 2 * np.pi, (E, n))
    sl = rng.uniform(0.1, 0.4, (E, n))
    sig = rng.uniform(0.01, 0.05, (E, n)).astype(np.float32)
    arr = dict(x=(sig * rng.normal(0, 1, (E, n))).astype(np.float32), y=(sig * rng.normal(0, 1, (E, n))).astype(np.float32), z=z,
               tx=(sl * np.cos(phi)).astype(np.float32), ty=(sl * np.sin(phi)).astype(np.float32),
               var_x=sig * sig, var_y=sig * sig, var_tx=np.full((E, n), 1e-6, np.float32), var_ty=np.full((E, n), 1e-6, np.float32))
    data = {k: v.reshape(-1) for k, v in arr.items()}
    data["offsets"] = (np.arange(E + 1) * n).astype(np.int32)
    data["n_events"] = E
    got, ref, rep = _both(pv, oracle, data, n_hist=400)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    H = ref["debug"]["hist"][:400]
    words = (H[:, : (H.shape[1] // 32) * 32].reshape(400, -1, 32) != 0).any(axis=2).sum(axis=1)
    assert words.mean() > 70 and words.mean() * 32 > 1.5 * 1333, words.mean()
    assert rep["hist_mismatch"] == 0 and rep["seed_z_mismatch"] == 0 and rep["trk_seed_mismatch"] == 0
    assert (ref["n_vtx"] >= 1).mean() > 0.9
    again = pv.find(data, pv.default_params(), debug=True, n_hist_events=400)
    for k in ("vtx_pos", "vtx_cov", "n_vtx", "trk_vertex", "trk_weight", "event_status"):
        assert np.array_equal(got[k], again[k]), k
    assert np.array_equal(got["debug"]["hist"], again["debug"]["hist"])


@pytest.mark.parametrize("n", [1000, 10000])
def test_batch_sweep_config4(pv, oracle, n):
    """configs[4] (seed 5, the configs[1] event model) at the batch sizes the oracle finishes in seconds; the
    larger sizes of the sweep are bench.py --config 4 --events N runs."""
    data = events.generate(events.config(4, n))
    got, ref, rep = _both(pv, oracle, data, n_hist=200)
    _assert_parity(rep)
    assert rep["assign_agreement"] >= 0.999


def test_batch_of_empty_events(pv):
    """Events but no tracks at all (null track pointers), both flavours and the IP consumer."""
    data = events.from_lists([{k: np.zeros(0, np.float32) for k in events.FIELDS}] * 5)
    for p in (pv.default_params(), pv.multivertex_params()):
        b = pv.DeviceBatch(data, p)
        b.find()
        b.track_ip()
        r = b.results()
        assert r["n_vtx"].tolist() == [0] * 5 and r["event_status"].tolist() == [0] * 5
        assert b.ip_results()["ip"].size == 0


def test_too_many_tracks_and_vertex_overflow(pv, oracle):
    """An event above PV_MAX_TRACKS_PER_EVENT is skipped with its flag; max_vtx_per_event smaller than the
    number of seeds keeps the first ones in z and flags the event."""
    big = events.generate(events.config(2, 40))
    n = int(big["offsets"][-1])
    assert n > 2047
    huge = {k: big[k][:2200] for k in events.FIELDS}
    exact = {k: big[k][:2047] for k in events.FIELDS}
    small = events.generate(events.config(0, 3))
    so = small["offsets"]
    lst = [huge, {k: small[k][so[0]:so[1]] for k in events.FIELDS}, exact, {k: small[k][so[1]:so[2]] for k in events.FIELDS}]
    data = events.from_lists(lst)
    got, ref, rep = _both(pv, oracle, data, max_vtx_per_event=32)
    _assert_parity(rep)
    assert got["event_status"][0] & 1 and got["n_vtx"][0] == 0
    assert np.all(got["trk_vertex"][:2200] == -1) and np.all(got["trk_weight"][:2200] == 0)
    assert got["n_vtx"][2] > 10                                   # 2047 tracks of 40 merged pile-up events
    got, ref, rep = _both(pv, oracle, events.generate(events.config(2, 300)), max_vtx_per_event=4)
    _assert_parity(rep)
    assert (got["event_status"] & 2).sum() > 100 and np.array_equal(got["event_status"] & 2, ref["event_status"] & 2)


def test_other_parameters(pv, oracle):
    """Displaced and tilted beamline, unit weights (chi2_max = inf), another binning, tighter
    convergence: the parameters travel through the ABI and both sides agree."""
    data = events.generate(events.config(1, 800))
    d2 = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in data.items()}
    d2["x"] = (d2["x"] + 0.8 + 1e-3 * d2["z"]).astype(np.float32)
    d2["y"] = (d2["y"] - 0.4 - 5e-4 * d2["z"]).astype(np.float32)
    _, _, rep = _both(pv, oracle, d2, n_hist=100, beam_x=0.8, beam_y=-0.4, beam_tx=1e-3, beam_ty=-5e-4)
    _assert_parity(rep)
    assert rep["n_vertices"] > 3000
    _, _, rep = _both(pv, oracle, data, n_hist=100, chi2_max=np.inf)
    _assert_parity(rep)
    _, _, rep = _both(pv, oracle, data, n_hist=100, dz=0.5, min_dip=0.5, min_bin_content=0.4)
    _assert_parity(rep)
    _, _, rep = _both(pv, oracle, data, n_hist=100, conv_dz=1e-4, conv_dchi2=1e-3, max_iter=16, merge_ratio=9.0)
    _assert_parity(rep)


def _both_mv(pv, oracle, data, n_hist=None, **over):
    from oracle import compare
    p = pv.multivertex_params(**over)
    po = oracle.mv_params(**over)
    E = data["offsets"].size - 1
    nh = E if n_hist is None else min(n_hist, E)
    got = pv.find(data, p, debug=True, n_hist_events=nh)
    ref = oracle.find(data, po, debug=True, n_hist_events=nh, trace=True, n_threads=NTHREADS)
    return got, ref, compare.compare(got, ref, np.asarray(data["offsets"]), p)


@pytest.mark.parametrize("idx,n", [(0, 1000), (1, 3000), (2, 1000), (3, 3000)])
def test_multivertex_flavour(pv, oracle, idx, n):
    """The paper's GPU flavour (implicit association, Eq. 19 weights, |dz| < 0.5 um):
    same a1-a3 (bit-exact seeds), fit within 1e-3 mm / 1e-3 rel, identical vertex counts, >= 99.9 % of the tracks
    follow the same vertex."""
    data = events.generate(events.config(idx, n))
    got, ref, rep = _both_mv(pv, oracle, data, n_hist=200)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    assert rep["seed_z_mismatch"] == 0 and rep["assign_agreement"] >= 0.999
    assert rep["n_vertices"] > 1000
    assert not (got["event_status"] & 8).any()


def test_multivertex_other_parameters_and_reproducibility(pv, oracle):
    """chi2_max = 4 (the value of Fig. 6), a narrower window, a tilted beamline; two runs are bit-identical."""
    data = events.generate(events.config(1, 800))
    _, _, rep = _both_mv(pv, oracle, data, n_hist=50, chi2_max=4.0, chi2_window=16.0)
    _assert_parity(rep)
    d2 = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in data.items()}
    d2["x"] = (d2["x"] + 0.8 + 1e-3 * d2["z"]).astype(np.float32)
    _, _, rep = _both_mv(pv, oracle, d2, n_hist=50, beam_x=0.8, beam_tx=1e-3)
    _assert_parity(rep)
    p = pv.multivertex_params()
    a = pv.find(data, p)
    b = pv.find(data, p)
    for k in a:
        assert np.array_equal(a[k], b[k], equal_nan=True), k


@pytest.mark.parametrize("idx,n", [(0, 1000), (1, 3000), (2, 1000)])
def test_track_ip(pv, oracle, idx, n):
    """pv_track_ip (NEXT-4) on the vertices pv_find just produced vs the oracle's IP on the SAME vertices
    (the kernel's fp32 outputs, fed to the oracle): same smallest-chi2 vertex for >= 99.9 % of the tracks (every
    other one a chi2 tie within 1e-3), IP within 1e-3 mm, IP chi2 within 2e-3 relative (floor 2e-3 absolute)."""
    data = events.generate(events.config(idx, n))
    p = pv.default_params()
    b = pv.DeviceBatch(data, p)
    b.find()
    b.track_ip()
    res, got = b.results(), b.ip_results()
    ref = oracle.track_ip(data, res["vtx_pos"], res["vtx_cov"], res["n_vtx"])
    same = got["ip_vertex"] == ref["ip_vertex"]
    assert same.mean() >= 0.999, same.mean()
    none = ref["ip_vertex"] < 0
    assert np.all(got["ip"][none] == -1.0) and np.all(got["ip_chi2"][none] == -1.0)
    m = same & ~none
    assert np.abs(got["ip"][m] - ref["ip"][m]).max() <= 1e-3
    dc = np.abs(got["ip_chi2"][m] - ref["ip_chi2"][m])
    assert np.all(dc <= 2e-3 * np.maximum(ref["ip_chi2"][m], 1.0)), (dc / np.maximum(ref["ip_chi2"][m], 1.0)).max()
    for i in np.flatnonzero(~same)[:20]:                     # near-ties of the argmin: the two chi2 agree
        assert abs(got["ip_chi2"][i] - ref["ip_chi2"][i]) <= 2e-3 * max(ref["ip_chi2"][i], 1.0), i
    # prompt tracks point to their own PV
    tv = res["trk_vertex"]
    assert (got["ip_vertex"][tv >= 0] == tv[tv >= 0]).mean() > 0.97


@pytest.mark.parametrize("idx,n,mv", [(3, 3000, False), (2, 1000, False), (2, 600, True)])
def test_recursive_splitter(pv, oracle, idx, n, mv):
    """split_mode = PV_SPLIT_RECURSIVE (the paper's x86 splitting, reading R-16) in both flavours: seeds
    bit-exact against the oracle in the same mode; on high pile-up some events split differently from the
    z-ordered variant."""
    from oracle import compare
    data = events.generate(events.config(idx, n))
    mk_p, mk_o = (pv.multivertex_params, oracle.mv_params) if mv else (pv.default_params, oracle.default_params)
    p, po = mk_p(split_mode=1), mk_o(split_mode=1)
    got = pv.find(data, p, debug=True, n_hist_events=100)
    ref = oracle.find(data, po, debug=True, n_hist_events=100, trace=True, n_threads=NTHREADS)
    rep = compare.compare(got, ref, np.asarray(data["offsets"]), p)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    assert rep["seed_bins_mismatch"] == 0 and rep["seed_z_mismatch"] == 0 and rep["n_seeds_mismatch"] == 0


def test_recursive_splitter_differs_on_a_small_middle_peak(pv, oracle):
    """A constructed event (two 6-track vertices two bins apart from a 1-track bump, on a background of three wide
    tracks): the z-ordered variant cuts at the first dip, the recursive one at the lower dip between the two largest
    maxima (hand-worked in tests/golden/peaks_x86_handbuilt.json for the same shape).  Both modes bit-exact vs oracle."""
    from oracle import compare
    f = np.float32

    rng = np.random.default_rng(3)

    def trk(b, sig_poca, n):                               # tracks through the beamline at the centre of bin b
        zc = -550 + 0.25 * (b + 0.5)
        phi = rng.uniform(0, 2 * np.pi, n)
        return dict(x=np.zeros(n, f), y=np.zeros(n, f), z=np.full(n, zc, f),
                    tx=(0.3 * np.cos(phi)).astype(f), ty=(0.3 * np.sin(phi)).astype(f),
                    var_x=np.full(n, (sig_poca * 0.3) ** 2, f), var_y=np.full(n, (sig_poca * 0.3) ** 2, f),
                    var_tx=np.full(n, 1e-6, f), var_ty=np.full(n, 1e-6, f))
    parts = [trk(2200, 0.01, 6), trk(2202, 0.01, 1), trk(2204, 0.01, 6), trk(2201, 0.3, 2), trk(2203, 0.3, 1)]
    ev = {k: np.concatenate([q[k] for q in parts]) for k in events.FIELDS}
    small = events.generate(events.config(0, 2))
    so = small["offsets"]
    data = events.from_lists([ev, {k: small[k][so[0]:so[1]] for k in events.FIELDS}, ev])
    seeds = {}
    for mode in (0, 1):
        p, po = pv.default_params(split_mode=mode), oracle.default_params(split_mode=mode)
        got = pv.find(data, p, debug=True, n_hist_events=3)
        ref = oracle.find(data, po, debug=True, n_hist_events=3, trace=True)
        rep = compare.compare(got, ref, np.asarray(data["offsets"]), p)
        _assert_parity(rep)
        assert rep["seed_bins_mismatch"] == 0 and rep["hist_mismatch"] == 0
        seeds[mode] = got["debug"]["seed_bins"][0][:got["debug"]["n_seeds_raw"][0]].tolist()
    assert seeds[0] == [[2200, 2201, 2200], [2201, 2205, 2204]]
    assert seeds[1] == [[2200, 2203, 2200], [2203, 2205, 2204]]


def test_runs_are_reproducible(pv, cfg0):
    """Integer histograms and a fixed summation order: two runs give bit-identical outputs."""
    a = pv.find(cfg0)
    b = pv.find(cfg0)
    for k in a:
        assert np.array_equal(a[k], b[k], equal_nan=True), k


@pytest.mark.parametrize("mode", ["explicit", "multivertex", "recursive"])
def test_repeated_runs_are_bit_identical_on_high_pileup(pv, mode):
    """Five launches over 3000 high pile-up events (multi-chunk events, many seeds, big-seed fit path): every output
    bit-identical -- a race in the shared-memory pool or an order-dependent sum would show up here."""
    data = events.generate(events.config(2, 3000))
    p = {"explicit": pv.default_params, "multivertex": pv.multivertex_params,
         "recursive": lambda: pv.default_params(split_mode=1)}[mode]()
    b = pv.DeviceBatch(data, p)
    ref = None
    for _ in range(5):
        b.find()
        r = b.results()
        if ref is None:
            ref = r
            continue
        m = np.arange(p.max_vtx_per_event)[None, :] < r["n_vtx"][:, None]
        for k in r:
            a, c = (r[k][m], ref[k][m]) if k.startswith("vtx_") else (r[k], ref[k])
            assert np.array_equal(a, c, equal_nan=True), k


@pytest.mark.parametrize("mv", [False, True])
def test_covariance_cross_terms(pv, oracle, mv):
    """NEXT-2: the x-tx / y-ty elements of Eq. 2 through pv_find_ext and pv_track_ip.  The track states of configs[1]
    are re-expressed at a z up to 150 mm away (x' = x + L tx, V_xx' = V_xx + L^2 V_tt, V_xtx' = L V_tt), which makes
    the cross terms essential; kernel vs oracle on the same inputs, both flavours, plus the IP consumer."""
    from oracle import compare
    d = events.generate(events.config(1, 2000))
    rng = np.random.default_rng(12)
    L = rng.uniform(-150, 150, d["x"].size)
    t = {k: np.asarray(d[k], np.float64) for k in events.FIELDS}
    m = dict(d)
    m["x"] = (t["x"] + L * t["tx"]).astype(np.float32); m["y"] = (t["y"] + L * t["ty"]).astype(np.float32)
    m["z"] = (t["z"] + L).astype(np.float32)
    m["var_x"] = (t["var_x"] + L * L * t["var_tx"]).astype(np.float32); m["cov_xtx"] = (L * t["var_tx"]).astype(np.float32)
    m["var_y"] = (t["var_y"] + L * L * t["var_ty"]).astype(np.float32); m["cov_yty"] = (L * t["var_ty"]).astype(np.float32)
    p, po = (pv.multivertex_params(), oracle.mv_params()) if mv else (pv.default_params(), oracle.default_params())
    b = pv.DeviceBatch(m, p, debug=True, n_hist_events=100)
    b.find()
    b.track_ip()
    got, gip = b.results(), b.ip_results()
    ref = oracle.find(m, po, debug=True, n_hist_events=100, trace=True, n_threads=NTHREADS)
    rep = compare.compare(got, ref, np.asarray(m["offsets"]), p)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    assert rep["n_vertices"] > 5000
    # without the cross terms the same inputs give clearly different covariances: the terms are exercised
    nocov = pv.find({k: v for k, v in m.items() if not k.startswith("cov_")}, p)
    k = np.arange(32)[None, :] < np.minimum(nocov["n_vtx"], got["n_vtx"])[:, None]
    assert np.median(np.abs(nocov["vtx_cov"][k][:, 5] / got["vtx_cov"][k][:, 5] - 1)) > 0.2
    rip = oracle.track_ip(m, got["vtx_pos"], got["vtx_cov"], got["n_vtx"])
    same = gip["ip_vertex"] == rip["ip_vertex"]
    assert same.mean() >= 0.999
    ok = same & (rip["ip_vertex"] >= 0)
    assert np.all(np.abs(gip["ip_chi2"][ok] - rip["ip_chi2"][ok]) <= 3e-3 * np.maximum(rip["ip_chi2"][ok], 1.0))


def test_beamline_offset_robustness_scan(pv):
    """Synthetic version of the paper's Fig. 8: the finder is told a beamline that is off by d from the
    true one (x direction).  "an efficiency of 99 % within a beamline position uncertainty of 50 um ... 99.9 %
    within 20 um": efficiency of reconstructible PVs (>= 4 tracks, matched within 5 sigma_z) relative
    to the zero-offset run, both flavours.  Far off (1 mm) the 0.3 mm beamline-distance cut removes the pp PVs."""
    data = events.generate(events.config(0, 3000), with_truth=True)
    tr = data["truth"]
    order = np.argsort(tr["pv_event"], kind="stable")
    pe, pz, pn = tr["pv_event"][order], tr["pv_z"][order], tr["pv_ntracks"][order]
    first = np.searchsorted(pe, np.arange(3001))

    def n_found(r):
        found = 0
        for e in range(3000):
            vz = r["vtx_pos"][e, :r["n_vtx"][e], 2]
            if not len(vz):
                continue
            vs = np.sqrt(r["vtx_cov"][e, :r["n_vtx"][e], 5])
            for z, n in zip(pz[first[e]:first[e + 1]], pn[first[e]:first[e + 1]]):
                if n >= 4:
                    j = int(np.argmin(np.abs(vz - z)))
                    found += abs(vz[j] - z) < 5 * vs[j]
        return found
    for mk in (pv.default_params, pv.multivertex_params):
        base = n_found(pv.find(data, mk()))
        assert base > 12000
        rel = {d: n_found(pv.find(data, mk(beam_x=d))) / base for d in (0.02, 0.05, 1.0)}
        print(mk.__name__, "relative efficiency vs beamline offset [mm]:", rel)
        assert rel[0.02] >= 0.999 and rel[0.05] >= 0.99 and rel[1.0] < 0.05


@pytest.mark.parametrize("mode", ["explicit", "multivertex"])
def test_full_size_throughput_config(pv, oracle, mode):
    """configs[1] at its full size (100 000 events) through the PRODUCT kernels (no taps), the launch configuration
    bench.py times: every final output against the oracle under the same rules as the tap tests -- the iteration
    count is an output, so rule N1 is applied exactly from vtx_niter and the oracle's trace; a differing vertex count
    or assignment is accepted only in events where the oracle's own deciding quantity is within 1 % of its cut."""
    from oracle import compare
    data = events.generate(events.config(1))
    p, po = (pv.default_params(), oracle.default_params()) if mode == "explicit" else (pv.multivertex_params(), oracle.mv_params())
    got = pv.find(data, p)
    info = pv.last_launch_info()
    assert info["n_kernels"] == 4 and info["grid"] >= 100
    ref = oracle.find(data, po, debug=True, trace=True, n_threads=NTHREADS)
    rep = compare.compare(got, ref, data["offsets"], p)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    assert rep["assign_agreement"] >= 0.999 and rep["n_vertices"] > 500_000
    # events excused from their first fragile seed on: 0 measured on B200 in either flavour (round 3)
    assert rep["n_fragile_events_excused"] <= 20


@pytest.mark.parametrize("mode", ["explicit", "multivertex"])
def test_one_million_events(pv, oracle, mode):
    """configs[4] at its largest batch (10^6 events, 1.15 10^8 tracks: track-record indices up to 1.15 10^8, twice that
    in the multi-vertex flavour) through the product kernels against the oracle run without taps or trace (the trace
    alone would be 45 GB).  Without the oracle's deciding quantities no near-tie can be explained, so the check is the
    one that holds at any size: the vertex count differs in fewer than 2 in 10^4 events (the near-tie rate measured with
    taps at 10^5 events), assignment agrees on >= 99.9 % of the tracks, and every vertex of an event with the same
    count and the same iteration counts meets the position and covariance tolerances."""
    from oracle import compare
    data = events.generate(events.config(4, 1_000_000))
    p, po = (pv.default_params(), oracle.default_params()) if mode == "explicit" else (pv.multivertex_params(), oracle.mv_params())
    got = pv.find(data, p)
    ref = oracle.find(data, po, n_threads=NTHREADS)
    E, mv = 1_000_000, p.max_vtx_per_event
    assert int(data["offsets"][-1]) > 100_000_000
    assert np.array_equal(got["event_status"] & ~np.uint32(4), ref["event_status"] & ~np.uint32(4))
    same_n = got["n_vtx"] == ref["n_vtx"]
    agree = float((got["trk_vertex"] == ref["trk_vertex"]).mean())
    m = (np.arange(mv)[None, :] < ref["n_vtx"][:, None]) & same_n[:, None]
    same_it = np.where(m, got["vtx_niter"] == ref["vtx_niter"], True).all(axis=1)
    m &= same_it[:, None]
    dpos = np.abs(got["vtx_pos"].astype(np.float64) - ref["vtx_pos"]).max(axis=-1)
    dcov = compare._cov_rel_err(got["vtx_cov"].astype(np.float64), ref["vtx_cov"])
    bad = m & ~((dpos <= compare.POS_TOL) & (dcov <= compare.COV_RTOL))
    summary = dict(test=f"test_one_million_events[{mode}]", events=E, vertices=int(ref["n_vtx"].sum()),
                   n_vtx_differs=int((~same_n).sum()), niter_differs_events=int((same_n & ~same_it).sum()),
                   assign_agreement=agree, vertices_compared=int(m.sum()), vertices_off=int(bad.sum()),
                   pos_max_err_mm=float(dpos[m & ~bad].max()), cov_max_rel_err=float(dcov[m & ~bad].max()))
    print("PARITY_1M", json.dumps(summary))
    if os.environ.get("PV_PARITY_LOG"):
        with open(os.environ["PV_PARITY_LOG"], "a") as f:
            f.write(json.dumps(summary) + "\n")
    assert (~same_n).sum() <= 2e-4 * E, summary
    assert agree >= 0.999, summary
    assert m.sum() >= 0.97 * ref["n_vtx"].sum(), summary
    # a vertex off with equal counts is an event whose cleanup paired the seeds differently (a near-tie upstream):
    # as rare as the differing counts
    assert bad.sum() <= 2e-4 * E, (summary, np.argwhere(bad)[:5].tolist())


@pytest.mark.parametrize("mode", ["explicit", "multivertex", "recursive", "recursive_multivertex", "template", "template_recursive_multivertex"])
def test_product_kernels_equal_the_tap_kernels(pv, mode):
    """pv_find (templates without taps) and pv_find_debug (the instantiations the tap tests check against the oracle)
    give bit-identical final outputs: ties every <false, ...> kernel to a tap-checked one.  High pile-up and SMOG2 events."""
    mk = pv.multivertex_params if "multivertex" in mode else pv.default_params
    p = mk(split_mode=1 if "recursive" in mode else 0, fill_mode=1 if "template" in mode else 0)
    for idx, n in ((2, 2000), (1, 4000)):
        data = events.generate(events.config(idx, n))
        a = pv.find(data, p)
        b = pv.find(data, p, debug=True, n_hist_events=10)
        m = np.arange(p.max_vtx_per_event)[None, :] < a["n_vtx"][:, None]
        for k in a:
            x, y = (a[k][m], b[k][m]) if k.startswith("vtx_") else (a[k], b[k])
            assert np.array_equal(x, y, equal_nan=True), (mode, idx, k)


def _select(res, E, T, ev_mask, trk_mask):
    """The per-event ([E, ...]) and per-track ([T]) arrays of a result dict restricted to the selected events."""
    out = {}
    for k, v in res.items():
        if isinstance(v, dict):
            out[k] = _select(v, E, T, ev_mask, trk_mask)
        elif isinstance(v, np.ndarray) and v.ndim >= 1 and v.shape[0] == E:
            out[k] = v[ev_mask]
        elif isinstance(v, np.ndarray) and v.ndim == 1 and v.shape[0] == T:
            out[k] = v[trk_mask]
    return out


def test_record_overflow_is_flagged_per_event(pv, oracle):
    """High pile-up events whose track errors are inflated tenfold, with chi2_window = 100: every track is inside the
    window of several candidates, far more (track, candidate) records than the 2 per track the workspace holds.
    Events that still got their records match the oracle (same inputs and window); the others carry
    PV_EVT_RECORD_OVERFLOW, no vertex, no assignment; the call itself succeeds."""
    from oracle import compare
    data = events.generate(events.config(2, 1500))
    data["var_x"] = data["var_x"] * 100.0
    data["var_y"] = data["var_y"] * 100.0
    off = np.asarray(data["offsets"])
    E, T = off.size - 1, int(off[-1])
    p, po = pv.multivertex_params(chi2_window=100.0), oracle.mv_params(chi2_window=100.0)
    got = pv.find(data, p)
    flagged = (got["event_status"] & 8) != 0
    print("events flagged with PV_EVT_RECORD_OVERFLOW:", int(flagged.sum()), "of", E)
    assert 50 < flagged.sum() < E - 50, flagged.sum()
    ev_of_trk = np.repeat(np.arange(E), np.diff(off))
    assert np.all(got["n_vtx"][flagged] == 0)
    assert np.all(got["trk_vertex"][flagged[ev_of_trk]] == -1) and np.all(got["trk_weight"][flagged[ev_of_trk]] == 0)
    ref = oracle.find(data, po, debug=True, trace=True, n_threads=NTHREADS)
    keep, tkeep = ~flagged, ~flagged[ev_of_trk]
    sub_off = np.concatenate([[0], np.cumsum(np.diff(off)[keep])]).astype(np.int32)
    g, r = _select(got, E, T, keep, tkeep), _select(ref, E, T, keep, tkeep)
    rep = compare.compare(g, r, sub_off, p)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    assert rep["n_vertices"] > 100


@pytest.mark.parametrize("mode", ["explicit", "multivertex"])
def test_n_tracks_smaller_than_the_offsets(pv, mode):
    """pv_find is told fewer tracks than offsets[n_events] holds, and gets a workspace sized for that smaller number:
    events inside the given count come out as in a correct call, the others carry PV_EVT_RECORD_OVERFLOW, no vertex,
    no assignment -- and nothing is written past the workspace (a guard area behind it keeps its pattern)."""
    import torch
    data = events.generate(events.config(1, 2000))
    off = np.asarray(data["offsets"])
    E = off.size - 1
    p = pv.default_params() if mode == "explicit" else pv.multivertex_params()
    want = pv.find(data, p)
    b = pv.DeviceBatch(data, p)
    T_given = int(off[E // 2]) + 3                           # ends inside event E/2
    need = pv.workspace_bytes(E, T_given, p)
    guard = 4 << 20
    b.workspace = torch.full((need + guard,), 0xA5, dtype=torch.uint8, device=b.device)
    b.T = T_given
    for _ in range(2):
        b.find()
    got = b.results()
    assert bool((b.workspace[need:] == 0xA5).all()), "the kernels wrote behind the workspace"
    inside = off[1:] <= T_given
    assert inside[:E // 2].all() and not inside[E // 2:].any()
    ev_of_trk = np.repeat(np.arange(E), np.diff(off))
    tin = inside[ev_of_trk]
    assert np.all((got["event_status"][~inside] & 8) != 0) and np.all(got["n_vtx"][~inside] == 0)
    assert np.all(got["trk_vertex"][~tin] == -1) and np.all(got["trk_weight"][~tin] == 0)
    assert np.array_equal(got["event_status"][inside], want["event_status"][inside])
    assert np.array_equal(got["n_vtx"][inside], want["n_vtx"][inside]) and want["n_vtx"][inside].sum() > 1000
    assert np.array_equal(got["trk_vertex"][tin], want["trk_vertex"][tin])
    assert np.array_equal(got["trk_weight"][tin], want["trk_weight"][tin])
    m = (np.arange(p.max_vtx_per_event)[None, :] < want["n_vtx"][:, None]) & inside[:, None]
    for k in ("vtx_pos", "vtx_cov", "vtx_chi2", "vtx_ntracks", "vtx_niter"):
        assert np.array_equal(got[k][m], want[k][m]), k


def test_unusual_parameters_reach_their_guards(pv, oracle):
    """min_tracks_seed = 0 keeps seeds without any track: they are singular fits on both sides, not stale slots;
    a sigma cut whose window would need more fill units than the list can number is refused (PV_E_PARAM)."""
    data = events.generate(events.config(0, 400))
    got, ref, rep = _both(pv, oracle, data, n_hist=50, min_tracks_seed=(0, 0), min_cluster_integral=(0.5, 0.5), min_tracks_pv=(1, 1))
    _assert_parity(rep)
    assert rep["n_vertices"] > 1500
    with pytest.raises(pv.PvError):
        pv.find(data, pv.default_params(max_sigma_poca=(1.5, 200.0)))


@pytest.mark.parametrize("mode", ["explicit", "multivertex"])
def test_host_pipeline_matches_device_path(pv, cfg0, mode):
    """pv_find_host (fixed-stride read-back) and pv_find_host_compact (packed vertices, int8 vertex index) return
    exactly what pv_find returns, for 1, 5 and 64 chunks, in both flavours; broken offsets are refused on the host."""
    p = pv.default_params() if mode == "explicit" else pv.multivertex_params()
    a = pv.find(cfg0, p)
    E, T = cfg0["offsets"].size - 1, int(cfg0["offsets"][-1])
    hp = pv.HostPipeline(E, T, p, n_streams=3)
    data = hp.pin_inputs(cfg0)
    for compact in (False, True):
        out = hp.alloc_outputs(E, T, compact=compact)
        for chunks in (1, 5, 64):
            for v in out.values():
                v.view(np.uint8)[...] = 0
            hp.find(data, out, n_chunks=chunks)
            assert hp.matches(out, a), (compact, chunks)
            if compact:
                nv = int(a["n_vtx"].sum())
                assert out["vtx_begin"][E] == nv and hp.bytes_per_call(data, out)[1] < 0.5 * (E * 32 * 48 + T * 8)
        bad = dict(data)
        bad["offsets"] = data["offsets"].copy()
        bad["offsets"][E // 2] = bad["offsets"][E // 2 + 1] + 7           # decreasing in the middle
        with pytest.raises(pv.PvError):
            hp.find(bad, out, n_chunks=4)
        bad["offsets"] = data["offsets"].copy()
        bad["offsets"][E] = T + 1000                                       # beyond the context's capacity
        with pytest.raises(pv.PvError):
            hp.find(bad, out, n_chunks=4)
    small = hp.alloc_outputs(E, T, compact=True)
    small["vertices"] = small["vertices"][:10]                            # too few vertex records: refused, nothing hangs
    with pytest.raises(pv.PvError):
        hp.find(data, small, n_chunks=4)
    hp.close()


@pytest.mark.parametrize("idx,n,mv", [(0, 1000, False), (1, 3000, False), (2, 1000, False), (3, 3000, False), (1, 1500, True)])
def test_template_fill(pv, oracle, idx, n, mv):
    """fill_mode = PV_FILL_TEMPLATE (the paper's x86 fill, reading R-17): histograms bit-exact against the
    oracle in the same mode (the table of templates is rebuilt on the device at every call), every later tap as for the
    polynomial fill; the product kernel equals the tap kernel."""
    from oracle import compare
    data = events.generate(events.config(idx, n))
    mk_p, mk_o = (pv.multivertex_params, oracle.mv_params) if mv else (pv.default_params, oracle.default_params)
    p, po = mk_p(fill_mode=1), mk_o(fill_mode=1)
    got = pv.find(data, p, debug=True, n_hist_events=400)
    assert pv.last_launch_info()["n_kernels"] == 5
    ref = oracle.find(data, po, debug=True, n_hist_events=400, trace=True, n_threads=NTHREADS)
    rep = compare.compare(got, ref, np.asarray(data["offsets"]), p)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    assert rep["hist_mismatch"] == 0 and rep["seed_bins_mismatch"] == 0 and rep["seed_z_mismatch"] == 0
    # it is another histogram than the polynomial fill's
    poly = oracle.find(data, mk_o(), debug=True, n_hist_events=400, n_threads=NTHREADS)
    assert (poly["debug"]["hist"] != ref["debug"]["hist"]).any()
    plain = pv.find(data, p)
    m = np.arange(p.max_vtx_per_event)[None, :] < plain["n_vtx"][:, None]
    for k in plain:
        x, y = (plain[k][m], got[k][m]) if k.startswith("vtx_") else (plain[k], got[k])
        assert np.array_equal(x, y, equal_nan=True), k


def test_template_fill_other_binning_and_wide_tracks(pv, oracle):
    """Another bin size (the classes are defined in bins), a larger sigma cut (more classes), recursive splitting, and
    p-gas tracks several mm wide whose templates span hundreds of bins and leave the range at its lower end."""
    data = events.generate(events.config(1, 1200))
    _, _, rep = _both(pv, oracle, data, n_hist=200, fill_mode=1, dz=0.5, split_mode=1)
    _assert_parity(rep)
    _, _, rep = _both(pv, oracle, data, n_hist=200, fill_mode=1, max_sigma_poca=(3.0, 20.0))
    _assert_parity(rep)
    rng = np.random.default_rng(17)
    n = 150
    sig = rng.uniform(0.2, 0.7, n).astype(np.float32)
    ev = dict(x=(sig * rng.normal(0, 1, n)).astype(np.float32), y=(sig * rng.normal(0, 1, n)).astype(np.float32),
              z=np.full(n, -535.0, np.float32), tx=rng.normal(0, 0.08, n).astype(np.float32),
              ty=rng.normal(0, 0.08, n).astype(np.float32), var_x=sig * sig, var_y=sig * sig,
              var_tx=np.full(n, 1e-6, np.float32), var_ty=np.full(n, 1e-6, np.float32))
    got, ref, rep = _both(pv, oracle, events.from_lists([ev, ev]), fill_mode=1)
    _assert_parity(rep)
    assert rep["hist_mismatch"] == 0 and (ref["debug"]["sigma_poca"][:n] > 4.0).sum() > 20 and ref["debug"]["hist"][0][:8].sum() > 0


def test_fill_and_splitting_variants_on_close_pairs(pv):
    """the alternatives of P:L131 / P:L137 compared on configs[3] -- the fraction of events in which
    two vertices are reconstructed, by pair separation (0.1 .. 5 mm), for polynomial / template fill and z-ordered /
    recursive splitting.  "the algorithm cannot separate vertices that are closer than about 2 mm"."""
    data = events.generate(events.config(3, 6000))
    sep = np.array([0.1, 0.2, 0.5, 1.0, 2.0, 5.0])
    which = np.arange(6000) % 6
    table = {}
    for fill in (0, 1):
        for split in (0, 1):
            r = pv.find(data, pv.default_params(fill_mode=fill, split_mode=split))
            table[(fill, split)] = [float((r["n_vtx"][which == q] >= 2).mean()) for q in range(6)]
            print("fill", ["polynomial", "template"][fill], "split", ["z-ordered", "recursive"][split],
                  dict(zip(sep.tolist(), np.round(table[(fill, split)], 3).tolist())))
    for key, frac in table.items():
        assert frac[0] < 0.02 and frac[1] < 0.05 and frac[5] > 0.97, (key, frac)   # merged at 0.1-0.2 mm, resolved at 5 mm
        assert frac[3] < frac[4] <= frac[5] + 1e-9                               # resolution turns on between 1 and 2 mm
    ref = np.array(table[(0, 0)])
    for key, frac in table.items():
        assert np.abs(np.array(frac) - ref).max() < 0.08, (key, frac)             # the variants agree to a few per cent


@pytest.mark.parametrize("mv", [False, True])
def test_seeds_of_every_group_size(pv, oracle, mv):
    """One vertex per event with 5 .. 1900 tracks: the fit handles a seed with 2, 4, 8, 16 or 32 lanes according to its
    track count (up to 28, 56, 112, 224, 448 tracks in the explicit flavour; 24 .. 384 in the multi-vertex one) and with
    the whole-warp global-memory loop beyond that; every size class must give the oracle's vertex."""
    from oracle import compare
    rng = np.random.default_rng(31)
    evs = []
    sizes = [5, 27, 28, 29, 40, 56, 57, 100, 112, 113, 200, 224, 225, 300, 384, 385, 448, 449, 700, 1200, 1900, 23, 24, 25, 48, 49, 96, 97, 192, 193]
    for n in sizes:
        z0 = rng.uniform(-100, 100)
        sig = rng.uniform(0.01, 0.1, n).astype(np.float32)
        evs.append(dict(x=(sig * rng.normal(0, 1, n)).astype(np.float32), y=(sig * rng.normal(0, 1, n)).astype(np.float32),
                        z=np.full(n, z0, np.float32), tx=np.clip(rng.normal(0, 0.25, n), -0.4, 0.4).astype(np.float32),
                        ty=np.clip(rng.normal(0, 0.25, n), -0.4, 0.4).astype(np.float32), var_x=sig * sig, var_y=sig * sig,
                        var_tx=np.full(n, 1e-6, np.float32), var_ty=np.full(n, 1e-6, np.float32)))
    small = events.generate(events.config(0, 40))
    so = small["offsets"]
    for e in range(40):                                       # ordinary events in between, so that windows mix the sizes
        evs.insert(rng.integers(0, len(evs) + 1), {k: small[k][so[e]:so[e + 1]] for k in events.FIELDS})
    data = events.from_lists(evs)
    p, po = (pv.multivertex_params(), oracle.mv_params()) if mv else (pv.default_params(), oracle.default_params())
    got = pv.find(data, p, debug=True, n_hist_events=len(evs))
    ref = oracle.find(data, po, debug=True, n_hist_events=len(evs), trace=True, n_threads=NTHREADS)
    rep = compare.compare(got, ref, np.asarray(data["offsets"]), p)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep)
    big = np.diff(data["offsets"]) >= 5
    nt = ref["debug"]["seed_ntrk"].max(axis=1)
    assert set(np.diff(data["offsets"])[big]) >= set(sizes) and nt.max() > 1500      # the large seeds really are single seeds
    plain = pv.find(data, p)
    m = np.arange(p.max_vtx_per_event)[None, :] < plain["n_vtx"][:, None]
    for k in plain:
        a, b = (plain[k][m], got[k][m]) if k.startswith("vtx_") else (plain[k], got[k])
        assert np.array_equal(a, b, equal_nan=True), k


@pytest.mark.parametrize("mv", [False, True])
def test_ill_conditioned_seeds_are_refitted_in_double(pv, oracle, mv):
    """Vertices made of 3 .. 8 NEARLY PARALLEL tracks (slopes equal within ~1e-3): the Hessian's third pivot is a few 1e-4
    of its diagonal, the case fp32 normal equations cannot resolve (C_zz would be off by more than 1e-3 relative).  The
    fit hands such seeds to ill_kernel; they must meet the same flat tolerances as every other seed.  Ordinary events
    in between, so that the fit's windows mix both kinds."""
    from oracle import compare
    rng = np.random.default_rng(41)
    small = events.generate(events.config(0, 300))
    so = small["offsets"]
    evs = []
    for e in range(300):
        ev = {k: small[k][so[e]:so[e + 1]] for k in events.FIELDS}
        n = int(rng.integers(3, 9))
        z0 = float(rng.uniform(180.0, 260.0))                    # far downstream of the luminous region: a seed of its own
        tx0, ty0 = rng.uniform(0.05, 0.3) * rng.choice([-1, 1]), rng.uniform(0.05, 0.3) * rng.choice([-1, 1])
        tx = (tx0 + 1e-3 * rng.normal(0, 1, n)).astype(np.float32)
        ty = (ty0 + 1e-3 * rng.normal(0, 1, n)).astype(np.float32)
        sig = rng.uniform(0.01, 0.03, n).astype(np.float32)
        zt = np.full(n, z0 + rng.uniform(-5, 5), np.float32)    # the states are given a few mm from the vertex
        extra = dict(x=((zt - z0) * tx + sig * rng.normal(0, 1, n)).astype(np.float32),
                     y=((zt - z0) * ty + sig * rng.normal(0, 1, n)).astype(np.float32), z=zt, tx=tx, ty=ty,
                     var_x=sig * sig, var_y=sig * sig, var_tx=np.full(n, 1e-6, np.float32), var_ty=np.full(n, 1e-6, np.float32))
        evs.append({k: np.concatenate([ev[k], extra[k]]) for k in events.FIELDS})
    data = events.from_lists(evs)
    p, po = (pv.multivertex_params(), oracle.mv_params()) if mv else (pv.default_params(), oracle.default_params())
    got = pv.find(data, p, debug=True, n_hist_events=10)
    ref = oracle.find(data, po, debug=True, n_hist_events=10, trace=True, n_threads=NTHREADS)
    rd = ref["debug"]
    fitted = (np.arange(p.max_vtx_per_event)[None, :] < rd["n_seeds"][:, None]) & (rd["seed_niter"] > 0)
    n_ill = int((fitted & (np.abs(rd["seed_pivot_min"]) < 1.0 / 256.0)).sum())
    n_very = int((fitted & (np.abs(rd["seed_pivot_min"]) < 1e-3)).sum())
    print("seeds with a relative pivot below 1/256:", n_ill, "below 1e-3:", n_very, "of", int(fitted.sum()))
    assert n_ill >= 150 and n_very >= 50, (n_ill, n_very)
    rep = compare.compare(got, ref, np.asarray(data["offsets"]), p)
    print({k: v for k, v in rep.items() if k not in ("failures", "near_ties")})
    _assert_parity(rep, allow_ties_frac=5e-3)                    # iterations near the cut are likelier on these flat minima
    assert rep["seed_cov_max_rel_err"] <= compare.COV_RTOL and rep["seed_pos_max_err_mm"] <= compare.POS_TOL
