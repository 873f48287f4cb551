"""Pins of the oracle's multi-vertex (GPU) flavour: implicit association and the weights of Eq. 19
(PAPER.md L234-239), convergence on |dz| alone.  CPU only."""
import numpy as np

from synth import events


def _tracks_from_point(rng, n, P, sigma=0.03, slope=0.25, noise=True):
    tx = rng.normal(0, slope, n); ty = rng.normal(0, slope, n)
    zt = P[2] + rng.uniform(-5, 5, n)
    sx = np.full(n, sigma)
    x = P[0] + (zt - P[2]) * tx + (sx * rng.normal(0, 1, n) if noise else 0.0)
    y = P[1] + (zt - P[2]) * ty + (sx * rng.normal(0, 1, n) if noise else 0.0)
    f = np.float32
    return dict(x=x.astype(f), y=y.astype(f), z=zt.astype(f), tx=tx.astype(f), ty=ty.astype(f), var_x=(sx * sx).astype(f),
                var_y=(sx * sx).astype(f), var_tx=np.full(n, 1e-6, f), var_ty=np.full(n, 1e-6, f))


def test_eq19_weight_properties(oracle):
    """chi2_max is "the chi2 value at which the weight is equal to 0.5 in the case of no other competing
    vertices"; a competing vertex lowers the weight; the weights of one track over all candidates sum to < 1."""
    w = oracle.mv_weight
    for cm in (4.0, 9.0, 12.0):
        assert abs(w(cm, cm) - 0.5) < 1e-15
    c = np.linspace(0, 40, 200)
    w0 = np.array([w(ci, 12.0) for ci in c])
    assert np.all(np.diff(w0) < 0) and w0[0] > 0.99 and w0[-1] < 1e-6            # monotone, "not a strict cut-off"
    assert w(2.0, 4.0, [9.0]) < w(2.0, 4.0) and w(2.0, 4.0, [3.0]) < w(2.0, 4.0, [9.0])   # Fig. 6 ordering
    assert abs(w(5.0, 4.0, [5.0]) - w(5.0, 4.0, [5.0])) == 0.0
    # a track seen from three candidates: sum_j w_ij = sum E / (e0 + sum E) < 1, and each is the Eq. 19 ratio
    chi = [1.0, 6.0, 15.0]
    ws = [w(chi[j], 4.0, [chi[k] for k in range(3) if k != j]) for j in range(3)]
    assert 0.0 < sum(ws) < 1.0
    assert abs(ws[0] / ws[1] - np.exp(-0.5 * (chi[0] - chi[1]))) < 1e-12         # ratio of two weights of one track
    # no competitor and chi2_max -> infinity: unit weights
    assert abs(w(30.0, 1e4) - 1.0) < 1e-12


def test_track_chi2_closed_forms(oracle):
    """Eq. 7 with W from Eq. 2: a track through the vertex has chi2 0; displaced by k sigma in x it has k^2; the
    slope variance enters with dz^2 (Eq. 2 diagonal)."""
    f = np.float32
    t = dict(x=np.array([0.5], f), y=np.array([-0.25], f), z=np.array([10.0], f), tx=np.array([0.125], f), ty=np.array([-0.0625], f),
             var_x=np.array([0.0009], f), var_y=np.array([0.0016], f), var_tx=np.array([1e-6], f), var_ty=np.array([4e-6], f))
    zv = 18.0
    on = [0.5 + 8 * 0.125, -0.25 - 8 * 0.0625, zv]
    assert abs(oracle.track_chi2(t, 0, on)) < 1e-12
    Vx = float(t["var_x"][0]) + 64 * float(t["var_tx"][0]); Vy = float(t["var_y"][0]) + 64 * float(t["var_ty"][0])
    assert abs(oracle.track_chi2(t, 0, [on[0] - 3 * np.sqrt(Vx), on[1], zv]) - 9.0) < 1e-9
    assert abs(oracle.track_chi2(t, 0, [on[0], on[1] + 2 * np.sqrt(Vy), zv]) - 4.0) < 1e-9
    t["var_x"][0] = 0.0
    t["var_tx"][0] = 0.0
    assert oracle.track_chi2(t, 0, on) < 0                                        # unusable (R-7)


def test_mv_fit_with_unit_weights_is_the_analytic_least_squares(oracle):
    """other = 0 makes every Eq. 19 weight exactly 1: the first Newton step then lands on the weighted
    least-squares point computed independently with numpy, and the second step is 0."""
    rng = np.random.default_rng(3)
    P = np.array([0.02, -0.03, 12.5])
    t = _tracks_from_point(rng, 25, P)
    idx = np.arange(25)
    seed = np.array([0.0, 0.0, 12.3])
    p = oracle.mv_params(max_iter=3, conv_dz=0.0)
    r = oracle.fit_mv(t, idx, seed, np.zeros(25), p)
    assert r["rc"] == 0 and np.all(r["w"] == 1.0) and r["ntrk"] == 25
    # independent weighted LSQ: rows (x: [1, 0, -tx], y: [0, 1, -ty]) alpha = (x - z tx, y - z ty), weights 1 / V(seed z)
    dz = seed[2] - t["z"].astype(float)
    Vx = t["var_x"].astype(float) + dz * dz * t["var_tx"].astype(float)
    Vy = t["var_y"].astype(float) + dz * dz * t["var_ty"].astype(float)
    A = np.zeros((50, 3)); b = np.zeros(50)
    A[:25, 0] = 1; A[:25, 2] = -t["tx"]; b[:25] = t["x"].astype(float) - t["z"].astype(float) * t["tx"]
    A[25:, 1] = 1; A[25:, 2] = -t["ty"]; b[25:] = t["y"].astype(float) - t["z"].astype(float) * t["ty"]
    sw = np.sqrt(np.concatenate([1 / Vx, 1 / Vy]))
    sol = np.linalg.lstsq(A * sw[:, None], b * sw, rcond=None)[0]
    assert np.allclose(r["trace"][0, :3], sol, atol=1e-10)
    assert np.abs(r["trace"][1, :3] - r["trace"][0, :3]).max() < 1e-10
    C = np.linalg.inv((A * sw[:, None]).T @ (A * sw[:, None]))
    assert np.allclose(r["cov"], [C[0, 0], C[0, 1], C[0, 2], C[1, 1], C[1, 2], C[2, 2]], rtol=1e-9)
    # and it is the explicit flavour's unit-weight fit
    r0 = oracle.fit(t, idx, seed, oracle.default_params(chi2_max=np.inf, max_iter=3, conv_dz=0.0))
    assert np.allclose(r0["pos"], r["pos"], atol=1e-12)


def test_mv_fit_downweights_a_track_claimed_by_another_vertex(oracle):
    """A track that is 2 sigma away counts less when another candidate explains it better (Eq. 19), and the fitted
    position moves away from it accordingly; weights are those of Eq. 19 at the position of the last iteration."""
    rng = np.random.default_rng(5)
    P = np.array([0.0, 0.0, 0.0])
    t = _tracks_from_point(rng, 12, P, noise=False)
    t["x"][0] += np.float32(0.06)                                                 # 2 sigma outlier
    idx = np.arange(12)
    p = oracle.mv_params()
    e0 = np.exp(-0.5 * 12.0)
    alone = oracle.fit_mv(t, idx, P, np.full(12, e0), p)
    other = np.full(12, e0); other[0] += np.exp(-0.5 * 0.1)                       # a competitor at chi2 = 0.1 for track 0
    shared = oracle.fit_mv(t, idx, P, other, p)
    assert alone["rc"] == 0 and shared["rc"] == 0
    assert shared["w"][0] < 0.5 * alone["w"][0] and np.allclose(shared["w"][1:], 1 / (1 + e0), atol=2e-3)
    assert abs(shared["pos"][0]) < abs(alone["pos"][0])
    # the reported weight is Eq. 19 evaluated at the position before the last step
    it = shared["niter"]
    prev = shared["trace"][it - 2, :3] if it >= 2 else P
    c2 = oracle.track_chi2(t, 0, [prev[0], prev[1], prev[2]])
    # W is frozen at the seed z while track_chi2 takes it at prev z: identical here because var_t dz^2 << var
    assert abs(shared["w"][0] - np.exp(-0.5 * c2) / (other[0] + np.exp(-0.5 * c2))) < 1e-5
    assert shared["ntrk"] == 11 and alone["ntrk"] == 12                            # w >= 1/2 counts as associated


def test_mv_pipeline_sanity_on_synthetic_events(oracle, cfg0):
    """Whole path in the multi-vertex flavour on configs[0]: efficiency and fakes like the explicit flavour
    ("98 % matched"), z pull width ~ 1, fits converge on |dz| < 0.5 um in a few iterations,
    thread-count invariance, and every followed track has a weight in (0, 1)."""
    p = oracle.mv_params()
    r = oracle.find(cfg0, p, debug=True, n_threads=1)
    r4 = oracle.find(cfg0, p, debug=True, n_threads=4)
    for k in ("vtx_pos", "n_vtx", "trk_vertex", "trk_weight"):
        assert np.array_equal(r[k], r4[k])
    r0 = oracle.find(cfg0, oracle.default_params())
    assert abs(int(r["n_vtx"].sum()) - int(r0["n_vtx"].sum())) < 0.01 * r0["n_vtx"].sum()
    # matching between the flavours: every explicit-flavour vertex has a multi-vertex one within 5 sigma_z
    mv = p.max_vtx_per_event
    matched = tot = 0
    pulls = []
    truth = cfg0["truth"]
    for e in range(300):
        za = r0["vtx_pos"][e, :r0["n_vtx"][e], 2]; zb = r["vtx_pos"][e, :r["n_vtx"][e], 2]
        sb = np.sqrt(r["vtx_cov"][e, :r["n_vtx"][e], 5])
        for z in za:
            tot += 1
            if zb.size and np.min(np.abs(zb - z) / np.maximum(sb, 1e-9)) < 5:
                matched += 1
        tz = truth["pv_z"][truth["pv_event"] == e]
        for k in range(zb.size):
            j = np.argmin(np.abs(tz - zb[k]))
            if abs(tz[j] - zb[k]) < 5 * sb[k]:
                pulls.append((zb[k] - tz[j]) / sb[k])
    assert matched / tot > 0.98
    pulls = np.array(pulls)
    assert 0.85 < np.std(pulls[np.abs(pulls) < 5]) < 1.25 and abs(np.mean(pulls)) < 0.1
    it = r["debug"]["seed_niter"]
    it = it[it > 0]
    assert np.median(it) <= 4 and (it == 10).mean() < 0.02
    w = r["trk_weight"][r["trk_vertex"] >= 0]
    assert np.all(w > 0) and np.all(w < 1)


def test_handworked_event_pins_the_association_glue(oracle):
    """tests/golden/mv_handworked.json: window membership, the 'other candidates' part of the denominator of Eq. 19
    (all candidates, listed or not), the followed candidate and the associated-track count of find_event."""
    import json
    import os
    from synth import events
    with open(os.path.join(os.path.dirname(__file__), "golden", "mv_handworked.json")) as f:
        g = json.load(f)
    ev = {k: np.asarray(g["event"][k], np.float32) for k in events.FIELDS}
    data = events.from_lists([ev])
    for c in g["cases"]:
        p = oracle.mv_params(chi2_window=c["chi2_window"], **g["params"])
        r = oracle.find(data, p, debug=True, n_hist_events=1)
        d = r["debug"]
        assert d["n_seeds"][0] == 2 and list(d["seed_z"][0, :2]) == [0.125, 10.125]          # delta = 0 (Eq. 5)
        assert list(d["seed_bins"][0, :2, 2]) == [2200, 2240]
        assert d["hist"][0, 2212] == 0                                                      # T5 is not histogrammed
        assert list(d["trk_seed"]) == c["trk_seed"], c["_why"]
        assert list(r["trk_vertex"]) == c["trk_seed"]
        assert np.allclose(r["trk_weight"], c["trk_weight"], atol=2e-6, rtol=0), (c["_why"], r["trk_weight"])
        assert np.allclose(d["trk_w2"], c["runner_up_weight"], atol=2e-6, rtol=0), (c["_why"], d["trk_w2"])
        assert r["n_vtx"][0] == 2 and list(r["vtx_ntracks"][0, :2]) == c["vtx_ntracks"], c["_why"]
