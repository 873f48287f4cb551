"""Pins of the x-tx / y-ty covariance terms of Eq. 2 in the oracle (NEXT-2).  CPU only."""
import numpy as np


def _tracks(rng, n, P, sigma=0.03, slope=0.25):
    tx = rng.normal(0, slope, n); ty = rng.normal(0, slope, n)
    zt = P[2] + rng.uniform(-5, 5, n)
    x = P[0] + (zt - P[2]) * tx + sigma * rng.normal(0, 1, n)
    y = P[1] + (zt - P[2]) * ty + sigma * rng.normal(0, 1, n)
    f = np.float64
    return dict(x=x.astype(f), y=y.astype(f), z=zt.astype(f), tx=tx.astype(f), ty=ty.astype(f),
                var_x=np.full(n, sigma * sigma, f), var_y=np.full(n, 1.5 * sigma * sigma, f),
                var_tx=np.full(n, 4e-6, f), var_ty=np.full(n, 1e-6, f))


def _transport(t, L):
    """The same straight-line tracks, their states re-expressed at z + L: x' = x + L tx, and by linear error
    propagation V_xx' = V_xx + 2 L V_xtx + L^2 V_txtx, V_xtx' = V_xtx + L V_txtx (V_txtx unchanged)."""
    c0x = t.get("cov_xtx", np.zeros_like(t["x"])); c0y = t.get("cov_yty", np.zeros_like(t["x"]))
    o = dict(t)
    o["x"] = t["x"] + L * t["tx"]; o["y"] = t["y"] + L * t["ty"]; o["z"] = t["z"] + L
    o["var_x"] = t["var_x"] + 2 * L * c0x + L * L * t["var_tx"]; o["cov_xtx"] = c0x + L * t["var_tx"]
    o["var_y"] = t["var_y"] + 2 * L * c0y + L * L * t["var_ty"]; o["cov_yty"] = c0y + L * t["var_ty"]
    return o


def _f32(t):
    return {k: np.asarray(v, np.float32) for k, v in t.items()}


def test_fit_is_invariant_under_transport_of_the_track_states(oracle):
    """The vertex must not depend on the z at which the track states are quoted: with the cross terms of Eq. 2 the
    extrapolated variance at the vertex is the same for a state and its transported copy.  (Dropping the term, its
    factor 2 or its sign breaks this by many sigma.)"""
    rng = np.random.default_rng(4)
    P = np.array([0.03, -0.02, 20.0])
    t = _tracks(rng, 18, P)
    L = rng.uniform(30, 120, 18) * rng.choice([-1, 1], 18)        # far enough for L^2 V_tt >> V_xx
    a, b = _f32(t), _f32(_transport(t, L))
    idx = np.arange(18)
    seed = np.array([0.0, 0.0, 19.5])
    for p in (oracle.default_params(), oracle.default_params(chi2_max=np.inf)):
        ra, rb = oracle.fit(a, idx, seed, p), oracle.fit(b, idx, seed, p)
        assert ra["rc"] == 0 and rb["rc"] == 0 and ra["niter"] == rb["niter"]
        assert np.abs(ra["pos"] - rb["pos"]).max() < 2e-4            # fp32 inputs: x' = x + L tx rounds at 1e-5 mm
        assert np.allclose(ra["cov"], rb["cov"], rtol=2e-3)
        assert np.allclose(ra["w"], rb["w"], atol=5e-3)
    # without the cross terms the transported states give a different (wrong) answer
    c = {k: v for k, v in b.items() if not k.startswith("cov_")}
    rc = oracle.fit(c, idx, seed, oracle.default_params(chi2_max=np.inf))
    assert np.abs(np.array(rc["cov"]) / np.array(ra["cov"]) - 1).max() > 0.5


def test_chi2_and_ip_with_cross_terms_closed_forms(oracle):
    """Eq. 2 for one coordinate: sigma^2(z) = V_xx + 2 dz V_xtx + dz^2 V_txtx; a track displaced by k sigma(z) has
    chi2 = k^2; the IP chi2 with C = 0 is the same number; negative extrapolated variance is unusable (R-7)."""
    f = np.float32
    t = dict(x=np.array([0.2], f), y=np.array([0.1], f), z=np.array([0.0], f), tx=np.array([0.25], f), ty=np.array([-0.125], f),
             var_x=np.array([0.01], f), var_y=np.array([0.04], f), var_tx=np.array([1e-4], f), var_ty=np.array([4e-4], f),
             cov_xtx=np.array([-5e-4], f), cov_yty=np.array([1e-3], f))
    dz = 8.0
    Vx = 0.01 + 2 * dz * (-5e-4) + dz * dz * 1e-4            # 0.0084
    Vy = 0.04 + 2 * dz * 1e-3 + dz * dz * 4e-4               # 0.0816
    on = np.array([0.2 + dz * 0.25, 0.1 - dz * 0.125, dz])
    assert abs(oracle.track_chi2(t, 0, on)) < 1e-10
    c2 = oracle.track_chi2(t, 0, [on[0] + 2 * np.sqrt(Vx), on[1] - 3 * np.sqrt(Vy), dz])
    assert abs(c2 - 13.0) < 1e-4
    rc, ip, ipc = oracle.ip_one(t, 0, [on[0] + 2 * np.sqrt(Vx), on[1] - 3 * np.sqrt(Vy), dz], np.zeros(6))
    assert rc == 0 and abs(ipc - c2) < 1e-9
    t["cov_xtx"][0] = f(-2e-3)                                # V_xx(8) = 0.01 - 0.032 + 0.0064 < 0
    assert oracle.track_chi2(t, 0, on) < 0


def test_unit_weight_fit_with_cross_terms_is_the_analytic_least_squares(oracle):
    rng = np.random.default_rng(6)
    P = np.array([0.0, 0.0, -3.0])
    t = _transport(_tracks(rng, 20, P), rng.uniform(-80, 80, 20))
    t32 = _f32(t)
    seed = np.array([0.0, 0.0, -3.2])
    r = oracle.fit(t32, np.arange(20), seed, oracle.default_params(chi2_max=np.inf, max_iter=3, conv_dz=0.0))
    T = {k: v.astype(np.float64) for k, v in t32.items()}
    dz = seed[2] - T["z"]
    Vx = T["var_x"] + 2 * dz * T["cov_xtx"] + dz * dz * T["var_tx"]
    Vy = T["var_y"] + 2 * dz * T["cov_yty"] + dz * dz * T["var_ty"]
    A = np.zeros((40, 3)); b = np.zeros(40)
    A[:20, 0] = 1; A[:20, 2] = -T["tx"]; b[:20] = T["x"] - T["z"] * T["tx"]
    A[20:, 1] = 1; A[20:, 2] = -T["ty"]; b[20:] = T["y"] - T["z"] * T["ty"]
    sw = np.sqrt(np.concatenate([1 / Vx, 1 / Vy]))
    sol = np.linalg.lstsq(A * sw[:, None], b * sw, rcond=None)[0]
    assert np.allclose(r["trace"][0, :3], sol, atol=1e-9)


def test_pipeline_with_cross_terms(oracle, cfg0):
    """Whole path: transporting every track state of configs[0] by a random L (sigma_poca of Eq. 3 is evaluated
    from V_xx at the state's own z, so it is kept by transporting only tracks' covariance reference, not their
    histogram inputs: here L is small, |L| < 2 mm) leaves the vertex count and the positions essentially unchanged,
    in both flavours; zero cross-term arrays are bit-identical to none."""
    from synth import events
    d = events.slice_events(cfg0, 0, 300)
    zero = dict(d); zero["cov_xtx"] = np.zeros_like(d["x"]); zero["cov_yty"] = np.zeros_like(d["x"])
    for p in (oracle.default_params(), oracle.mv_params()):
        r0, rz = oracle.find(d, p), oracle.find(zero, p)
        for k in ("vtx_pos", "vtx_cov", "n_vtx", "trk_weight", "trk_vertex"):
            assert np.array_equal(r0[k], rz[k])
    rng = np.random.default_rng(8)
    L = rng.uniform(-2, 2, d["x"].size)
    t = _transport({k: np.asarray(d[k], np.float64) for k in ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")}, L)
    moved = _f32(t); moved["offsets"] = d["offsets"]
    r0, r1 = oracle.find(d, oracle.default_params()), oracle.find(moved, oracle.default_params())
    same = r0["n_vtx"] == r1["n_vtx"]
    assert same.mean() > 0.97
    m = (np.arange(32)[None, :] < r0["n_vtx"][:, None]) & same[:, None]
    assert np.median(np.abs(r0["vtx_pos"][m] - r1["vtx_pos"][m]).max(axis=-1)) < 2e-3
