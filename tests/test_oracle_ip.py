"""Pins of the oracle's impact parameter and IP chi2.  CPU only."""
import numpy as np

from synth import events


def _tracks(rng, n, P, sigma=0.03, slope=0.25):
    tx = rng.normal(0, slope, n); ty = rng.normal(0, slope, n)
    zt = P[2] + rng.uniform(-5, 5, n)
    x = P[0] + (zt - P[2]) * tx + sigma * rng.normal(0, 1, n)
    y = P[1] + (zt - P[2]) * ty + sigma * rng.normal(0, 1, n)
    f = np.float32
    return dict(x=x.astype(f), y=y.astype(f), z=zt.astype(f), tx=tx.astype(f), ty=ty.astype(f),
                var_x=np.full(n, sigma * sigma, f), var_y=np.full(n, sigma * sigma, f),
                var_tx=np.full(n, 1e-6, f), var_ty=np.full(n, 1e-6, f))


def test_ip_is_the_distance_of_closest_approach_brute_force(oracle):
    """"the distance of closest approach of a track to a vertex": scan the straight line on a fine grid."""
    rng = np.random.default_rng(1)
    t = _tracks(rng, 20, np.array([0.1, -0.2, 30.0]), sigma=0.5, slope=0.3)
    for i in range(20):
        P = np.array([rng.normal(0, 0.3), rng.normal(0, 0.3), 30.0 + rng.normal(0, 2)])
        rc, ip, _ = oracle.ip_one(t, i, P, np.zeros(6))
        assert rc == 0
        zz = np.linspace(P[2] - 3, P[2] + 3, 600001)
        px = float(t["x"][i]) + (zz - float(t["z"][i])) * float(t["tx"][i])
        py = float(t["y"][i]) + (zz - float(t["z"][i])) * float(t["ty"][i])
        d = np.sqrt((px - P[0]) ** 2 + (py - P[1]) ** 2 + (zz - P[2]) ** 2).min()
        assert abs(ip - d) < 1e-8 + 1e-6 * d
    # a track through the vertex
    t0 = {k: v[:1].copy() for k, v in t.items()}
    P = [float(t0["x"][0]) + 2.0 * float(t0["tx"][0]), float(t0["y"][0]) + 2.0 * float(t0["ty"][0]), float(t0["z"][0]) + 2.0]
    rc, ip, c2 = oracle.ip_one(t0, 0, P, np.zeros(6))
    assert rc == 0 and ip < 1e-6 and c2 < 1e-6


def test_ip_chi2_is_the_chi2_difference_with_and_without_the_track(oracle):
    """"the chi2 difference of a PV reconstructed with and without the track": with unit weights the vertex
    fit is linear least squares, and r^T (V + H C H^T)^-1 r evaluated at the vertex fitted WITHOUT the track
    equals chi2(with) - chi2(without), both from the oracle's Newton fit."""
    rng = np.random.default_rng(2)
    P = np.array([0.0, 0.0, 5.0])
    t = _tracks(rng, 15, P)
    t["x"][14] += np.float32(0.12)                        # the track under test sits 4 sigma off
    p = oracle.default_params(chi2_max=np.inf, max_iter=4, conv_dz=0.0, conv_dchi2=0.0)
    seed = np.array([0.0, 0.0, 5.0])
    first = oracle.fit(t, np.arange(14), seed, p)
    # Eq. 2 is evaluated at the seed z in the fit and at the vertex z in the IP: seed both fits at the
    # converged vertex, so that the two coincide; chi2 is reported at the start of the last iteration = the minimum
    seed = first["pos"].copy()
    without = oracle.fit(t, np.arange(14), seed, p)
    with_ = oracle.fit(t, np.arange(15), seed, p)
    assert without["rc"] == 0 and with_["rc"] == 0 and np.abs(without["pos"] - seed).max() < 1e-4
    rc, ip, c2 = oracle.ip_one(t, 14, without["pos"], without["cov"])
    assert rc == 0
    delta = with_["chi2"] - without["chi2"]
    assert abs(c2 - delta) < 1e-4 * delta, (c2, delta)
    assert 3 < c2 < 25
    # C = 0 reduces to Eq. 7
    rc, _, c0 = oracle.ip_one(t, 14, without["pos"], np.zeros(6))
    assert abs(c0 - oracle.track_chi2(t, 14, without["pos"])) < 1e-12 * max(c0, 1)
    assert c0 > c2                                          # the vertex uncertainty can only lower the chi2


def test_track_ip_picks_the_smallest_chi2_vertex(oracle, cfg0, cfg0_oracle):
    """Whole batch: tracks that belong to a PV have their own PV as the smallest-IP-chi2 vertex (>= 98 %), prompt
    tracks have small IP chi2 and ghosts large; events without vertices give -1."""
    o = cfg0_oracle
    r = oracle.track_ip(cfg0, o["vtx_pos"], o["vtx_cov"], o["n_vtx"])
    tv = o["trk_vertex"]
    m = tv >= 0
    assert (r["ip_vertex"][m] == tv[m]).mean() > 0.98
    assert np.median(r["ip_chi2"][m]) < 3.0 and np.median(r["ip"][m]) < 0.1
    ghosts = cfg0["truth"]["trk_pv"] < 0
    assert np.median(r["ip_chi2"][ghosts & (r["ip_vertex"] >= 0)]) > 50
    empty = {k: (v.copy() if isinstance(v, np.ndarray) else v) for k, v in cfg0.items() if k != "truth"}
    nv = o["n_vtx"].copy(); nv[:10] = 0
    r2 = oracle.track_ip(empty, o["vtx_pos"], o["vtx_cov"], nv)
    t1 = cfg0["offsets"][10]
    assert np.all(r2["ip_vertex"][:t1] == -1) and np.all(r2["ip_chi2"][:t1] == -1.0)
    assert np.array_equal(r2["ip_vertex"][t1:], r["ip_vertex"][t1:])
