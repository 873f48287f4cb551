"""Pins of the oracle's peak search (O4), seed position (O5) and association (O6) against
hand-worked cases (tests/golden/peaks_handbuilt.json) and invariants.  PAPER.md L133-163."""
import json
import os

import numpy as np

S = 1 << 20
GOLD = os.path.join(os.path.dirname(__file__), "golden", "peaks_handbuilt.json")


def _hist(first, content):
    H = np.zeros(3400, np.int64)
    H[first:first + len(content)] = np.rint(np.asarray(content) * S).astype(np.int64)
    return H.astype(np.int32)


def test_handbuilt_histograms(oracle):
    p = oracle.default_params()
    with open(GOLD) as f:
        cases = json.load(f)["cases"]
    assert len(cases) >= 12
    for c in cases:
        H = _hist(c["first_bin"], c["content"])
        b, e, k, n = oracle.peaks(H, p)
        got = [list(map(int, t)) for t in zip(b, e, k)]
        assert got == c["clusters"], c["name"]
        assert n == len(c["clusters"])
        if c["seed_z"] is not None:
            for kk, zexp in zip(k, c["seed_z"]):
                assert abs(oracle.seed_z(H, int(kk), p) - zexp) < 1e-4, c["name"]


def test_handbuilt_histograms_x86_splitter(oracle):
    """R-16, the recursive x86 variant, against hand-worked cases; the same file also pins what the
    z-ordered variant gives on them (they differ when a small peak sits between the two largest)."""
    with open(os.path.join(os.path.dirname(GOLD), "peaks_x86_handbuilt.json")) as f:
        cases = json.load(f)["cases"]
    differ = 0
    for c in cases:
        H = _hist(c["first_bin"], c["content"])
        for mode, key in ((1, "clusters"), (0, "clusters_gpu")):
            b, e, k, n = oracle.peaks(H, oracle.default_params(split_mode=mode))
            got = [list(map(int, t)) for t in zip(b, e, k)]
            assert got == c[key], (c["name"], mode)
            assert n == len(c[key])
        differ += c["clusters"] != c["clusters_gpu"]
    assert differ >= 1


def test_x86_splitter_invariants_on_events(oracle, cfg0):
    """On real histograms: clusters disjoint, z-ordered, each with the minimum integral, within one proto-cluster
    contiguous; both variants cover the same bins whenever they keep a proto-cluster, and agree on most events."""
    from synth import events
    p0, p1 = oracle.default_params(), oracle.default_params(split_mode=1)
    data = events.generate(events.config(3, 600))                 # close pairs: many multi-peak proto-clusters
    r0 = oracle.find(data, p0, debug=True, n_hist_events=600)
    H = r0["debug"]["hist"]
    same = 0
    for e in range(600):
        b0, e0, k0, _ = oracle.peaks(H[e], p0)
        b1, e1, k1, _ = oracle.peaks(H[e], p1)
        assert np.all(b1[1:] >= e1[:-1]) and np.all(e1 > b1) and np.all((k1 >= b1) & (k1 < e1))
        for b, en, k in zip(b1, e1, k1):
            region = 1 if (-550 + 0.25 * (k + 0.5)) < -300 else 0
            assert H[e][b:en].astype(np.int64).sum() >= int(round((1.75 if region else 2.5) * S))
            assert H[e][k] == H[e][b:en].max() and (H[e][b:k] < H[e][k]).all()
        cover0 = np.zeros(3400, bool); cover1 = np.zeros(3400, bool)
        for b, en in zip(b0, e0): cover0[b:en] = True
        for b, en in zip(b1, e1): cover1[b:en] = True
        assert np.array_equal(cover0, cover1)
        same += (len(b0) == len(b1)) and np.array_equal(b0, b1)
    assert same > 500


def test_seed_delta_properties(oracle):
    """Eq. 5: symmetric peak -> delta = 0; N_{i+1} -> N_i gives delta -> +1/2; delta in [-1/2, 1/2]."""
    p = oracle.default_params()
    zi = -550 + 0.25 * 2200.5
    assert oracle.seed_z(_hist(2199, [1.0, 3.0, 1.0]), 2200, p) == np.float32(zi)
    assert abs(oracle.seed_z(_hist(2199, [1.0, 3.0, 3.0]), 2200, p) - (zi + 0.125)) < 1e-6
    assert abs(oracle.seed_z(_hist(2199, [2.999999, 3.0, 1.0]), 2200, p) - (zi - 0.125)) < 1e-5
    rng = np.random.default_rng(1)
    for _ in range(200):
        n0 = rng.uniform(1, 20); nm = rng.uniform(0, n0 * 0.999); npl = rng.uniform(0, n0)
        d = (oracle.seed_z(_hist(2199, [nm, n0, npl]), 2200, p) - zi) / 0.25
        assert -0.5 - 1e-6 <= d <= 0.5 + 1e-6
        assert abs(d - 0.5 * (npl - nm) / (2 * n0 - npl - nm)) < 1e-4


def test_seed_recovers_gaussian_mean(oracle):
    """A Gaussian-shaped peak sampled on the bins: the parabola-like correction recovers its mean to << dz."""
    p = oracle.default_params()
    rng = np.random.default_rng(2)
    worst = 0.0
    for _ in range(100):
        mu = np.float32(rng.uniform(-50, 50)); sg = np.float32(rng.uniform(0.15, 0.4))
        # 30 identical tracks -> a clean Gaussian-shaped peak, filled by the oracle's own contract fill
        H = oracle.fill(np.full(30, mu, np.float32), np.full(30, sg, np.float32), np.full(30, 3, np.int32), p)
        b, e, k, n = oracle.peaks(H, p)
        assert n == 1
        worst = max(worst, abs(oracle.seed_z(H, int(k[0]), p) - float(mu)))
    assert worst < 0.05                                # dz = 0.25


def test_peak_invariants_on_events(oracle, cfg0_oracle):
    """Clusters disjoint and z-ordered, integral above the cut, peak inside, peaks >= 2 bins apart (L125)."""
    p = oracle.default_params()
    Hs = cfg0_oracle["debug"]["hist"]
    nseen = 0
    for ev in range(0, 1000, 5):
        H = Hs[ev]
        b, e, k, n = oracle.peaks(H, p)
        nseen += n
        for j in range(n):
            assert 0 <= b[j] <= k[j] < e[j] <= 3400
            assert H[b[j]:e[j]].astype(np.int64).sum() >= int(round((2.5 if k[j] >= 1000 else 1.75) * S))
            assert H[k[j]] == H[b[j]:e[j]].max() and k[j] == b[j] + int(np.argmax(H[b[j]:e[j]]))
            assert np.all(H[b[j]:e[j]] > 0.25 * S)
            if j:
                assert b[j] >= e[j - 1] and k[j] - k[j - 1] >= 2
    assert nseen > 800


def test_assign_partition_points_and_unassignable(oracle):
    """Partition point = floor((end_k + begin_{k+1}) / 2) (L163, R-11); bins < p -> k, >= p -> k+1."""
    p = oracle.default_params(min_tracks_seed=(1, 1))
    begin, end, peak = [2100, 2120, 2131], [2110, 2131, 2140], [2105, 2125, 2135]
    zs = [0.0, 1.0, 2.0]
    bins = [2114, 2115, 2130, 2131, 0, 3399, 2000]
    flags = [1, 1, 1, 1, 1, 1, 0]
    ts, *_ = oracle.assign(bins, flags, begin, end, peak, zs, p)
    assert list(ts) == [0, 1, 1, 2, 0, 2, -1]
    ts, *_ = oracle.assign([2114, 2115], [1, 1], [2100, 2120], [2111, 2131], [2105, 2125], [0.0, 1.0], p)
    assert list(ts) == [0, 1]                          # (2111 + 2120) // 2 = 2115


def test_assign_removal_order(oracle):
    """Seeds under 3 (pp) / 2 (SMOG2) tracks are removed one at a time, least populated first,
    ties at lowest z, and the tracks are re-distributed (L163)."""
    p = oracle.default_params()
    begin, end, peak = [2100, 2120, 2140], [2110, 2130, 2150], [2105, 2125, 2145]
    zs = [-24.0, -19.0, -14.0]
    # counts A=1, B=5, C=2 -> A removed first (its track goes to B), then C (2 < 3): all 8 end in B
    bins = [2105] + [2125] * 5 + [2145] * 2
    ts, b, e, k, z = oracle.assign(bins, [1] * 8, begin, end, peak, zs, p)
    assert list(b) == [2120] and list(ts) == [0] * 8
    # tie A=2, C=2: lowest z first; after A is gone B has 5 and C still 2 -> removed too
    bins = [2105] * 2 + [2125] * 3 + [2145] * 2
    ts, b, e, k, z = oracle.assign(bins, [1] * 7, begin, end, peak, zs, p)
    assert list(b) == [2120]
    # after removing the weakest the neighbour may pass: A=2, B=2 -> A removed, B becomes 4, stays
    ts, b, e, k, z = oracle.assign([2105] * 2 + [2125] * 2, [1] * 4, begin[:2], end[:2], peak[:2], zs[:2], p)
    assert list(b) == [2120] and list(ts) == [0, 0, 0, 0]
    # SMOG2 region: 2 tracks are enough (z_seed < -300)
    ts, b, e, k, z = oracle.assign([400, 401], [1, 1], [398], [404], [400], [-449.9], p)
    assert list(b) == [398] and list(ts) == [0, 0]
    ts, b, e, k, z = oracle.assign([2200, 2201], [1, 1], [2198], [2204], [2200], [0.1], p)
    assert len(b) == 0 and list(ts) == [-1, -1]
