"""Pins of the oracle's fixed-point histogram fill (O3).  PAPER.md L125-131."""
import math

import numpy as np
from scipy.special import ndtr

S = 1 << 20
HIST = 1 | 2


def test_layout(oracle):
    """3400 bins of 0.25 mm over [-550, 300] (L125)."""
    p = oracle.default_params()
    assert oracle.nbins(p) == 3400


def test_cdf_limits_symmetry_monotone(oracle):
    p = oracle.default_params()
    zp, sp = 0.125, 0.4
    ks = np.arange(2150, 2260)
    q = np.array([oracle.edge_q(int(k), zp, sp, p) for k in ks])
    assert q[0] == 0 and q[-1] == S
    assert np.all(np.diff(q) >= 0)
    # edges beyond +-3 sigma are exactly 0 / S (compact support, reading R-6)
    e = -550 + 0.25 * ks
    assert np.all(q[e <= zp - 3 * sp - 1e-4] == 0) and np.all(q[e >= zp + 3 * sp + 1e-4] == S)
    # odd polynomial: Q(+s) + Q(-s) = S up to one rounding; track centred on an edge (k=2200 -> z=0)
    qs = np.array([oracle.edge_q(2200 + d, 0.0, 0.5, p) for d in range(-7, 8)])
    assert np.all(np.abs(qs + qs[::-1] - S) <= 1)
    assert qs[7] == S // 2


def test_single_track_vs_closed_form(oracle):
    """Bin contents of one track against Phi differences: (i) the truncated-renormalised Gaussian the
    contract approximates (|err| <= 1e-5 per edge), (ii) the exact integral of P:L129 within the
    truncation bound 2 Phi(-3) / (1 - 2 Phi(-3)) + 1e-5."""
    p = oracle.default_params()
    rng = np.random.default_rng(3)
    tail = ndtr(-3.0)
    for _ in range(40):
        zp = np.float32(rng.uniform(-100, 100)); sp = np.float32(rng.uniform(0.03, 1.5))
        H = oracle.fill([zp], [sp], [HIST], p).astype(np.float64) / S
        edges = -550.0 + 0.25 * np.arange(3401)
        u = (edges - float(zp)) / float(sp)
        F = np.clip((ndtr(u) - tail) / (1 - 2 * tail), 0, 1)
        F[u <= -3] = 0; F[u >= 3] = 1
        assert np.abs(H - np.diff(F)).max() < 2.0e-5
        exact = np.diff(ndtr(u))
        assert np.abs(H - exact).max() <= 2 * tail / (1 - 2 * tail) + 1e-5
        H0 = oracle.fill_exact([zp], [sp], [HIST], p)
        assert np.abs(H0 - exact).max() < 1e-12
        assert H.sum() == 1.0                         # "contributions of a single track add up to unity"


def test_mass_conservation_exact(oracle, cfg0_oracle):
    """Sum of all bins == sum over histogrammed tracks of Q(top edge) - Q(bottom edge), exactly."""
    p = oracle.default_params()
    d = cfg0_oracle["debug"]
    H = d["hist"].astype(np.int64)
    from synth import events
    off = events.generate(events.config(0))["offsets"]
    for e in range(0, 1000, 37):
        sl = slice(off[e], off[e + 1])
        fl, zp, sp = d["trk_flags"][sl], d["z_poca"][sl], d["sigma_poca"][sl]
        acc = (fl & 2) != 0
        mass = sum(oracle.edge_q(3400, float(a), float(b), p) - oracle.edge_q(0, float(a), float(b), p)
                   for a, b in zip(zp[acc], sp[acc]))
        assert H[e].sum() == mass
        inside = acc & (zp - 3 * sp > -550) & (zp + 3 * sp < 300)
        assert mass >= inside.sum() * S


def test_mass_at_the_range_edge(oracle):
    """A track centred on the upper range limit keeps half of its mass."""
    p = oracle.default_params()
    H = oracle.fill([np.float32(299.999)], [np.float32(0.5)], [HIST], p)
    assert abs(H.sum() / S - 0.5) < 2e-3
    assert H[:3390].sum() == 0


def test_permutation_invariance_bitwise(oracle):
    rng = np.random.default_rng(5)
    p = oracle.default_params()
    n = 300
    zp = rng.normal(0, 40, n).astype(np.float32); sp = rng.uniform(0.02, 1.4, n).astype(np.float32)
    fl = np.full(n, HIST, np.int32)
    H = oracle.fill(zp, sp, fl, p)
    for _ in range(3):
        perm = rng.permutation(n)
        assert np.array_equal(H, oracle.fill(zp[perm], sp[perm], fl, p))


def test_whole_bin_shift(oracle):
    """Shifting every z_poca by a whole number of bins shifts the histogram (exact for dyadic inputs)."""
    rng = np.random.default_rng(6)
    p = oracle.default_params()
    n = 200
    zp = (rng.integers(-40 * 1024, 40 * 1024, n) / 1024.0).astype(np.float32)    # multiples of 2^-10
    sp = (rng.integers(8, 256, n) / 256.0).astype(np.float32)
    fl = np.full(n, HIST, np.int32)
    H = oracle.fill(zp, sp, fl, p)
    for shift_bins in (1, 7, -33, 400):
        H2 = oracle.fill(zp + np.float32(0.25 * shift_bins), sp, fl, p)
        assert np.array_equal(np.roll(H, shift_bins), H2)


def test_window_equals_full_range(oracle, cfg0_oracle):
    """The finite window is only an optimisation: evaluating every edge gives the same bins."""
    p = oracle.default_params()
    d = cfg0_oracle["debug"]
    sl = slice(0, 5000)
    a = oracle.fill(d["z_poca"][sl], d["sigma_poca"][sl], d["trk_flags"][sl], p, full_range=False)
    b = oracle.fill(d["z_poca"][sl], d["sigma_poca"][sl], d["trk_flags"][sl], p, full_range=True)
    assert np.array_equal(a, b)
    # including wide gas-cell tracks and tracks hugging both range limits
    zp = np.array([-549.9, -540.0, 299.9, 295.0, -450.0], np.float32)
    sp = np.array([5.0, 9.9, 1.4, 0.7, 10.0], np.float32)
    fl = np.full(5, HIST, np.int32)
    assert np.array_equal(oracle.fill(zp, sp, fl, p, False), oracle.fill(zp, sp, fl, p, True))


def test_l1_vs_l0_bound_on_events(oracle, cfg0_oracle):
    """Contract histogram vs exact erf integrals on real events: per-bin error bounded by
    m_i * (2 Phi(-3)/(1-2 Phi(-3)) + 1e-5), m_i = tracks overlapping bin i."""
    p = oracle.default_params()
    d = cfg0_oracle["debug"]
    from synth import events
    off = events.generate(events.config(0))["offsets"]
    tail = ndtr(-3.0)
    per_track = 2 * tail / (1 - 2 * tail) + 1e-5
    for e in (0, 1, 2, 500, 999):
        sl = slice(off[e], off[e + 1])
        zp, sp, fl = d["z_poca"][sl], d["sigma_poca"][sl], d["trk_flags"][sl]
        H0 = oracle.fill_exact(zp, sp, fl, p)
        H1 = d["hist"][e].astype(np.float64) / S
        acc = (fl & 2) != 0
        edges = -550.0 + 0.25 * np.arange(3401)
        m = np.zeros(3400)
        for a, b in zip(zp[acc].astype(np.float64), sp[acc].astype(np.float64)):
            m += (edges[1:] > a - 10 * b) & (edges[:-1] < a + 10 * b)
        assert np.all(np.abs(H1 - H0) <= m * per_track + 1e-12)
        assert np.abs(H1 - H0).max() < 0.06


def test_frozen_cdf_coefficients_are_the_documented_fit(oracle):
    """The seven fp32 literals of the CDF contract (R-6) are the least-squares fit oracle/fit_cdf_poly.py
    describes: recompute them from scipy's Phi and compare with the literals in pv_oracle.c bit by bit."""
    import os
    import re
    from oracle import fit_cdf_poly
    src = open(os.path.join(os.path.dirname(fit_cdf_poly.__file__), "pv_oracle.c")).read()
    body = re.search(r"PVO_G\[7\]\s*=\s*\{(.*?)\}", src, flags=re.S).group(1)
    frozen = np.array([float.fromhex(t.strip().rstrip("f")) for t in body.split(",")], dtype=np.float32)
    assert frozen.size == 7
    assert np.array_equal(frozen.view(np.uint32), fit_cdf_poly.fit().view(np.uint32))
    # and the polynomial stays within 1e-5 of its target over the whole support, in fp32 arithmetic
    s = np.linspace(-1, 1, 20001).astype(np.float32)
    t = s * s
    g = np.full_like(s, frozen[6])
    for j in range(5, -1, -1):
        g = (g * t + frozen[j]).astype(np.float32)
    F = (s * g + np.float32(0.5)).astype(np.float64)
    tail = ndtr(-3.0)
    assert np.abs(F - (ndtr(3.0 * s.astype(np.float64)) - tail) / (1 - 2 * tail)).max() < 1e-5

