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



# ---- x86 variant: template histograms selected by sigma_poca (reading R-17) ------------------------------------

def test_template_class_is_the_nearest_in_log_sigma(oracle):
    """Class k has its centre at 0.08 dz 2^(k/4); a sigma takes the class nearest in log sigma, clamped to
    [0, class of the largest sigma cut].  The expectation is the closed form round(4 log2(sigma / (0.08 dz)))."""
    p = oracle.default_params()
    dz = 0.25
    kmax = round(4 * math.log2(10.0 / (0.08 * dz)))
    assert kmax == 36
    for k in range(0, kmax + 1):
        centre = 0.08 * dz * 2.0 ** (k / 4)
        assert oracle.tmpl_class(centre, p) == k
        assert oracle.tmpl_class(centre * 2.0 ** (0.124), p) == k                    # just below the upper class edge
        assert oracle.tmpl_class(centre * 2.0 ** (0.126), p) == min(k + 1, kmax)     # just above it
        assert oracle.tmpl_halfwidth(k) == math.ceil(3 * float(np.float32(0.08) * np.float32(2.0 ** (k / 4))) - 1e-9)
    assert oracle.tmpl_class(1e-6, p) == 0 and oracle.tmpl_class(0.0, p) == 0
    assert oracle.tmpl_class(1e9, p) == kmax
    rng = np.random.default_rng(4)
    for s in np.exp(rng.uniform(np.log(0.02), np.log(10.0), 500)):
        x = 4 * math.log2(s / (0.08 * dz))
        if abs(x - math.floor(x) - 0.5) > 1e-4:                                      # away from a class edge
            assert oracle.tmpl_class(float(np.float32(s)), p) == min(max(round(x), 0), kmax)
    # another binning and cut: the finite set follows the largest sigma cut
    q = oracle.default_params(dz=0.5, max_sigma_poca=(1.5, 3.0))
    assert oracle.tmpl_class(100.0, q) == round(4 * math.log2(3.0 / (0.08 * 0.5)))


def test_templates_are_gaussian_bin_integrals_of_unit_mass(oracle):
    """Every template sums to exactly 2^20 ("the contributions for a single track add up to unity"), is
    non-negative, is the mirror image of the template for the mirrored position inside the bin (to the rounding of the
    two edges), and equals the Phi
    differences of a Gaussian of width sigma_k centred on the j-th eighth of the central bin (truncated at +-3 sigma and
    renormalised, as the contract of reading R-6) to 2e-5."""
    tail = ndtr(-3.0)
    for k in range(0, 37):
        W = oracle.tmpl_halfwidth(k)
        u = float(np.float32(0.08) * np.float32(2.0 ** (k / 4)))
        for j in range(8):
            T = oracle.tmpl(k, j)
            assert T.size == 2 * W + 1 and T.sum() == S and T.min() >= 0
            assert np.abs(T[::-1] - oracle.tmpl(k, 7 - j)).max() <= 2      # Q(s) + Q(-s) = 2^20 up to one rounding per edge
            if k % 5 == 0 or k == 36:
                zrel = (j + 0.5) / 8
                edges = np.arange(-W, W + 2) - zrel
                F = np.clip((ndtr(edges / u) - tail) / (1 - 2 * tail), 0, 1)
                F[edges / u <= -3] = 0; F[edges / u >= 3] = 1
                assert np.abs(T / S - np.diff(F)).max() < 2.0e-5, (k, j)
    # a narrow track keeps (almost) all its mass in the central bin; a wide one spreads it
    assert oracle.tmpl(0, 4)[oracle.tmpl_halfwidth(0)] > 0.99 * S
    assert oracle.tmpl(30, 4).max() < 0.05 * S


def test_template_fill_places_the_selected_template(oracle):
    """One track: the histogram is template (class of its sigma, eighth of its z_poca) centred on its central bin;
    bins beyond the range are dropped; the fill is an integer sum, so track order does not matter."""
    p = oracle.default_params(fill_mode=1)
    rng = np.random.default_rng(8)
    for _ in range(60):
        b = int(rng.integers(5, 3390)); j = int(rng.integers(0, 8))
        zp = np.float32(-550 + 0.25 * (b + (j + rng.uniform(0.05, 0.95)) / 8))
        sp = np.float32(np.exp(rng.uniform(np.log(0.02), np.log(9.0))))
        k = round(4 * math.log2(float(sp) / 0.02))
        if abs(4 * math.log2(float(sp) / 0.02) - k) > 0.49:
            continue
        H = oracle.fill_template([zp], [sp], [b], [HIST], p).astype(np.int64)
        W = oracle.tmpl_halfwidth(k)
        T = oracle.tmpl(k, j)
        lo, hi = max(b - W, 0), min(b + W + 1, 3400)
        exp = np.zeros(3400, np.int64)
        exp[lo:hi] = T[lo - (b - W):hi - (b - W)]
        assert np.array_equal(H, exp), (b, j, k)
    # at the lower end of the range part of the template is dropped
    H = oracle.fill_template([np.float32(-549.9)], [np.float32(0.5)], [0], [HIST], p)
    assert 0.4 * S < H.sum() < 0.7 * S and H[0] > 0
    # tracks that are not histogrammed contribute nothing; permutation invariance
    zp = rng.uniform(-50, 50, 200).astype(np.float32); sp = rng.uniform(0.03, 1.2, 200).astype(np.float32)
    bins = np.floor((zp - np.float32(-550)) * np.float32(4)).astype(np.int32)
    fl = np.where(rng.random(200) < 0.9, HIST, 1).astype(np.int32)
    H1 = oracle.fill_template(zp, sp, bins, fl, p)
    perm = rng.permutation(200)
    assert np.array_equal(H1, oracle.fill_template(zp[perm], sp[perm], bins[perm], fl[perm], p))
    assert H1.astype(np.int64).sum() == int((fl == HIST).sum()) * S


def test_template_fill_against_the_exact_integrals(oracle, cfg0):
    """On events: the template histogram stays within the bound that its two quantisations allow around the exact erf
    integrals of P:L129 -- sigma is replaced by a class centre at most 2^(1/8) away (|d sigma / sigma| <= 9.05 %, which
    moves at most 0.0905 max|u phi(u)| = 0.022 of a track across any edge), z_poca by the centre of its eighth of a bin
    (at most dz / 16, moving at most min(1, 0.399 / 16 / sigma_bins)), plus the +-3 sigma truncation of R-6 -- and the
    seeds it gives are those of the per-track polynomial fill on most events (the two variants are alternatives)."""
    from synth import events
    p0, p1 = oracle.default_params(), oracle.default_params(fill_mode=1)
    data = events.slice_events(cfg0, 0, 200)
    r0 = oracle.find(data, p0, debug=True, n_hist_events=200)
    r1 = oracle.find(data, p1, debug=True, n_hist_events=200)
    d = r0["debug"]
    off = data["offsets"]
    tail = 2 * ndtr(-3.0) / (1 - 2 * ndtr(-3.0)) + 1e-5
    worst = 0.0
    for e in range(0, 200, 4):
        sl = slice(off[e], off[e + 1])
        zp, sp, fl = d["z_poca"][sl], d["sigma_poca"][sl], d["trk_flags"][sl]
        H0 = oracle.fill_exact(zp, sp, fl, p0)
        H1 = r1["debug"]["hist"][e].astype(np.float64) / S
        bound = np.zeros(3400)
        for z, s, f in zip(zp, sp, fl):
            if not (f & 2):
                continue
            u = float(s) / 0.25
            per = 0.0905 * 0.242 + min(1.0, 0.399 / 16 / u) + tail
            lo = max(int(math.floor((float(z) + 550 - 6 * float(s)) / 0.25)) - 1, 0)      # the exact integral has tails
            hi = min(int(math.floor((float(z) + 550 + 6 * float(s)) / 0.25)) + 2, 3400)
            bound[lo:hi] += per
        assert np.all(np.abs(H1 - H0) <= bound + 1e-8), e
        worst = max(worst, np.abs(H1 - H0).max())
    assert 0.01 < worst < 1.0                                   # the approximation is visible, and small
    assert np.array_equal(r0["debug"]["z_poca"], r1["debug"]["z_poca"])          # only the fill differs
    same = sum(int(r0["n_vtx"][e] == r1["n_vtx"][e]) for e in range(200))
    assert same >= 190
    m = (r0["n_vtx"] == r1["n_vtx"])
    k = np.arange(32)[None, :] < r0["n_vtx"][:, None]
    dz = np.abs(r0["vtx_pos"][..., 2] - r1["vtx_pos"][..., 2])[k & m[:, None]]
    assert np.median(dz) < 1e-3 and np.quantile(dz, 0.95) < 0.05   # the fit does not depend on the histogram details
