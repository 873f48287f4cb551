"""Pins of the oracle's projection (O1/O2) against geometry, not against itself.
PAPER.md Eq. 1 (L87), Eq. 3 (L116), acceptance (L129, Table 2)."""
import numpy as np


def _line_dist2(zs, trk, beam):
    """Squared transverse distance between track line and beamline at z (double)."""
    x, y, z, tx, ty = trk
    bx, by, btx, bty = beam
    dx = (x + (zs - z) * tx) - (bx + btx * zs)
    dy = (y + (zs - z) * ty) - (by + bty * zs)
    return dx * dx + dy * dy


def test_noiseless_tracks_through_beamline_point(oracle):
    """A straight line through a point P on the beamline has its POCA at P_z (Eq. 1 is exact there)."""
    rng = np.random.default_rng(7)
    for beam in [(0, 0, 0, 0), (1.092, 0.472, 0, 0), (0.3, -0.2, 2e-4, -1.5e-4)]:
        p = oracle.default_params(beam_x=beam[0], beam_y=beam[1], beam_tx=beam[2], beam_ty=beam[3])
        n = 500
        pz = rng.uniform(-500, 250, n)
        px, py = beam[0] + beam[2] * pz, beam[1] + beam[3] * pz
        tx, ty = rng.normal(0, 0.2, n), rng.normal(0, 0.2, n)
        z = pz + rng.uniform(-30, 30, n)             # state quoted away from the vertex
        x, y = px + (z - pz) * tx, py + (z - pz) * ty
        zp, sp, b, fl = oracle.project(x, y, z, tx, ty, np.full(n, 1e-3), p)
        slope = np.hypot(tx - beam[2], ty - beam[3])
        # fp32 inputs carry ~|x| * 6e-8 of rounding, amplified by 1/slope
        tol = 2e-5 / np.maximum(slope, 1e-3) + 1e-4
        assert np.all(np.abs(zp - pz) < tol)
        assert np.all(b[fl & 1 == 1] == np.floor((zp[fl & 1 == 1] - (-550.0)) / 0.25).astype(int))


def test_poca_is_the_distance_minimiser_brute_force(oracle):
    """Brute force: scan z on a fine grid for the minimum track-beamline distance."""
    rng = np.random.default_rng(8)
    beam = (0.05, -0.03, 3e-4, 2e-4)
    p = oracle.default_params(beam_x=beam[0], beam_y=beam[1], beam_tx=beam[2], beam_ty=beam[3])
    n = 60
    x, y = rng.normal(0, 0.2, n), rng.normal(0, 0.2, n)
    z = rng.uniform(-100, 100, n)
    tx, ty = rng.normal(0, 0.2, n), rng.normal(0, 0.2, n)
    zp, sp, b, fl = oracle.project(x, y, z, tx, ty, np.full(n, 1e-3), p)
    x32, y32, z32, tx32, ty32 = (a.astype(np.float32).astype(np.float64) for a in (x, y, z, tx, ty))
    for i in range(n):
        grid = zp[i] + np.linspace(-0.05, 0.05, 20001)          # 5 nm steps
        d2 = _line_dist2(grid, (x32[i], y32[i], z32[i], tx32[i], ty32[i]), beam)
        zmin = grid[np.argmin(d2)]
        assert abs(zmin - zp[i]) < 2e-4 + 2e-5 / np.hypot(tx32[i], ty32[i])
        # and the scanned minimum is interior (so the window contained it)
        assert 0 < np.argmin(d2) < grid.size - 1


def test_sigma_poca_matches_monte_carlo_of_eq1(oracle):
    """Eq. 3 is linear error propagation of Eq. 1 under equal, uncorrelated x/y errors: check by MC."""
    rng = np.random.default_rng(9)
    p = oracle.default_params()
    for (tx, ty, sig) in [(0.1, 0.0, 0.05), (0.05, -0.12, 0.02), (0.3, 0.3, 0.1)]:
        n = 200_000
        x = rng.normal(0, sig, n); y = rng.normal(0, sig, n)
        zp, sp, _, _ = oracle.project(x, y, np.zeros(n), np.full(n, tx), np.full(n, ty), np.full(n, sig ** 2), p)
        assert abs(np.std(zp) / sp[0] - 1.0) < 0.01
        assert abs(sp[0] - sig / np.hypot(tx, ty)) < 1e-5 * sp[0] + 1e-7


def test_sigma_inverse_to_slope(oracle):
    """'The uncertainty is approximately inversely proportional to the track slope' (L119)."""
    p = oracle.default_params()
    t = np.array([0.01, 0.02, 0.04, 0.08, 0.16])
    _, sp, _, _ = oracle.project(np.zeros(5), np.zeros(5), np.zeros(5), t, np.zeros(5), np.full(5, 1e-4), p)
    assert np.allclose(sp * t, sp[0] * t[0], rtol=1e-5)


def test_validity_range_and_sigma_cuts(oracle):
    p = oracle.default_params()
    A, Hh = oracle.TRK_ASSIGNABLE, oracle.TRK_HISTOGRAMMED
    # parallel to the beamline: invalid (R-3)
    _, _, b, fl = oracle.project([0.1], [0.1], [0.0], [0.0], [0.0], [1e-4], p)
    assert fl[0] == 0 and b[0] == -1
    # POCA outside [-550, 300): x = -0.1*tx -> z_poca = z + ... ; place it at +400 and -600
    for zt, ok in [(400.0, False), (-600.0, False), (299.9, True), (-549.9, True)]:
        _, _, b, fl = oracle.project([0.0], [0.0], [zt], [0.1], [0.0], [1e-4], p)
        assert bool(fl[0] & A) == ok
    # sigma cut 1.5 mm in pp, 10 mm in the gas region (Table 2): sigma = 0.2/0.1 = 2 mm
    _, sp, _, fl = oracle.project([0.0, 0.0], [0.0, 0.0], [0.0, -400.0], [0.1, 0.1], [0.0, 0.0], [0.04, 0.04], p)
    assert abs(sp[0] - 2.0) < 1e-5
    assert fl[0] == A                      # pp: assignable but not histogrammed
    assert fl[1] == A | Hh                 # gas cell: histogrammed
    # last bin index
    zp, _, b, fl = oracle.project([0.0], [0.0], [299.99], [0.1], [0.0], [1e-4], p)
    assert b[0] == 3399 and oracle.nbins(p) == 3400
