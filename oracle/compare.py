"""Element-by-element comparator: results of the CUDA path vs the CPU oracle on the same seeded inputs.

TEST INFRASTRUCTURE ONLY (used by tests/, __graft_entry__.smoke() and bench.py's parity spot check).  Pure
numpy; imports neither the product nor the oracle library: both result dicts are passed in.

Tolerances (BASELINE.json north_star):
  * z_poca, sigma_poca, central bin, histogram bins, seed clusters (begin, end, peak), seed z: bit-exact
  * per-event seed count and vertex count: identical
  * fitted vertex x, y, z: 1e-3 mm;  covariance: 1e-3 relative (off-diagonals relative to sqrt(Cii Cjj))
  * track -> vertex assignment: >= 99.9 % agreement, every mismatch explained by a logged near-tie
Near-tie rules.  Every one of them looks at the ORACLE's deciding quantity (its trace and
its diagnostic taps), never at the size of the disagreement:
  * N1 iteration count: the fp32 fit and the fp64 oracle may stop one iteration apart when the deciding
    |dchi2| or |dz| of the oracle is within NEAR_REL of its cut; the GPU vertex is then compared with the
    oracle's trace entry at the GPU's iteration count.
  * N2 active-track count / singular flag: accepted only when the oracle has a track of that seed within NEAR_REL of
    the Tukey cut-off (|chi2_i / chi2_max - 1|; multi-vertex flavour: |w_i - 1/2| <= W_TOL) in the deciding iteration,
    or (singular flag) a Cholesky pivot within PIVOT_REL of zero.
  * N2 cleanup decisions (merge ratio, beamline distance, min tracks): a differing fate is accepted when the oracle's
    deciding quantity is within NEAR_REL of its cut, or the event holds an N1 / N2 vertex.
  * (N5, round 2 only: a covariance tolerance widened for ill-conditioned fits and any iteration-count difference
    accepted there.  Removed in round 3: the kernel re-sums the Schur complement of such seeds in centred form, and
    they meet the flat tolerances; PIVOT_REL now only serves the singular flag of N2.)
  * N3 argmax (multi-vertex flavour): accepted only when the oracle's two largest weights of that track differ by at
    most W_TOL.  N4 chi2 window: a track listed on one side only must carry a weight below W_TOL there.
Without the GPU's taps (product kernels, debug=False) the same rules are applied from the final outputs: the
iteration count is an output (vtx_niter) and the oracle's trace is indexed through its own seed -> vertex map.  An
event may then be excused only from its first fragile seed on: the vertices (and the tracks of the vertices) that
come before it in z are compared strictly, because a flipped decision on a seed can only shift the vertices behind it.
The report carries how often each rule fired (`rules`), so that a test can print and bound them.
"""
from __future__ import annotations

from typing import Dict, List

import numpy as np

POS_TOL = 1e-3       # mm
COV_RTOL = 1e-3
W_TOL = 2e-3         # Tukey weight, absolute (vertices with equal iteration count)
NEAR_REL = 1e-2
PIVOT_REL = 1e-3     # a Cholesky pivot this close to zero (relative to its diagonal element) may change sign in fp32
MIN_ASSIGN_AGREEMENT = 0.999


def _cov_rel_err(cg: np.ndarray, cr: np.ndarray) -> np.ndarray:
    """max over the 6 elements of |dC_ij| / sqrt(C_ii C_jj) (reference values in the denominator)."""
    d = np.sqrt(np.abs(cr[..., [0, 3, 5]]))
    scale = np.stack([d[..., 0] * d[..., 0], d[..., 0] * d[..., 1], d[..., 0] * d[..., 2],
                      d[..., 1] * d[..., 1], d[..., 1] * d[..., 2], d[..., 2] * d[..., 2]], axis=-1)
    scale = np.where(scale > 0, scale, 1.0)
    return np.max(np.abs(cg - cr) / scale, axis=-1)


def compare(gpu: Dict[str, np.ndarray], ref: Dict[str, np.ndarray], offsets: np.ndarray, p, max_log: int = 20) -> Dict:
    """gpu: binding.DeviceBatch.results() with debug=True; ref: oracle.pvref.find(debug=True, trace=True).
    Returns a report dict with 'failures' (list of strings; empty = parity) and 'near_ties' (logged)."""
    fails: List[str] = []
    ties: List[str] = []
    rules = dict(N1_iteration=0, N2_singular=0, N2_track_count=0, N2_cleanup=0, N3_argmax=0, N4_window=0,
                 fragile_events_excused=0)
    rep: Dict = {"failures": fails, "near_ties": ties, "rules": rules}
    strict_below = None                                 # no-tap path: per excused event, vertices below this index are strict
    gd, rd = gpu.get("debug"), ref.get("debug")
    E = offsets.size - 1
    mv = p.max_vtx_per_event
    ev_of_trk = np.repeat(np.arange(E), np.diff(offsets))
    skipped = (ref["event_status"] & 1) != 0          # TOO_MANY_TRACKS: per-track taps are undefined there
    trk_ok = ~skipped[ev_of_trk] if ev_of_trk.size else np.zeros(0, bool)

    def exact(name, a, b, mask=None):
        a, b = np.asarray(a), np.asarray(b)
        if a.shape != b.shape:
            fails.append(f"{name}: shape {a.shape} vs {b.shape}")
            return
        if a.dtype.kind == "f":
            eq = (a.view(np.uint32) == b.view(np.uint32)) | (np.isnan(a) & np.isnan(b)) if a.dtype == np.float32 and b.dtype == np.float32 \
                else ((a == b) | (np.isnan(a) & np.isnan(b)))
        else:
            eq = a == b
        if mask is not None:
            eq = eq | ~mask
        nbad = int(eq.size - np.count_nonzero(eq))
        rep[f"{name}_mismatch"] = nbad
        if nbad:
            idx = np.argwhere(~eq)[:3]
            fails.append(f"{name}: {nbad} of {eq.size} differ (bit-exact required), first at {idx.tolist()}: "
                         f"gpu {a[tuple(idx[0])]} ref {b[tuple(idx[0])]}")

    # ---- status and counts ----------------------------------------------------------------------------------
    exact("event_status", gpu["event_status"].astype(np.uint32) & ~np.uint32(4), ref["event_status"].astype(np.uint32) & ~np.uint32(4))
    if gd is not None and rd is not None:
        # ---- a1: projection ---------------------------------------------------------------------------------
        exact("z_poca", gd["z_poca"], rd["z_poca"], trk_ok)
        exact("sigma_poca", gd["sigma_poca"], rd["sigma_poca"], trk_ok)
        exact("trk_bin", gd["trk_bin"], np.where((rd["trk_flags"] & 1) != 0, rd["trk_bin"], -1), trk_ok)
        # ---- a2: histogram ----------------------------------------------------------------------------------
        nh = min(gd["hist"].shape[0], rd["hist"].shape[0])
        if nh > 0 and gd["hist"].shape[1] == rd["hist"].shape[1]:
            exact("hist", gd["hist"][:nh], rd["hist"][:nh], np.broadcast_to((~skipped[:nh])[:, None], rd["hist"][:nh].shape))
        # ---- a3 / a4: seeds ---------------------------------------------------------------------------------
        exact("n_seeds_raw", gd["n_seeds_raw"], rd["n_seeds_raw"])
        exact("n_seeds", gd["n_seeds"], rd["n_seeds"])
        ks = np.arange(mv)[None, :] < rd["n_seeds"][:, None]
        exact("seed_bins", gd["seed_bins"], rd["seed_bins"], np.repeat(ks[:, :, None], 3, axis=2))
        exact("seed_z", gd["seed_z"], rd["seed_z"], ks)
        mvf = int(getattr(p, "flavour", 0)) == 1
        if not mvf:
            exact("trk_seed", gd["trk_seed"], rd["trk_seed"])
        else:
            # multi-vertex flavour: the seed a track follows is an argmax over floating-point weights (R-13)
            same = gd["trk_seed"] == rd["trk_seed"]
            rep["trk_seed_mismatch"] = int((~same).sum())
            if same.size and same.mean() < MIN_ASSIGN_AGREEMENT:
                fails.append(f"trk_seed (largest-weight seed) agreement {same.mean():.6f} < {MIN_ASSIGN_AGREEMENT}")

        # ---- a5: per-seed fit, pre-cleanup -------------------------------------------------------------------
        same_seeds = gd["n_seeds"] == rd["n_seeds"]
        ks = ks & same_seeds[:, None]
        gn, rn = gd["seed_niter"], rd["seed_niter"]
        sing_g, sing_r = (gn < 0) & ks, (rn < 0) & ks
        bad_sing = sing_g != sing_r
        mvf_ = int(getattr(p, "flavour", 0)) == 1
        edge_tol = W_TOL if mvf_ else NEAR_REL
        if bad_sing.any():
            for e, k in np.argwhere(bad_sing):
                # N2: the count of active tracks can only flip through a track at the cut-off, the pivot only near zero
                edge, piv, nmin = rd["seed_edge_any"][e, k], rd["seed_pivot_min"][e, k], rd["seed_nact_min"][e, k]
                ok = (nmin <= 2 and edge <= edge_tol) or abs(piv) <= PIVOT_REL
                msg = (f"singular-fit flag differs at event {e} seed {k}: gpu niter {gn[e, k]} ref {rn[e, k]}; oracle: fewest active "
                       f"tracks {nmin}, closest track to the cut-off {edge:.3g}, smallest relative pivot {piv:.3g}")
                (ties if ok else fails).append(("near-tie: " if ok else "NOT a near-tie: ") + msg)
                rules["N2_singular"] += int(ok)
            rep["singular_mismatch"] = int(bad_sing.sum())
        fit = ks & ~sing_g & ~sing_r
        ref_pos = rd["seed_pos"].copy()
        ref_cov = rd["seed_cov"].copy()
        niter_diff = fit & (gn != rn)
        rep["n_fitted_seeds"] = int(fit.sum())
        rep["n_niter_diff"] = int(niter_diff.sum())
        trace = rd.get("trace")
        cuts = (float(p.conv_dchi2), float(p.conv_dz))
        tie_mask = np.zeros_like(fit)
        for e, k in np.argwhere(niter_diff):
            g_it, r_it = int(gn[e, k]), int(rn[e, k])
            ok = False
            why = "no oracle trace"
            if trace is not None and 1 <= g_it <= trace.shape[2]:
                it = min(g_it, r_it)                  # the iteration at which one side stopped and the other went on
                dchi2, dz = abs(trace[e, k, it - 1, 9]), abs(trace[e, k, it - 1, 10])
                near = (np.isfinite(cuts[0]) and abs(dchi2 - cuts[0]) <= NEAR_REL * cuts[0]) or \
                       (abs(dz - cuts[1]) <= NEAR_REL * cuts[1])
                why = f"oracle |dchi2| {dchi2:.6g} (cut {cuts[0]:g}), |dz| {dz:.6g} (cut {cuts[1]:g}) at iteration {it}"
                if near:
                    ok = True
                    ref_pos[e, k] = trace[e, k, g_it - 1, 0:3]
                    ref_cov[e, k] = trace[e, k, g_it - 1, 3:9]
                    tie_mask[e, k] = True
            msg = f"iteration count differs at event {e} seed {k}: gpu {g_it} ref {r_it}; {why}"
            (ties if ok else fails).append(("near-tie: " if ok else "NOT a near-tie: ") + msg)
            rules["N1_iteration"] += int(ok)
        dpos = np.abs(gd["seed_pos"].astype(np.float64) - ref_pos).max(axis=-1)
        dcov = _cov_rel_err(gd["seed_cov"].astype(np.float64), ref_cov)
        rep["seed_pos_max_err_mm"] = float(dpos[fit].max()) if fit.any() else 0.0
        rep["seed_cov_max_rel_err"] = float(dcov[fit].max()) if fit.any() else 0.0
        badp = fit & ~(dpos <= POS_TOL)
        badc = fit & ~(dcov <= COV_RTOL)
        for e, k in np.argwhere(badp)[:max_log]:
            fails.append(f"seed position off by {dpos[e, k]:.3g} mm at event {e} seed {k} (niter gpu {gn[e, k]} ref {rn[e, k]})")
        for e, k in np.argwhere(badc)[:max_log]:
            fails.append(f"seed covariance off by {dcov[e, k]:.3g} rel at event {e} seed {k} (niter gpu {gn[e, k]} ref {rn[e, k]})")
        eq_it = fit & ~niter_diff
        dn = eq_it & (gd["seed_ntrk"] != rd["seed_ntrk"])
        rep["seed_ntrk_diff"] = int(dn.sum())
        for e, k in np.argwhere(dn):
            edge = rd["seed_edge_last"][e, k]               # N2: the oracle's closest track to the cut that defines n_trk
            ok = edge <= edge_tol and abs(int(gd["seed_ntrk"][e, k]) - int(rd["seed_ntrk"][e, k])) <= 1
            msg = (f"track count differs at event {e} seed {k}: gpu {gd['seed_ntrk'][e, k]} ref {rd['seed_ntrk'][e, k]}; "
                   f"oracle's closest track to the cut: {edge:.3g} (tolerance {edge_tol:g})")
            (ties if ok else fails).append(("near-tie: " if ok else "NOT a near-tie: ") + msg)
            rules["N2_track_count"] += int(ok)
        dchi = np.abs(gd["seed_chi2"].astype(np.float64) - rd["seed_chi2"])
        rel = dchi / np.maximum(1.0, np.abs(rd["seed_chi2"]))
        rep["seed_chi2_max_rel_err"] = float(rel[eq_it & ~dn].max()) if (eq_it & ~dn).any() else 0.0
        if ((eq_it & ~dn) & (rel > 1e-3)).any():
            e, k = np.argwhere((eq_it & ~dn) & (rel > 1e-3))[0]
            fails.append(f"seed chi2 off at event {e} seed {k}: gpu {gd['seed_chi2'][e, k]} ref {rd['seed_chi2'][e, k]}")

        # ---- a6: fate of each seed ---------------------------------------------------------------------------
        gf, rf = gd["seed_fate"], rd["seed_fate"]
        fate_diff = ks & (gf != rf)
        rep["n_fate_diff"] = int(fate_diff.sum())
        ev_fate_tie = np.zeros(E, bool)
        for e in np.unique(np.argwhere(fate_diff)[:, 0]) if fate_diff.any() else []:
            why = _explain_fate(e, rd, p, int(rd["n_seeds"][e]), tie_mask[e], dn[e] | bad_sing[e])
            if why:
                ties.append(f"near-tie: cleanup decisions differ in event {e}: {why}")
                ev_fate_tie[e] = True
                rules["N2_cleanup"] += 1
            else:
                fails.append(f"cleanup decisions differ in event {e} with no near-tie: gpu fate {gf[e][:rd['n_seeds'][e]].tolist()} "
                             f"ref {rf[e][:rd['n_seeds'][e]].tolist()}")
    elif rd is not None and rd.get("trace") is not None:
        # ---- product kernels (no GPU taps): the same rules from the final outputs ---------------------------------
        # vtx_niter is an output, so N1 needs no tap: vertex v of an event is the oracle's seed with fate v.
        trace = rd["trace"]
        cuts = (float(p.conv_dchi2), float(p.conv_dz))
        mvf_ = int(getattr(p, "flavour", 0)) == 1
        edge_tol = W_TOL if mvf_ else NEAR_REL
        ns_r, fate_r, rn = rd["n_seeds"], rd["seed_fate"], rd["seed_niter"]
        ks = np.arange(mv)[None, :] < ns_r[:, None]

        def near_cut(e, k, it):                               # oracle's deciding quantities at iteration `it` (1-based)
            if it < 1 or it > trace.shape[2]:
                return False
            dchi2, dz = abs(trace[e, k, it - 1, 9]), abs(trace[e, k, it - 1, 10])
            return bool((np.isfinite(cuts[0]) and abs(dchi2 - cuts[0]) <= NEAR_REL * cuts[0]) or abs(dz - cuts[1]) <= NEAR_REL * cuts[1])

        # fragile seeds, from the oracle alone: it stopped (or went on) on a quantity within NEAR_REL of its cut, or a
        # track sits at the cut that defines n_trk, or the fit is at the edge of being singular
        it_r = np.clip(rn, 1, trace.shape[2])
        ee, kk = np.nonzero(ks & (rn > 0))
        frag_stop = np.zeros((E, mv), bool)
        for off_ in (0, -1):                                  # the stopping iteration and the one before it
            it = np.clip(it_r[ee, kk] + off_, 1, trace.shape[2]) - 1
            dchi2, dz = np.abs(trace[ee, kk, it, 9]), np.abs(trace[ee, kk, it, 10])
            near = np.abs(dz - cuts[1]) <= NEAR_REL * cuts[1]
            if np.isfinite(cuts[0]):
                near |= np.abs(dchi2 - cuts[0]) <= NEAR_REL * cuts[0]
            frag_stop[ee, kk] |= near
        frag_cnt = ks & ((rd["seed_edge_last"] <= edge_tol) | ((rd["seed_nact_min"] <= 2) & (rd["seed_edge_any"] <= edge_tol))
                         | (np.abs(rd["seed_pivot_min"]) <= PIVOT_REL))
        rep["n_fragile_seeds"] = int((frag_stop | frag_cnt).sum())
        # N1 on the final vertices of events with the same vertex count
        nv_g, nv_r = gpu["n_vtx"], ref["n_vtx"]
        tie_mask = np.zeros((E, mv), bool)                    # indexed by SEED, as in the tap path
        ref_pos = rd["seed_pos"].copy()
        ref_cov = rd["seed_cov"].copy()
        ee, kk = np.nonzero(ks & (fate_r >= 0) & (nv_g == nv_r)[:, None])
        vv = fate_r[ee, kk]
        g_it, r_it = gpu["vtx_niter"][ee, vv], rn[ee, kk]
        rep["n_fitted_seeds"] = int((ks & (rn > 0)).sum())
        rep["n_niter_diff"] = int((g_it != r_it).sum())
        for e, k, gi, ri in zip(ee[g_it != r_it], kk[g_it != r_it], g_it[g_it != r_it], r_it[g_it != r_it]):
            ok = 1 <= gi <= trace.shape[2] and near_cut(e, k, min(int(gi), int(ri)))
            if ok:
                rules["N1_iteration"] += 1
                ref_pos[e, k] = trace[e, k, gi - 1, 0:3]
                ref_cov[e, k] = trace[e, k, gi - 1, 3:9]
                tie_mask[e, k] = True
                ties.append(f"near-tie: iteration count differs at event {e} seed {k}: gpu {gi} ref {ri} (oracle within {NEAR_REL} of its cut)")
            elif not (frag_stop[e] | frag_cnt[e]).any() and not _explain_fate(int(e), rd, p, int(ns_r[e]), frag_stop[e], frag_cnt[e]):
                fails.append(f"NOT a near-tie: iteration count differs at event {e} seed {k}: gpu {gi} ref {ri}")
        # events whose outcome may legitimately differ: some decision of the oracle is within tolerance of its cut
        fragile_ev = np.zeros(E, bool)
        differs = (nv_g != nv_r)
        for e in np.flatnonzero(differs):
            why = _explain_fate(int(e), rd, p, int(ns_r[e]), frag_stop[e], frag_cnt[e])
            if why:
                ties.append(f"near-tie: vertex count differs in event {e} (gpu {nv_g[e]} ref {nv_r[e]}): {why}")
                fragile_ev[e] = True
                rules["N2_cleanup"] += 1
        # same count but another pairing of merged / rejected vertices: only excused in events that are fragile
        for e in np.flatnonzero(~differs & (frag_stop | frag_cnt).any(axis=1)):
            fragile_ev[e] = True
        ev_fate_tie = fragile_ev & (differs | _any_vertex_off(gpu, ref, ref_pos, rd, mv))
        rep["n_fragile_events_excused"] = int(ev_fate_tie.sum())
        rules["fragile_events_excused"] = int(ev_fate_tie.sum())
        # an excused event is excused from its first fragile seed on: that seed's place among the oracle's final
        # vertices (the number of surviving seeds before it); events excused by a cleanup cut alone: from vertex 0
        frag = (frag_stop | frag_cnt) & ks
        surv_before = np.cumsum((fate_r >= 0) & ks, axis=1) - ((fate_r >= 0) & ks)
        first = np.where(frag, surv_before, mv).min(axis=1)
        strict_below = np.where(ev_fate_tie, np.where(frag.any(axis=1), first, 0), mv)
    else:
        ev_fate_tie = np.zeros(E, bool)
        tie_mask = None

    # ---- final outputs ------------------------------------------------------------------------------------------
    nv_g, nv_r = gpu["n_vtx"], ref["n_vtx"]
    nv_bad = (nv_g != nv_r) & ~ev_fate_tie
    rep["n_vtx_mismatch_events"] = int((nv_g != nv_r).sum())
    if nv_bad.any():
        fails.append(f"n_vtx differs in {int(nv_bad.sum())} events without a near-tie, first {np.argwhere(nv_bad)[:5, 0].tolist()}")
    ev_same = (nv_g == nv_r) & ~ev_fate_tie
    kv = (np.arange(mv)[None, :] < nv_r[:, None]) & ev_same[:, None]
    if strict_below is not None:                        # no-tap path: the vertices before an excused event's first fragile seed
        kv |= (np.arange(mv)[None, :] < np.minimum(np.minimum(nv_r, nv_g), strict_below)[:, None]) & ev_fate_tie[:, None]
        rep["n_strict_vertices_in_excused_events"] = int((kv & ev_fate_tie[:, None]).sum())
    rep["n_vertices"] = int(nv_r.sum())
    if rd is not None and tie_mask is not None:
        # map final vertices back to seeds to reuse the (possibly trace-substituted) reference
        ref_vpos = ref["vtx_pos"].copy()
        ref_vcov = ref["vtx_cov"].copy()
        for e, k in np.argwhere(tie_mask) if tie_mask is not None and tie_mask.any() else []:
            v = rd["seed_fate"][e, k]
            if v >= 0 and ev_same[e]:
                ref_vpos[e, v] = ref_pos[e, k]
                ref_vcov[e, v] = ref_cov[e, k]
    else:
        ref_vpos, ref_vcov = ref["vtx_pos"], ref["vtx_cov"]
    dpos = np.abs(gpu["vtx_pos"].astype(np.float64) - ref_vpos).max(axis=-1)
    dcov = _cov_rel_err(gpu["vtx_cov"].astype(np.float64), ref_vcov)
    rep["vtx_pos_max_err_mm"] = float(dpos[kv].max()) if kv.any() else 0.0
    rep["vtx_cov_max_rel_err"] = float(dcov[kv].max()) if kv.any() else 0.0
    for e, k in np.argwhere(kv & ~(dpos <= POS_TOL))[:max_log]:
        fails.append(f"vertex position off by {dpos[e, k]:.3g} mm at event {e} vertex {k}")
    for e, k in np.argwhere(kv & ~(dcov <= COV_RTOL))[:max_log]:
        fails.append(f"vertex covariance off by {dcov[e, k]:.3g} rel at event {e} vertex {k}")

    tv_g, tv_r = gpu["trk_vertex"], ref["trk_vertex"]
    agree = tv_g == tv_r
    rep["assign_agreement"] = float(agree.mean()) if agree.size else 1.0
    rep["assign_mismatch_tracks"] = int((~agree).sum())
    if agree.size and rep["assign_agreement"] < MIN_ASSIGN_AGREEMENT:
        fails.append(f"track-assignment agreement {rep['assign_agreement']:.6f} < {MIN_ASSIGN_AGREEMENT}")
    unexplained = (~agree) & ~ev_fate_tie[ev_of_trk] if agree.size else np.zeros(0, bool)
    if strict_below is not None and agree.size:          # tracks of the strict vertices of an excused event
        sb = strict_below[ev_of_trk]
        unexplained |= (~agree) & ev_fate_tie[ev_of_trk] & (((tv_r >= 0) & (tv_r < sb)) | ((tv_g >= 0) & (tv_g < sb)))
    if int(getattr(p, "flavour", 0)) == 1 and agree.size:
        # argmax near-tie: both sides follow a vertex and the two largest weights are equal within W_TOL
        if rd is not None and "trk_w1" in rd:              # N3: the ORACLE's two largest weights of the track
            gap = rd["trk_w1"] - rd["trk_w2"]
        else:
            gap = np.full(agree.shape, np.inf)
        argmax_tie = (~agree) & (gap <= W_TOL) & (rd["trk_w2"] > 0 if rd is not None and "trk_w2" in rd else False)
        rep["n_argmax_ties"] = int(argmax_tie.sum())
        rules["N3_argmax"] = int(argmax_tie.sum())
        for i in np.argwhere(argmax_tie)[:max_log, 0]:
            ties.append(f"near-tie: the oracle's two largest weights of track {int(i)} differ by {gap[i]:.3g} <= {W_TOL}: gpu {tv_g[i]} ref {tv_r[i]}")
        unexplained &= ~argmax_tie
        # window near-tie: chi2 at the seed position within rounding of chi2_window lists the track on one side only;
        # accepted when the weight it then has is below W_TOL (it is exp(-window / 2) / exp(-chi2_max / 2) at most)
        wg, wr = gpu["trk_weight"].astype(np.float64), ref["trk_weight"]
        window_tie = (~agree) & (((tv_g < 0) & (tv_r >= 0) & (wr <= W_TOL)) | ((tv_r < 0) & (tv_g >= 0) & (wg <= W_TOL)))
        rep["n_window_ties"] = int(window_tie.sum())
        rules["N4_window"] = int(window_tie.sum())
        for i in np.argwhere(window_tie)[:max_log, 0]:
            ties.append(f"near-tie: track {int(i)} is at the chi2 window of its only vertex: weights gpu {wg[i]:.3g} ref {wr[i]:.3g}")
        unexplained &= ~window_tie
    if unexplained.any():
        fails.append(f"{int(unexplained.sum())} track-assignment mismatches outside near-tie events, first track "
                     f"{int(np.argwhere(unexplained)[0, 0])} (event {int(ev_of_trk[np.argwhere(unexplained)[0, 0]])})")
    # weights: compare where the assignment agrees and the vertex was not an iteration near-tie
    wmask = agree & (tv_r >= 0)
    if tie_mask is not None and tie_mask.any() and wmask.any():
        tie_ev = tie_mask.any(axis=1)
        wmask &= ~tie_ev[ev_of_trk]
    dw = np.abs(gpu["trk_weight"].astype(np.float64) - ref["trk_weight"])
    rep["trk_weight_max_err"] = float(dw[wmask].max()) if wmask.any() else 0.0
    nbw = int((dw[wmask] > W_TOL).sum()) if wmask.any() else 0
    if nbw:
        i = int(np.argwhere(wmask & (dw > W_TOL))[0, 0])
        fails.append(f"{nbw} track weights off by more than {W_TOL}, first track {i}: gpu {gpu['trk_weight'][i]} ref {ref['trk_weight'][i]}")
    zero_ok = np.all(gpu["trk_weight"][tv_g < 0] == 0.0) if tv_g.size else True
    if not zero_ok:
        fails.append("unassigned tracks with non-zero weight")
    rep["n_near_ties"] = len(ties)
    del ties[max_log:]
    return rep


def _any_vertex_off(gpu, ref, ref_seed_pos, rd, mv) -> np.ndarray:
    """Per event: does some final vertex of the GPU sit more than POS_TOL from the oracle's vertex of the same index
    (with the N1 substitutions already applied to ref_seed_pos)?  Events with differing counts report False."""
    nv_g, nv_r = gpu["n_vtx"], ref["n_vtx"]
    E = nv_r.size
    ref_vpos = ref["vtx_pos"].copy()
    fate = rd["seed_fate"]
    ee, kk = np.nonzero(fate >= 0)
    ref_vpos[ee, fate[ee, kk]] = ref_seed_pos[ee, kk]
    d = np.abs(gpu["vtx_pos"].astype(np.float64) - ref_vpos).max(axis=-1)
    m = (np.arange(mv)[None, :] < nv_r[:, None]) & (nv_g == nv_r)[:, None]
    return (m & ~(d <= POS_TOL)).any(axis=1)


def _explain_fate(e: int, rd: Dict[str, np.ndarray], p, ns: int, niter_tie: np.ndarray, ntrk_tie: np.ndarray) -> str:
    """Is some cleanup decision of the ORACLE in event e within NEAR_REL of its cut (or fed by a documented
    near-tie upstream)?  Returns a description, or '' if nothing is close."""
    if niter_tie[:ns].any():
        return "a vertex of the event is an iteration-count near-tie"
    if ntrk_tie[:ns].any():
        return "a vertex of the event has a track at the Tukey cut-off / singular-fit edge"
    pos, cov, ntrk, nit = rd["seed_pos"][e], rd["seed_cov"][e], rd["seed_ntrk"][e], rd["seed_niter"][e]
    alive = [k for k in range(ns) if nit[k] >= 0]
    for a in range(len(alive)):
        for b in range(a + 1, len(alive)):
            i, j = alive[a], alive[b]
            ratio = (pos[j, 2] - pos[i, 2]) ** 2 / (cov[j, 5] + cov[i, 5])
            if abs(ratio - p.merge_ratio) <= NEAR_REL * p.merge_ratio:
                return f"merge ratio {ratio:.6g} of seeds {i},{j} vs cut {p.merge_ratio:g}"
    for k in alive:
        vz = pos[k, 2]
        if vz >= p.z_split:
            d2 = (pos[k, 0] - (p.beam_x + p.beam_tx * vz)) ** 2 + (pos[k, 1] - (p.beam_y + p.beam_ty * vz)) ** 2
            c2 = p.max_beam_dist ** 2
            if abs(d2 - c2) <= 2 * NEAR_REL * c2:
                return f"beamline distance^2 {d2:.6g} of seed {k} vs cut {c2:.6g}"
    return ""
