"""Seeded synthetic event generator shared by the oracle tests and the CUDA path.

This module holds NONE of the method's arithmetic (no projection, no histogram, no fit):
it only draws track states shaped like the paper's Run 3 pp + SMOG2 workloads
("mu = 5", L51 track state (x, y, z, tx, ty) + covariance, L333-335 SMOG2 cell)
following the recipe in /root/repo/BASELINE.json `configs` and DESIGN.md "Input recipe".

Output layout (what both `pv_find` and the oracle read): nine fp32 SoA arrays of length T
(x, y, z, tx, ty, var_x, var_y, var_tx, var_ty) and int32 `offsets[E+1]`.

Determinism: events are generated in blocks of BLOCK events; block j of a config with seed s uses
numpy.random.default_rng([s, j]).  The result does not depend on how many blocks are requested at once.
"""
from __future__ import annotations

import dataclasses
from typing import Dict, Optional

import numpy as np

BLOCK = 10_000

FIELDS = ("x", "y", "z", "tx", "ty", "var_x", "var_y", "var_tx", "var_ty")


@dataclasses.dataclass
class EventModel:
    """Parameters of one BASELINE.json config."""
    name: str
    seed: int
    n_events: int
    mu_pp: float = 5.0                 # Poisson mean of pp vertices
    min_one_pp: bool = True            # N_pv = max(1, Poisson(mu))
    fixed_n_pp: Optional[int] = None   # exactly this many pp PVs (configs[3])
    trk_pp_mean: float = 20.0          # tracks per PV = 1 + Poisson(.)
    fixed_trk_pp: Optional[int] = None
    slope_pp: float = 0.25
    ghost_frac: float = 0.05
    smog_prob: float = 0.0             # Bernoulli probability of one p-gas vertex
    trk_smog_mean: float = 15.0
    slope_smog: float = 0.15
    pair_separations: Optional[tuple] = None  # configs[3]: dz sweep, by event index mod len
    aniso: bool = False                # per-track var_y = k var_x, k in [1/4, 4]; var_tx, var_ty in [0.5, 2] x 1e-6, independent


def config(idx: int, n_events: Optional[int] = None) -> EventModel:
    """The five BASELINE.json configs (idx 0..4). configs[4] takes n_events from the caller."""
    if idx == 0:
        m = EventModel("tiny_pp", seed=1, n_events=1_000)
    elif idx == 1:
        m = EventModel("throughput_pp_smog2", seed=2, n_events=100_000, smog_prob=0.3)
    elif idx == 2:
        m = EventModel("high_pileup", seed=3, n_events=50_000, mu_pp=10.0, min_one_pp=False,
                       trk_pp_mean=25.0, ghost_frac=0.10)
    elif idx == 3:
        m = EventModel("close_pairs", seed=4, n_events=20_000, fixed_n_pp=2, fixed_trk_pp=30,
                       pair_separations=(0.1, 0.2, 0.5, 1.0, 2.0, 5.0))
    elif idx == 4:
        m = EventModel("batch_sweep", seed=5, n_events=100_000, smog_prob=0.3)
    else:
        raise ValueError("config index must be 0..4")
    if n_events is not None:
        m = dataclasses.replace(m, n_events=int(n_events))
    return m


def _gen_block(m: EventModel, block: int, n_ev: int, ev0: int):
    rng = np.random.default_rng([m.seed, block])
    # ---- vertices -------------------------------------------------------------------------
    if m.fixed_n_pp is not None:
        n_pp = np.full(n_ev, m.fixed_n_pp, dtype=np.int64)
    else:
        n_pp = rng.poisson(m.mu_pp, n_ev)
        if m.min_one_pp:
            n_pp = np.maximum(n_pp, 1)
    n_gas = (rng.random(n_ev) < m.smog_prob).astype(np.int64) if m.smog_prob > 0 else np.zeros(n_ev, np.int64)

    pv_ev_pp = np.repeat(np.arange(n_ev), n_pp)
    npp_tot = pv_ev_pp.size
    pv_z_pp = rng.normal(0.0, 45.0, npp_tot)
    if m.pair_separations is not None:
        # exactly two PVs per event, centre ~ N(0,45), separation by event index
        centre = rng.normal(0.0, 45.0, n_ev)
        sep = np.asarray(m.pair_separations)[(ev0 + np.arange(n_ev)) % len(m.pair_separations)]
        pv_z_pp = np.empty(npp_tot)
        pv_z_pp[0::2] = centre - 0.5 * sep
        pv_z_pp[1::2] = centre + 0.5 * sep
    pv_ev_gas = np.nonzero(n_gas)[0]
    ngas_tot = pv_ev_gas.size
    pv_z_gas = rng.uniform(-541.0, -341.0, ngas_tot)

    pv_ev = np.concatenate([pv_ev_pp, pv_ev_gas])
    pv_z = np.concatenate([pv_z_pp, pv_z_gas])
    pv_is_gas = np.concatenate([np.zeros(npp_tot, bool), np.ones(ngas_tot, bool)])
    npv = pv_ev.size
    pv_x = rng.normal(0.0, 0.04, npv)
    pv_y = rng.normal(0.0, 0.04, npv)
    if m.fixed_trk_pp is not None:
        ntrk_pp = np.full(npp_tot, m.fixed_trk_pp, dtype=np.int64)
    else:
        ntrk_pp = 1 + rng.poisson(m.trk_pp_mean, npp_tot)
    ntrk_gas = 1 + rng.poisson(m.trk_smog_mean, ngas_tot)
    pv_ntrk = np.concatenate([ntrk_pp, ntrk_gas])

    # ---- real tracks ----------------------------------------------------------------------
    t_pv = np.repeat(np.arange(npv), pv_ntrk)
    nreal = t_pv.size
    t_ev = pv_ev[t_pv]
    slope_sigma = np.where(pv_is_gas[t_pv], m.slope_smog, m.slope_pp)
    tx_true = np.clip(rng.normal(0.0, 1.0, nreal) * slope_sigma, -0.4, 0.4)
    ty_true = np.clip(rng.normal(0.0, 1.0, nreal) * slope_sigma, -0.4, 0.4)
    sig = rng.uniform(0.01, 0.1, nreal)
    sig_y = sig * np.sqrt(np.exp(rng.uniform(np.log(0.25), np.log(4.0), nreal))) if m.aniso else sig
    x = pv_x[t_pv] + sig * rng.normal(0.0, 1.0, nreal)
    y = pv_y[t_pv] + sig_y * rng.normal(0.0, 1.0, nreal)
    z = pv_z[t_pv]
    tx = tx_true + rng.normal(0.0, 1e-3, nreal)
    ty = ty_true + rng.normal(0.0, 1e-3, nreal)

    # ---- ghosts: Poisson(f * n_real) per event ----------------------------------------------
    n_real_ev = np.bincount(t_ev, minlength=n_ev)
    n_ghost_ev = rng.poisson(m.ghost_frac * n_real_ev)
    g_ev = np.repeat(np.arange(n_ev), n_ghost_ev)
    ng = g_ev.size
    g_tx = np.clip(rng.normal(0.0, m.slope_pp, ng), -0.4, 0.4) + rng.normal(0.0, 1e-3, ng)
    g_ty = np.clip(rng.normal(0.0, m.slope_pp, ng), -0.4, 0.4) + rng.normal(0.0, 1e-3, ng)
    g_sig = rng.uniform(0.01, 0.1, ng)
    g_sig_y = g_sig * np.sqrt(np.exp(rng.uniform(np.log(0.25), np.log(4.0), ng))) if m.aniso else g_sig
    g_x = rng.uniform(-0.5, 0.5, ng)
    g_y = rng.uniform(-0.5, 0.5, ng)
    g_z = rng.uniform(-300.0, 300.0, ng)

    ev = np.concatenate([t_ev, g_ev])
    truth_pv = np.concatenate([t_pv, np.full(ng, -1, dtype=np.int64)])
    cols = {
        "x": np.concatenate([x, g_x]), "y": np.concatenate([y, g_y]), "z": np.concatenate([z, g_z]),
        "tx": np.concatenate([tx, g_tx]), "ty": np.concatenate([ty, g_ty]),
    }
    s_all = np.concatenate([sig, g_sig])
    s_all_y = np.concatenate([sig_y, g_sig_y])
    if m.aniso:
        v_tx = 1e-6 * np.exp(rng.uniform(np.log(0.5), np.log(2.0), ev.size))
        v_ty = 1e-6 * np.exp(rng.uniform(np.log(0.5), np.log(2.0), ev.size))
    else:
        v_tx = v_ty = np.full(ev.size, 1e-6)
    # ---- shuffle inside each event ----------------------------------------------------------
    key = rng.random(ev.size)
    order = np.lexsort((key, ev))
    out = {k: v[order].astype(np.float32) for k, v in cols.items()}
    out["var_x"] = (s_all[order] ** 2).astype(np.float32)
    out["var_y"] = (s_all_y[order] ** 2).astype(np.float32)
    out["var_tx"] = v_tx[order].astype(np.float32)
    out["var_ty"] = v_ty[order].astype(np.float32)
    counts = np.bincount(ev, minlength=n_ev).astype(np.int64)
    truth = {
        "pv_event": pv_ev + ev0, "pv_x": pv_x, "pv_y": pv_y, "pv_z": pv_z,
        "pv_ntracks": pv_ntrk, "pv_is_gas": pv_is_gas,
        # per-track truth PV index local to this block (-1 = ghost); made global by the caller
        "trk_pv": truth_pv[order],
    }
    return out, counts, truth


def generate(m: EventModel, with_truth: bool = False) -> Dict[str, np.ndarray]:
    """Generate all events of a model. Returns dict with the nine fp32 arrays, int32 `offsets`,
    `n_events`, and (optionally) `truth`."""
    parts = {k: [] for k in FIELDS}
    counts = []
    truths = []
    pv_base = 0
    ev0 = 0
    block = 0
    while ev0 < m.n_events:
        n_ev = min(BLOCK, m.n_events - ev0)
        if n_ev < BLOCK:
            # a partial block is the prefix of the full block (generate full, cut) so that
            # n_events only truncates the sequence
            full, cnt, tr = _gen_block(m, block, BLOCK, ev0)
            ntr = int(cnt[:n_ev].sum())
            full = {k: v[:ntr] for k, v in full.items()}
            cnt = cnt[:n_ev]
            keep_pv = tr["pv_event"] < ev0 + n_ev
            tr = {k: (v[keep_pv] if k != "trk_pv" else v[:ntr]) for k, v in tr.items()}
        else:
            full, cnt, tr = _gen_block(m, block, n_ev, ev0)
        for k in FIELDS:
            parts[k].append(full[k])
        counts.append(cnt)
        if with_truth:
            tp = tr["trk_pv"].copy()
            tp[tp >= 0] += pv_base
            tr["trk_pv"] = tp
            pv_base += tr["pv_z"].size
            truths.append(tr)
        ev0 += n_ev
        block += 1
    out = {k: np.ascontiguousarray(np.concatenate(parts[k])) if parts[k] else np.zeros(0, np.float32)
           for k in FIELDS}
    cnt = np.concatenate(counts) if counts else np.zeros(0, np.int64)
    off = np.zeros(m.n_events + 1, dtype=np.int64)
    np.cumsum(cnt, out=off[1:])
    if off[-1] >= 2 ** 31:
        raise ValueError("track count exceeds int32 offsets")
    out["offsets"] = off.astype(np.int32)
    out["n_events"] = m.n_events
    if with_truth:
        out["truth"] = {k: np.concatenate([t[k] for t in truths]) for k in truths[0]} if truths else {}
    return out


def generate_range(m: EventModel, e0: int, e1: int, cache: Optional[dict] = None) -> Dict[str, np.ndarray]:
    """The events [e0, e1) of model m as a stand-alone batch (offsets rebased to 0), drawing only the generator
    blocks that overlap the range: identical to slice_events(generate(m), e0, e1) for e1 <= m.n_events.
    `cache` (block index -> block) lets a caller reuse blocks between calls (bench.py --gpus N: every rank draws its
    own share of one large batch)."""
    if not 0 <= e0 <= e1:
        raise ValueError("need 0 <= e0 <= e1")
    parts = {k: [] for k in FIELDS}
    counts = []
    for block in range(e0 // BLOCK, (e1 + BLOCK - 1) // BLOCK if e1 > e0 else e0 // BLOCK):
        if cache is not None and block in cache:
            full, cnt = cache[block]
        else:
            full, cnt, _tr = _gen_block(m, block, BLOCK, block * BLOCK)
            if cache is not None:
                cache[block] = (full, cnt)
        a, b = max(e0, block * BLOCK) - block * BLOCK, min(e1, (block + 1) * BLOCK) - block * BLOCK
        first = np.concatenate([[0], np.cumsum(cnt)])
        for k in FIELDS:
            parts[k].append(full[k][first[a]:first[b]])
        counts.append(cnt[a:b])
    out = {k: np.ascontiguousarray(np.concatenate(parts[k])) if parts[k] else np.zeros(0, np.float32) for k in FIELDS}
    cnt = np.concatenate(counts) if counts else np.zeros(0, np.int64)
    off = np.zeros(e1 - e0 + 1, dtype=np.int64)
    np.cumsum(cnt, out=off[1:])
    if off[-1] >= 2 ** 31:
        raise ValueError("track count exceeds int32 offsets")
    out["offsets"] = off.astype(np.int32)
    out["n_events"] = e1 - e0
    return out


def slice_events(data: Dict[str, np.ndarray], e0: int, e1: int) -> Dict[str, np.ndarray]:
    """Contiguous event range [e0, e1) as a stand-alone batch (offsets rebased to 0)."""
    off = data["offsets"]
    t0, t1 = int(off[e0]), int(off[e1])
    out = {k: np.ascontiguousarray(data[k][t0:t1]) for k in FIELDS}
    out["offsets"] = (off[e0:e1 + 1] - off[e0]).astype(np.int32)
    out["n_events"] = e1 - e0
    return out


def from_lists(events) -> Dict[str, np.ndarray]:
    """Build a batch from a list of events, each a dict of equal-length sequences for FIELDS
    (hand-made test events)."""
    out = {k: [] for k in FIELDS}
    off = [0]
    for ev in events:
        n = len(ev["x"])
        for k in FIELDS:
            a = np.asarray(ev[k], dtype=np.float32)
            assert a.shape == (n,)
            out[k].append(a)
        off.append(off[-1] + n)
    res = {k: (np.concatenate(v) if v else np.zeros(0, np.float32)).astype(np.float32) for k, v in out.items()}
    res["offsets"] = np.asarray(off, dtype=np.int32)
    res["n_events"] = len(events)
    return res
