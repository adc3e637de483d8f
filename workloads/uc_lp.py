"""Synthetic DC unit-commitment LP generator (BASELINE.json configs[0..3]).

Stands in for the paper's 6,049-bus ARPA-E cases (Table I l.107-114,
Table VII l.236-246), which are not in this container.  The recipe is BASELINE.json
configs[0] made concrete as in SURVEY.md 8(d); every choice BASELINE.json leaves open is
listed in DESIGN.md ("Input recipe").  Only problem DATA is produced here.

Variables, period-major, per period t:  p(G) u(G) su(G) sd(G) r(G) f(L) theta(B) shed(B)
Rows, period-major, per period t:
    balance (E, B)  sum_{g@i} p - sum_{l:from=i} f + sum_{l:to=i} f + shed_i = d_{i,t}
    flow    (E, L)  f - b (theta_from - theta_to) = 0
    pmin    (G, G)  p - Pmin u >= 0
    pmax    (G, G)  Pmax u - p - r >= 0
    rampup  (G, G)  p_{t-1} - p_t >= -ramp           (t >= 1)
    rampdn  (G, G)  p_t - p_{t-1} >= -ramp           (t >= 1)
    logic   (E, G)  u_t - u_{t-1} - su_t + sd_t = 0  (t = 0: u_0 - su_0 + sd_0 = u_init)
    reserve (G, 1)  sum_g r_{g,t} >= 0.05 sum_i d_{i,t}
    minup   (G, G)  u_t - sum_{s=max(0,t-UT+1)}^{t} su_s >= 0        (configs 2-3)
    mindn   (G, G)  -u_t - sum_{s=max(0,t-DT+1)}^{t} sd_s >= -1      (configs 2-3)
"""
from __future__ import annotations

import numpy as np

from .lp import LP, from_coo

# name -> (B, L, G, T, hours per period, min-up/down rows, seed)
UC_CONFIGS = {
    0: dict(B=14, L=20, G=5, T=24, dt_hours=1.0, min_updown=False, seed=0),
    1: dict(B=500, L=700, G=90, T=48, dt_hours=1.0, min_updown=False, seed=1),
    2: dict(B=2000, L=3200, G=300, T=48, dt_hours=1.0, min_updown=True, seed=2),
    3: dict(B=6049, L=8000, G=800, T=96, dt_hours=0.25, min_updown=True, seed=3),
    # not a BASELINE.json config: the SHAPE of the LP the paper's tuned presolve hands to PDHG, 38,238 x 44,822
    # (Table VII l.241-246; Table VI l.221-226: the GPU loses all 45 races there) -> 38,168 x 44,928 here
    "tuned_presolve": dict(B=138, L=200, G=92, T=48, dt_hours=1.0, min_updown=False, seed=5),
}

SHED_PENALTY = 1e4
RESERVE_FRACTION = 0.05


def uc_config(i) -> LP:
    cfg = UC_CONFIGS[i]
    lp = uc_lp(**cfg)
    lp.name = f"uc_config{i}" if isinstance(i, int) else f"uc_{i}"
    return lp


def _topology(rng, B, L):
    """Random spanning tree (parent ~ U{0..i-1}) plus L-(B-1) extra edges between near indices."""
    frm = np.empty(L, dtype=np.int64)
    to = np.empty(L, dtype=np.int64)
    parents = np.array([rng.integers(0, i) for i in range(1, B)], dtype=np.int64) if B > 1 else np.zeros(0, np.int64)
    frm[:B - 1] = parents
    to[:B - 1] = np.arange(1, B)
    have = set(zip(frm[:B - 1].tolist(), to[:B - 1].tolist()))
    k = B - 1
    guard = 0
    while k < L:
        guard += 1
        assert guard < 1000 * L + 1000, "cannot place extra edges"
        i = int(rng.integers(0, B))
        j = i + int(rng.integers(2, 11))
        if j >= B or (i, j) in have or (j, i) in have:
            continue
        have.add((i, j))
        frm[k], to[k] = i, j
        k += 1
    return frm, to


def uc_lp(B, L, G, T, dt_hours=1.0, min_updown=False, seed=0, commitment=None) -> LP:
    """Build the relaxed DC-UC LP.  `commitment` (G x T array of 0/1) fixes u instead of relaxing it."""
    rng = np.random.default_rng(seed)
    assert L >= B - 1
    frm, to = _topology(rng, B, L)
    react = rng.uniform(0.01, 0.2, L)
    susc = 1.0 / react
    flim = rng.uniform(0.5, 3.0, L)

    gbus = rng.integers(0, B, G)
    pmax = rng.uniform(0.2, 5.0, G)
    pmin = rng.uniform(0.2, 0.5, G) * pmax
    cost = rng.uniform(10.0, 80.0, G)
    startup = rng.uniform(100.0, 2000.0, G)
    ramp = rng.uniform(0.2, 1.0, G) * pmax
    u_init = (np.arange(G) % 2 == 0).astype(np.float64)
    if min_updown:
        UT = rng.integers(2, 7, G)
        DT = rng.integers(2, 7, G)

    base = rng.lognormal(0.0, 0.5, B)
    hours = np.arange(T) * dt_hours
    shape = 1.0 + 0.3 * np.sin(2.0 * np.pi * hours / 24.0)
    scale = pmax.sum() / (1.3 * (base.sum() * shape).max())
    load = scale * np.outer(shape, base)                       # T x B

    # ---- variable layout -------------------------------------------------------------
    V = 5 * G + L + 2 * B
    oP, oU, oSU, oSD, oR, oF, oTH, oSH = 0, G, 2 * G, 3 * G, 4 * G, 5 * G, 5 * G + L, 5 * G + L + B
    n = V * T
    tt = np.arange(T)[:, None]

    def var(off, idx, t=tt):
        return (t * V + off + np.asarray(idx)[None, :]).astype(np.int64)

    lo = np.zeros((T, V))
    hi = np.zeros((T, V))
    cc = np.zeros((T, V))
    hi[:, oP:oP + G] = pmax
    hi[:, oU:oU + G] = 1.0
    hi[:, oSU:oSU + G] = 1.0
    hi[:, oSD:oSD + G] = 1.0
    hi[:, oR:oR + G] = pmax
    lo[:, oF:oF + L] = -flim
    hi[:, oF:oF + L] = flim
    lo[:, oTH:oTH + B] = -np.inf
    hi[:, oTH:oTH + B] = np.inf
    lo[:, oTH] = 0.0
    hi[:, oTH] = 0.0                                           # reference bus angle fixed
    hi[:, oSH:oSH + B] = np.inf
    cc[:, oP:oP + G] = cost
    cc[:, oSU:oSU + G] = startup
    cc[:, oSH:oSH + B] = SHED_PENALTY
    if commitment is not None:
        commitment = np.asarray(commitment, dtype=np.float64).reshape(G, T)
        lo[:, oU:oU + G] = commitment.T
        hi[:, oU:oU + G] = commitment.T

    # ---- row layout --------------------------------------------------------------------
    per0 = B + L + 2 * G + G + 1 + (2 * G if min_updown else 0)      # rows in period 0
    per = per0 + 2 * G                                               # rows in periods >= 1
    rbase = np.where(np.arange(T) == 0, 0, per0 + (np.arange(T) - 1) * per).astype(np.int64)
    m = int(per0 + (T - 1) * per) if T > 0 else 0

    def blocks(t_has_ramp):
        o = {}
        k = 0
        o["bal"] = k; k += B
        o["flow"] = k; k += L
        o["pmin"] = k; k += G
        o["pmax"] = k; k += G
        if t_has_ramp:
            o["rup"] = k; k += G
            o["rdn"] = k; k += G
        o["logic"] = k; k += G
        o["res"] = k; k += 1
        if min_updown:
            o["mup"] = k; k += G
            o["mdn"] = k; k += G
        return o

    o0, o1 = blocks(False), blocks(True)

    def row(name, idx, ts=None):
        ts = np.arange(T) if ts is None else np.asarray(ts)
        off = np.where(ts == 0, o0.get(name, 0), o1[name]).astype(np.int64)
        return (rbase[ts] + off)[:, None] + np.asarray(idx)[None, :]

    R, C, Vv = [], [], []

    def add(r, c, v):
        r = np.asarray(r); c = np.asarray(c)
        v = np.broadcast_to(np.asarray(v, dtype=np.float64), r.shape)
        R.append(r.ravel()); C.append(c.ravel()); Vv.append(v.ravel())

    sense = np.empty(m, dtype=np.uint8)
    rhs = np.zeros(m)
    E, Gs = ord("E"), ord("G")
    gi, li, bi = np.arange(G), np.arange(L), np.arange(B)

    # balance
    rb = row("bal", bi)
    sense[rb.ravel()] = E
    rhs[rb.ravel()] = load.ravel()
    add(row("bal", gbus), var(oP, gi), 1.0)
    add(row("bal", frm), var(oF, li), -1.0)
    add(row("bal", to), var(oF, li), 1.0)
    add(rb, var(oSH, bi), 1.0)
    # flow
    rf = row("flow", li)
    sense[rf.ravel()] = E
    add(rf, var(oF, li), 1.0)
    add(rf, var(oTH, frm), -susc[None, :])
    add(rf, var(oTH, to), susc[None, :])
    # pmin / pmax
    r1 = row("pmin", gi)
    sense[r1.ravel()] = Gs
    add(r1, var(oP, gi), 1.0)
    add(r1, var(oU, gi), -pmin[None, :])
    r2 = row("pmax", gi)
    sense[r2.ravel()] = Gs
    add(r2, var(oU, gi), pmax[None, :])
    add(r2, var(oP, gi), -1.0)
    add(r2, var(oR, gi), -1.0)
    # ramps (t >= 1)
    if T > 1:
        ts = np.arange(1, T)
        tcol = ts[:, None]
        ru = row("rup", gi, ts)
        sense[ru.ravel()] = Gs
        rhs[ru.ravel()] = np.broadcast_to(-ramp, ru.shape).ravel()
        add(ru, var(oP, gi, tcol - 1), 1.0)
        add(ru, var(oP, gi, tcol), -1.0)
        rd = row("rdn", gi, ts)
        sense[rd.ravel()] = Gs
        rhs[rd.ravel()] = np.broadcast_to(-ramp, rd.shape).ravel()
        add(rd, var(oP, gi, tcol), 1.0)
        add(rd, var(oP, gi, tcol - 1), -1.0)
    # logic
    rl = row("logic", gi)
    sense[rl.ravel()] = E
    rhs[rl[0]] = u_init
    add(rl, var(oU, gi), 1.0)
    add(rl, var(oSU, gi), -1.0)
    add(rl, var(oSD, gi), 1.0)
    if T > 1:
        ts = np.arange(1, T)
        add(row("logic", gi, ts), var(oU, gi, ts[:, None] - 1), -1.0)
    # reserve
    rr = row("res", np.zeros(1, dtype=np.int64))
    sense[rr.ravel()] = Gs
    rhs[rr.ravel()] = RESERVE_FRACTION * load.sum(axis=1)
    add(np.broadcast_to(rr, (T, G)), var(oR, gi), 1.0)
    # min up / down
    if min_updown:
        rmu = row("mup", gi)
        rmd = row("mdn", gi)
        sense[rmu.ravel()] = Gs
        sense[rmd.ravel()] = Gs
        rhs[rmd.ravel()] = -1.0
        add(rmu, var(oU, gi), 1.0)
        add(rmd, var(oU, gi), -1.0)
        for w in range(int(max(UT.max(), DT.max()))):            # s = t - w
            ts = np.arange(w, T)
            if ts.size == 0:
                break
            sel = np.nonzero(UT > w)[0]
            if sel.size:
                add(row("mup", sel, ts), var(oSU, sel, (ts - w)[:, None]), -1.0)
            sel = np.nonzero(DT > w)[0]
            if sel.size:
                add(row("mdn", sel, ts), var(oSD, sel, (ts - w)[:, None]), -1.0)

    meta = dict(B=B, L=L, G=G, T=T, V=V, dt_hours=dt_hours, min_updown=min_updown, seed=seed,
                offsets=dict(p=oP, u=oU, su=oSU, sd=oSD, r=oR, f=oF, theta=oTH, shed=oSH),
                total_load=float(load.sum()), pmax_sum=float(pmax.sum()),
                peak_load=float(load.sum(axis=1).max()), rows_period0=int(per0), rows_period=int(per))
    lp = from_coo(m, n, np.concatenate(R), np.concatenate(C), np.concatenate(Vv), sense, rhs,
                  cc.ravel(), lo.ravel(), hi.ravel(), name=f"uc_B{B}_L{L}_G{G}_T{T}_s{seed}", meta=meta)
    return lp


def fix_commitment(lp: LP, commitment) -> LP:
    """Same LP with u fixed to a 0/1 pattern (north_star: 'commitment relaxed to [0,1] or fixed')."""
    G, T, V = lp.meta["G"], lp.meta["T"], lp.meta["V"]
    oU = lp.meta["offsets"]["u"]
    commitment = np.asarray(commitment, dtype=np.float64).reshape(G, T)
    l = lp.l.copy().reshape(T, V)
    u = lp.u.copy().reshape(T, V)
    l[:, oU:oU + G] = commitment.T
    u[:, oU:oU + G] = commitment.T
    return LP(m=lp.m, n=lp.n, row_ptr=lp.row_ptr, col_idx=lp.col_idx, val=lp.val, sense=lp.sense,
              b=lp.b, c=lp.c, l=l.ravel(), u=u.ravel(), name=lp.name + "_fixed", meta=dict(lp.meta))
