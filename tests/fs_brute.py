"""Brute-force evaluators for the oracle's pins (tests only).

Written independently of oracle/festina_oracle.cpp: flat enumeration of EVERY candidate of the
finite candidate set with numpy float32 scalars (each operation is one binary32 rounding), the
result taken by an explicit lexicographic minimum over (value, flat index).  No early exits, no
shared structure with the oracle's loops.
"""
from __future__ import annotations

import itertools
from math import comb

import numpy as np

f32 = np.float32
INF = f32(np.inf)


def _slot(lat, pow_, m, p, phi, sg, beta, q, wait, slo):
    if q == 0:
        return True, f32(0), f32(0)
    rounds = -(-int(q) // (int(beta) + 1))
    l = lat[m, p, phi, sg, beta]
    t = f32(f32(rounds) * l)
    ok = bool(f32(f32(wait) + t) <= f32(slo)) if p == 0 else bool(l <= f32(slo))
    e = f32(t * pow_[m, p, phi, sg, beta])
    return ok, t, e


def _tenant(lat, pow_, B, t, phi, sg, bump):
    b1 = int(t["beta"][1]) + (1 if (bump and t["q"][1] > 0) else 0)
    if b1 >= B:
        return False, INF
    ok0, _, e0 = _slot(lat, pow_, int(t["model"]), 0, phi, sg, int(t["beta"][0]), int(t["q"][0]), 0.0, t["slo_ms"][0])
    ok1, _, e1 = _slot(lat, pow_, int(t["model"]), 1, phi, sg, b1, int(t["q"][1]), 0.0, t["slo_ms"][1])
    return ok0 and ok1, f32(e0 + e1)


def _sum_left(vals):
    acc = vals[0]
    for v in vals[1:]:
        acc = f32(acc + v)
    return acc


def place_candidates(cl, r):
    """All feasible (dE, flat, k, sigma, phi) of request r, in no particular order."""
    lat, pow_ = cl.lat, cl.pow
    rq = cl.requests[r]
    m = int(rq["model"])
    O = (21 * int(rq["o_pred"]) + 19) // 20
    mem = f32(f32(int(rq["L"]) + O) * cl.models["kv_mb_per_token"][m])
    out = []
    for k, phi, sg in itertools.product(range(cl.K), range(cl.F), range(cl.S)):
        g = cl.states[k]
        n = int(g["n_res"])
        if n < 1 or not (mem <= g["mem_free_mb"]):
            continue
        used = sum(int(g["t"][i]["sigma"]) + 1 for i in range(n))
        if sg >= cl.S - used:
            continue
        js = [i for i in range(n) if int(g["t"][i]["model"]) == m]
        j = js[0] if js else -1
        if j < 0 and n >= 4:
            continue
        wait = g["t_avail_ms"] if j >= 0 else f32(g["t_avail_ms"] + cl.models["load_ms"][m])
        br0 = min(int(rq["L"]), cl.B) - 1
        br1 = int(g["t"][j]["beta"][1]) + 1 if (j >= 0 and g["t"][j]["q"][1] > 0) else 0
        if br1 >= cl.B:
            continue
        te = [_tenant(lat, pow_, cl.B, g["t"][i], phi, int(g["t"][i]["sigma"]), i == j) for i in range(n)]
        if not all(ok for ok, _ in te):
            continue
        A = _sum_left([e for _, e in te])
        Ecur = _sum_left([_tenant(lat, pow_, cl.B, g["t"][i], int(g["f_cur"]), int(g["t"][i]["sigma"]), False)[1] for i in range(n)])
        ok0, t0, e0 = _slot(lat, pow_, m, 0, phi, sg, max(br0, 0), int(rq["L"]), wait, rq["slo_ttft_ms"])
        ok1, _, e1 = _slot(lat, pow_, m, 1, phi, sg, br1, O, 0.0, rq["slo_tbt_ms"])
        if not (ok0 and ok1):
            continue
        dE = f32(f32(A + f32(e0 + e1)) - Ecur)
        if not dE < INF:
            continue
        flat = (k * cl.S + sg) * cl.F + phi
        out.append((float(dE) + 0.0, flat, k, sg, phi, br1, f32(wait + t0), lat[m, 1, phi, sg, br1]))
    return out


def place_best(cl, r):
    c = place_candidates(cl, r)
    if not c:
        return None
    return min(c, key=lambda x: (x[0], x[1]))


def compositions(S, n):
    """All (sigma_0..sigma_{n-1}) with sum(sigma_i+1) == S, lexicographic."""
    for parts in itertools.product(range(S), repeat=n):
        if sum(parts) + n == S:
            yield parts


def local_slot_costs(cl, g, i, p, phi, sg, obj_power):
    """[(cost, beta, e, pw)] over every feasible beta of slot (i,p) at (phi, sg)."""
    t = g["t"][i]
    q = int(t["q"][p])
    if q == 0:
        return [(f32(0), 0, f32(0), f32(0))]
    res = []
    for beta in range(min(cl.B, q)):
        ok, _, e = _slot(cl.lat, cl.pow, int(t["model"]), p, phi, sg, beta, q, 0.0, t["slo_ms"][p])
        if ok:
            pw = cl.pow[int(t["model"]), p, phi, sg, beta]
            res.append((pw if obj_power else e, beta, e, pw))
    return res


def local_best(cl, k, obj_power, minsm):
    """Hierarchical definition, by exhaustive enumeration.  Returns (C, flat, phi, sigmas, betas)."""
    g = cl.states[k]
    n = int(g["n_res"])
    best = None
    NS = comb(cl.S - 1, n - 1)
    for phi in range(cl.F):
        G = {}
        for i in range(n):
            for sg in range(cl.S):
                c0 = local_slot_costs(cl, g, i, 0, phi, sg, obj_power)
                c1 = local_slot_costs(cl, g, i, 1, phi, sg, obj_power)
                if c0 and c1:
                    b0 = min(c0, key=lambda x: (x[0], x[1]))
                    b1 = min(c1, key=lambda x: (x[0], x[1]))
                    G[i, sg] = (f32(b0[0] + b1[0]), b0[1], b1[1])
        if minsm:
            sig = []
            for i in range(n):
                feas = [sg for sg in range(cl.S) if (i, sg) in G and G[i, sg][0] < INF]
                if not feas:
                    break
                sig.append(min(feas))
            if len(sig) < n or sum(sig) + n > cl.S:
                continue
            cands = [(tuple(sig), phi)]
        else:
            cands = [(sp, phi * NS + rank) for rank, sp in enumerate(compositions(cl.S, n))]
        for sp, flat in cands:
            if any((i, sp[i]) not in G for i in range(n)):
                continue
            C = _sum_left([G[i, sp[i]][0] for i in range(n)])
            if not C < INF:
                continue
            key = (float(C), flat)
            if best is None or key < best[0]:
                best = (key, phi, sp, [(G[i, sp[i]][1], G[i, sp[i]][2]) for i in range(n)])
    return best


def consolidate_all(cl):
    """[(dst, phi, score)] per source by full enumeration; dst=-1 if none."""
    P = cl.params
    K, F, S = cl.K, cl.F, cl.S
    S_eff = (S * (100 - P.delta_pct)) // 100
    M_eff = f32(f32(f32(P.mem_cap_mb) * f32(100 - P.delta_pct)) / f32(100.0))
    need = np.full((K, F), 1 << 20, dtype=np.int64)
    E = np.full((K, F), INF, dtype=np.float32)
    mem = np.zeros(K, dtype=np.float32)
    for g in range(K):
        st = cl.states[g]
        n = int(st["n_res"])
        if n < 1:
            continue
        mem[g] = _sum_left([st["t"][i]["mem_used_mb"] for i in range(n)])
        for phi in range(F):
            tot, es = 0, []
            for i in range(n):
                feas = [(sg, _tenant(cl.lat, cl.pow, cl.B, st["t"][i], phi, sg, False)) for sg in range(S)]
                feas = [(sg, te[1]) for sg, te in feas if te[0]]
                if not feas:
                    break
                tot += feas[0][0] + 1
                es.append(feas[0][1])
            if len(es) == n:
                need[g, phi] = tot
                E[g, phi] = _sum_left(es)
    Cstar = np.array([min([E[g, phi] for phi in range(F) if need[g, phi] <= S_eff], default=INF) for g in range(K)], dtype=np.float32)
    res = []
    for a in range(K):
        cands = []
        na = int(cl.states[a]["n_res"])
        for b in range(K):
            nb = int(cl.states[b]["n_res"])
            if a == b or na < 1 or nb < 1 or na + nb > 4:
                continue
            if not f32(mem[a] + mem[b]) <= M_eff or not Cstar[b] < INF:
                continue
            per_phi = [(float(f32(E[b, phi] + E[a, phi])), phi) for phi in range(F) if need[a, phi] + need[b, phi] <= S_eff]
            per_phi = [x for x in per_phi if x[0] < np.inf]
            if not per_phi:
                continue
            cab, phis = min(per_phi)
            cands.append((float(f32(f32(cab) - Cstar[b])), b, phis))
        if cands:
            sc, b, phis = min(cands)
            res.append((b, phis, f32(sc), Cstar[a]))
        else:
            res.append((-1, -1, INF, Cstar[a]))
    return res
