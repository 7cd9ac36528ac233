"""ORACLE (test infrastructure, not product): coefficient construction, Algorithm 1 l.1-8 with
Eq.(2), in plain Python / fp64, written from the text.  Shares no code with the CUDA path.

  v_n      = Psi(role(n), s_n, fanin(n))
  q        = Q^(s_n, m, p)
  tau      = sum_{a in S_p} max_{j in C_a} g^{a,j}(s_n, m, p) / theta_dec(m, d, b0) + tau_pre     Eq.(2)
             "Serial stage durations add, while each parallel stage contributes its longest nominal call duration."
  c        = normalized token count across all base and verification calls, including those that execute in parallel
                                                                               PAPER.md:162
Readings: tau is reported in integer microseconds (round half to even of the fp64 value, theta_dec in tokens/s); the
normaliser of c is a parameter; the fan-in bucket is min(fan-in, F-1).  The policy catalogue of Table 4
 fixes the stage STRUCTURES used by the pins; token counts, rates and Psi values are measured
quantities the paper does not print (parity unpinned for constants).
"""
from __future__ import annotations

import math

import numpy as np


def bind_option(tokens_aj, theta_dec: float, tau_pre_us: float, token_norm: float):
    """tokens_aj: list of stages, each a list of per-call token counts.  Returns (tau_us, cost, total_tokens)."""
    serial = 0.0
    total = 0.0
    for stage in tokens_aj:
        longest = 0.0
        for g in stage:
            longest = max(longest, float(g))
            total += float(g)
        serial += longest
    tau = 1e6 * serial / float(theta_dec) + float(tau_pre_us)
    return int(np.rint(tau)), total / float(token_norm), total


def bind(dims: dict, quality, tokens, theta_dec, tau_pre_us, psi, token_norm, opt_off, pred_mask, skill, role, model,
         backend, policy):
    S, M, P, D, A, J, ROLES, F = (dims[k] for k in ("S", "M", "P", "D", "A", "J", "ROLES", "F"))
    q = np.asarray(quality, np.float32).reshape(S, M, P)
    g = np.asarray(tokens, np.float32).reshape(S, M, P, A, J)
    th = np.asarray(theta_dec, np.float32).reshape(M, D)
    tp = np.asarray(tau_pre_us, np.float32).reshape(M, D)
    ps = np.asarray(psi, np.float32).reshape(ROLES, S, F)
    NN = len(skill)
    KK = len(model)
    vuln = np.full(NN, np.nan, np.float32)
    acc = np.full(KK, np.nan, np.float32)
    lat = np.full(KK, -1, np.int32)
    cost = np.full(KK, np.nan, np.float32)
    dem = np.full(KK, -1, np.int32)
    for n in range(NN):
        s, ro = int(skill[n]), int(role[n])
        node_ok = s < S and ro < ROLES
        if node_ok:
            fan = bin(int(pred_mask[n])).count("1")
            vuln[n] = ps[ro, s, min(fan, F - 1)]
        for o in range(int(opt_off[n]), int(opt_off[n + 1])):
            m, d, p = int(model[o]), int(backend[o]), int(policy[o])
            if not (node_ok and m < M and d < D and p < P and float(th[m, d]) > 0.0):
                continue
            stages = [[float(x) for x in g[s, m, p, a]] for a in range(A)]
            t, c, tot = bind_option(stages, float(th[m, d]), float(tp[m, d]), float(np.float32(token_norm)))
            acc[o] = q[s, m, p]
            lat[o] = t if 0 <= t <= 2**31 - 1 else -1
            cost[o] = np.float32(c)
            dem[o] = int(np.rint(tot)) if tot <= 2**31 - 1 else -1
    return dict(vuln=vuln, acc=acc, lat_us=lat, cost=cost, demand=dem)
