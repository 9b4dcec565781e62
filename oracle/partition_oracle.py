"""Brute-force oracle of the skip-aware balanced partitioning.  TEST INFRASTRUCTURE ONLY (see pulse_oracle.py).

PAPER.md:L140-L150 (sec. IV-B) states the problem; this file is that statement written out, for small n:
  * the model is a sequence of operations l_1 .. l_n, cut into p contiguous stages S_1 .. S_p;
  * "if a skip connection exists between operations l_i and l_j such that |i-j| > 1, and l_i is assigned to partition
    q, then l_j must be assigned to partition p-q+1";
  * minimise max_m ( T_f(S_m) + lambda * (t_lat + M_a(S_m) / B_inter) )   (Eq. 1, with the communication term of Eq. 2-3:
    M_a of an encoder-side stage (m <= p/2) is the activation its LAST operation sends on; of a decoder-side stage
    (m > p/2) the activation that arrives from the operation BEFORE its first one).
Every set of p-1 cut positions is enumerated (itertools.combinations); nothing is shared with csrc/partition.cpp.
"""
from __future__ import annotations

import itertools
import math


def stage_costs(t_f, act_bytes, cuts, p, lam=0.0, t_lat=0.0, b_inter=1.0):
    """cuts: 1-based index of the last operation of stages 1 .. p-1 (increasing)."""
    n = len(t_f)
    ends = list(cuts) + [n]
    costs, start = [], 1
    for m, end in enumerate(ends, start=1):
        t = sum(t_f[l - 1] for l in range(start, end + 1))
        if lam != 0.0:
            a = act_bytes[end - 1] if m <= p // 2 else (act_bytes[start - 2] if start >= 2 else 0.0)
            t += lam * (t_lat + a / b_inter)
        costs.append(t)
        start = end + 1
    return costs


def stage_of(cuts, n, l):
    for m, end in enumerate(list(cuts) + [n], start=1):
        if l <= end:
            return m
    raise ValueError(l)


def feasible(cuts, n, p, skips):
    for a, b in skips:
        if abs(a - b) > 1 and stage_of(cuts, n, b) != p - stage_of(cuts, n, a) + 1:
            return False
    return True


def brute_force(t_f, skips, p, act_bytes=None, lam=0.0, t_lat=0.0, b_inter=1.0):
    """Returns (best bottleneck, list of all optimal cut tuples); (inf, []) if nothing is feasible."""
    n = len(t_f)
    best, arg = math.inf, []
    for cuts in itertools.combinations(range(1, n), p - 1):
        if not feasible(cuts, n, p, skips):
            continue
        c = max(stage_costs(t_f, act_bytes, cuts, p, lam, t_lat, b_inter))
        if c < best - 1e-12:
            best, arg = c, [cuts]
        elif abs(c - best) <= 1e-12:
            arg.append(cuts)
    return best, arg
