"""Skip-aware balanced partitioning (sec. IV-B): the native O(p n^3) table of libpulse.so
against the brute-force oracle (every set of cuts enumerated, constraint and objective written from the paper's
sentences), plus pins of that oracle on cases with a known answer.  Host code only: runs without a GPU."""
import math

import numpy as np
import pytest

from oracle import partition_oracle as PO
from paper_2606_19163_b200 import workloads as W


@pytest.fixture(scope="module")
def B():
    from paper_2606_19163_b200 import binding
    return binding


# ------------------------------------------------------------------ pins of the brute-force oracle
def test_oracle_without_skips_is_classical_linear_partition():
    # 6 equal operations into 2 stages: the balanced cut
    assert PO.brute_force([1] * 6, [], 2) == (3.0, [(3,)])
    # 1 2 ... 9 into 4 stages: 1-5 | 6-7 | 8 | 9 -> 15 (no stage can hold less than 9, and 6+7 forces >= 13; 1-5 = 15
    # cannot be split without a fifth stage: {1..4} = 10, then 5-6 = 11, 7-8 = 15)
    best, arg = PO.brute_force(list(range(1, 10)), [], 4)
    assert best == 15.0 and (5, 7, 8) in arg
    # the textbook instance of the linear partition problem: 1 .. 9 into 3 -> 1-5 | 6-7 | 8-9 = 17 (the oracle does not
    # require an even p; the native table does)
    assert PO.brute_force(list(range(1, 10)), [], 3) == (17.0, [(5, 7)])


def test_oracle_skip_constraint_by_hand():
    # UNet of 6 operations with nested skips 1->6, 2->5: with p = 2 any cut between 2 and 5 keeps both pairs collocated
    # (stage 1 with stage 2); with p = 4 operation 1 must sit in stage 1 and 6 in stage 4, 2 with 5 in (1,4) or (2,3)
    t = [1, 1, 4, 4, 1, 1]
    best2, arg2 = PO.brute_force(t, [(1, 6), (2, 5)], 2)
    assert best2 == 6.0 and arg2 == [(3,)]
    best4, arg4 = PO.brute_force(t, [(1, 6), (2, 5)], 4)
    assert best4 == 4.0 and arg4 == [(2, 3, 4)]
    # a cut that separates a pair from its mirror stage is infeasible: skip 1->4 with cuts (1, 2, 4): op 4 in stage 3, needs 4
    assert not PO.feasible((1, 2, 4), 6, 4, [(1, 4)])
    assert PO.feasible((1, 2, 3), 6, 4, [(1, 4)])
    # adjacent operations (|i - j| = 1) do not constrain
    assert PO.feasible((1, 2, 3), 6, 4, [(3, 4)])


def test_oracle_communication_term():
    # lambda = 1, t_lat = 0.5, B = 2: stage 1 pays act[last]/B, stage 2 (decoder side) act[op before its first]/B
    c = PO.stage_costs([1, 2, 3, 4], [10, 20, 30, 40], (2,), 2, lam=1.0, t_lat=0.5, b_inter=2.0)
    assert c == [1 + 2 + 0.5 + 20 / 2, 3 + 4 + 0.5 + 20 / 2]


# ------------------------------------------------------------------ native table vs brute force
def _random_case(rng, n, p):
    t = rng.uniform(0.2, 5.0, n).round(3).tolist()
    act = rng.uniform(1.0, 50.0, n).round(2).tolist()
    # nested UNet-style skips around a random centre, plus (sometimes) nothing
    k = int(rng.integers(0, n // 2))
    mid = int(rng.integers(2, n - 1))
    skips = []
    for d in range(1, k + 1):
        a, b = mid - d, mid + d
        if a >= 1 and b <= n and rng.random() < 0.8:
            skips.append((a, b))
    return t, act, skips


@pytest.mark.parametrize("seed", range(40))
def test_native_matches_brute_force(B, seed):
    rng = np.random.default_rng(seed)
    n = int(rng.integers(4, 13))
    p = int(rng.choice([q for q in (2, 4, 6) if q <= n]))
    t, act, skips = _random_case(rng, n, p)
    lam = float(rng.choice([0.0, 0.7]))
    want, args = PO.brute_force(t, skips, p, act, lam, 0.3, 7.0)
    if math.isinf(want):
        with pytest.raises(B.PulseError) as ei:
            B.partition(t, skips, p, act, lam, 0.3, 7.0)
        assert ei.value.status == 2
        return
    cuts, best = B.partition(t, skips, p, act, lam, 0.3, 7.0)
    assert abs(best - want) <= 1e-9 * max(1.0, want), (best, want)
    # the returned cuts are a feasible partition that attains the optimum (several may tie)
    assert PO.feasible(tuple(cuts), n, p, skips)
    assert abs(max(PO.stage_costs(t, act, cuts, p, lam, 0.3, 7.0)) - want) <= 1e-9 * max(1.0, want)
    assert all(a < b for a, b in zip(cuts, cuts[1:])) and 1 <= cuts[0] and cuts[-1] < n


def test_non_nested_skips(B):
    # crossing skips 1->5, 2->6 (not LIFO): both must satisfy the mirror rule
    t = [1, 2, 3, 1, 2, 3, 1]
    for p in (2, 4):
        want, _ = PO.brute_force(t, [(1, 5), (2, 6)], p)
        if math.isinf(want):
            with pytest.raises(B.PulseError):
                B.partition(t, [(1, 5), (2, 6)], p)
        else:
            assert abs(B.partition(t, [(1, 5), (2, 6)], p)[1] - want) < 1e-12


def test_argument_errors(B):
    with pytest.raises(B.PulseError) as ei:
        B.partition([1, 2, 3], [], 3)
    assert ei.value.status == 3          # odd p
    with pytest.raises(B.PulseError) as ei:
        B.partition([1, 2], [], 4)
    assert ei.value.status == 2          # more stages than operations
    with pytest.raises(B.PulseError) as ei:
        B.partition([1, 2, 3, 4], [(3, 2)], 2)
    assert ei.value.status == 2          # src >= dst


def test_config4_unet_partition_beats_blockwise(B):
    """configs[3]'s op list (27 operations, 12 skips) with FLOP-proportional costs: the balanced partition into 4 / 8
    stages is feasible and at least as good as cutting into equal operation counts (the paper's block-wise baseline)."""
    desc = W.config(4)
    ops = desc["enc_ops"] + desc["mid_ops"] + desc["dec_ops"]
    n = len(ops)
    # forward conv FLOPs per op
    h = desc["h"]
    t, hh = [], h
    pushes, skips = [], []
    for i, op in enumerate(ops, start=1):
        if op["kind"] == "down":
            hh //= 2
        if op["kind"] == "up":
            hh *= 2
        ci, co = op["cin"] + op["skip"], op["cout"]
        f = 2.0 * desc["n"] * hh * hh * co * ci * 9
        if op["kind"] == "resblock":
            f += 2.0 * desc["n"] * hh * hh * co * co * 9
        t.append(f / 1e12)
        if op.get("push"):
            pushes.append(i)
        if op["skip"]:
            skips.append((pushes.pop(), i))
    assert len(skips) == 12 and not pushes
    for p in (2, 4, 8):
        cuts, best = B.partition(t, skips, p)
        assert PO.feasible(tuple(cuts), n, p, skips)
        assert abs(max(PO.stage_costs(t, None, cuts, p)) - best) < 1e-12
        assert best >= sum(t) / p - 1e-12           # lower bound: perfect balance
        # block-wise: mirror-symmetric equal operation counts (feasible for this symmetric op list only if it pairs skips)
        block = [round(n * m / p) for m in range(1, p)]
        if PO.feasible(tuple(block), n, p, skips):
            assert best <= max(PO.stage_costs(t, None, block, p)) + 1e-12
