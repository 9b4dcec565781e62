"""Kernel-level GPU parity of GroupNorm + SiLU through the single-operator C-ABI entry
points pulse_groupnorm_silu / pulse_groupnorm_silu_backward, against the oracle's definition: single source and
virtual concat, groups that straddle the x0|x1 boundary, channel-per-group counts that are not vector multiples
(10, 30), ragged pixel counts, the one-pass cluster kernel and the two-kernel form, `add` and `+=` destinations,
and the launch shapes of configs[1] (4 x 64 x 64 x 320 and 320|320)."""
import numpy as np
import pytest
import torch

from oracle import pulse_oracle as O
from paper_2606_19163_b200 import workloads as W

pytestmark = pytest.mark.gpu

EPS = 1e-5


def _B():
    from paper_2606_19163_b200 import binding
    return binding


def grid(rng, *shape, scale=1.0, shift=0.0):
    return W.to_bf16_grid(rng.standard_normal(shape) * scale + shift)


def close_stored(got_nchw, ref, what, dtype, acc_tol=2e-3):
    """A value computed in fp32 and stored once: bf16 |err| <= 2^-8 |ref| + acc_tol RMS(ref); fp32: 1e-4 RMS(ref)
    (north_star's fp32 bar)."""
    ref = ref.to(torch.float64)
    err = (got_nchw.to(torch.float64) - ref).abs()
    rms = float(ref.pow(2).mean().sqrt())
    allow = ref.abs() * 2.0 ** -8 + acc_tol * rms if dtype == torch.bfloat16 else torch.full_like(ref, 1e-4 * rms)
    worst = float((err / allow).max())
    assert worst <= 1.0, f"{what}: worst err/allowance {worst:.3f}, max err {float(err.max()):.3e}, rms {rms:.3e}"


def close_sum(got, ref, what, rel=1e-3):
    """fp32 sums over n*h*w terms of fp32 products (fast-math sigmoid): within rel of the RMS of the vector."""
    ref = ref.to(torch.float64)
    err = float((got.double().cpu() - ref).abs().max())
    rms = float(ref.pow(2).mean().sqrt())
    assert err <= rel * rms + 1e-6, f"{what}: max err {err:.3e} vs rms {rms:.3e}"


CASES = [
    # n, h, w, c0, c1, groups
    (2, 16, 16, 64, 0, 8),        # 8 channels per group: one vector per group
    (3, 8, 8, 320, 0, 32),        # 10 channels per group (configs[1]): slices of lcm(10, 8) = 40 channels
    (2, 8, 8, 64, 32, 4),         # 24 channels per group, group 2 straddles the x0|x1 boundary
    (1, 8, 8, 640, 320, 32),      # configs[2] decoder: 30 channels per group, group 21 straddles 640|320
    (2, 5, 7, 32, 32, 8),         # 35 pixels: ragged pixel rows
    (1, 1, 1, 32, 0, 4),          # one pixel: statistics over the channels of a group only
    (2, 32, 32, 128, 128, 32),    # virtual concat on group boundaries, several CTAs per image
]


def _run_case(case, dtype, two_pass=False, with_add=False, accumulate=False, seed=0, shift=0.3, scale=1.5):
    B = _B()
    n, h, w, c0, c1, groups = case
    C = c0 + c1
    rng = np.random.default_rng(abs(hash((case, seed))) % 2 ** 31)
    x = grid(rng, n, C, h, w, scale=scale, shift=shift)
    gamma, beta = grid(rng, C, scale=0.5, shift=1.0), grid(rng, C, scale=0.3)
    g_a = grid(rng, n, C, h, w)
    add = grid(rng, n, C, h, w) if with_add else None
    base = grid(rng, n, C, h, w) if accumulate else None

    xt, gt, bt = (torch.as_tensor(v).double() for v in (x, gamma, beta))
    a_ref, ctx = O.gn_silu_fwd(xt, gt, bt, groups, EPS)
    gx_ref, dgam_ref, dbet_ref = O.gn_silu_bwd(torch.as_tensor(g_a).double(), ctx, gt)
    if with_add:
        gx_ref = gx_ref + torch.as_tensor(add).double()
    if accumulate:
        gx_ref = gx_ref + torch.as_tensor(base).double()

    dev = lambda a: B.nhwc(a, dtype)
    vec = lambda v: torch.as_tensor(v).to("cuda", dtype)
    x0, x1 = dev(x[:, :c0]), (dev(x[:, c0:]) if c1 else None)
    a, stats = B.groupnorm_silu(x0, vec(gamma), vec(beta), groups, EPS, x1=x1)
    a2, _ = B.groupnorm_silu(x0, vec(gamma), vec(beta), groups, EPS, x1=x1, stats=stats)     # statistics reused
    g0, g1 = (dev(base[:, :c0]), dev(base[:, c0:]) if c1 else None) if accumulate else (None, None)
    g0, g1, dgam, dbet = B.groupnorm_silu_backward(dev(g_a), x0, vec(gamma), vec(beta), groups, stats, EPS, x1=x1,
                                                   add=None if add is None else dev(add), two_pass=two_pass,
                                                   g_x0=g0, g_x1=g1)
    torch.cuda.synchronize()
    what = f"{case} {dtype} two_pass={two_pass} add={with_add} acc={accumulate}"
    close_stored(B.nchw(a), a_ref, "a " + what, dtype)
    assert torch.equal(a, a2), "forward with reused statistics differs: " + what
    gx = B.nchw(g0) if not c1 else torch.cat([B.nchw(g0), B.nchw(g1)], 1)
    # with += the destination's own rounding adds half an ulp of the sum
    close_stored(gx, gx_ref, "g_x " + what, dtype, acc_tol=4e-3 if accumulate else 2e-3)
    close_sum(dgam, dgam_ref, "dgamma " + what)
    close_sum(dbet, dbet_ref, "dbeta " + what)


@pytest.mark.parametrize("two_pass", [False, True])
@pytest.mark.parametrize("case", CASES)
def test_groupnorm_silu_bf16(case, two_pass):
    _run_case(case, torch.bfloat16, two_pass=two_pass)


@pytest.mark.parametrize("case", CASES[:5])
def test_groupnorm_silu_fp32(case):
    _run_case(case, torch.float32)


@pytest.mark.parametrize("two_pass", [False, True])
@pytest.mark.parametrize("case", [CASES[1], CASES[3], CASES[6]])
def test_groupnorm_silu_backward_add_and_accumulate(case, two_pass):
    _run_case(case, torch.bfloat16, two_pass=two_pass, with_add=True, seed=1)
    _run_case(case, torch.bfloat16, two_pass=two_pass, with_add=True, accumulate=True, seed=2)


@pytest.mark.parametrize("dtype", [torch.bfloat16, torch.float32])
@pytest.mark.parametrize("case", [CASES[1], CASES[6]])
def test_groupnorm_silu_large_mean(case, dtype):
    """|mean| = 20 sigma: the statistics travel as per-channel sums of x and x^2 (variance = E[x^2] - E[x]^2, reading
    R22), which cancels 400:1 here; the bars of the other cases must still hold."""
    _run_case(case, dtype, seed=3, shift=20.0, scale=1.0)


@pytest.mark.parametrize("case", [(4, 64, 64, 320, 0, 32), (4, 64, 64, 320, 320, 32)])
def test_groupnorm_silu_config2_launch_shapes(case):
    """The GroupNorm sites of configs[1] at full size, in the launch configuration bench.py times."""
    _run_case(case, torch.bfloat16, with_add=True)


def test_groupnorm_group_statistics_on_device():
    """Invariant at any size: the saved mean / r reproduce per-group mean 0, variance 1 of xhat."""
    B = _B()
    n, h, w, c, groups = 2, 24, 40, 160, 32
    rng = np.random.default_rng(5)
    x = grid(rng, n, c, h, w, scale=2.0, shift=-0.7)
    one, zero = torch.ones(c, device="cuda", dtype=torch.bfloat16), torch.zeros(c, device="cuda", dtype=torch.bfloat16)
    _, stats = B.groupnorm_silu(B.nhwc(x, torch.bfloat16), one, zero, groups, EPS)
    torch.cuda.synchronize()
    mr = stats[n * 2 * c:].view(n, 2, groups).double().cpu()
    xg = torch.as_tensor(x).double().reshape(n, groups, -1)
    xhat = (xg - mr[:, 0, :, None]) * mr[:, 1, :, None]
    assert float(xhat.mean(2).abs().max()) < 1e-4
    assert float((xhat.var(2, unbiased=False) - 1).abs().max()) < 1e-3
