"""Kernel-level GPU parity: the single-operator C-ABI entry points (tcgen05 and CUDA-core
kernels) against the oracle's conv definitions, on shapes that span several tiles, ragged
tails (tile rows / images beyond the tensor), dual sources, strides and every epilogue input."""
import numpy as np
import pytest
import torch

from oracle import pulse_oracle as O
from paper_2606_19163_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _B():
    from paper_2606_19163_b200 import binding
    return binding


def grid(rng, *shape, scale=1.0):
    return W.to_bf16_grid(rng.standard_normal(shape) * scale)


def dev_nhwc(a):
    return _B().nhwc(a, torch.bfloat16)


def dev_w(w):      # [Cout,Cin,k,k] -> [Cout,k,k,Cin]
    return torch.as_tensor(w).permute(0, 2, 3, 1).contiguous().to("cuda", torch.bfloat16)


def assert_bf16_close(got_nchw, ref, what, acc_tol=2e-3):
    """fp32-accumulated result stored once in bf16: |err| <= 2^-8 |ref| + acc_tol * RMS(ref)."""
    ref = ref.to(torch.float64)
    err = (got_nchw.to(torch.float64) - ref).abs()
    rms = float(ref.pow(2).mean().sqrt())
    allow = ref.abs() * 2.0 ** -8 + acc_tol * rms
    worst = float((err / allow).max())
    assert worst <= 1.0, f"{what}: worst err/allowance {worst:.3f}, max err {float(err.max()):.3e}, rms {rms:.3e}"


FPROP_CASES = [
    # n, h, w, c0, c1, cout, k, stride, extras
    (3, 8, 8, 64, 0, 160, 3, 1, False),        # 192 pixels: 1.5 tiles, image box beyond N
    (2, 16, 16, 128, 64, 320, 3, 1, True),     # dual source (virtual concat), 2 N tiles, all epilogue inputs
    (1, 32, 32, 64, 0, 160, 1, 1, True),       # 1x1
    (2, 16, 16, 128, 192, 160, 1, 1, False),   # 1x1 shortcut on a concat
    (2, 16, 16, 128, 0, 160, 3, 2, True),      # stride-2 down conv
    (1, 24, 32, 64, 0, 160, 3, 1, False),      # H not a multiple of the tile rows (ragged tail rows)
    (1, 64, 64, 64, 0, 320, 3, 1, False),
    (1, 8, 128, 64, 0, 160, 3, 1, False),      # W = 128: one row per tile
    (5, 8, 8, 320, 0, 128, 3, 1, False),       # BN = 128 path, odd image count
    (5, 16, 16, 64, 64, 320, 3, 1, True),      # 10 M tiles = 5 pair tiles, 1280 pixels: even pairs, every epilogue input
    (3, 16, 16, 64, 0, 320, 3, 1, True),       # 6 M tiles: 3 pair tiles
    (1, 24, 16, 128, 0, 160, 3, 1, True),      # 3 M tiles: the last pair has no second tile (mt >= tiles_m on rank 1)
    (3, 8, 16, 64, 0, 640, 3, 1, False),       # 3 M tiles x 2 N tiles, image boxes (bn > 1 is 8x8 only; here bh = 8)
    (3, 16, 16, 64, 0, 160, 3, 2, True),       # stride 2: 8x8 outputs, 192 pixels, image box beyond N on the pair's rank 1
]
KERNELS = ["pair", "1cta", "simt"]


def _or_skip(B, fn):
    try:
        return fn()
    except B.PulseError as e:
        if e.status == 3:
            pytest.skip("this tcgen05 kernel does not cover the shape")
        raise


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("case", FPROP_CASES)
def test_conv_fprop(case, kernel):
    B = _B()
    n, h, w, c0, c1, cout, k, stride, extras = case
    rng = np.random.default_rng(hash(case) % 2 ** 31)
    x0, x1 = grid(rng, n, c0, h, w), (grid(rng, n, c1, h, w) if c1 else None)
    wt = grid(rng, cout, c0 + c1, k, k, scale=(2.0 / ((c0 + c1) * k * k)) ** 0.5)
    bias = grid(rng, cout, scale=0.1) if extras else None
    pn = rng.standard_normal((n, cout)).astype(np.float32) if extras else None
    res = grid(rng, n, cout, h // stride, w // stride) if extras else None
    xin = torch.as_tensor(x0 if x1 is None else np.concatenate([x0, x1], 1)).double()
    ref = O.conv_fwd(xin, torch.as_tensor(wt).double(), None if bias is None else torch.as_tensor(bias).double(), stride)
    if extras:
        ref = ref + torch.as_tensor(pn).double()[:, :, None, None] + torch.as_tensor(res).double()
    cst = torch.zeros((n, 2, cout), dtype=torch.float32, device="cuda")
    got = _or_skip(B, lambda: B.conv2d(dev_nhwc(x0), dev_w(wt), None if x1 is None else dev_nhwc(x1),
                                       None if bias is None else torch.as_tensor(bias).to("cuda", torch.bfloat16),
                                       None if pn is None else torch.as_tensor(pn).cuda(),
                                       None if res is None else dev_nhwc(res), stride=stride, kernel=kernel,
                                       chan_stats=cst))
    torch.cuda.synchronize()
    assert_bf16_close(B.nchw(got), ref, f"fprop {case} kernel={kernel}")
    # statistics hand-off (fused into the pair kernel's epilogue, masked on ragged tiles): sums of the STORED values
    stored = got.double()                                         # [n, h, w, cout]
    want = torch.stack([stored.sum((1, 2)), stored.pow(2).sum((1, 2))], 1).cpu()
    tol = 1e-4 * float(want[:, 1].abs().max()) + 1e-3
    assert float((cst.double().cpu() - want).abs().max()) <= tol, f"chan stats {case} kernel={kernel}"


DGRAD_CASES = [
    (3, 8, 8, 128, 160, 3, 1), (2, 16, 16, 320, 64, 3, 1), (1, 32, 32, 160, 128, 1, 1),
    (2, 16, 16, 160, 128, 3, 2), (3, 32, 32, 320, 64, 3, 2),
    (3, 16, 16, 320, 128, 3, 1),               # 6 M tiles = 3 pair tiles
    (1, 24, 16, 160, 64, 3, 1),                # 3 M tiles: odd count
    (3, 16, 16, 160, 64, 3, 2),                # stride-2 dgrad phases on 8x8 grids of 3 images (1.5 tiles per phase)
]


@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("case", DGRAD_CASES)
def test_conv_dgrad(case, kernel):
    B = _B()
    n, h, w, cin, cout, k, stride = case       # h, w: input (g_in) size
    rng = np.random.default_rng(hash(case) % 2 ** 31)
    g = grid(rng, n, cout, h // stride, w // stride)
    wt = grid(rng, cout, cin, k, k, scale=(2.0 / (cin * k * k)) ** 0.5)
    ref = O.conv_dgrad(torch.as_tensor(g).double(), torch.as_tensor(wt).double(), (h, w), stride)
    got = _or_skip(B, lambda: B.conv2d_dgrad(dev_nhwc(g), dev_w(wt), (h, w), stride=stride, kernel=kernel))
    torch.cuda.synchronize()
    assert_bf16_close(B.nchw(got), ref, f"dgrad {case} kernel={kernel}")
    # accumulate: g_in += ... on top of a seeded tensor
    base = grid(rng, n, cin, h, w)
    acc = B.conv2d_dgrad(dev_nhwc(g), dev_w(wt), (h, w), stride=stride, kernel=kernel, g_in=dev_nhwc(base))
    torch.cuda.synchronize()
    assert_bf16_close(B.nchw(acc), ref + torch.as_tensor(base).double(), f"dgrad+= {case} kernel={kernel}")


WGRAD_CASES = [
    (3, 8, 8, 64, 0, 320, 3, 1), (2, 16, 16, 128, 64, 320, 3, 1), (1, 32, 32, 64, 0, 320, 1, 1),
    (2, 16, 16, 128, 0, 320, 3, 2), (1, 64, 64, 128, 0, 640, 3, 1), (2, 16, 16, 192, 128, 320, 1, 1),
]


@pytest.mark.parametrize("simt", [False, True])
@pytest.mark.parametrize("case", WGRAD_CASES)
def test_conv_wgrad(case, simt):
    B = _B()
    n, h, w, c0, c1, cout, k, stride = case
    rng = np.random.default_rng(hash(case) % 2 ** 31)
    x0, x1 = grid(rng, n, c0, h, w), (grid(rng, n, c1, h, w) if c1 else None)
    g = grid(rng, n, cout, h // stride, w // stride)
    xin = torch.as_tensor(x0 if x1 is None else np.concatenate([x0, x1], 1)).double()
    ref, _ = O.conv_wgrad(xin, torch.as_tensor(g).double(), (cout, c0 + c1, k, k), stride)
    got = B.conv2d_wgrad(dev_nhwc(x0), dev_nhwc(g), k, None if x1 is None else dev_nhwc(x1), stride=stride,
                         force_simt=simt)
    torch.cuda.synchronize()
    got = got.permute(0, 3, 1, 2).double().cpu()
    rms = float(ref.pow(2).mean().sqrt())
    err = float((got - ref).abs().max())
    assert err <= 1e-4 * rms * 10, f"wgrad {case} simt={simt}: max err {err:.3e} vs rms {rms:.3e}"   # fp32 sums of exact products
