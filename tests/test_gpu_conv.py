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
    # cluster split-K of the pair kernel (few tiles, long K; conv_tc2.cu): 2 or 4 pairs share a tile
    (2, 8, 8, 256, 0, 320, 3, 1, True),        # 1 M tile (the pair's rank 1 idle), 36 K blocks over 4 pairs
    (3, 16, 16, 320, 0, 640, 3, 1, False),     # 3 pair tiles x 2 N tiles, 45 K blocks over 4 pairs (11 + 11 + 11 + 12)
    (8, 8, 8, 640, 640, 1280, 3, 1, True),     # the 8x8 decoder shape: virtual concat, 180 K blocks over 4 pairs, every epilogue input
    (8, 16, 16, 320, 0, 1280, 3, 1, False),    # the 16x16 shape: 32 tiles, 45 K blocks over 2 pairs
]
KERNELS = ["pair", "1cta", "simt"]


def _or_auto(B, kernel, fn, may_refuse=False):
    """fn(kernel) with the forced kernel; a forced tcgen05 kernel that does not cover the shape must refuse it with
    PULSE_ERR_UNSUPPORTED (status 3, nothing launched) - the case then runs through the selector ("auto"), which has to
    cover every shape of the plain convs.  may_refuse: operators that exist only as tcgen05 kernels (the 4-phase upsample
    forms; the stage then takes the materialised form) may be refused by the selector as well: None is returned."""
    try:
        return fn(kernel)
    except B.PulseError as e:
        if e.status != 3 or kernel == "auto":
            raise
    try:
        return fn("auto")
    except B.PulseError as e:
        if e.status != 3 or not may_refuse:
            raise
    return None


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
    got = _or_auto(B, kernel, lambda kn: B.conv2d(dev_nhwc(x0), dev_w(wt), None if x1 is None else dev_nhwc(x1),
                                       None if bias is None else torch.as_tensor(bias).to("cuda", torch.bfloat16),
                                       None if pn is None else torch.as_tensor(pn).cuda(),
                                       None if res is None else dev_nhwc(res), stride=stride, kernel=kn,
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
    (8, 8, 8, 1280, 640, 3, 1),                # split-K over 4 pairs (90 K blocks), also with += on top of a tensor
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
    got = _or_auto(B, kernel, lambda kn: B.conv2d_dgrad(dev_nhwc(g), dev_w(wt), (h, w), stride=stride, kernel=kn))
    torch.cuda.synchronize()
    assert_bf16_close(B.nchw(got), ref, f"dgrad {case} kernel={kernel}")
    # accumulate: g_in += ... on top of a seeded tensor
    base = grid(rng, n, cin, h, w)
    acc = _or_auto(B, kernel, lambda kn: B.conv2d_dgrad(dev_nhwc(g), dev_w(wt), (h, w), stride=stride, kernel=kn, g_in=dev_nhwc(base)))
    torch.cuda.synchronize()
    assert_bf16_close(B.nchw(acc), ref + torch.as_tensor(base).double(), f"dgrad+= {case} kernel={kernel}")


WGRAD_CASES = [
    (3, 8, 8, 64, 0, 320, 3, 1), (2, 16, 16, 128, 64, 320, 3, 1), (1, 32, 32, 64, 0, 320, 1, 1),
    (2, 16, 16, 128, 0, 320, 3, 2), (1, 64, 64, 128, 0, 640, 3, 1), (2, 16, 16, 192, 128, 320, 1, 1),
    # whole-tile ownership (at least as many output tiles as CTA pairs: stores instead of reduce-adds)
    (2, 8, 8, 1280, 0, 1280, 3, 1),            # 180 output tiles: runs of 2 - 3 tiles per pair
    (2, 8, 8, 1280, 640, 640, 3, 1),           # virtual concat, 68 x 2 = 136 tiles, last unit block ragged (270 units)
    (3, 8, 8, 1280, 0, 1280, 1, 1),            # 1x1: 20 units x 4 = 20 tiles < pairs: the shared-tile (reduce-add) path
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
    # += on top of a seeded gradient (the accumulating backwards of a wave)
    base = torch.as_tensor(rng.standard_normal((cout, k, k, c0 + c1)).astype(np.float32))
    acc = B.conv2d_wgrad(dev_nhwc(x0), dev_nhwc(g), k, None if x1 is None else dev_nhwc(x1), stride=stride,
                         force_simt=simt, dw=base.cuda())
    torch.cuda.synchronize()
    err = float((acc.permute(0, 3, 1, 2).double().cpu() - ref - base.permute(0, 3, 1, 2).double()).abs().max())
    assert err <= 1e-4 * rms * 10 + 1e-6, f"wgrad += {case} simt={simt}: max err {err:.3e} vs rms {rms:.3e}"


# ------------------------------------------------------------------ nearest-2x upsample + conv, 4-phase form (row a6)
UP_CASES = [
    # n, h, w (low resolution), cin, cout
    (2, 8, 8, 64, 320),          # 128 low-res pixels: one tile, image box
    (3, 8, 8, 128, 160),         # 192 pixels: ragged tile, image box beyond N
    (1, 16, 16, 64, 640),        # two N tiles
    (3, 16, 16, 128, 320),       # 6 M tiles
    (1, 24, 16, 64, 320),        # 3 M tiles: odd count
    (2, 32, 32, 64, 320),        # configs[2]'s up: 32x32 -> 64x64
]


def phase_form(x, wt, bias, round_weights):
    """The 4-phase identity written out on the CPU (fp64): out[2y+py, 2x+px] = sum_{a,b} Wp[py,px][a,b] x[y+a-1+py, x+b-1+px],
    Wp = sum of W[r][s] over r in R(py,a), s in R(px,b); round_weights: Wp rounded to bf16 as the kernels hold it."""
    R = {(0, 0): [0], (0, 1): [1, 2], (1, 0): [0, 1], (1, 1): [2]}
    n, c, h, w = x.shape
    xp = torch.nn.functional.pad(x, (1, 1, 1, 1))
    out = torch.zeros((n, wt.shape[0], 2 * h, 2 * w), dtype=torch.float64)
    for py in range(2):
        for px in range(2):
            acc = torch.zeros((n, wt.shape[0], h, w), dtype=torch.float64)
            for a in range(2):
                for b in range(2):
                    wp = sum(wt[:, :, r, s_] for r in R[(py, a)] for s_ in R[(px, b)])
                    if round_weights:
                        wp = wp.float().to(torch.bfloat16).double()
                    dy, dx = a - 1 + py, b - 1 + px
                    acc += torch.einsum("oc,nchw->nohw", wp, xp[:, :, 1 + dy:1 + dy + h, 1 + dx:1 + dx + w])
            out[:, :, py::2, px::2] = acc + (0 if bias is None else bias.view(1, -1, 1, 1))
    return out


def test_phase_form_is_the_upsample_conv_identity():
    """No GPU needed in principle (kept here beside its use): with exact weights the 4-phase form IS conv3x3(upsample2(x))."""
    rng = np.random.default_rng(11)
    x, wt, b = (torch.as_tensor(rng.standard_normal(s)) for s in ((2, 3, 4, 5), (6, 3, 3, 3), (6,)))
    assert torch.allclose(phase_form(x, wt, b, False), O.conv_fwd(O.upsample2(x), wt, b), atol=1e-12)


@pytest.mark.parametrize("kernel", ["pair", "1cta"])
@pytest.mark.parametrize("case", UP_CASES)
def test_upsample_conv_fprop_dgrad(case, kernel):
    """The 4-phase form against the oracle's definition conv3x3(upsample2(x)) and its adjoint
    upsample2_bwd(conv_dgrad(g)).  The kernels hold the pre-summed weights in bf16: one rounding of the WEIGHTS (2^-9
    relative per product; it does not average out of the K = 4 c sum the way independent operand errors would), measured
    as <= 1e-2 x RMS max-abs = the size of one bf16 store of the output.  Against the same identity with the weights
    rounded the same way the kernels must be as tight as every other conv (2e-3)."""
    B = _B()
    n, h, w, cin, cout = case
    rng = np.random.default_rng(hash(case) % 2 ** 31)
    x = grid(rng, n, cin, h, w)
    wt = grid(rng, cout, cin, 3, 3, scale=(2.0 / (cin * 9)) ** 0.5)
    bias = grid(rng, cout, scale=0.1)
    ref = O.conv_fwd(O.upsample2(torch.as_tensor(x).double()), torch.as_tensor(wt).double(), torch.as_tensor(bias).double())
    cst = torch.zeros((n, 2, cout), dtype=torch.float32, device="cuda")
    got = _or_auto(B, kernel, lambda kn: B.upsample_conv2d(dev_nhwc(x), dev_w(wt), torch.as_tensor(bias).to("cuda", torch.bfloat16),
                                                kernel=kn, chan_stats=cst))
    torch.cuda.synchronize()
    assert_bf16_close(B.nchw(got), ref, f"up fprop {case} kernel={kernel}", acc_tol=1e-2)
    ref_q = phase_form(torch.as_tensor(x).double(), torch.as_tensor(wt).double(), torch.as_tensor(bias).double(), True)
    assert_bf16_close(B.nchw(got), ref_q, f"up fprop (rounded phase weights) {case} kernel={kernel}")
    stored = got.double()
    want = torch.stack([stored.sum((1, 2)), stored.pow(2).sum((1, 2))], 1).cpu()
    assert float((cst.double().cpu() - want).abs().max()) <= 1e-4 * float(want[:, 1].abs().max()) + 1e-3
    g = grid(rng, n, cout, 2 * h, 2 * w)
    ref_g = O.upsample2_bwd(O.conv_dgrad(torch.as_tensor(g).double(), torch.as_tensor(wt).double(), (2 * h, 2 * w)))
    got_g = _or_auto(B, kernel, lambda kn: B.upsample_conv2d_dgrad(dev_nhwc(g), dev_w(wt), kernel=kn), may_refuse=True)
    if got_g is None:                        # no tcgen05 tile covers the adjoint's shape (e.g. N = cin = 64): refused cleanly
        return
    torch.cuda.synchronize()
    assert_bf16_close(B.nchw(got_g), ref_g, f"up dgrad {case} kernel={kernel}", acc_tol=1e-2)
    # adjoint of the rounded-weight phase form, by autograd of the CPU identity above (fp64)
    xg = torch.zeros((n, cin, h, w), dtype=torch.float64, requires_grad=True)
    (phase_form(xg, torch.as_tensor(wt).double(), None, True) * torch.as_tensor(g).double()).sum().backward()
    assert_bf16_close(B.nchw(got_g), xg.grad, f"up dgrad (rounded phase weights) {case} kernel={kernel}")


@pytest.mark.parametrize("case", [c for c in UP_CASES if c[4] % 320 == 0])
def test_upsample_conv_wgrad(case):
    B = _B()
    n, h, w, cin, cout = case
    rng = np.random.default_rng(hash(case) % 2 ** 31 + 1)
    x, g = grid(rng, n, cin, h, w), grid(rng, n, cout, 2 * h, 2 * w)
    ref, _ = O.conv_wgrad(O.upsample2(torch.as_tensor(x).double()), torch.as_tensor(g).double(), (cout, cin, 3, 3))
    got = B.upsample_conv2d_wgrad(dev_nhwc(x), dev_nhwc(g)).permute(0, 3, 1, 2).double().cpu()
    torch.cuda.synchronize()
    rms = float(ref.pow(2).mean().sqrt())
    err = float((got - ref).abs().max())
    assert err <= 1e-3 * rms, f"up wgrad {case}: max err {err:.3e} vs rms {rms:.3e}"      # fp32 sums of exact bf16 products
