"""Pins for oracle/pulse_oracle.py against things other than itself (no GPU).

The paper prints no worked numeric example of a stage (SURVEY.md 8c last row), so the
pins are: brute-force direct sums on tiny inputs, closed forms, invariants, adjoint
identities, fp64 central differences, and an independently composed library+autograd
run that recomputes every skip (tests/naive_autograd.py)."""
import itertools
import math

import numpy as np
import pytest
import torch

from oracle import pulse_oracle as O
from paper_2606_19163_b200 import workloads as W
from tests import naive_autograd as NA

torch.manual_seed(0)
D = torch.float64


def rnd(*s):
    return torch.randn(*s, dtype=D)


# ------------------------------------------------------------------ conv: brute force

def conv_direct(x, w, b, stride):
    """SURVEY 8c item 2 written as loops (gather form)."""
    x, w = x.numpy(), w.numpy()
    n, ci, H, Wd = x.shape
    co, _, k, _ = w.shape
    pad = (k - 1) // 2
    Ho, Wo = (H + 2 * pad - k) // stride + 1, (Wd + 2 * pad - k) // stride + 1
    out = np.zeros((n, co, Ho, Wo))
    for nn, o, y, xx in itertools.product(range(n), range(co), range(Ho), range(Wo)):
        acc = b[o].item() if b is not None else 0.0
        for c, r, s in itertools.product(range(ci), range(k), range(k)):
            iy, ix = y * stride + r - pad, xx * stride + s - pad
            if 0 <= iy < H and 0 <= ix < Wd:
                acc += w[o, c, r, s] * x[nn, c, iy, ix]
        out[nn, o, y, xx] = acc
    return torch.from_numpy(out)


def dgrad_scatter(g, w, in_hw, stride):
    """scatter form: g_in[n,ci,y st+r-pad,x st+s-pad] += W g_out[n,co,y,x]."""
    g, w = g.numpy(), w.numpy()
    n, co, Ho, Wo = g.shape
    _, ci, k, _ = w.shape
    pad = (k - 1) // 2
    out = np.zeros((n, ci, in_hw[0], in_hw[1]))
    for nn, o, y, xx, c, r, s in itertools.product(range(n), range(co), range(Ho), range(Wo),
                                                   range(ci), range(k), range(k)):
        iy, ix = y * stride + r - pad, xx * stride + s - pad
        if 0 <= iy < in_hw[0] and 0 <= ix < in_hw[1]:
            out[nn, c, iy, ix] += w[o, c, r, s] * g[nn, o, y, xx]
    return torch.from_numpy(out)


def wgrad_direct(x, g, k, stride):
    x, g = x.numpy(), g.numpy()
    n, ci, H, Wd = x.shape
    _, co, Ho, Wo = g.shape
    pad = (k - 1) // 2
    dw = np.zeros((co, ci, k, k))
    for o, c, r, s in itertools.product(range(co), range(ci), range(k), range(k)):
        acc = 0.0
        for nn, y, xx in itertools.product(range(n), range(Ho), range(Wo)):
            iy, ix = y * stride + r - pad, xx * stride + s - pad
            if 0 <= iy < H and 0 <= ix < Wd:
                acc += g[nn, o, y, xx] * x[nn, c, iy, ix]
        dw[o, c, r, s] = acc
    return torch.from_numpy(dw)


@pytest.mark.parametrize("k,stride,hw", [(3, 1, (5, 4)), (3, 2, (6, 4)), (1, 1, (3, 5))])
def test_conv_matches_direct_sums(k, stride, hw):
    x, w, b = rnd(2, 3, *hw), rnd(4, 3, k, k), rnd(4)
    out = O.conv_fwd(x, w, b, stride)
    assert torch.allclose(out, conv_direct(x, w, b, stride), atol=1e-12)
    g = rnd(*out.shape)
    assert torch.allclose(O.conv_dgrad(g, w, hw, stride), dgrad_scatter(g, w, hw, stride), atol=1e-12)
    dw, db = O.conv_wgrad(x, g, w.shape, stride)
    assert torch.allclose(dw, wgrad_direct(x, g, k, stride), atol=1e-12)
    assert torch.allclose(db, g.sum((0, 2, 3)), atol=1e-12)


def test_conv_closed_forms():
    x = rnd(2, 5, 6, 6)
    # 1x1 conv == matmul over channels
    w1 = rnd(7, 5, 1, 1)
    assert torch.allclose(O.conv_fwd(x, w1, None), torch.einsum("oc,nchw->nohw", w1[:, :, 0, 0], x), atol=1e-12)
    # delta kernel == identity
    wd = torch.zeros(5, 5, 3, 3, dtype=D)
    for c in range(5):
        wd[c, c, 1, 1] = 1.0
    assert torch.equal(O.conv_fwd(x, wd, None), x)
    # constant input: interior output == sum of weights (+ bias)
    w, b = rnd(4, 5, 3, 3), rnd(4)
    out = O.conv_fwd(torch.ones(1, 5, 6, 6, dtype=D), w, b)
    assert torch.allclose(out[0, :, 2, 3], w.sum((1, 2, 3)) + b, atol=1e-12)
    # corner sees only 4 taps
    assert torch.allclose(out[0, :, 0, 0], w[:, :, 1:, 1:].sum((1, 2, 3)) + b, atol=1e-12)
    # stride 2 == stride 1 sampled at even pixels (reading R11)
    assert torch.allclose(O.conv_fwd(x, w, b, 2), O.conv_fwd(x, w, b, 1)[:, :, ::2, ::2], atol=1e-12)


@pytest.mark.parametrize("stride", [1, 2])
def test_conv_adjoint_identities(stride):
    x, w = rnd(2, 6, 8, 8), rnd(5, 6, 3, 3)
    y = rnd(*O.conv_fwd(x, w, None, stride).shape)
    lhs = (O.conv_fwd(x, w, None, stride) * y).sum()
    assert abs(lhs - (x * O.conv_dgrad(y, w, x.shape[2:], stride)).sum()) < 1e-10 * abs(lhs)
    assert abs(lhs - (w * O.conv_wgrad(x, y, w.shape, stride)[0]).sum()) < 1e-10 * abs(lhs)


# ------------------------------------------------------------------ GroupNorm + SiLU

def test_silu_closed_forms():
    z = torch.zeros(1, dtype=D)
    assert O.silu(z).item() == 0.0 and O.silu_grad(z).item() == 0.5
    # minimum of SiLU: x* solves 1 + x(1-s) = 0 -> x* = -1.2784645..., SiLU(x*) = -0.2784645...
    xs = torch.tensor([-1.2784645427610738], dtype=D)
    assert abs(O.silu_grad(xs).item()) < 1e-12
    assert abs(O.silu(xs).item() + 0.2784645427610738) < 1e-12
    big = torch.tensor([40.0], dtype=D)
    assert abs(O.silu(big).item() - 40.0) < 1e-12 and abs(O.silu(-big).item()) < 1e-12
    y = rnd(100)
    eps = 1e-6
    fd = (O.silu(y + eps) - O.silu(y - eps)) / (2 * eps)
    assert torch.allclose(O.silu_grad(y), fd, atol=1e-8)


def test_groupnorm_invariants():
    n, c, G, eps = 3, 12, 4, 1e-5
    x = rnd(n, c, 5, 5) * 3 + 2
    ones, zeros = torch.ones(c, dtype=D), torch.zeros(c, dtype=D)
    _, ctx = O.gn_silu_fwd(x, ones, zeros, G, eps)
    xh = ctx["xhat"].reshape(n, G, -1)
    var = x.reshape(n, G, -1).var(dim=2, unbiased=False)
    assert xh.mean(2).abs().max() < 1e-12                     # per-group mean 0
    assert torch.allclose(xh.var(dim=2, unbiased=False), var / (var + eps), atol=1e-12)  # ~1 before affine
    # GN(alpha x + beta) == GN(x) for alpha > 0 when eps scales with alpha^2
    _, ctx2 = O.gn_silu_fwd(2.5 * x + 7.0, ones, zeros, G, eps * 2.5 ** 2)
    assert torch.allclose(ctx2["xhat"], ctx["xhat"], atol=1e-10)
    # affine + SiLU applied on top of xhat
    gamma, beta = rnd(c), rnd(c)
    a, _ = O.gn_silu_fwd(x, gamma, beta, G, eps)
    y = gamma.view(1, c, 1, 1) * ctx["xhat"] + beta.view(1, c, 1, 1)
    assert torch.allclose(a, y / (1 + torch.exp(-y)), atol=1e-12)
    # channel c belongs to group c // (C/G): perturbing one group leaves the others' xhat alone
    x2 = x.clone()
    x2[:, 3:6] += 5.0
    _, ctx3 = O.gn_silu_fwd(x2, ones, zeros, G, eps)
    assert torch.equal(ctx3["xhat"][:, :3], ctx["xhat"][:, :3]) and torch.equal(ctx3["xhat"][:, 6:], ctx["xhat"][:, 6:])
    # backward: per group sum g_x = 0 and sum g_x xhat = 0
    g_a = rnd(n, c, 5, 5)
    a, ctxg = O.gn_silu_fwd(x, gamma, beta, G, eps)
    g_x, dg, db = O.gn_silu_bwd(g_a, ctxg, gamma)
    gx = g_x.reshape(n, G, -1)
    assert gx.sum(2).abs().max() < 1e-10
    # sum g_x xhat = r B (m - sum xhat^2) = r B m eps/(var+eps): zero only as eps -> 0
    m = xh.shape[2]
    q = (g_a * O.silu_grad(ctxg["y"]) * gamma.view(1, c, 1, 1)).reshape(n, G, -1)
    Bq = (q * xh).mean(2)
    want = ctxg["r"][:, :, 0] * Bq * m * eps / (var + eps)
    assert torch.allclose((gx * xh).sum(2), want, atol=1e-10)
    # library cross-check incl. autograd
    xr = x.clone().requires_grad_(True)
    gr, br = gamma.clone().requires_grad_(True), beta.clone().requires_grad_(True)
    ar = torch.nn.functional.silu(torch.nn.functional.group_norm(xr, G, gr, br, eps))
    ar.backward(g_a)
    assert torch.allclose(a, ar.detach(), atol=1e-12)
    assert torch.allclose(g_x, xr.grad, atol=1e-10) and torch.allclose(dg, gr.grad, atol=1e-10)
    assert torch.allclose(db, br.grad, atol=1e-10)


def test_sinusoidal_and_upsample():
    e = O.sinusoidal(torch.tensor([0, 3, 999]), 16)
    assert torch.equal(e[0, :8], torch.ones(8, dtype=D)) and torch.equal(e[0, 8:], torch.zeros(8, dtype=D))
    assert abs(e[1, 0].item() - math.cos(3.0)) < 1e-14 and abs(e[1, 8].item() - math.sin(3.0)) < 1e-14  # f_0 = 1
    assert abs(e[2, 4].item() - math.cos(999 * 10000 ** (-4 / 8))) < 1e-12                              # f_i
    d = rnd(2, 3, 3, 4)
    u = O.upsample2(d)
    for Y, X in itertools.product(range(6), range(8)):
        assert torch.equal(u[:, :, Y, X], d[:, :, Y // 2, X // 2])
    g = rnd(*u.shape)
    assert abs((u * g).sum() - (d * O.upsample2_bwd(g)).sum()) < 1e-10      # adjoint == 2x2 sum
    assert torch.allclose(O.upsample2_bwd(g)[:, :, 1, 2], g[:, :, 2:4, 4:6].sum((2, 3)), atol=1e-12)


# ------------------------------------------------------------------ whole stage

KINDS = ["pair", "level", "updown", "straddle", "unet", "attn", "attn_unet", "uvit"]


@pytest.mark.parametrize("kind", KINDS)
def test_stage_matches_naive_recompute_autograd(kind):
    """Skip locality: cached-skip result == naive sequential run that recomputes the skip;
    hand-written backward == autograd of the library-composed forward."""
    desc = W.mini(kind)
    data = W.draw(desc, seed=1, with_g_e_out=True)
    mb = data["microbatches"][0]
    r = O.run_stage(desc, data["params"], mb)
    ref = NA.run(desc, data["params"], mb)
    for k in ["loss", "d_out", "g_x_in", "g_h_in", "e_out", "g_emb"]:
        if k in ref and not (ref[k] is None and r[k] is None):      # g_emb: None on both sides where no block takes the embedding
            assert torch.allclose(r[k], ref[k], rtol=1e-9, atol=1e-11), k
    for k, v in ref["param_grads"].items():
        assert torch.allclose(r["param_grads"][k], v, rtol=1e-8, atol=1e-11), k
    assert set(r["param_grads"]) == set(ref["param_grads"])


@pytest.mark.parametrize("kind", ["updown", "unet", "attn", "uvit"])
def test_stage_central_differences(kind):
    """fp64 central finite differences along random directions, every input and parameter
    tensor, rel err <= 1e-3 (BASELINE.json north_star)."""
    desc = W.mini(kind)
    data = W.draw(desc, seed=2, with_g_e_out=True)
    mb = data["microbatches"][0]

    def loss_of(params, mbx):
        r = O.run_stage(desc, params, mbx)
        L = r["loss"]
        if "g_e_out" in mbx:
            L = L + (r["e_out"] * torch.as_tensor(mbx["g_e_out"], dtype=D)).sum()
        return float(L)

    base = O.run_stage(desc, data["params"], mb)
    rng = np.random.default_rng(0)
    eps = 1e-5
    checks = [("param", k) for k in data["params"]] + [("in", "x_in")] + ([("in", "h_in")] if "h_in" in mb else [])
    for where, k in checks:
        src = data["params"] if where == "param" else mb
        d = rng.standard_normal(src[k].shape)
        d /= np.linalg.norm(d)
        plus, minus = dict(src), dict(src)
        plus[k] = src[k].astype(np.float64) + eps * d
        minus[k] = src[k].astype(np.float64) - eps * d
        if where == "param":
            fd = (loss_of(plus, mb) - loss_of(minus, mb)) / (2 * eps)
            an = float((base["param_grads"][k] * torch.from_numpy(d)).sum())
        else:
            fd = (loss_of(data["params"], plus) - loss_of(data["params"], minus)) / (2 * eps)
            an = float((base["g_" + k] * torch.from_numpy(d)).sum())
        assert abs(fd - an) <= 1e-3 * max(abs(an), abs(fd)) + 1e-9, (k, fd, an)


def test_linearity_and_microbatch_independence():
    desc = W.mini("level")
    data = W.draw(desc, seed=3, with_g_e_out=True)
    mb = data["microbatches"][0]
    r1 = O.run_stage(desc, data["params"], mb, loss_scale=1.0)
    mb2 = dict(mb)
    mb2["g_e_out"] = 2 * mb["g_e_out"]
    r2 = O.run_stage(desc, data["params"], mb2, loss_scale=2.0)
    for k in r1["param_grads"]:
        assert torch.allclose(2 * r1["param_grads"][k], r2["param_grads"][k], rtol=1e-10, atol=1e-12)
    assert torch.allclose(2 * r1["g_x_in"], r2["g_x_in"], rtol=1e-10, atol=1e-12)
    # per-sample independence: sample 0 alone gives the same d_out row (GroupNorm is per sample)
    d1 = W.scaled(desc, n=1)
    mb_s = {k: (v[:1] if k != "t" else v[:1]) for k, v in mb.items()}
    rs = O.run_stage(d1, data["params"], mb_s)
    assert torch.allclose(rs["d_out"][0], r1["d_out"][0], atol=1e-12)
    assert torch.allclose(rs["e_out"][0], r1["e_out"][0], atol=1e-12)


def test_wave_equals_per_microbatch_and_peak():
    desc = W.mini("wave")
    data = W.draw(desc, seed=4)
    wave = O.run_wave(desc, data["params"], data["microbatches"])
    M = desc["microbatches"]
    acc = {}
    for mb in data["microbatches"]:
        r = NA.run(desc, data["params"], mb, loss_scale=1.0 / M)
        for k, v in r["param_grads"].items():
            acc[k] = v if k not in acc else acc[k] + v
    for k in acc:
        assert torch.allclose(wave["param_grads"][k], acc[k], rtol=1e-8, atol=1e-11), k
    per = sum(c * h * w for c, h, w in W.skip_channels_pushed(desc)) * desc["n"]
    assert wave["skip_elements_per_mb"] == per and wave["peak_skip_elements"] == per * M


def test_skip_cache_bytes_closed_forms():
    """tests/golden/skip_cache_bytes.txt: closed forms of BASELINE.md sec. 4 / SURVEY App. A."""
    import os
    want = {}
    with open(os.path.join(os.path.dirname(__file__), "golden", "skip_cache_bytes.txt")) as f:
        for line in f:
            if line.strip() and not line.startswith("#"):
                k, v = line.split()
                want[int(k)] = float(v)
    for i in range(1, 6):
        desc = W.config(i)
        elem = sum(c * h * w for c, h, w in W.skip_channels_pushed(desc)) * desc["n"]
        nbytes = elem * (4 if desc["dtype"] == "fp32" else 2) * desc["microbatches"]
        assert nbytes / 2 ** 20 == want[i], (i, nbytes / 2 ** 20)
    assert len(W.skip_channels_pushed(W.config(4))) == 12      # configs[3]: "12 skip connections"
    assert len(W.skip_channels_pushed(W.config(5))) == 9


def test_boundary_traffic_has_no_skip_bytes():
    """PULSE moves 2(D-1)a per microbatch - only stage outputs cross; the
    skip tensors of a collocated stage never appear among its boundary tensors."""
    for i in (2, 3):
        desc = W.config(i)
        assert set(W.boundary_shapes(desc)) == {"x_in", "h_in", "e_out", "d_out"}


# ------------------------------------------------------------------ the oracle's second instantiations
# (a) storage-precision mode (stored_in / st): DESIGN.md "Store points".  (b) the float32 instantiation that the
# GPU parity tests of configs 3-5 compare with (the exact-mode pins above all run at float64).

def _store_point_count(desc):
    """Closed form of DESIGN.md "Store points": tensors written between operators per microbatch.
    ResBlock forward a1, h1, a2, out (+ shortcut output) and backward g_a2, g_h1, g_a1 (+ shortcut input gradient)
    = 7 (+ 2); its input gradient is one stored write (encoder / mid) or two (decoder: g_h and g_skip);
    conv_in / down: out, g_in = 2; up: out, g_u, g_in = 3; head: a, out, g_a, g_in = 4; the loss gradient g_d = 1."""
    n = 1
    for phase in ("enc_ops", "mid_ops", "dec_ops"):
        for op in desc[phase]:
            if op["kind"] == "resblock":
                sc = (op["cin"] + op["skip"]) != op["cout"]
                n += 7 + (2 if sc else 0) + (2 if phase == "dec_ops" else 1)
            elif op["kind"] in ("conv_in", "down"):
                n += 2
            elif op["kind"] == "up":
                n += 3
            elif op["kind"] == "head":
                n += 4
            elif op["kind"] == "attn":
                n += 8          # xn, qkv, o, out; g_o, g_qkv, g_xn; the input gradient
            elif op["kind"] == "tblock":
                # l1, qkv, o, x1, l2, f1, g, out; g_g, g_f1, g_l2, g_x1, g_o, g_qkv, g_l1; the input gradient
                # with a long skip: xs forward, g_xs backward, and a second input-gradient write (g_skip)
                n += 16 + (3 if op["skip"] else 0)
    return n


@pytest.mark.parametrize("kind", KINDS)
def test_stored_in_store_points(kind, monkeypatch):
    desc = W.mini(kind)
    data = W.draw(desc, seed=6, with_g_e_out=True)
    mb = data["microbatches"][0]
    exact = O.run_stage(desc, data["params"], mb)
    # storing in the compute dtype rounds nothing: bit-for-bit the plain definition
    with O.stored_in(torch.float64):
        same = O.run_stage(desc, data["params"], mb)
    for k in ["loss", "d_out", "g_x_in", "g_h_in", "e_out", "g_emb"]:
        if exact.get(k) is not None:
            assert torch.equal(torch.as_tensor(exact[k]), torch.as_tensor(same[k])), k
    for k, v in exact["param_grads"].items():
        assert torch.equal(v, same["param_grads"][k]), k
    # the number of st() applications is the closed form of the "Store points" table
    calls = []
    real_st = O.st
    monkeypatch.setattr(O, "st", lambda x: (calls.append(1), real_st(x))[1])
    with O.stored_in(torch.bfloat16):
        q = O.run_stage(desc, data["params"], mb)
    assert len(calls) == _store_point_count(desc), (len(calls), _store_point_count(desc))
    # every boundary activation / gradient the stage hands out has been stored: it lies on the bf16 grid
    for k in ["d_out", "e_out", "g_x_in", "g_h_in"]:
        if q.get(k) is not None:
            assert torch.equal(q[k].to(torch.bfloat16).to(D), q[k]), k
    # statistics, weight gradients and the timestep path are NOT stored in bf16 (fp32 accumulate, north_star)
    assert any(not torch.equal(v.to(torch.bfloat16).to(D), v) for v in q["param_grads"].values())
    assert q["g_emb"] is None or not torch.equal(q["g_emb"].to(torch.bfloat16).to(D), q["g_emb"])
    # and the rounded run stays a small perturbation of the exact one (<= 2^-8 relative per store point)
    rms = float(exact["d_out"].pow(2).mean().sqrt())
    assert 0 < float((q["d_out"] - exact["d_out"]).abs().max()) < 0.05 * rms


def test_st_is_round_to_nearest_even_and_idempotent():
    x = torch.tensor([1.0, 1.0 + 2.0 ** -8, 1.0 + 2.0 ** -7, 1.0 + 3 * 2.0 ** -8, -3.3, 1e-3, 70000.0], dtype=D)
    assert torch.equal(O.st(x), x)                                   # outside the context: nothing is rounded
    with O.stored_in(torch.bfloat16):
        y = O.st(x)
        assert torch.equal(O.st(y), y)                               # idempotent
    # bf16 has 8 significand bits: spacing 2^-7 in [1, 2); ties go to the even neighbour
    assert y[0].item() == 1.0 and y[1].item() == 1.0 and y[2].item() == 1.0 + 2.0 ** -7
    assert y[3].item() == 1.0 + 2.0 ** -6
    assert torch.equal(y, torch.from_numpy(W.to_bf16_grid(x.numpy().astype(np.float32))).to(D))   # == the input recipe's grid
    assert ((y - x).abs() <= x.abs() * 2.0 ** -8 + 1e-300).all()     # relative rounding error <= 2^-8 (half a spacing)


@pytest.mark.parametrize("kind", KINDS + ["wave"])
def test_float32_instantiation_matches_float64(kind):
    """The float32 oracle (used for configs 3-5 on the GPU box to bound the test time) against the pinned float64
    one: max |err| <= 5e-5 x RMS per tensor (measured <= 3.6e-5 on these structures: fp32 rounding 6e-8 through 40-100
    operators in series with sums of 10^2-10^3 terms), three orders below the bf16 bar it serves and below north_star's own
    1e-4 bar for an fp32 evaluation of the stage."""
    desc = W.mini(kind)
    data = W.draw(desc, seed=7, with_g_e_out=True)

    def run(dtype):
        if desc["microbatches"] == 1:
            r = O.run_stage(desc, data["params"], data["microbatches"][0], 1.0, dtype)
            per, grads = [r], r["param_grads"]
        else:
            w = O.run_wave(desc, data["params"], data["microbatches"], dtype)
            per, grads = w["per_mb"], w["param_grads"]
        out = {"grad." + k: v for k, v in grads.items()}
        for m, r in enumerate(per):
            for k in ["loss", "d_out", "e_out", "g_x_in", "g_h_in", "emb", "g_emb"]:
                if r.get(k) is not None:
                    out[f"mb{m}.{k}"] = torch.as_tensor(r[k]).reshape(-1)
        return out

    a, b = run(torch.float64), run(torch.float32)
    assert set(a) == set(b)
    for k, v in a.items():
        assert b[k].dtype == torch.float32, k
        rms = max(float(v.pow(2).mean().sqrt()), 1e-30)
        assert float((b[k].to(D) - v).abs().max()) <= 5e-5 * rms, (k, float((b[k].to(D) - v).abs().max()) / rms)


def test_one_bf16_store_of_a_config2_tensor_is_at_the_bar():
    """Why tests/golden/bf16_floor.json exists: north_star's bf16 bar is max|err| <= 2e-2 x RMS per
    tensor.  ONE round-to-nearest bf16 store of an N(0,1) tensor of configs[1]'s size (4 x 320 x 64 x 64 = 5.2 M
    elements, max |x| = 5.9 sigma) already has max|err| = 1.6e-2 x RMS: 2^-9..2^-8 relative at the largest element.
    Two stores in series pass the bar; a stage output has 20-100 in series."""
    g = torch.Generator().manual_seed(0)
    x = torch.randn(4 * 320 * 64 * 64, generator=g, dtype=D)
    rms = float(x.pow(2).mean().sqrt())
    with O.stored_in(torch.bfloat16):
        e1 = float((O.st(x) - x).abs().max()) / rms
        y = O.st(O.st(x) * 1.3371) / 1.3371            # a second store after any operator that moves the grid
        e2 = float((y - x).abs().max()) / rms
    assert 1.4e-2 < e1 <= 2.0 ** -8 * float(x.abs().max()) / rms
    assert e2 > 2e-2


# ------------------------------------------------------------------ attention

def test_attention_core_matches_brute_force_and_closed_forms():
    B_, T, d = 3, 7, 5
    q, k, v = rnd(B_, T, d), rnd(B_, T, d), rnd(B_, T, d)
    o, p = O.attn_core_fwd(q, k, v)
    # the definition as loops: o[b,i] = sum_j softmax_j(q_i . k_j / sqrt(d)) v_j
    want = torch.zeros(B_, T, d, dtype=D)
    for b, i in itertools.product(range(B_), range(T)):
        e = [math.exp(sum(q[b, i, c].item() * k[b, j, c].item() for c in range(d)) / math.sqrt(d)) for j in range(T)]
        z = sum(e)
        for j in range(T):
            want[b, i] += (e[j] / z) * v[b, j]
    assert torch.allclose(o, want, atol=1e-12)
    assert torch.allclose(p.sum(2), torch.ones(B_, T, dtype=D), atol=1e-14) and (p > 0).all()       # rows sum to 1
    # permuting keys and values together changes nothing; permuting queries permutes the output rows
    perm = torch.randperm(T)
    assert torch.allclose(O.attn_core_fwd(q, k[:, perm], v[:, perm])[0], o, atol=1e-12)
    assert torch.allclose(O.attn_core_fwd(q[:, perm], k, v)[0], o[:, perm], atol=1e-12)
    # equal keys -> uniform weights -> the mean of v; one dominant key -> its value
    ku = k[:, :1].expand(B_, T, d)
    assert torch.allclose(O.attn_core_fwd(q, ku, v)[0], v.mean(1, keepdim=True).expand(B_, T, d), atol=1e-12)
    kb = torch.zeros(B_, T, d, dtype=D)
    kb[:, 2] = 200.0 * torch.sign(q[:, 0])                   # query 0 sees key 2 with score >> all others
    assert torch.allclose(O.attn_core_fwd(q, kb, v)[0][:, 0], v[:, 2], atol=1e-9)
    # shift invariance of softmax: adding a constant vector to every key's score (q . c) changes nothing
    assert torch.allclose(O.attn_core_fwd(q, k + 3.0, v)[0], o, atol=1e-10)
    # the library routine
    assert torch.allclose(o, torch.nn.functional.scaled_dot_product_attention(q, k, v), atol=1e-12)


def test_attention_core_backward_finite_differences_and_autograd():
    B_, T, d = 2, 6, 4
    q, k, v, g = rnd(B_, T, d), rnd(B_, T, d), rnd(B_, T, d), rnd(B_, T, d)
    o, p = O.attn_core_fwd(q, k, v)
    g_q, g_k, g_v = O.attn_core_bwd(g, q, k, v, p)
    qa, ka, va = (t.clone().requires_grad_(True) for t in (q, k, v))
    (torch.nn.functional.scaled_dot_product_attention(qa, ka, va) * g).sum().backward()
    assert torch.allclose(g_q, qa.grad, atol=1e-11) and torch.allclose(g_k, ka.grad, atol=1e-11)
    assert torch.allclose(g_v, va.grad, atol=1e-11)
    eps = 1e-6
    for name, t, an in (("q", q, g_q), ("k", k, g_k), ("v", v, g_v)):
        dirn = rnd(B_, T, d)
        args = {"q": q, "k": k, "v": v}
        plus, minus = dict(args), dict(args)
        plus[name], minus[name] = t + eps * dirn, t - eps * dirn
        fd = ((O.attn_core_fwd(**plus)[0] - O.attn_core_fwd(**minus)[0]) * g).sum() / (2 * eps)
        assert abs(fd - (an * dirn).sum()) <= 1e-6 * max(1.0, abs(fd)), name
    # softmax Jacobian: the score gradient of every query row sums to zero -> g_q, g_k are invariant to adding a constant to g_P
    assert torch.allclose(O.attn_core_bwd(g, q, k, v, p)[0], g_q)


def test_plain_groupnorm_matches_library_autograd():
    n, c, G, eps = 2, 12, 4, 1e-5
    x, gamma, beta, g_y = rnd(n, c, 3, 5) * 2 + 1, rnd(c), rnd(c), rnd(n, c, 3, 5)
    y, ctx = O.gn_fwd(x, gamma, beta, G, eps)
    g_x, dg, db = O.gn_bwd(g_y, ctx, gamma)
    xr, gr, br = (t.clone().requires_grad_(True) for t in (x, gamma, beta))
    yr = torch.nn.functional.group_norm(xr, G, gr, br, eps)
    yr.backward(g_y)
    assert torch.allclose(y, yr.detach(), atol=1e-12) and torch.allclose(g_x, xr.grad, atol=1e-10)
    assert torch.allclose(dg, gr.grad, atol=1e-10) and torch.allclose(db, br.grad, atol=1e-10)
    # same statistics as the fused GroupNorm + SiLU: a = SiLU(y)
    a, _ = O.gn_silu_fwd(x, gamma, beta, G, eps)
    assert torch.allclose(a, O.silu(y), atol=1e-12)


def test_attention_heads_layout():
    """Head h owns channels [h d, (h+1) d); tokens are pixels in row-major order (reading R24)."""
    n, heads, d, h, w = 2, 3, 4, 2, 5
    x = rnd(n, heads * d, h, w)
    t = O._heads(x, heads)
    assert t.shape == (n * heads, h * w, d)
    assert torch.equal(t[1 * heads + 2, 1 * w + 3], x[1, 2 * d:3 * d, 1, 3])
    assert torch.equal(O._unheads(t, n, heads, h, w), x)


# ------------------------------------------------------------------ transformer block pieces

def test_layernorm_and_gelu_match_library_and_closed_forms():
    n, c = 2, 10
    x, gamma, beta, g_y = rnd(n, c, 3, 4) * 2 + 1, rnd(c), rnd(c), rnd(n, c, 3, 4)
    y, ctx = O.ln_fwd(x, gamma, beta, 1e-5)
    g_x, dg, db = O.ln_bwd(g_y, ctx, gamma)
    xr, gr, br = (t.clone().requires_grad_(True) for t in (x, gamma, beta))
    yr = torch.nn.functional.layer_norm(xr.permute(0, 2, 3, 1), (c,), gr, br, 1e-5).permute(0, 3, 1, 2)
    yr.backward(g_y)
    assert torch.allclose(y, yr.detach(), atol=1e-12) and torch.allclose(g_x, xr.grad, atol=1e-10)
    assert torch.allclose(dg, gr.grad, atol=1e-10) and torch.allclose(db, br.grad, atol=1e-10)
    # per token: mean 0, variance var / (var + eps) before the affine; the input gradient sums to zero over the channels
    assert ctx["xhat"].mean(1).abs().max() < 1e-12 and g_x.sum(1).abs().max() < 1e-10
    # GELU: x Phi(x); GELU(0) = 0, GELU'(0) = 1/2, GELU(x) -> x, GELU(-x) -> 0; the library's erf form; finite differences
    z = torch.zeros(1, dtype=D)
    assert O.gelu(z).item() == 0.0 and O.gelu_grad(z).item() == 0.5
    big = torch.tensor([12.0], dtype=D)
    assert abs(O.gelu(big).item() - 12.0) < 1e-12 and abs(O.gelu(-big).item()) < 1e-12
    assert abs(O.gelu(torch.tensor([1.0], dtype=D)).item() - 0.8413447460685429) < 1e-12      # Phi(1)
    t = rnd(50)
    assert torch.allclose(O.gelu(t), torch.nn.functional.gelu(t), atol=1e-12)
    assert torch.allclose(O.gelu_grad(t), (O.gelu(t + 1e-6) - O.gelu(t - 1e-6)) / 2e-6, atol=1e-8)


def test_long_skip_is_concat_then_linear():
    """the long skip of a transformer stage is concat + Linear: with the Linear = [I | 0] the block ignores
    the skip, with [0 | I] it runs on the skip instead of on h."""
    desc = W.mini("uvit")
    data = W.draw(desc, seed=8)
    P = {k: torch.as_tensor(v, dtype=D) for k, v in data["params"].items()}
    x, sk = rnd(2, 16, 4, 4), rnd(2, 16, 4, 4)
    eye = torch.eye(16, dtype=D)
    Pa = dict(P); Pa["dec0.skip.w"] = torch.cat([eye, torch.zeros(16, 16, dtype=D)], 1)[:, :, None, None]; Pa["dec0.skip.b"] = torch.zeros(16, dtype=D)
    Pb = dict(P); Pb["dec0.skip.w"] = torch.cat([torch.zeros(16, 16, dtype=D), eye], 1)[:, :, None, None]; Pb["dec0.skip.b"] = torch.zeros(16, dtype=D)
    Pn = {k.replace("dec0.", "enc0."): v for k, v in P.items() if k.startswith("dec0.") and "skip" not in k}
    base_x, _ = O.tblock_fwd(Pn, "enc0.", x, None, 1e-5, 2)
    base_s, _ = O.tblock_fwd(Pn, "enc0.", sk, None, 1e-5, 2)
    assert torch.allclose(O.tblock_fwd(Pa, "dec0.", x, sk, 1e-5, 2)[0], base_x, atol=1e-12)
    assert torch.allclose(O.tblock_fwd(Pb, "dec0.", x, sk, 1e-5, 2)[0], base_s, atol=1e-12)
