"""CPU oracle for one PULSE skip-local (collocated) UNet stage.  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
legs may import this file.  It shares no code with the CUDA path and never imports
it.  Plain PyTorch CPU ops, fp64 by default (fp32 selectable for the two largest
configs).

What it follows
  * PAPER.md:L91 (sec. III): "we allocate local buffers for skip activations and their
    gradients.  Skip activations are stored locally during the forward pass, and
    these values are retrieved for gradient computation in the backward pass."
  * PAPER.md:L142 (sec. IV-B): the model is a linear sequence of operations whose
    I/O carries "an additional field for storing skip connections".
  * PAPER.md:L49 (sec. II-A): "Each block contains Attention and ResNet layers"; the
    inside of a ResNet layer is not in the paper; BASELINE.json north_star fixes it
    (GroupNorm, SiLU, timestep-embedding add, 3x3 conv, residual add, concat with the
    cached skip) and SURVEY.md 8c items 1-7 / readings R1-R20 give the formulas.
Because the stage is an exact reformulation (fusion, virtual concat, caching), the
oracle is the plain definition: materialise the concat, run ops one at a time on
[N,C,H,W] tensors, keep every intermediate, back-propagate by the chain rule written
out below (no autograd anywhere in this file).

Library primitives used as single steps: conv2d / conv_transpose2d / conv2d_weight
(cross-correlation, its adjoint in the input and in the weight), matmul.  They are
pinned in tests/test_oracle_pins.py against brute-force direct sums, adjoint
identities, closed forms and fp64 central differences.  The two further instantiations
are pinned there as well: the float32 one (configs 3-5 on the GPU box) against the float64
one, and the storage-precision mode `stored_in` / `st` (bit-identical to the exact mode
when storing in the compute dtype, number of store points = the closed form of DESIGN.md
"Store points", round-to-nearest-even, idempotent).  Parity status: pinned (no function
here is "parity unpinned").
"""
from __future__ import annotations

import math
import torch
import torch.nn.functional as F

DT = torch.float64


# --------------------------------------------------------------------------- elementary pieces

def sigmoid(y):
    return 1.0 / (1.0 + torch.exp(-y))


def silu(y):
    """SiLU(y) = y * s(y), s = logistic."""
    return y * sigmoid(y)


def silu_grad(y):
    """d SiLU / dy = s(y) (1 + y (1 - s(y)))."""
    s = sigmoid(y)
    return s * (1.0 + y * (1.0 - s))


def gn_silu_fwd(x, gamma, beta, groups, eps):
    """a = SiLU(gamma * xhat + beta), xhat = (x - mu) r, per (n, group) biased variance,
    r = 1/sqrt(var + eps)  (reading R5)."""
    n, c, h, w = x.shape
    xg = x.reshape(n, groups, -1)
    mu = xg.mean(dim=2, keepdim=True)
    var = ((xg - mu) ** 2).mean(dim=2, keepdim=True)
    r = 1.0 / torch.sqrt(var + eps)
    xhat = ((xg - mu) * r).reshape(n, c, h, w)
    y = gamma.view(1, c, 1, 1) * xhat + beta.view(1, c, 1, 1)
    return silu(y), {"xhat": xhat, "r": r, "y": y, "groups": groups}


def gn_silu_bwd(g_a, ctx, gamma):
    """g_y = g_a SiLU'(y); dgamma = sum g_y xhat; dbeta = sum g_y; q = g_y gamma;
    A = mean_S q; B = mean_S q xhat; g_x = r (q - A - xhat B)."""
    xhat, r, y, groups = ctx["xhat"], ctx["r"], ctx["y"], ctx["groups"]
    n, c, h, w = xhat.shape
    g_y = g_a * silu_grad(y)
    dgamma = (g_y * xhat).sum(dim=(0, 2, 3))
    dbeta = g_y.sum(dim=(0, 2, 3))
    q = (g_y * gamma.view(1, c, 1, 1)).reshape(n, groups, -1)
    xh = xhat.reshape(n, groups, -1)
    A = q.mean(dim=2, keepdim=True)
    B = (q * xh).mean(dim=2, keepdim=True)
    g_x = (r * (q - A - xh * B)).reshape(n, c, h, w)
    return g_x, dgamma, dbeta


def conv_fwd(x, w, b, stride=1):
    """out[n,co,y,x] = b[co] + sum_{ci,r,s} W[co,ci,r,s] in[n,ci,y st+r-pad,x st+s-pad],
    zero outside, pad = (k-1)/2."""
    return F.conv2d(x, w, b, stride=stride, padding=(w.shape[-1] - 1) // 2)


def conv_dgrad(g, w, in_hw, stride=1):
    """Adjoint of conv_fwd in its input (scatter of the same sum)."""
    pad = (w.shape[-1] - 1) // 2
    k = w.shape[-1]
    oph = in_hw[0] - ((g.shape[2] - 1) * stride - 2 * pad + k)
    opw = in_hw[1] - ((g.shape[3] - 1) * stride - 2 * pad + k)
    return F.conv_transpose2d(g, w, None, stride=stride, padding=pad, output_padding=(oph, opw))


def conv_wgrad(x, g, w_shape, stride=1):
    """dW[co,ci,r,s] = sum_{n,y,x} g[n,co,y,x] in[n,ci,y st+r-pad,x st+s-pad]; db = sum g."""
    pad = (w_shape[-1] - 1) // 2
    dw = torch.nn.grad.conv2d_weight(x, w_shape, g, stride=stride, padding=pad)
    return dw, g.sum(dim=(0, 2, 3))


def upsample2(d):
    """u[n,c,Y,X] = d[n,c,Y//2,X//2]."""
    return d.repeat_interleave(2, dim=2).repeat_interleave(2, dim=3)


def upsample2_bwd(g_u):
    """g_d[y,x] = sum_{i,j in {0,1}} g_u[2y+i, 2x+j]."""
    n, c, h, w = g_u.shape
    return g_u.reshape(n, c, h // 2, 2, w // 2, 2).sum(dim=(3, 5))


# --------------------------------------------------------------------------- attention

def gn_fwd(x, gamma, beta, groups, eps):
    """Plain GroupNorm (no activation): y = gamma xhat + beta, statistics as in gn_silu_fwd."""
    n, c, h, w = x.shape
    xg = x.reshape(n, groups, -1)
    mu = xg.mean(dim=2, keepdim=True)
    var = ((xg - mu) ** 2).mean(dim=2, keepdim=True)
    r = 1.0 / torch.sqrt(var + eps)
    xhat = ((xg - mu) * r).reshape(n, c, h, w)
    return gamma.view(1, c, 1, 1) * xhat + beta.view(1, c, 1, 1), {"xhat": xhat, "r": r, "groups": groups}


def gn_bwd(g_y, ctx, gamma):
    """dgamma = sum g_y xhat; dbeta = sum g_y; q = g_y gamma; g_x = r (q - mean_S q - xhat mean_S (q xhat))."""
    xhat, r, groups = ctx["xhat"], ctx["r"], ctx["groups"]
    n, c, h, w = xhat.shape
    dgamma = (g_y * xhat).sum(dim=(0, 2, 3))
    dbeta = g_y.sum(dim=(0, 2, 3))
    q = (g_y * gamma.view(1, c, 1, 1)).reshape(n, groups, -1)
    xh = xhat.reshape(n, groups, -1)
    g_x = (r * (q - q.mean(dim=2, keepdim=True) - xh * (q * xh).mean(dim=2, keepdim=True))).reshape(n, c, h, w)
    return g_x, dgamma, dbeta


def attn_core_fwd(q, k, v):
    """Scaled dot-product attention, the plain definition: q, k, v [B, T, d] (B = samples x heads, T tokens);
    S = q k^T / sqrt(d); P = softmax over keys (each row of P sums to 1); o = P v."""
    d = q.shape[-1]
    s = q @ k.transpose(1, 2) / math.sqrt(d)
    p = torch.exp(s - s.max(dim=2, keepdim=True).values)
    p = p / p.sum(dim=2, keepdim=True)
    return p @ v, p


def attn_core_bwd(g_o, q, k, v, p):
    """g_v = P^T g_o; g_P = g_o v^T; g_S = P (g_P - rowsum(P g_P))  (softmax Jacobian); g_q = g_S k / sqrt(d);
    g_k = g_S^T q / sqrt(d)."""
    d = q.shape[-1]
    g_v = p.transpose(1, 2) @ g_o
    g_p = g_o @ v.transpose(1, 2)
    g_s = p * (g_p - (p * g_p).sum(dim=2, keepdim=True))
    return g_s @ k / math.sqrt(d), g_s.transpose(1, 2) @ q / math.sqrt(d), g_v


def _heads(t, heads):
    """[N, C, H, W] -> [N heads, H W, C / heads]: head h owns channels [h d, (h+1) d), tokens are pixels in row-major order."""
    n, c, h, w = t.shape
    return t.reshape(n, heads, c // heads, h * w).permute(0, 1, 3, 2).reshape(n * heads, h * w, c // heads)


def _unheads(t, n, heads, h, w):
    d = t.shape[-1]
    return t.reshape(n, heads, h * w, d).permute(0, 1, 3, 2).reshape(n, heads * d, h, w)


def attn_block_fwd(P, p, x, groups, eps, heads):
    """Self-attention block of a UNet level ("Each block contains Attention and ResNet layers"; the inside
    is not in the paper: reading R24, the SD form): xn = GN(x); [q|k|v] = conv1x1(xn) (C -> 3C); o = attention per head
    over the H W pixels; out = x + conv1x1(o).  st() marks the stored tensors."""
    n, c, h, w = x.shape
    xn, cg = gn_fwd(x, P[p + "gn.gamma"], P[p + "gn.beta"], groups, eps)
    xn = st(xn)
    qkv = st(conv_fwd(xn, P[p + "qkv.w"], P[p + "qkv.b"]))
    q, k, v = (_heads(qkv[:, i * c:(i + 1) * c], heads) for i in range(3))
    o, pr = attn_core_fwd(q, k, v)
    o = st(_unheads(o, n, heads, h, w))
    out = st(conv_fwd(o, P[p + "proj.w"], P[p + "proj.b"]) + x)
    return out, {"x": x, "xn": xn, "cg": cg, "qkv": qkv, "q": q, "k": k, "v": v, "p": pr, "o": o, "heads": heads}


def attn_block_bwd(P, p, ctx, g_out, G):
    """Chain rule of attn_block_fwd; adds parameter grads into G, returns g_x before it is stored."""
    x, heads = ctx["x"], ctx["heads"]
    n, c, h, w = x.shape
    G[p + "proj.w"], G[p + "proj.b"] = conv_wgrad(ctx["o"], g_out, P[p + "proj.w"].shape)
    g_o = st(conv_dgrad(g_out, P[p + "proj.w"], (h, w)))
    g_q, g_k, g_v = attn_core_bwd(_heads(g_o, heads), ctx["q"], ctx["k"], ctx["v"], ctx["p"])
    g_qkv = st(torch.cat([_unheads(t, n, heads, h, w) for t in (g_q, g_k, g_v)], dim=1))
    G[p + "qkv.w"], G[p + "qkv.b"] = conv_wgrad(ctx["xn"], g_qkv, P[p + "qkv.w"].shape)
    g_xn = st(conv_dgrad(g_qkv, P[p + "qkv.w"], (h, w)))
    g_x, G[p + "gn.gamma"], G[p + "gn.beta"] = gn_bwd(g_xn, ctx["cg"], P[p + "gn.gamma"])
    return g_x + g_out


# --------------------------------------------------------------------------- transformer block with a long skip

def ln_fwd(x, gamma, beta, eps):
    """LayerNorm over the channels of every token (pixel): y = gamma xhat + beta, biased variance, eps inside the sqrt."""
    c = x.shape[1]
    mu = x.mean(dim=1, keepdim=True)
    var = ((x - mu) ** 2).mean(dim=1, keepdim=True)
    r = 1.0 / torch.sqrt(var + eps)
    xhat = (x - mu) * r
    return gamma.view(1, c, 1, 1) * xhat + beta.view(1, c, 1, 1), {"xhat": xhat, "r": r}


def ln_bwd(g_y, ctx, gamma):
    """dgamma = sum g_y xhat; dbeta = sum g_y; q = g_y gamma; g_x = r (q - mean_c q - xhat mean_c (q xhat))."""
    xhat, r = ctx["xhat"], ctx["r"]
    c = xhat.shape[1]
    q = g_y * gamma.view(1, c, 1, 1)
    g_x = r * (q - q.mean(dim=1, keepdim=True) - xhat * (q * xhat).mean(dim=1, keepdim=True))
    return g_x, (g_y * xhat).sum(dim=(0, 2, 3)), g_y.sum(dim=(0, 2, 3))


def gelu(x):
    """GELU(x) = x Phi(x), Phi the standard normal CDF (the exact erf form)."""
    return 0.5 * x * (1.0 + torch.erf(x / math.sqrt(2.0)))


def gelu_grad(x):
    """Phi(x) + x phi(x)."""
    return 0.5 * (1.0 + torch.erf(x / math.sqrt(2.0))) + x * torch.exp(-0.5 * x * x) / math.sqrt(2.0 * math.pi)


def tblock_fwd(P, p, x, skip, eps, heads):
    """Transformer block of a U-ViT / Hunyuan-DiT style stage (long skips between early and late
    transformer blocks; reading R26): tokens are the H W pixels, Linear layers are 1x1 convs.
      xs  = Linear_skip(concat_C(x, skip))      only where a cached skip is consumed ("concat + Linear")
      x1  = xs + proj(attention(qkv(LN1(xs))))
      out = x1 + fc2(GELU(fc1(LN2(x1))))        fc1: C -> 4C
    st() marks the stored tensors."""
    n, _, h, w = x.shape
    xin = x if skip is None else torch.cat([x, skip], dim=1)
    xs = x if skip is None else st(conv_fwd(xin, P[p + "skip.w"], P[p + "skip.b"]))
    c = xs.shape[1]
    l1, c1 = ln_fwd(xs, P[p + "ln1.gamma"], P[p + "ln1.beta"], eps)
    l1 = st(l1)
    qkv = st(conv_fwd(l1, P[p + "qkv.w"], P[p + "qkv.b"]))
    q, k, v = (_heads(qkv[:, i * c:(i + 1) * c], heads) for i in range(3))
    o, pr = attn_core_fwd(q, k, v)
    o = st(_unheads(o, n, heads, h, w))
    x1 = st(conv_fwd(o, P[p + "proj.w"], P[p + "proj.b"]) + xs)
    l2, c2 = ln_fwd(x1, P[p + "ln2.gamma"], P[p + "ln2.beta"], eps)
    l2 = st(l2)
    f1 = st(conv_fwd(l2, P[p + "fc1.w"], P[p + "fc1.b"]))
    g = st(gelu(f1))
    out = st(conv_fwd(g, P[p + "fc2.w"], P[p + "fc2.b"]) + x1)
    return out, {"xin": xin, "has_skip": skip is not None, "xs": xs, "c1": c1, "l1": l1, "q": q, "k": k, "v": v, "p": pr,
                 "o": o, "x1": x1, "c2": c2, "l2": l2, "f1": f1, "g": g, "heads": heads, "ch": x.shape[1]}


def tblock_bwd(P, p, ctx, g_out, G):
    """Chain rule of tblock_fwd; adds parameter grads into G; returns the gradient of the block's input before it is
    stored (of concat_C(x, skip) where a skip was consumed)."""
    heads = ctx["heads"]
    n, c, h, w = ctx["xs"].shape
    hw = (h, w)
    G[p + "fc2.w"], G[p + "fc2.b"] = conv_wgrad(ctx["g"], g_out, P[p + "fc2.w"].shape)
    g_g = st(conv_dgrad(g_out, P[p + "fc2.w"], hw))
    g_f1 = st(g_g * gelu_grad(ctx["f1"]))
    G[p + "fc1.w"], G[p + "fc1.b"] = conv_wgrad(ctx["l2"], g_f1, P[p + "fc1.w"].shape)
    g_l2 = st(conv_dgrad(g_f1, P[p + "fc1.w"], hw))
    g_x1, G[p + "ln2.gamma"], G[p + "ln2.beta"] = ln_bwd(g_l2, ctx["c2"], P[p + "ln2.gamma"])
    g_x1 = st(g_x1 + g_out)
    G[p + "proj.w"], G[p + "proj.b"] = conv_wgrad(ctx["o"], g_x1, P[p + "proj.w"].shape)
    g_o = st(conv_dgrad(g_x1, P[p + "proj.w"], hw))
    g_q, g_k, g_v = attn_core_bwd(_heads(g_o, heads), ctx["q"], ctx["k"], ctx["v"], ctx["p"])
    g_qkv = st(torch.cat([_unheads(t, n, heads, h, w) for t in (g_q, g_k, g_v)], dim=1))
    G[p + "qkv.w"], G[p + "qkv.b"] = conv_wgrad(ctx["l1"], g_qkv, P[p + "qkv.w"].shape)
    g_l1 = st(conv_dgrad(g_qkv, P[p + "qkv.w"], hw))
    g_xs, G[p + "ln1.gamma"], G[p + "ln1.beta"] = ln_bwd(g_l1, ctx["c1"], P[p + "ln1.gamma"])
    g_xs = g_xs + g_x1
    if not ctx["has_skip"]:
        return g_xs
    g_xs = st(g_xs)
    G[p + "skip.w"], G[p + "skip.b"] = conv_wgrad(ctx["xin"], g_xs, P[p + "skip.w"].shape)
    return conv_dgrad(g_xs, P[p + "skip.w"], hw)


# --------------------------------------------------------------------------- time embedding

def sinusoidal(t, d, dtype=DT):
    """emb0[n,i] = cos(t_n f_i), emb0[n,half+i] = sin(t_n f_i), f_i = exp(-ln(10000) i/half)
    (reading R15)."""
    half = d // 2
    f = torch.exp(-math.log(10000.0) * torch.arange(half, dtype=dtype) / half)
    a = t.to(dtype).view(-1, 1) * f.view(1, -1)
    return torch.cat([torch.cos(a), torch.sin(a)], dim=1)


def temb_fwd(desc, P, t, dtype=DT):
    """emb = emb0 (config 1) or W2 SiLU(W1 emb0 + b1) + b2 (configs 2-5)."""
    emb0 = sinusoidal(t, desc["temb"]["d0"], dtype)
    if desc["temb"]["kind"] == "sinusoidal":
        return emb0, {"emb0": emb0}
    z1 = emb0 @ P["temb.w1"].T + P["temb.b1"]
    emb = silu(z1) @ P["temb.w2"].T + P["temb.b2"]
    return emb, {"emb0": emb0, "z1": z1}


def temb_bwd(desc, P, ctx, g_emb):
    grads = {}
    if desc["temb"]["kind"] == "sinusoidal":
        return grads
    a1 = silu(ctx["z1"])
    grads["temb.w2"] = g_emb.T @ a1
    grads["temb.b2"] = g_emb.sum(0)
    g_z1 = (g_emb @ P["temb.w2"]) * silu_grad(ctx["z1"])
    grads["temb.w1"] = g_z1.T @ ctx["emb0"]
    grads["temb.b1"] = g_z1.sum(0)
    return grads


# --------------------------------------------------------------------------- storage precision

_STORE = None      # None: exact (every intermediate kept in the compute dtype)


class stored_in:
    """`with stored_in(torch.bfloat16): ...` rounds every tensor the method STORES between
    operators (north_star: "bf16 in with fp32 accumulate": activations, their gradients and
    the skip buffers are bf16 tensors) to that dtype, round-to-nearest-even, at exactly the
    points listed in DESIGN.md "Store points"; sums, statistics, weight gradients and the
    timestep path stay in the compute dtype.  Outside the context nothing is rounded: that
    is the plain definition.  Used by the parity tests to measure the rounding floor of the
    bf16 protocol (reading R18)."""

    def __init__(self, dtype):
        self.dtype = dtype

    def __enter__(self):
        global _STORE
        self.prev, _STORE = _STORE, self.dtype

    def __exit__(self, *a):
        global _STORE
        _STORE = self.prev


def st(x):
    return x if _STORE is None else x.to(_STORE).to(x.dtype)


# --------------------------------------------------------------------------- ResBlock

def resblock_fwd(P, p, x, emb, groups, eps):
    """a1 = SiLU(GN1(x)); h1 = conv1(a1) + pr[n,c]; a2 = SiLU(GN2(h1));
    out = conv2(a2) + sc(x); pr = Wt SiLU(emb) + bt; sc = identity if Cin == Cout else 1x1 conv
    (readings R1, R2).  st() marks the stored tensors."""
    a1, c1 = gn_silu_fwd(x, P[p + "gn1.gamma"], P[p + "gn1.beta"], groups, eps)
    a1 = st(a1)
    pr = silu(emb) @ P[p + "temb.w"].T + P[p + "temb.b"]
    h1 = st(conv_fwd(a1, P[p + "conv1.w"], P[p + "conv1.b"]) + pr[:, :, None, None])
    a2, c2 = gn_silu_fwd(h1, P[p + "gn2.gamma"], P[p + "gn2.beta"], groups, eps)
    a2 = st(a2)
    if (p + "sc.w") in P:
        res = st(conv_fwd(x, P[p + "sc.w"], P[p + "sc.b"]))
    else:
        res = x
    out = st(conv_fwd(a2, P[p + "conv2.w"], P[p + "conv2.b"]) + res)
    return out, {"x": x, "a1": a1, "c1": c1, "h1": h1, "a2": a2, "c2": c2, "emb": emb}


def resblock_bwd(P, p, ctx, g_out, G):
    """Chain rule of resblock_fwd.  Adds parameter grads into G,
    returns (g_x before it is stored, g_emb contribution)."""
    x, emb = ctx["x"], ctx["emb"]
    hw = x.shape[2:]
    G[p + "conv2.w"], G[p + "conv2.b"] = conv_wgrad(ctx["a2"], g_out, P[p + "conv2.w"].shape)
    g_a2 = st(conv_dgrad(g_out, P[p + "conv2.w"], hw))
    g_h1, G[p + "gn2.gamma"], G[p + "gn2.beta"] = gn_silu_bwd(g_a2, ctx["c2"], P[p + "gn2.gamma"])
    g_h1 = st(g_h1)
    g_p = g_h1.sum(dim=(2, 3))
    G[p + "temb.w"] = g_p.T @ silu(emb)
    G[p + "temb.b"] = g_p.sum(0)
    g_emb = (g_p @ P[p + "temb.w"]) * silu_grad(emb)
    G[p + "conv1.w"], G[p + "conv1.b"] = conv_wgrad(ctx["a1"], g_h1, P[p + "conv1.w"].shape)
    g_a1 = st(conv_dgrad(g_h1, P[p + "conv1.w"], hw))
    g_x, G[p + "gn1.gamma"], G[p + "gn1.beta"] = gn_silu_bwd(g_a1, ctx["c1"], P[p + "gn1.gamma"])
    if (p + "sc.w") in P:
        G[p + "sc.w"], G[p + "sc.b"] = conv_wgrad(x, g_out, P[p + "sc.w"].shape)
        g_x = g_x + st(conv_dgrad(g_out, P[p + "sc.w"], hw))
    else:
        g_x = g_x + g_out
    return g_x, g_emb


# --------------------------------------------------------------------------- the collocated stage

def stage_forward(desc, P, x_in, h_in, emb):
    """Encoder ops then (closed: mid ops) then decoder ops of one collocated stage.
    Pushed encoder outputs go to the local skip buffers `skips`; each
    decoder ResBlock pops the most recent one (LIFO, reading R7) and runs on the
    materialised concat [h, skip] along C, h first (reading R6)."""
    G_, eps = desc["groups"], desc["eps"]
    skips, tape = [], {"enc": [], "mid": [], "dec": []}
    x = x_in
    if desc["x_in_is_skip"]:
        skips.append((("e", -1), x))
    for i, op in enumerate(desc["enc_ops"]):
        p = f"enc{i}."
        if op["kind"] == "resblock":
            x, c = resblock_fwd(P, p, x, emb, G_, eps)
        elif op["kind"] == "attn":
            x, c = attn_block_fwd(P, p, x, G_, eps, op["heads"])
        elif op["kind"] == "tblock":
            x, c = tblock_fwd(P, p, x, None, eps, op["heads"])
        elif op["kind"] in ("conv_in", "down"):
            s = 2 if op["kind"] == "down" else 1
            c = {"x": x, "stride": s}
            x = st(conv_fwd(x, P[p + "conv.w"], P[p + "conv.b"], stride=s))
        else:
            raise ValueError(op["kind"])
        c["out_shape"] = x.shape
        if op["push"]:
            skips.append((("e", i), x))
        tape["enc"].append(c)
    skip_list = [s for _, s in skips]          # what the skip cache holds, in push order
    outs = {}
    if desc["link"] == "closed":
        h = x
        for i, op in enumerate(desc["mid_ops"]):
            if op["kind"] == "attn":
                h, c = attn_block_fwd(P, f"mid{i}.", h, G_, eps, op["heads"])
            else:
                h, c = resblock_fwd(P, f"mid{i}.", h, emb, G_, eps)
            tape["mid"].append(c)
    else:
        outs["e_out"] = x
        h = h_in
    for i, op in enumerate(desc["dec_ops"]):
        p = f"dec{i}."
        if op["kind"] == "resblock":
            key, s = skips.pop()
            assert s.shape[1] == op["skip"] and h.shape[1] == op["cin"], (p, s.shape, h.shape)
            h, c = resblock_fwd(P, p, torch.cat([h, s], dim=1), emb, G_, eps)
            c["pop"], c["ch"] = key, op["cin"]
        elif op["kind"] == "attn":
            h, c = attn_block_fwd(P, p, h, G_, eps, op["heads"])
        elif op["kind"] == "tblock":
            sk = None
            if op["skip"]:
                key, sk = skips.pop()
                assert sk.shape[1] == op["skip"] and h.shape[1] == op["cin"], (p, sk.shape, h.shape)
            h, c = tblock_fwd(P, p, h, sk, eps, op["heads"])
            if op["skip"]:
                c["pop"] = key
        elif op["kind"] == "up":
            u = upsample2(h)
            c = {"u": u}
            h = st(conv_fwd(u, P[p + "conv.w"], P[p + "conv.b"]))
        elif op["kind"] == "head":
            a, cg = gn_silu_fwd(h, P[p + "gn.gamma"], P[p + "gn.beta"], G_, eps)
            a = st(a)
            c = {"a": a, "cg": cg}
            h = st(conv_fwd(a, P[p + "conv.w"], P[p + "conv.b"]))
        else:
            raise ValueError(op["kind"])
        tape["dec"].append(c)
    assert not skips, "every cached skip is consumed exactly once"
    outs["d_out"] = h
    return outs, {"tape": tape, "skips": skip_list}


def stage_backward(desc, P, ctx, g_d_out, g_e_out=None):
    """Reverse of stage_forward.  `gbuf` holds one gradient buffer per tensor of the stage
    ("local buffers for skip activations and their gradients"): a decoder
    ResBlock's input gradient is split into g_h and g_skip, g_skip goes into the buffer of
    the encoder output it popped, and that buffer also receives the gradient from the
    tensor's encoder-chain consumer.  Each write stores (st); a second
    write into a buffer adds to the stored value, in the order the stage runs them
    (decoder first, then mid, then encoder, last to first)."""
    tape = ctx["tape"]
    G, g_emb, gbuf = {}, None, {}
    n_enc, n_mid, n_dec = len(desc["enc_ops"]), len(desc["mid_ops"]), len(desc["dec_ops"])

    def acc(key, v):
        gbuf[key] = st(v) if key not in gbuf else st(gbuf[key] + v)

    def add_emb(ge):
        nonlocal g_emb
        g_emb = ge if g_emb is None else g_emb + ge

    last_enc = ("e", n_enc - 1)
    closed = desc["link"] == "closed"
    dec_in0 = (("m", n_mid - 1) if n_mid else last_enc) if closed else ("hin",)
    gbuf[("d", n_dec - 1) if n_dec else dec_in0] = g_d_out
    if not closed and g_e_out is not None:
        gbuf[last_enc] = g_e_out
    for i in reversed(range(n_dec)):
        op, c, p = desc["dec_ops"][i], tape["dec"][i], f"dec{i}."
        g, kin = gbuf[("d", i)], (("d", i - 1) if i else dec_in0)
        if op["kind"] == "resblock":
            g_x, ge = resblock_bwd(P, p, c, g, G)
            add_emb(ge)
            acc(kin, g_x[:, :c["ch"]])
            acc(c["pop"], g_x[:, c["ch"]:])
        elif op["kind"] == "attn":
            acc(kin, attn_block_bwd(P, p, c, g, G))
        elif op["kind"] == "tblock":
            g_x = tblock_bwd(P, p, c, g, G)
            acc(kin, g_x[:, :c["ch"]])
            if c["has_skip"]:
                acc(c["pop"], g_x[:, c["ch"]:])
        elif op["kind"] == "up":
            G[p + "conv.w"], G[p + "conv.b"] = conv_wgrad(c["u"], g, P[p + "conv.w"].shape)
            acc(kin, upsample2_bwd(st(conv_dgrad(g, P[p + "conv.w"], c["u"].shape[2:]))))
        elif op["kind"] == "head":
            G[p + "conv.w"], G[p + "conv.b"] = conv_wgrad(c["a"], g, P[p + "conv.w"].shape)
            g_a = st(conv_dgrad(g, P[p + "conv.w"], c["a"].shape[2:]))
            g_x, G[p + "gn.gamma"], G[p + "gn.beta"] = gn_silu_bwd(g_a, c["cg"], P[p + "gn.gamma"])
            acc(kin, g_x)
    grads_out = {}
    if closed:
        for i in reversed(range(n_mid)):
            if desc["mid_ops"][i]["kind"] == "attn":
                g_x = attn_block_bwd(P, f"mid{i}.", tape["mid"][i], gbuf[("m", i)], G)
            else:
                g_x, ge = resblock_bwd(P, f"mid{i}.", tape["mid"][i], gbuf[("m", i)], G)
                add_emb(ge)
            acc(("m", i - 1) if i else last_enc, g_x)
    else:
        grads_out["g_h_in"] = gbuf[("hin",)]
    for i in reversed(range(n_enc)):
        op, c, p = desc["enc_ops"][i], tape["enc"][i], f"enc{i}."
        g = gbuf.get(("e", i))
        if g is None:
            g = torch.zeros(c["out_shape"], dtype=c["x"].dtype)
        if op["kind"] == "resblock":
            g_x, ge = resblock_bwd(P, p, c, g, G)
            add_emb(ge)
            acc(("e", i - 1), g_x)
        elif op["kind"] == "attn":
            acc(("e", i - 1), attn_block_bwd(P, p, c, g, G))
        elif op["kind"] == "tblock":
            acc(("e", i - 1), tblock_bwd(P, p, c, g, G))
        else:
            G[p + "conv.w"], G[p + "conv.b"] = conv_wgrad(c["x"], g, P[p + "conv.w"].shape, c["stride"])
            acc(("e", i - 1), conv_dgrad(g, P[p + "conv.w"], c["x"].shape[2:], c["stride"]))
    grads_out["g_x_in"] = gbuf[("e", -1)]
    grads_out["g_emb"] = g_emb
    return grads_out, G


def mse(d, target, scale=1.0):
    """L = scale * mean((d - T)^2); g_d = scale * 2 (d - T) / numel."""
    diff = d - target
    return scale * (diff ** 2).mean(), st(scale * 2.0 * diff / diff.numel())


def _to(x, dtype):
    return None if x is None else torch.as_tensor(x).to(dtype)


def run_stage(desc, params, mb, loss_scale=1.0, dtype=DT):
    """One microbatch: temb -> stage forward -> MSE(d_out, target) -> stage backward ->
    temb backward.  `params`, `mb` as produced by workloads.draw (numpy / tensors)."""
    P = {k: _to(v, dtype) for k, v in params.items()}
    x_in, h_in = _to(mb["x_in"], dtype), _to(mb.get("h_in"), dtype)
    emb, tctx = temb_fwd(desc, P, torch.as_tensor(mb["t"]), dtype)
    outs, ctx = stage_forward(desc, P, x_in, h_in, emb)
    loss, g_d = mse(outs["d_out"], _to(mb["target"], dtype), loss_scale)
    gi, G = stage_backward(desc, P, ctx, g_d, _to(mb.get("g_e_out"), dtype))
    G.update(temb_bwd(desc, P, tctx, gi["g_emb"]))
    res = {"loss": loss, "emb": emb, "skips": ctx["skips"], "param_grads": G}
    res.update(outs)
    res.update(gi)
    return res


def run_wave(desc, params, mbs, dtype=DT):
    """configs[4]: forwards F0..F{M-1} then backwards B{M-1}..B0; L_total = mean over
    microbatches, weight grads summed (reading R16).  The oracle has no notion of
    time, so the wave order only matters for which skip sets are alive; it reports
    the peak number of bytes the skip buffers would hold."""
    M = len(mbs)
    results = [run_stage(desc, params, mb, 1.0 / M, dtype) for mb in mbs]
    total = {}
    for r in results:
        for k, v in r["param_grads"].items():
            total[k] = v if k not in total else total[k] + v
    elem = sum(s.numel() for s in results[0]["skips"])
    return {"per_mb": results, "param_grads": total, "loss": sum(r["loss"] for r in results),
            "skip_elements_per_mb": elem, "peak_skip_elements": elem * M}
