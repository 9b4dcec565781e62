"""Independent pin for the oracle (CPU tests only): a *naive sequential* run of the same
stage that keeps no skip buffers - whenever a decoder ResBlock needs a skip it
recomputes the encoder prefix that produces it (BASELINE.json north_star: "cached-skip
result equals a naive sequential run that recomputes the skip") - composed from
library modules (F.group_norm, F.silu, F.interpolate, torch.cat) and differentiated by
torch.autograd.  It shares no code with oracle/pulse_oracle.py."""
import math

import torch
import torch.nn.functional as F


def _temb(desc, P, t):
    d = desc["temb"]["d0"]
    half = d // 2
    freqs = torch.pow(torch.tensor(10000.0, dtype=torch.float64), -torch.arange(half, dtype=torch.float64) / half)
    ang = t.double()[:, None] * freqs[None, :]
    e = torch.cat([ang.cos(), ang.sin()], 1)
    if desc["temb"]["kind"] == "mlp":
        e = F.linear(F.silu(F.linear(e, P["temb.w1"], P["temb.b1"])), P["temb.w2"], P["temb.b2"])
    return e


def _rb(desc, P, p, x, emb):
    h = F.conv2d(F.silu(F.group_norm(x, desc["groups"], P[p + "gn1.gamma"], P[p + "gn1.beta"], desc["eps"])),
                 P[p + "conv1.w"], P[p + "conv1.b"], padding=1)
    h = h + F.linear(F.silu(emb), P[p + "temb.w"], P[p + "temb.b"])[:, :, None, None]
    h = F.conv2d(F.silu(F.group_norm(h, desc["groups"], P[p + "gn2.gamma"], P[p + "gn2.beta"], desc["eps"])),
                 P[p + "conv2.w"], P[p + "conv2.b"], padding=1)
    sc = F.conv2d(x, P[p + "sc.w"], P[p + "sc.b"]) if (p + "sc.w") in P else x
    return h + sc


def _attn(desc, P, p, x, heads):
    """Self-attention block from library pieces: F.group_norm, 1x1 convs, F.scaled_dot_product_attention."""
    n, c, h, w = x.shape
    qkv = F.conv2d(F.group_norm(x, desc["groups"], P[p + "gn.gamma"], P[p + "gn.beta"], desc["eps"]), P[p + "qkv.w"], P[p + "qkv.b"])
    q, k, v = (t.reshape(n, heads, c // heads, h * w).transpose(2, 3) for t in qkv.chunk(3, dim=1))    # [n, heads, T, d]
    o = F.scaled_dot_product_attention(q, k, v)
    o = o.transpose(2, 3).reshape(n, c, h, w)
    return x + F.conv2d(o, P[p + "proj.w"], P[p + "proj.b"])


def _tblock(desc, P, p, x, skip, heads):
    """Transformer block with an optional long skip from library pieces (F.layer_norm on channels-last tokens, F.gelu,
    F.scaled_dot_product_attention, F.linear)."""
    n, _, h, w = x.shape
    tok = lambda t: t.flatten(2).transpose(1, 2)                  # [n, T, c]
    lin = lambda t, name: F.linear(t, P[p + name + ".w"][:, :, 0, 0], P[p + name + ".b"])
    z = tok(x)
    if skip is not None:
        z = lin(torch.cat([z, tok(skip)], dim=2), "skip")
    c = z.shape[2]
    qkv = lin(F.layer_norm(z, (c,), P[p + "ln1.gamma"], P[p + "ln1.beta"], desc["eps"]), "qkv")
    q, k, v = (t.reshape(n, h * w, heads, c // heads).transpose(1, 2) for t in qkv.chunk(3, dim=2))
    o = F.scaled_dot_product_attention(q, k, v).transpose(1, 2).reshape(n, h * w, c)
    z = z + lin(o, "proj")
    z = z + lin(F.gelu(lin(F.layer_norm(z, (c,), P[p + "ln2.gamma"], P[p + "ln2.beta"], desc["eps"]), "fc1")), "fc2")
    return z.transpose(1, 2).reshape(n, c, h, w)


def _enc_prefix(desc, P, x_in, emb, upto_push):
    """Recompute the encoder from x_in until push number `upto_push` exists; return it."""
    k = 0
    x = x_in
    if desc["x_in_is_skip"]:
        if upto_push == 0:
            return x
        k = 1
    for i, op in enumerate(desc["enc_ops"]):
        p = f"enc{i}."
        if op["kind"] == "resblock":
            x = _rb(desc, P, p, x, emb)
        elif op["kind"] == "attn":
            x = _attn(desc, P, p, x, op["heads"])
        elif op["kind"] == "tblock":
            x = _tblock(desc, P, p, x, None, op["heads"])
        else:
            x = F.conv2d(x, P[p + "conv.w"], P[p + "conv.b"], stride=2 if op["kind"] == "down" else 1, padding=1)
        if op["push"]:
            if k == upto_push:
                return x
            k += 1
    if upto_push is None:
        return x
    raise AssertionError("push index not found")


def run(desc, params, mb, loss_scale=1.0, extra_e_loss=False):
    P = {k: torch.tensor(v, dtype=torch.float64, requires_grad=True) for k, v in params.items()}
    x_in = torch.tensor(mb["x_in"], dtype=torch.float64, requires_grad=True)
    h_in = torch.tensor(mb["h_in"], dtype=torch.float64, requires_grad=True) if "h_in" in mb else None
    emb = _temb(desc, P, torch.as_tensor(mb["t"]))
    if not emb.requires_grad:
        emb.requires_grad_(True)
    emb.retain_grad()
    n_push = desc["x_in_is_skip"] + sum(op["push"] for op in desc["enc_ops"])
    e_last = _enc_prefix(desc, P, x_in, emb, None)
    if desc["link"] == "closed":
        h = e_last
        for i, op in enumerate(desc["mid_ops"]):
            h = _attn(desc, P, f"mid{i}.", h, op["heads"]) if op["kind"] == "attn" else _rb(desc, P, f"mid{i}.", h, emb)
    else:
        h = h_in
    top = n_push
    for i, op in enumerate(desc["dec_ops"]):
        p = f"dec{i}."
        if op["kind"] == "resblock":
            top -= 1
            skip = _enc_prefix(desc, P, x_in, emb, top)      # recomputed, never cached
            h = _rb(desc, P, p, torch.cat([h, skip], 1), emb)
        elif op["kind"] == "attn":
            h = _attn(desc, P, p, h, op["heads"])
        elif op["kind"] == "tblock":
            sk = None
            if op["skip"]:
                top -= 1
                sk = _enc_prefix(desc, P, x_in, emb, top)      # recomputed, never cached
            h = _tblock(desc, P, p, h, sk, op["heads"])
        elif op["kind"] == "up":
            h = F.conv2d(F.interpolate(h, scale_factor=2, mode="nearest"), P[p + "conv.w"], P[p + "conv.b"], padding=1)
        else:
            h = F.conv2d(F.silu(F.group_norm(h, desc["groups"], P[p + "gn.gamma"], P[p + "gn.beta"], desc["eps"])),
                         P[p + "conv.w"], P[p + "conv.b"], padding=1)
    loss = loss_scale * F.mse_loss(h, torch.tensor(mb["target"], dtype=torch.float64))
    total = loss
    if "g_e_out" in mb and desc["link"] == "open":
        total = total + (e_last * torch.tensor(mb["g_e_out"], dtype=torch.float64)).sum()
    total.backward()
    out = {"loss": loss.detach(), "d_out": h.detach(), "g_x_in": x_in.grad, "g_emb": emb.grad,
           "param_grads": {k: v.grad for k, v in P.items()}}
    if h_in is not None:
        out["g_h_in"] = h_in.grad
        out["e_out"] = e_last.detach()
    return out
