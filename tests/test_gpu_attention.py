"""Kernel-level GPU parity of the attention core through pulse_attention /
pulse_attention_backward against the oracle's plain definition (softmax(q k^T / sqrt(d)) v and its hand-written
chain rule): several 64-token tiles with a ragged tail, one token, head widths 8 ... 128, fp32 and bf16 storage."""
import numpy as np
import pytest
import torch

from oracle import pulse_oracle as O
from paper_2606_19163_b200 import workloads as W

pytestmark = pytest.mark.gpu


def _B():
    from paper_2606_19163_b200 import binding
    return binding


CASES = [
    # n, tokens, channels, heads
    (2, 64, 64, 2),        # one tile, d = 32
    (1, 200, 48, 3),       # 3.125 tiles: ragged keys and queries, d = 16
    (3, 1, 32, 4),         # a single token: P = 1, o = v
    (1, 130, 128, 1),      # d = 128 (the widest head)
    (2, 96, 80, 2),        # d = 40 (the SD1.5 head width), 1.5 tiles
    (1, 1024, 128, 2),     # 32 x 32 pixels, d = 64: 16 tiles
    (2, 300, 320, 5),      # d = 64, 2.3 tiles of 128 queries / keys: the tcgen05 forward with ragged tails
    (3, 64, 256, 2),       # d = 128, fewer tokens than one tile
]


def _split(t, c, heads):       # [n, T, c] -> [n heads, T, d]
    n, T, _ = t.shape
    return t.reshape(n, T, heads, c // heads).permute(0, 2, 1, 3).reshape(n * heads, T, c // heads)


def _merge(t, n, heads):       # [n heads, T, d] -> [n, T, c]
    _, T, d = t.shape
    return t.reshape(n, heads, T, d).permute(0, 2, 1, 3).reshape(n, T, heads * d)


@pytest.mark.parametrize("dtype", [torch.float32, torch.bfloat16, "bf16_simt"])
@pytest.mark.parametrize("case", CASES)
def test_attention_core(case, dtype):
    """bf16 with 64 / 128 channels per head runs the tcgen05 forward; "bf16_simt" forces the CUDA-core forward on the same
    inputs."""
    B = _B()
    force_simt = dtype == "bf16_simt"
    dtype = torch.bfloat16 if force_simt else dtype
    n, T, c, heads = case
    rng = np.random.default_rng(hash(case) % 2 ** 31)
    draw = (lambda *s: W.to_bf16_grid(rng.standard_normal(s))) if dtype == torch.bfloat16 else \
        (lambda *s: rng.standard_normal(s).astype(np.float32))
    qkv, g_o = draw(n, T, 3 * c) * 1.5, draw(n, T, c)
    if dtype == torch.bfloat16:
        qkv = W.to_bf16_grid(qkv)
    qt = torch.as_tensor(qkv).double()
    q, k, v = (_split(qt[:, :, i * c:(i + 1) * c], c, heads) for i in range(3))
    o_ref, p = O.attn_core_fwd(q, k, v)
    gq, gk, gv = O.attn_core_bwd(_split(torch.as_tensor(g_o).double(), c, heads), q, k, v, p)
    g_ref = torch.cat([_merge(t, n, heads) for t in (gq, gk, gv)], dim=2)
    dq = torch.as_tensor(qkv).to("cuda", dtype)
    o, stats = B.attention(dq, heads, force_simt=force_simt)
    g = B.attention_backward(dq, torch.as_tensor(g_o).to("cuda", dtype), heads, stats, force_simt=force_simt)
    torch.cuda.synchronize()

    # the tcgen05 forward feeds P to the tensor cores as bf16 (as every flash-attention kernel does): each probability carries
    # a 2^-9 relative rounding, o = sum_j p_j v_j / l inherits at most 2^-9 (1 + 1) max|v| of it
    tc = dtype == torch.bfloat16 and not force_simt and (c // heads) in (64, 128)
    p_round = 2.0 ** -8 * float(v.abs().max()) if tc else 0.0

    def close(got, ref, what):
        ref = ref.double()
        err = (got.double().cpu() - ref).abs()
        rms = float(ref.pow(2).mean().sqrt())
        allow = ref.abs() * 2.0 ** -8 + 3e-3 * rms if dtype == torch.bfloat16 else torch.full_like(ref, 1e-4 * rms)
        if what == "o":
            allow = allow + p_round
        elif tc:       # P and g_S reach the tensor cores as bf16: 2^-9 per product on sums of |g_S| |k| (or |P| |g_o|) terms
            allow = allow + 2.0 ** -8 * float(ref.abs().max())
        worst = float((err / allow).max())
        assert worst <= 1.0, f"{what} {case} {dtype}: worst err/allowance {worst:.3f}, max err {float(err.max()):.3e}, rms {rms:.3e}"

    close(o, _merge(o_ref, n, heads), "o")
    close(g, g_ref, "g_qkv")
    # log-sum-exp of the scaled scores, per (image, head, query)
    lse = stats[: n * heads * T].view(n * heads, T).double().cpu()
    want = torch.logsumexp(q @ k.transpose(1, 2) / (c // heads) ** 0.5, dim=2)
    assert float((lse - want).abs().max()) < 1e-3
