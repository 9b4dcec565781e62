"""Stage structures of the five BASELINE.json configs and the seeded synthetic inputs.

This module holds NO arithmetic of the method (no conv, norm, activation, loss):
only the op lists that describe a collocated stage ("linear sequence
of operations" with a skip field; L91 local skip buffers) and the recipe that draws
parameters and inputs from a seed.  It is
the one module both the oracle's tests and the CUDA binding's tests may use.

Logical layouts produced here (the oracle's): activations [N,C,H,W], conv weights
[Cout,Cin,kh,kw], linear weights [out,in].  The binding permutes to the device
layout (NHWC / [Cout,kh,kw,Cin]).
"""
from __future__ import annotations

import copy
import numpy as np

CONV_IN, RESBLOCK, DOWN, UP, HEAD, ATTN, TBLOCK = "conv_in", "resblock", "down", "up", "head", "attn", "tblock"


def _op(kind, cin, cout, skip=0, push=0, heads=0):
    return {"kind": kind, "cin": cin, "cout": cout, "skip": skip, "push": push, "heads": heads}


def attn(c, heads, push=0):
    """Self-attention block on c channels: GN -> 1x1 conv to q|k|v -> attention per head over the
    H W pixels -> 1x1 conv, + residual."""
    return _op(ATTN, c, c, 0, push, heads)


def rb(cin, cout, skip=0, push=0):
    return _op(RESBLOCK, cin, cout, skip, push)


def _stage(name, dtype, n, h, w, c_in, groups, temb, link, x_in_is_skip, enc, mid, dec,
           microbatches=1, eps=1e-5):
    return {"name": name, "dtype": dtype, "n": n, "h": h, "w": w, "c_in": c_in,
            "groups": groups, "eps": eps, "temb": temb, "link": link,
            "x_in_is_skip": int(x_in_is_skip), "enc_ops": enc, "mid_ops": mid, "dec_ops": dec,
            "microbatches": microbatches}


def _unet(name, n, hw, levels, microbatches=1, dtype="bf16", groups=32, temb=None, c_lat=4):
    """Conv-only SD-shaped UNet, every skip pair local (configs[3], configs[4])."""
    temb = temb or {"kind": "mlp", "d0": levels[0], "dim": 4 * levels[0]}
    enc = [_op(CONV_IN, c_lat, levels[0], push=1)]
    skips = [levels[0]]
    c = levels[0]
    for li, ch in enumerate(levels):
        for _ in range(2):
            enc.append(rb(c, ch, push=1)); c = ch; skips.append(c)
        if li != len(levels) - 1:
            enc.append(_op(DOWN, c, c, push=1)); skips.append(c)
    mid = [rb(c, c), rb(c, c)]
    dec = []
    for li in reversed(range(len(levels))):
        ch = levels[li]
        for _ in range(3):
            s = skips.pop()
            dec.append(rb(c, ch, skip=s)); c = ch
        if li != 0:
            dec.append(_op(UP, c, c))
    dec.append(_op(HEAD, c, c_lat))
    assert not skips
    return _stage(name, dtype, n, hw, hw, c_lat, groups, temb, "closed", 0, enc, mid, dec,
                  microbatches=microbatches)


def config(i: int) -> dict:
    """The five configs of BASELINE.json, 1-based, read as SURVEY.md 8c R1-R20; 6 = attn_level() (row f1)."""
    mlp = {"kind": "mlp", "d0": 320, "dim": 1280}
    if i == 6:
        return attn_level()
    if i == 1:
        return _stage("config1", "fp32", 2, 16, 16, 32, 8, {"kind": "sinusoidal", "d0": 128, "dim": 128},
                      "open", 0, [rb(32, 32, push=1)], [], [rb(32, 32, skip=32)])
    if i == 2:
        return _stage("config2", "bf16", 4, 64, 64, 320, 32, mlp, "open", 1,
                      [rb(320, 320, push=1), rb(320, 320, push=1)], [],
                      [rb(320, 320, skip=320) for _ in range(3)])
    if i == 3:
        return _stage("config3", "bf16", 8, 32, 32, 320, 32, mlp, "open", 1,
                      [rb(320, 640, push=1), rb(640, 640, push=1), _op(DOWN, 640, 640)], [],
                      [rb(640, 640, skip=640), rb(640, 640, skip=640), rb(640, 640, skip=320),
                       _op(UP, 640, 640)])
    if i == 4:
        return _unet("config4", 8, 64, [320, 640, 1280, 1280])
    if i == 5:
        return _unet("config5", 2, 128, [320, 640, 1280], microbatches=8)
    raise ValueError(i)


def tblock(c, heads, skip=0, push=0):
    """Transformer block on c channels: [Linear on concat(x, skip) where a skip is consumed ->]
    LN -> qkv -> attention -> proj + residual -> LN -> fc1 (c -> 4c) -> GELU -> fc2 + residual."""
    return _op(TBLOCK, c, c, skip, push, heads)


def uvit_stage(name, n, hw, c, heads, depth, dtype="bf16") -> dict:
    """U-ViT style stage: `depth` early blocks whose outputs are cached, `depth` late blocks that each
    consume one of them through concat + Linear (LIFO); OPEN (tokens in, tokens out on both sides)."""
    temb = {"kind": "sinusoidal", "d0": 16, "dim": 16}      # the blocks take no timestep input (reading R26)
    return _stage(name, dtype, n, hw, hw, c, 1, temb, "open", 0, [tblock(c, heads, push=1) for _ in range(depth)], [],
                  [tblock(c, heads, skip=c) for _ in range(depth)])


def attn_level() -> dict:
    """configs[2]'s level-2 stage with a self-attention block (640 channels = 10 heads x 64, 1024
    tokens) after every ResBlock, as in an SD-shaped UNet level; skips are pushed after the attention."""
    mlp = {"kind": "mlp", "d0": 320, "dim": 1280}
    return _stage("attn_level", "bf16", 8, 32, 32, 320, 32, mlp, "open", 1,
                  [rb(320, 640), attn(640, 10, push=1), rb(640, 640), attn(640, 10, push=1), _op(DOWN, 640, 640)], [],
                  [rb(640, 640, skip=640), attn(640, 10), rb(640, 640, skip=640), attn(640, 10), rb(640, 640, skip=320),
                   attn(640, 10), _op(UP, 640, 640)])


def mini(kind: str, dtype: str = "fp32") -> dict:
    """Small structures with the same op patterns, for the CPU pins and quick GPU parity."""
    sin = {"kind": "sinusoidal", "d0": 16, "dim": 16}
    mlp = {"kind": "mlp", "d0": 8, "dim": 16}
    if kind == "pair":          # config-1 pattern, smaller
        return _stage("mini_pair", dtype, 2, 4, 4, 8, 4, sin, "open", 0,
                      [rb(8, 8, push=1)], [], [rb(8, 8, skip=8)])
    if kind == "level":         # config-2 pattern: x_in is a skip, 2 enc + 3 dec RBs
        return _stage("mini_level", dtype, 2, 4, 4, 8, 4, mlp, "open", 1,
                      [rb(8, 8, push=1), rb(8, 8, push=1)], [],
                      [rb(8, 8, skip=8) for _ in range(3)])
    if kind == "updown":        # config-3 pattern incl. a straddling GroupNorm group (16|8, G=4)
        return _stage("mini_updown", dtype, 2, 4, 4, 8, 4, mlp, "open", 1,
                      [rb(8, 16, push=1), rb(16, 16, push=1), _op(DOWN, 16, 16)], [],
                      [rb(16, 16, skip=16), rb(16, 16, skip=16), rb(16, 16, skip=8), _op(UP, 16, 16)])
    if kind == "straddle":      # h 32 ch | skip 16 ch, G=8 -> cpg 6, group 5 straddles
        return _stage("mini_straddle", dtype, 1, 4, 4, 16, 8, sin, "open", 1,
                      [rb(16, 16)], [], [rb(32, 16, skip=16)])
    if kind == "unet":          # config-4/5 pattern: closed, conv_in, down/up, mid, head
        return _unet("mini_unet", 2, 8, [8, 16], dtype=dtype, groups=4, temb=mlp, c_lat=4)
    if kind == "wave":
        d = _unet("mini_wave", 1, 8, [8, 16], dtype=dtype, groups=4, temb=mlp, c_lat=4)
        d["microbatches"] = 3
        return d
    if kind == "attn":          # ResBlock + self-attention per block, skips pushed after the attention
        return _stage("mini_attn", dtype, 2, 4, 4, 8, 4, mlp, "open", 1,
                      [rb(8, 16), attn(16, 2, push=1), rb(16, 16), attn(16, 4, push=1)], [],
                      [rb(16, 16, skip=16), attn(16, 2), rb(16, 16, skip=16), attn(16, 1), rb(16, 16, skip=8)])
    if kind == "uvit":          # transformer blocks with long skips (concat + Linear)
        return uvit_stage("mini_uvit", 2, 4, 16, 2, 2, dtype=dtype)
    if kind == "attn_unet":     # closed: attention in the mid block as well
        d = _unet("mini_attn_unet", 2, 8, [8, 16], dtype=dtype, groups=4, temb=mlp, c_lat=4)
        d["mid_ops"] = [rb(16, 16), attn(16, 2), rb(16, 16)]
        return d
    raise ValueError(kind)


def gpu_mid(kind: str) -> dict:
    """bf16 structures wide enough for the tensor-core path (C % 64 == 0, Cout % 160 == 0)
    and small enough for the oracle in seconds; spatial sizes chosen to span several
    128-pixel tiles with a ragged tail (N*H*W not a multiple of 128)."""
    mlp = {"kind": "mlp", "d0": 64, "dim": 128}
    if kind == "level":         # 3 images of 8x8 -> 192 pixels = 1.5 tiles
        return _stage("mid_level", "bf16", 3, 8, 8, 320, 32, mlp, "open", 1,
                      [rb(320, 320, push=1), rb(320, 320, push=1)], [],
                      [rb(320, 320, skip=320) for _ in range(3)])
    if kind == "updown":        # 16x16 -> 8x8 down, 16x16 -> 32x32 up, 960-ch straddling GN
        return _stage("mid_updown", "bf16", 3, 16, 16, 320, 32, mlp, "open", 1,
                      [rb(320, 640, push=1), rb(640, 640, push=1), _op(DOWN, 640, 640)], [],
                      [rb(640, 640, skip=640), rb(640, 640, skip=640), rb(640, 640, skip=320),
                       _op(UP, 640, 640)])
    if kind == "unet":
        return _unet("mid_unet", 1, 32, [320, 640], temb=mlp)
    if kind == "uvit":          # 320 channels = 5 heads x 64, 3 images of 64 tokens (192 pixels = 1.5 tiles), 2 + 2 blocks
        return uvit_stage("mid_uvit", 3, 8, 320, 5, 2)
    if kind == "attn":          # SD-style level with attention: 320 channels = 5 heads x 64, 64 tokens per image, 192 pixels = 1.5 tiles
        return _stage("mid_attn", "bf16", 3, 8, 8, 320, 32, mlp, "open", 1,
                      [rb(320, 320), attn(320, 5, push=1)], [],
                      [rb(320, 320, skip=320), attn(320, 5), rb(320, 320, skip=320)])
    raise ValueError(kind)


def split_closed(desc: dict, k_enc: int) -> tuple:
    """Cut a CLOSED whole-model structure into an OPEN outer stage and a CLOSED inner stage for two pipeline devices
    (a stage pair = a contiguous encoder-side op range plus the decoder-side range that
    consumes its skips).  The outer stage takes enc_ops[:k_enc] and the decoder suffix that pops exactly their skips.
    Returns (outer, inner, name map): map[stage][stage param prefix] = whole-model param prefix."""
    enc, dec = desc["enc_ops"], desc["dec_ops"]
    pushes = desc["x_in_is_skip"] + sum(op["push"] for op in enc[:k_enc])
    j, pops = len(dec), 0
    while pops < pushes:
        j -= 1
        pops += 1 if dec[j]["skip"] else 0
    assert pops == pushes and j > 0, "cut does not separate whole skip pairs"
    h = w = desc["h"]
    for op in enc[:k_enc]:
        if op["kind"] == DOWN:
            h, w = h // 2, w // 2
    outer = _stage(desc["name"] + "_outer", desc["dtype"], desc["n"], desc["h"], desc["w"], desc["c_in"], desc["groups"],
                   desc["temb"], "open", desc["x_in_is_skip"], copy.deepcopy(enc[:k_enc]), [], copy.deepcopy(dec[j:]),
                   microbatches=desc["microbatches"], eps=desc["eps"])
    inner = _stage(desc["name"] + "_inner", desc["dtype"], desc["n"], h, w, enc[k_enc - 1]["cout"], desc["groups"], desc["temb"],
                   "closed", 0, copy.deepcopy(enc[k_enc:]), copy.deepcopy(desc["mid_ops"]), copy.deepcopy(dec[:j]),
                   microbatches=desc["microbatches"], eps=desc["eps"])
    names = {"outer": {f"enc{i}.": f"enc{i}." for i in range(k_enc)}, "inner": {f"enc{i}.": f"enc{k_enc + i}." for i in range(len(enc) - k_enc)}}
    names["outer"].update({f"dec{i}.": f"dec{j + i}." for i in range(len(dec) - j)})
    names["inner"].update({f"dec{i}.": f"dec{i}." for i in range(j)})
    names["inner"].update({f"mid{i}.": f"mid{i}." for i in range(len(desc["mid_ops"]))})
    for k in names:
        names[k]["temb."] = "temb."
    return outer, inner, names


def stage_params(whole_params: dict, names: dict) -> dict:
    """Parameters of one stage of split_closed() out of the whole model's (same arrays, renamed)."""
    out = {}
    for sp, wp in names.items():
        for k, v in whole_params.items():
            if k.startswith(wp):
                out[sp + k[len(wp):]] = v
    return out


# ----------------------------------------------------------------------------- structure walks

def skip_channels_pushed(desc) -> list:
    """Channel count, and spatial size, of every pushed skip in push order."""
    out = []
    h, w = desc["h"], desc["w"]
    if desc["x_in_is_skip"]:
        out.append((desc["c_in"], h, w))
    for op in desc["enc_ops"]:
        if op["kind"] == DOWN:
            h, w = h // 2, w // 2
        if op["push"]:
            out.append((op["cout"], h, w))
    return out


def boundary_shapes(desc) -> dict:
    """Logical [N,C,H,W] shapes of the tensors that cross the stage boundary."""
    n, h, w = desc["n"], desc["h"], desc["w"]
    shapes = {"x_in": (n, desc["c_in"], h, w)}
    c = desc["c_in"]
    for op in desc["enc_ops"]:
        if op["kind"] == DOWN:
            h, w = h // 2, w // 2
        c = op["cout"]
    if desc["link"] == "open":
        shapes["e_out"] = (n, c, h, w)
        sk = skip_channels_pushed(desc)
        hh, ww = (sk[-1][1], sk[-1][2]) if sk else (h, w)
        shapes["h_in"] = (n, desc["dec_ops"][0]["cin"], hh, ww)
        h, w = hh, ww
    for op in desc["dec_ops"]:
        if op["kind"] == UP:
            h, w = 2 * h, 2 * w
        c = op["cout"]
    shapes["d_out"] = (n, c, h, w)
    return shapes


def param_specs(desc) -> list:
    """(name, logical shape, kind, fan_in) in the fixed draw order (also the C-ABI's
    pulse_stage_param_info order).  kind in {weight, bias, gamma, beta}."""
    specs = []
    T = desc["temb"]["dim"]
    if desc["temb"]["kind"] == "mlp":
        d0 = desc["temb"]["d0"]
        specs += [("temb.w1", (T, d0), "weight", d0), ("temb.b1", (T,), "bias", 0),
                  ("temb.w2", (T, T), "weight", T), ("temb.b2", (T,), "bias", 0)]
    for phase in ("enc", "mid", "dec"):
        for i, op in enumerate(desc[phase + "_ops"]):
            p = f"{phase}{i}."
            k, ci, co = op["kind"], op["cin"] + op["skip"], op["cout"]
            if k == RESBLOCK:
                specs += [(p + "gn1.gamma", (ci,), "gamma", 0), (p + "gn1.beta", (ci,), "beta", 0),
                          (p + "conv1.w", (co, ci, 3, 3), "weight", ci * 9), (p + "conv1.b", (co,), "bias", 0),
                          (p + "temb.w", (co, T), "weight", T), (p + "temb.b", (co,), "bias", 0),
                          (p + "gn2.gamma", (co,), "gamma", 0), (p + "gn2.beta", (co,), "beta", 0),
                          (p + "conv2.w", (co, co, 3, 3), "weight", co * 9), (p + "conv2.b", (co,), "bias", 0)]
                if ci != co:
                    specs += [(p + "sc.w", (co, ci, 1, 1), "weight", ci), (p + "sc.b", (co,), "bias", 0)]
            elif k in (CONV_IN, DOWN, UP):
                specs += [(p + "conv.w", (co, ci, 3, 3), "weight", ci * 9), (p + "conv.b", (co,), "bias", 0)]
            elif k == TBLOCK:
                c = co
                if op["skip"]:
                    specs += [(p + "skip.w", (c, ci, 1, 1), "weight", ci), (p + "skip.b", (c,), "bias", 0)]
                specs += [(p + "ln1.gamma", (c,), "gamma", 0), (p + "ln1.beta", (c,), "beta", 0),
                          (p + "qkv.w", (3 * c, c, 1, 1), "weight", c), (p + "qkv.b", (3 * c,), "bias", 0),
                          (p + "proj.w", (c, c, 1, 1), "weight", c), (p + "proj.b", (c,), "bias", 0),
                          (p + "ln2.gamma", (c,), "gamma", 0), (p + "ln2.beta", (c,), "beta", 0),
                          (p + "fc1.w", (4 * c, c, 1, 1), "weight", c), (p + "fc1.b", (4 * c,), "bias", 0),
                          (p + "fc2.w", (c, 4 * c, 1, 1), "weight", 4 * c), (p + "fc2.b", (c,), "bias", 0)]
            elif k == ATTN:
                specs += [(p + "gn.gamma", (ci,), "gamma", 0), (p + "gn.beta", (ci,), "beta", 0),
                          (p + "qkv.w", (3 * ci, ci, 1, 1), "weight", ci), (p + "qkv.b", (3 * ci,), "bias", 0),
                          (p + "proj.w", (ci, ci, 1, 1), "weight", ci), (p + "proj.b", (ci,), "bias", 0)]
            elif k == HEAD:
                specs += [(p + "gn.gamma", (ci,), "gamma", 0), (p + "gn.beta", (ci,), "beta", 0),
                          (p + "conv.w", (co, ci, 3, 3), "weight", ci * 9), (p + "conv.b", (co,), "bias", 0)]
            else:
                raise ValueError(k)
    return specs


# ----------------------------------------------------------------------------- seeded draws

def to_bf16_grid(a: np.ndarray) -> np.ndarray:
    """Round-to-nearest-even onto the bf16 grid, returned as float32 (input recipe R18:
    both sides receive identical, bf16-representable values)."""
    a = np.ascontiguousarray(a, dtype=np.float32)
    u = a.view(np.uint32).astype(np.uint64)
    u = (u + 0x7FFF + ((u >> 16) & 1)) & 0xFFFF0000
    return u.astype(np.uint32).view(np.float32).reshape(a.shape)


def draw(desc, seed: int = 0, with_g_e_out: bool = False) -> dict:
    """Parameters then inputs from numpy default_rng(seed), fixed order:
    params in param_specs order (weights N(0,2/fan_in); biases 0.1 N(0,1); gamma
    1+0.1 N(0,1); beta 0.1 N(0,1)), then per microbatch x_in, h_in (open), t, target,
    optional g_e_out.  bf16 configs get values on the bf16 grid."""
    rng = np.random.default_rng(seed)
    q = to_bf16_grid if desc["dtype"] == "bf16" else (lambda a: np.asarray(a, np.float32))
    params = {}
    for name, shape, kind, fan_in in param_specs(desc):
        z = rng.standard_normal(shape)
        if kind == "weight":
            v = z * np.sqrt(2.0 / fan_in)
        elif kind == "gamma":
            v = 1.0 + 0.1 * z
        else:
            v = 0.1 * z
        params[name] = q(v)
    shapes = boundary_shapes(desc)
    mbs = []
    for _ in range(desc["microbatches"]):
        mb = {"x_in": q(rng.standard_normal(shapes["x_in"]))}
        if desc["link"] == "open":
            mb["h_in"] = q(rng.standard_normal(shapes["h_in"]))
        mb["t"] = rng.integers(0, 1000, size=(desc["n"],), dtype=np.int64)
        mb["target"] = q(rng.standard_normal(shapes["d_out"]))
        if with_g_e_out and desc["link"] == "open":
            mb["g_e_out"] = q(rng.standard_normal(shapes["e_out"]) / np.prod(shapes["e_out"]))
        mbs.append(mb)
    return {"params": params, "microbatches": mbs}


def scaled(desc, **kw) -> dict:
    d = copy.deepcopy(desc)
    d.update(kw)
    return d
