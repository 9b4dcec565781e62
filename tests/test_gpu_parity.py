"""GPU parity: libpulse.so (through the C-ABI binding) vs the CPU oracle, element by
element on the same seeded inputs.  Bars (BASELINE.json north_star): fp32 debug path
max|err| <= 1e-4 * RMS(ref); bf16 max|err| <= 2e-2 * RMS(ref), per tensor.

The bf16 bar is the PLAIN 2e-2 for every tensor except those named in tests/golden/bf16_floor.json (written by
tests/golden/make_bf16_floor.py from the oracle alone): tensors for which the plain definition evaluated with bf16
storage (oracle.stored_in) is itself more than 1e-2 away from the exact result.  Those
may reach 2 x their storage floor (capped at CAP unless the floor itself is above CAP / 2: attention stages, whose
max-abs floor is heavy-tailed) and must then stay within 1.5 x the floor in rms.  A tensor that
is not on the committed list and exceeds 2e-2 fails the test."""
import json
import os

import numpy as np
import pytest
import torch

from oracle import pulse_oracle as O
from paper_2606_19163_b200 import workloads as W

pytestmark = pytest.mark.gpu

TOL = {"fp32": 1e-4, "bf16": 2e-2}


def _binding():
    from paper_2606_19163_b200 import binding
    return binding


def rel_err(got, ref):
    """north_star's metric: max |err| / RMS(ref)."""
    ref = ref.to(torch.float64)
    rms = float(ref.pow(2).mean().sqrt())
    return float((got.to(torch.float64) - ref).abs().max()) / max(rms, 1e-30)


def rms_err(got, ref):
    ref = ref.to(torch.float64)
    rms = float(ref.pow(2).mean().sqrt())
    return float((got.to(torch.float64) - ref).pow(2).mean().sqrt()) / max(rms, 1e-30)


REPORT = os.environ.get("PULSE_PARITY_REPORT")
with open(os.path.join(os.path.dirname(os.path.abspath(__file__)), "golden", "bf16_floor.json")) as _f:
    GOLD = json.load(_f)
CAP = 0.15          # allowance cap for tensors whose own storage floor is below CAP / 2


def run_gpu(desc, data, flags=0, with_g_e_out=False, order=None, max_inflight=None, steps=1):
    """order: list of ("F", m) / ("B", m) events (default: one step, or the wave F0..F{M-1}, B{M-1}..B0)."""
    B = _binding()
    st = B.Stage(desc, flags=flags, max_inflight=max_inflight)
    st.load_params(data["params"])
    M = desc["microbatches"]
    outs = []
    devs = [st.to_device(mb) for mb in data["microbatches"]]
    if order is not None:
        fw, done, first = {}, {}, True
        half = {}                    # split stages: per microbatch state between the half calls
        for ev, m in order:
            if ev == "FE":           # the two-call forms of a split (pipeline) stage
                emb, tst = st.temb_forward(devs[m]["t"])
                half[m] = {"emb": emb, "tst": tst, "e_out": st.forward_enc(m, devs[m]["x_in"], emb)}
                assert st.cache_stats()["live_slots"] <= st.max_inflight
            elif ev == "FD":
                half[m]["d_out"] = st.forward_dec(m, devs[m]["h_in"])
            elif ev == "BD":
                h = half[m]
                h["loss"], g_d = st.mse(h["d_out"], devs[m]["target"], 1.0 / M)
                h["g_emb"] = torch.zeros_like(h["emb"])
                h["g_h_in"] = st.backward_dec(m, g_d, h["g_emb"], accumulate=not first)
                h["first"], first = first, False
            elif ev == "BE":
                h = half.pop(m)
                h["g_x_in"] = st.backward_enc(m, devs[m].get("g_e_out"), h["g_emb"])
                st.temb_backward(h["g_emb"], h.pop("tst"), accumulate=not h.pop("first"))
                done[m] = h
            elif ev == "F":
                emb, tst = st.temb_forward(devs[m]["t"])
                fw[m] = (emb, tst) + st.forward(m, devs[m]["x_in"], devs[m].get("h_in"), emb)
                assert st.cache_stats()["live_slots"] <= st.max_inflight
            else:
                emb, tst, e_out, d_out = fw.pop(m)
                loss, g_d = st.mse(d_out, devs[m]["target"], 1.0 / M)
                g_temb = torch.zeros_like(emb)
                g_x_in, g_h_in = st.backward(m, g_d, devs[m].get("g_e_out"), True, g_temb, accumulate=not first)
                st.temb_backward(g_temb, tst, accumulate=not first)
                first = False
                done[m] = {"loss": loss, "e_out": e_out, "d_out": d_out, "g_x_in": g_x_in, "g_h_in": g_h_in,
                           "g_emb": g_temb, "emb": emb}
        outs = [done[m] for m in range(M)]
        assert st.cache_stats()["live_slots"] == 0
    elif M == 1:
        for rep in range(steps):       # steps > 1: the later steps run what the first backward of a stage prepares
            if rep:                    # (weight gradients stored whole into a buffer that is no longer zeroed): poison it
                st.d_grads.fill_(255)
            r = st.step(0, devs[0], 1.0, accumulate=False)
        outs.append(r)
    else:       # wave: F0..F{M-1}, B{M-1}..B0 (configs[4])
        for rep in range(steps):
            if rep:
                st.d_grads.fill_(255)
                outs = []
            fw = []
            for m, dev in enumerate(devs):
                emb, tst = st.temb_forward(dev["t"])
                e_out, d_out = st.forward(m, dev["x_in"], dev.get("h_in"), emb)
                fw.append((emb, tst, e_out, d_out))
            peak = st.cache_stats()
            assert peak["live_slots"] == M and peak["peak_bytes"] == M * st.skip_bytes
            for m in reversed(range(M)):
                emb, tst, e_out, d_out = fw[m]
                loss, g_d = st.mse(d_out, devs[m]["target"], 1.0 / M)
                g_temb = torch.zeros_like(emb)
                first = m == M - 1
                g_x_in, g_h_in = st.backward(m, g_d, None, True, g_temb, accumulate=not first)
                st.temb_backward(g_temb, tst, accumulate=not first)
                outs.append({"loss": loss, "e_out": e_out, "d_out": d_out, "g_x_in": g_x_in, "g_h_in": g_h_in,
                             "g_emb": g_temb, "emb": emb})
            outs.reverse()
            assert st.cache_stats()["live_slots"] == 0
    torch.cuda.synchronize()
    res = {"per_mb": [], "param_grads": st.grads(), "stage": st}
    for r in outs:
        o = {}
        for k, v in r.items():
            if v is None:
                continue
            o[k] = B.nchw(v) if v.dim() == 4 else v.to(torch.float64).cpu()
        res["per_mb"].append(o)
    return res


def oracle_run(desc, data, dtype):
    M = desc["microbatches"]
    if M == 1:
        r = O.run_stage(desc, data["params"], data["microbatches"][0], 1.0, dtype)
        return [r], r["param_grads"]
    wave = O.run_wave(desc, data["params"], data["microbatches"], dtype)
    return wave["per_mb"], wave["param_grads"]


def flatten(per_mb, grads):
    out = {}
    for m, r in enumerate(per_mb):
        for k in ["d_out", "e_out", "g_x_in", "g_h_in", "emb", "g_emb"]:
            if r.get(k) is not None:
                out[f"mb{m}.{k}"] = r[k]
        out[f"mb{m}.loss"] = torch.as_tensor(float(r["loss"]), dtype=torch.float64).reshape(1)
    for k, v in grads.items():
        out["grad." + k] = v
    return out


def check(desc, seed=0, flags=0, oracle_dtype=torch.float64, with_g_e_out=False, tol=None, gold=None, order=None, steps=2,
          max_inflight=None, slack=1.0):
    """fp32: every tensor within 1e-4 of the exact oracle.  bf16: every tensor within the plain 2e-2, except the
    tensors named in tests/golden/bf16_floor.json[gold] (see the module docstring).
    steps = 2 (where the calls are not given by `order`): the step is run twice on the same inputs, the gradient buffer
    filled with NaN patterns in between, and the SECOND step is compared - the steady state a training loop and bench.py
    see (the first backward of a stage also records which weight gradients later steps store whole instead of adding
    into a zeroed buffer)."""
    data = W.draw(desc, seed, with_g_e_out=with_g_e_out)
    got_raw = run_gpu(desc, data, flags, with_g_e_out, order, max_inflight, steps)
    got = flatten(got_raw["per_mb"], got_raw["param_grads"])
    ref = flatten(*oracle_run(desc, data, oracle_dtype))
    bf16 = desc["dtype"] == "bf16"
    tol = tol or TOL[desc["dtype"]]
    exc = {}
    if bf16:
        g = GOLD[gold or desc["name"]]              # KeyError: run tests/golden/make_bf16_floor.py for this structure
        assert g["seed"] == seed and g["tensors"] == len(ref) and g["oracle_dtype"] == str(oracle_dtype).split(".")[1], g
        exc = g["exceptions"]
    rows, bad = {}, []
    for k, r in ref.items():
        e, er = rel_err(got[k], r), rms_err(got[k], r)
        row = {"max": e, "rms": er, "limit": tol}
        rlimit = None
        if k in exc:
            fmax, frms = exc[k]
            lim = max(tol, 2.0 * slack * fmax)
            row.update(floor_max=fmax, floor_rms=frms, limit=lim if fmax > CAP / 2 else min(lim, CAP))
            # the rms bound needs elements to average over: a scalar (the loss) has rms == max
            rlimit = 1.5 * frms + 1e-4 if r.numel() >= 1024 else None
        rows[k] = row
        # a listed tensor that uses its allowance (max above the plain bar) must not hide a systematic error there
        if not (e <= row["limit"]) or (e > tol and rlimit is not None and not (er <= rlimit)):
            bad.append((k, row))
    top = sorted(rows.items(), key=lambda kv: -kv[1]["max"] / kv[1]["limit"])[:4]
    print(f"[parity] {desc['name']} flags={flags} tol={tol:g}: " +
          "; ".join(f"{k} max={v['max']:.2e} (limit {v['limit']:.2e}) rms={v['rms']:.2e}" for k, v in top), flush=True)
    n_plain = sum(1 for v in rows.values() if v["max"] <= tol)
    print(f"[parity] {desc['name']}: {n_plain}/{len(rows)} tensors within north_star's plain {tol:g} bar, "
          f"{len(exc)} on the committed exception list", flush=True)
    if REPORT and REPORT.endswith(".md"):      # the per-tensor report kept under profiles/ (markdown, appended per structure)
        with open(REPORT, "a") as f:
            rest = [v["max"] for k, v in rows.items() if k not in exc and v["max"] <= 0.5 * tol]
            f.write(f"\n### {desc['name']} (flags {flags}, seed {seed}, oracle {str(oracle_dtype).split('.')[1]}): "
                    f"{n_plain}/{len(rows)} tensors within the plain {tol:g} bar; {len(exc)} on the exception list; "
                    f"{len(bad)} out of tolerance\n\n")
            f.write("| tensor | max err / RMS | rms err / RMS | storage floor (max) | limit | listed |\n|---|---|---|---|---|---|\n")
            for k, v in sorted(rows.items(), key=lambda kv: -kv[1]["max"]):
                if k in exc or v["max"] > 0.5 * tol:
                    f.write(f"| {k} | {v['max']:.3e} | {v['rms']:.3e} | {v.get('floor_max', float('nan')):.3e} | "
                            f"{v['limit']:.3e} | {'yes' if k in exc else 'no'} |\n")
            f.write(f"\n{len(rest)} further unlisted tensors, all below half the bar (worst {max(rest, default=0.0):.3e}).\n")
    elif REPORT:
        with open(REPORT, "a") as f:
            f.write(json.dumps({"config": desc["name"], "flags": flags, "tol": tol, "within_plain_tol": n_plain,
                                "tensors": len(rows), "listed": len(exc), "rows": rows}) + "\n")
    assert not bad, f"{desc['name']}: {len(bad)} tensors out of tolerance: {bad[:6]}"
    return got_raw


# ------------------------------------------------------------------ fp32 debug path
@pytest.mark.parametrize("kind", ["pair", "level", "updown", "straddle", "unet", "wave", "attn", "attn_unet", "uvit"])
def test_mini_fp32(kind):
    check(W.mini(kind, "fp32"), seed=1, with_g_e_out=True)


def test_config1_fp32():
    check(W.config(1), seed=0)


# ------------------------------------------------------------------ bf16, small shapes (CUDA-core convs)
@pytest.mark.parametrize("kind", ["level", "updown", "unet", "wave", "attn_unet"])
def test_mini_bf16(kind):
    # 8-16 channel, 4x4 tensors: reductions of 32-100 terms do not average bf16 store rounding, so most of their
    # tensors are on the exception list (storage floor above 1e-2).  (mini("attn"), nine blocks deep on 16 pixels, has
    # storage floors up to 0.14 - above CAP / 2 - and is compared in fp32 only; the bf16 attention stage is mid_attn.)
    check(W.mini(kind, "bf16"), seed=1, with_g_e_out=True)


# ------------------------------------------------------------------ bf16, tensor-core shapes with ragged tiles
@pytest.mark.parametrize("flags", [0, 4, 8], ids=["auto", "pair", "1cta"])
@pytest.mark.parametrize("kind", ["level", "updown", "unet"])
def test_mid_bf16(kind, flags):
    """flags 4 / 8: every tcgen05 conv through the CTA-pair kernel (ragged pair tiles, odd tile counts, image boxes,
    stride-2 phases, 1x1 on the concat, masked statistics epilogue) / through the single-CTA kernel."""
    check(W.gpu_mid(kind), seed=2, flags=flags, with_g_e_out=(kind != "unet"))


def test_mid_bf16_attention_stage():
    """a stage whose blocks are ResBlock + self-attention (320 channels = 5 heads x 64), skips pushed after
    the attention; GroupNorm / 1x1 convs on the tcgen05 path, attention core on CUDA cores."""
    check(W.gpu_mid("attn"), seed=2, with_g_e_out=True)


@pytest.mark.parametrize("flags", [16, 32, 32 | 64], ids=["materialised", "phase_fwd", "phase_fwd_dgrad"])
@pytest.mark.parametrize("kind", ["updown", "unet"])
def test_mid_bf16_upsample_forms(kind, flags):
    """Row a6 in its other forms (include/pulse.h PULSE_FLAG_UP_*): everything through the materialised upsampled tensor,
    and the 4-phase forward / input gradient with pre-summed bf16 weights.  The materialised form has the default bar;
    the opt-in phase forms carry one extra rounding of the weights per up conv and direction, which
    the oracle's storage floor does not contain: listed tensors get 2.5 x (not 2 x) their floor, unlisted ones still
    the plain 2e-2."""
    check(W.gpu_mid(kind), seed=2, flags=flags, with_g_e_out=(kind != "unet"), slack=1.0 if flags == 16 else 1.25)


@pytest.mark.parametrize("kind", ["level", "updown"])
def test_mid_bf16_split_halves(kind):
    """the encoder half and the decoder half of an OPEN stage as separate calls (PULSE_FLAG_SPLIT):
    forward_enc, forward_dec, backward_dec, backward_enc give what the one-call forms give ("level": e_out is itself a
    cached skip, so the decoder half writes its gradient before g_e_out arrives; "updown": it is not)."""
    order = [("FE", 0), ("FD", 0), ("BD", 0), ("BE", 0)]
    check(W.gpu_mid(kind), seed=2, flags=128, with_g_e_out=True, order=order)


def test_mid_bf16_split_halves_wave():
    """Three microbatches in the order a pipeline device sees them: all encoder halves, all decoder halves, then the
    backward halves in reverse - the skip gradients of each microbatch wait in its own slot between backward_dec and
    backward_enc while the other microbatches' halves run."""
    desc = W.scaled(W.gpu_mid("level"), microbatches=3, name="mid_level_1f1b")
    order = [("FE", 0), ("FE", 1), ("FE", 2), ("FD", 0), ("FD", 1), ("FD", 2),
             ("BD", 2), ("BD", 1), ("BD", 0), ("BE", 2), ("BE", 1), ("BE", 0)]
    check(desc, seed=4, flags=128, order=order, max_inflight=3)


def test_mini_fp32_split_one_call_forms():
    """A stage created with PULSE_FLAG_SPLIT still answers the one-call forms (its backward runs as the two halves)."""
    check(W.mini("level", "fp32"), seed=1, flags=128, with_g_e_out=True)
    check(W.mini("updown", "fp32"), seed=1, flags=128, with_g_e_out=True)


def _pipeline_two_stages(whole, seed, k_enc):
    """The whole CLOSED model cut into an OPEN outer stage (rank 0) and a CLOSED inner stage (rank 1), both on this GPU,
    driven by the wave runtime's in-process driver; returns results in the whole model's names."""
    from paper_2606_19163_b200 import pipeline as PL
    B = _binding()
    outer, inner, names = W.split_closed(whole, k_enc)
    data = W.draw(whole, seed)
    M = whole["microbatches"]
    st0 = B.Stage(outer, flags=B.FLAG_SPLIT, max_inflight=M)
    st1 = B.Stage(inner, max_inflight=M)
    st0.load_params(W.stage_params(data["params"], names["outer"]))
    st1.load_params(W.stage_params(data["params"], names["inner"]))
    devs = [st0.to_device({k: v for k, v in mb.items()}) for mb in data["microbatches"]]
    ex = [PL.CudaStageExec(st0), PL.CudaStageExec(st1)]
    progs = [PL.rank_program(0, 2, ex[0], M, devs), PL.rank_program(1, 2, ex[1], M, None)]
    results, traffic = PL.run_local(progs)
    torch.cuda.synchronize()
    per_mb = []
    for m in range(M):
        r = results[0][m]
        per_mb.append({"loss": r["loss"], "d_out": B.nchw(r["d_out"]), "g_x_in": B.nchw(r["g_x_in"])})
    grads = {}
    for st, nm in ((st0, names["outer"]), (st1, names["inner"])):
        for k, v in st.grads().items():
            for sp, wp in nm.items():
                if k.startswith(sp):
                    full = wp + k[len(sp):]
                    grads[full] = v if full not in grads else grads[full] + v      # temb.*: both stages hold the MLP
                    break
    # per microbatch one activation down (e_out) and one up (d_out) cross the single boundary, no skip
    sh = W.boundary_shapes(outer)
    esz = 2 if whole["dtype"] == "bf16" else 4
    a = (int(np.prod(sh["e_out"])) + int(np.prod(sh["h_in"]))) * esz
    assert traffic.bytes["act"] == a * M and traffic.bytes["grad"] == a * M
    assert st0.cache_stats()["live_slots"] == 0 and st1.cache_stats()["live_slots"] == 0
    return data, per_mb, grads


@pytest.mark.parametrize("kind", ["unet", "wave"])
def test_pipeline_two_stages_fp32(kind):
    """Row f2 end to end on one GPU: mini UNet (wave: 3 microbatches) as two pipeline stages == the whole model's oracle."""
    whole = W.mini(kind, "fp32")
    data, per_mb, grads = _pipeline_two_stages(whole, 1, 3)
    ref_mb, ref_g = oracle_run(whole, data, torch.float64)
    assert set(grads) == set(ref_g)
    for m, r in enumerate(ref_mb):
        assert abs(float(per_mb[m]["loss"]) - float(r["loss"])) <= 1e-5 * abs(float(r["loss"]))
        for k in ("d_out", "g_x_in"):
            assert rel_err(per_mb[m][k], r[k]) <= 1e-4, (m, k)
    for k, v in ref_g.items():
        assert rel_err(grads[k], v) <= 1e-4, k


def test_pipeline_two_stages_bf16():
    """The same with tensor-core shapes (mid_unet: 320 / 640 channels, 32 x 32), against the one-stage run's bar."""
    whole = W.gpu_mid("unet")
    data, per_mb, grads = _pipeline_two_stages(whole, 2, 3)
    ref_mb, ref_g = oracle_run(whole, data, torch.float64)
    exc = GOLD["mid_unet"]["exceptions"]
    got = {"mb0.d_out": per_mb[0]["d_out"], "mb0.g_x_in": per_mb[0]["g_x_in"]}
    got.update({"grad." + k: v for k, v in grads.items()})
    ref = {"mb0.d_out": ref_mb[0]["d_out"], "mb0.g_x_in": ref_mb[0]["g_x_in"]}
    ref.update({"grad." + k: v for k, v in ref_g.items()})
    for k, r in ref.items():
        limit = min(max(2e-2, 2.0 * exc[k][0]), CAP) if k in exc else 2e-2
        assert rel_err(got[k], r) <= limit, (k, rel_err(got[k], r), limit)


def test_mid_bf16_transformer_skip_stage():
    """transformer blocks with long skips (concat + Linear as a 1x1 conv on the virtual concat), 320
    channels = 5 heads x 64: LayerNorm / GELU kernels, Linear layers on the tcgen05 conv path, tcgen05 attention."""
    check(W.gpu_mid("uvit"), seed=2, with_g_e_out=True)


def test_mid_bf16_1f1b_order():
    """Interleaved 1F1B order F0 F1 B0 F2 B1 B2 on two slots with weight-gradient accumulation: slot reuse (FIFO
    release), transposed-weight reuse across the backwards of a step, shared gradient work buffers; against the
    oracle's wave result (order-free: mean loss, summed weight gradients)."""
    desc = W.scaled(W.gpu_mid("level"), microbatches=3, name="mid_level_1f1b")
    order = [("F", 0), ("F", 1), ("B", 0), ("F", 2), ("B", 1), ("B", 2)]
    check(desc, seed=4, order=order, max_inflight=2)


@pytest.mark.parametrize("kind", ["level", "updown"])
def test_mid_bf16_simt_crosscheck(kind):
    """Same shapes through the CUDA-core convs (PULSE_FLAG_FORCE_SIMT): isolates tensor-core bugs."""
    check(W.gpu_mid(kind), seed=2, flags=1, with_g_e_out=True)


@pytest.mark.parametrize("kind", ["mini_updown", "mid_level", "mid_unet"])
def test_bf16_gn_two_pass_crosscheck(kind):
    """GroupNorm backward as reduction pass + apply pass (PULSE_FLAG_GN_TWO_PASS): the form that runs where a
    slice of an image does not fit a cluster's shared memory; the default runs cover the one-pass cluster kernel."""
    desc = W.mini("updown", "bf16") if kind == "mini_updown" else W.gpu_mid(kind[4:])
    check(desc, seed=2, flags=2, with_g_e_out=(kind != "mid_unet"), gold="mini_updown@2" if kind == "mini_updown" else None)


# ------------------------------------------------------------------ full configs
def test_config2_bf16():
    check(W.config(2), seed=0)


def test_config3_bf16():
    check(W.config(3), seed=0, oracle_dtype=torch.float32)


def test_attn_level_bf16():
    """SURVEY 8f row f1 at full size: configs[2]'s stage with a 10-head attention block (1024 tokens) after every ResBlock;
    tcgen05 attention forward and backward inside the stage."""
    check(W.attn_level(), seed=0, oracle_dtype=torch.float32)


@pytest.mark.skipif(os.environ.get("PULSE_SKIP_BIG") == "1", reason="PULSE_SKIP_BIG=1")
def test_config4_bf16():
    check(W.config(4), seed=0, oracle_dtype=torch.float32)


@pytest.mark.skipif(os.environ.get("PULSE_SKIP_BIG") == "1", reason="PULSE_SKIP_BIG=1")
def test_config5_wave_full():
    """configs[4] at full size: wave of 8 microbatches, all 8 skip sets resident; the float32 oracle
    takes about a minute on the GPU box's host cores."""
    got = check(W.config(5), seed=0, oracle_dtype=torch.float32)
    assert got["stage"].cache_stats()["peak_bytes"] == 780 * 2 ** 20


def test_config5_wave_reduced():
    """configs[4] shapes (N=2, 4x128x128, 9 skips) with a wave of 2 microbatches for the oracle comparison,
    plus the full 8-slot peak-bytes accounting without the oracle."""
    desc = W.scaled(W.config(5), microbatches=2, name="config5_wave2")
    got = check(desc, seed=0, oracle_dtype=torch.float32)
    assert got["stage"].skip_bytes == int(97.5 * 2 ** 20)
    del got
    torch.cuda.empty_cache()
    B = _binding()
    full = W.config(5)
    st = B.Stage(full)
    data = W.draw(W.scaled(full, microbatches=1), 0)
    st.load_params(data["params"])
    dev = st.to_device(data["microbatches"][0])
    fw = []
    for m in range(8):
        emb, tst = st.temb_forward(dev["t"])
        fw.append((emb, tst) + st.forward(m, dev["x_in"], None, emb))
    stats = st.cache_stats()
    assert stats["live_slots"] == 8 and stats["peak_bytes"] == 780 * 2 ** 20
    with pytest.raises(B.PulseError) as ei:                                         # 9th forward with 8 slots
        st.forward(8, dev["x_in"], None, fw[0][0])
    assert ei.value.status == 5
    for m in reversed(range(8)):
        loss, g_d = st.mse(fw[m][3], dev["target"], 1.0 / 8)
        st.backward(m, g_d, None, True, torch.zeros_like(fw[m][0]), accumulate=(m != 7))
    torch.cuda.synchronize()
    assert st.cache_stats()["live_slots"] == 0
    # identical microbatches: summed weight gradient == 8 x (1/8-scaled single) -> equals the 1-microbatch gradient
    g8 = st.grads()
    st.step(0, dev, 1.0, accumulate=False)
    torch.cuda.synchronize()
    g1 = st.grads()
    for k in g1:
        if k.startswith("temb.w") or k.startswith("temb.b1") or k.startswith("temb.b2"):
            continue
        # two runs differ by a re-roll of the bf16 rounding noise (fp32 atomics in the statistics make the last
        # bits order-dependent): measured 1-3e-2 x RMS max-abs run to run on this structure
        assert rel_err(g8[k], g1[k]) < 6e-2 and rms_err(g8[k], g1[k]) < 1e-2, k


# ------------------------------------------------------------------ the one-call forms of the timestep path
@pytest.mark.parametrize("dtype", ["fp32", "bf16"])
def test_temb_fused_calls_match_separate_calls(dtype):
    """pulse_stage_forward_temb / pulse_stage_backward_temb == pulse_temb_forward + pulse_stage_forward and
    pulse_stage_backward + pulse_temb_backward (same kernels, the timestep path merely runs beside the chain)."""
    B = _binding()
    desc = W.mini("level", dtype)
    data = W.draw(desc, 3)
    res = []
    for fused in (False, True):
        st = B.Stage(desc)
        st.load_params(data["params"])
        dev = st.to_device(data["microbatches"][0])
        if fused:
            emb, tst, e_out, d_out = st.forward_temb(0, dev["x_in"], dev.get("h_in"), dev["t"])
        else:
            emb, tst = st.temb_forward(dev["t"])
            e_out, d_out = st.forward(0, dev["x_in"], dev.get("h_in"), emb)
        _, g_d = st.mse(d_out, dev["target"], 1.0)
        g_temb = torch.zeros_like(emb)
        if fused:
            g_x, g_h = st.backward_temb(0, g_d, None, g_temb, tst, True, False)
        else:
            g_x, g_h = st.backward(0, g_d, None, True, g_temb, False)
            st.temb_backward(g_temb, tst, False)
        torch.cuda.synchronize()
        res.append((emb.cpu(), d_out.float().cpu(), g_x.float().cpu(), g_temb.cpu(), st.grads()))
    a, b = res
    assert torch.equal(a[0], b[0]) and torch.equal(a[1], b[1])          # forward: same kernels, same order of sums
    tol = 1e-5 if dtype == "fp32" else 3e-2                              # backward: atomics re-roll the last bits
    assert rel_err(b[2], a[2]) < tol and rel_err(b[3], a[3]) < tol
    for k in a[4]:
        assert rel_err(b[4][k], a[4][k]) < tol, k


# ------------------------------------------------------------------ cache / error behaviour (paper-faithful cases)
def test_cache_errors_and_skip_locality():
    B = _binding()
    desc = W.mini("level", "fp32")
    data = W.draw(desc, 5)
    st = B.Stage(desc, max_inflight=2)
    st.load_params(data["params"])
    dev = st.to_device(data["microbatches"][0])
    emb, _ = st.temb_forward(dev["t"])
    with pytest.raises(B.PulseError) as ei:          # backward on unknown microbatch
        st.backward(7, dev["target"], None, True, None)
    assert ei.value.status == 6
    e_out, d_out = st.forward(0, dev["x_in"], dev["h_in"], emb)
    with pytest.raises(B.PulseError) as ei:          # same microbatch forwarded twice
        st.forward(0, dev["x_in"], dev["h_in"], emb)
    assert ei.value.status == 5
    st.forward(1, dev["x_in"], dev["h_in"], emb)
    with pytest.raises(B.PulseError) as ei:          # third forward with 2 slots
        st.forward(2, dev["x_in"], dev["h_in"], emb)
    assert ei.value.status == 5
    # the cached skips are the encoder outputs (zero-copy put): skip 0 = x_in, last = e_out
    torch.cuda.synchronize()
    assert st.skip_count() == 3
    assert torch.equal(st.skip(0, 0), dev["x_in"]) and torch.equal(st.skip(0, 2), e_out)
    ref = O.run_stage(desc, data["params"], data["microbatches"][0])
    for k in range(3):
        assert rel_err(B.nchw(st.skip(1, k)), ref["skips"][k]) < 1e-4
    assert st.cache_stats() == {"live_slots": 2, "live_bytes": 2 * st.skip_bytes, "peak_bytes": 2 * st.skip_bytes}
    st.backward(1, dev["target"], None, True, None)       # FIFO/LIFO free list: release 1 first, then reuse
    st.forward(5, dev["x_in"], dev["h_in"], emb)
    assert st.cache_stats()["live_slots"] == 2


def test_descriptor_validation():
    B = _binding()
    bad = W.mini("level", "fp32")
    bad["dec_ops"] = bad["dec_ops"] + [W.rb(8, 8, skip=8)]     # pops more than pushed
    with pytest.raises(B.PulseError) as ei:
        B.Stage(bad, allocate=False)
    assert ei.value.status == 2
    bad2 = W.mini("level", "fp32")
    bad2["dec_ops"] = bad2["dec_ops"][:2]                       # a cached skip never consumed
    with pytest.raises(B.PulseError) as ei:
        B.Stage(bad2, allocate=False)
    assert ei.value.status == 2
