#!/usr/bin/env python
"""bench.py - one "step" = the whole hot path (temb -> stage forward -> MSE -> stage backward
-> temb backward; for configs[4] the wave F0..F7,B7..B0) over one batch of synthetic input.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 2] [--impl ours|reference]

Prints ONE JSON line (contract in the task statement / DESIGN.md "Measurement").  N > 1 runs
N independent replicas (the path has no exchange step - "replicas only").
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402
import torch  # noqa: E402

from paper_2606_19163_b200 import workloads as W  # noqa: E402

METRIC = "stage fwd+bwd samples/s"
WORKLOADS = {1: "configs[0]: tiny collocated pair, fp32 debug path", 2: "configs[1]: SD1.5-shaped level-1 stage, "
             "2 enc + 3 dec ResBlocks 320ch, microbatch 4, 64x64", 3: "configs[2]: level-2 stage with down/up, "
             "microbatch 8, 32x32", 4: "configs[3]: full conv-only SD1.5-shaped UNet, microbatch 8, 4x64x64",
             5: "configs[4]: SDXL-shaped stage, wave of 8 microbatches of 2, 4x128x128",
             6: "SURVEY 8f f1: configs[2]'s level-2 stage with a self-attention block (10 heads x 64, 1024 tokens) after "
                "every ResBlock, microbatch 8, 32x32"}


def conv_flops_fwd(desc) -> float:
    """Algorithmic forward FLOPs of the convs + linears of one microbatch: 2 N Ho Wo Cout Cin k^2
    (SURVEY.md 8d); the nominal 9-tap count for the up conv."""
    n, h, w = desc["n"], desc["h"], desc["w"]
    T = desc["temb"]["dim"]
    fl = 0.0
    if desc["temb"]["kind"] == "mlp":
        fl += 2.0 * n * T * (desc["temb"]["d0"] + T)
    sk = W.skip_channels_pushed(desc)
    hh, ww = h, w
    for op in desc["enc_ops"] + desc["mid_ops"]:
        if op["kind"] == "down":
            hh, ww = hh // 2, ww // 2
        fl += _op_flops(op, n, hh, ww, T)
    if desc["link"] == "open" and sk:
        hh, ww = sk[-1][1], sk[-1][2]
    for op in desc["dec_ops"]:
        if op["kind"] == "up":
            hh, ww = 2 * hh, 2 * ww
        fl += _op_flops(op, n, hh, ww, T)
    return fl


def _op_flops(op, n, h, w, T):
    ci, co = op["cin"] + op["skip"], op["cout"]
    pix = 2.0 * n * h * w
    if op["kind"] == "resblock":
        f = pix * co * ci * 9 + pix * co * co * 9 + 2.0 * n * co * T
        if ci != co:
            f += pix * co * ci
        return f
    if op["kind"] == "attn":      # qkv and proj 1x1 convs + Q K^T and P V (4 n tokens^2 c)
        return pix * ci * 3 * ci + pix * ci * ci + 4.0 * n * (h * w) ** 2 * ci
    return pix * co * ci * 9


class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.lines, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.perf_counter(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        rows = [l.split(",") for t, l in self.lines if t0 <= t <= t1] or [l.split(",") for _, l in self.lines[-3:]]
        sm, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in rows:
            try:
                sm.append(float(r[0])); mx = max(mx, float(r[1]))
                for nm, v in zip(names, r[3:7]):
                    if v.strip().lower() == "active":
                        reasons.add(nm)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx or None, "reasons": sorted(reasons),
                "samples": len(sm)}


def max_over_ranks(x: float, dist, device="cuda") -> float:
    """Replicas only: the job's time is the slowest replica's (max over ranks)."""
    if dist is None:
        return float(x)
    t = torch.tensor([x], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def job_throughput(samples_per_rank: int, world: int, seconds_max: float) -> float:
    """Whole-job samples/s of `world` independent replicas (weak scaling)."""
    return world * samples_per_rank / seconds_max


def oracle_time(desc, data, budget_note):
    from oracle import pulse_oracle as O
    t0 = time.perf_counter()
    if desc["microbatches"] == 1:
        O.run_stage(desc, data["params"], data["microbatches"][0])
    else:
        O.run_wave(desc, data["params"], data["microbatches"])
    dt = time.perf_counter() - t0
    samples = desc["n"] * desc["microbatches"]
    return {"value": samples / dt, "unit": "samples/s", "cores": torch.get_num_threads(), "kind": "oracle",
            "sample": budget_note, "seconds": dt}


def reference_sample(desc, full=False):
    """Bounded sample of the workload for the CPU oracle: the stage structure and spatial size of the
    config with the microbatch cut to 1 sample (GroupNorm and every conv are per-sample, so cost
    scales linearly with N) and, for the wave, one microbatch."""
    n = desc["n"] if (full and desc["name"] in ("config1", "config2")) else 1
    d = W.scaled(desc, n=n, microbatches=1)
    return d, f"{desc['name']} structure at N={n} sample(s), 1 microbatch, fp64 oracle as it stands"


def run_reference(args):
    """The oracle as it stands on the host cores: configs 1-2 at the SAME microbatch as our arm, configs 3-5 on the
    bounded sample (one sample of one microbatch); every step is one oracle forward + backward."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    desc = W.config(args.config)
    d1, note = reference_sample(desc, full=True)
    data = W.draw(d1, 0)
    for _ in range(args.warmup):
        oracle_time(d1, data, note)
    ts = []
    for _ in range(args.steps):
        r = oracle_time(d1, data, note)
        ts.append(r["seconds"])
    dt = float(np.mean(ts))
    val = d1["n"] / dt
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": "samples/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic (seeded N(0,1), DESIGN.md)",
            "config": {"workload": WORKLOADS[args.config], "sample": note, "samples_per_step": d1["n"],
                       "microbatches": 1},
            "cpu_baseline": {"value": val, "unit": "samples/s", "cores": torch.get_num_threads(), "kind": "oracle",
                             "sample": note},
            "e2e": {"value": val, "unit": "samples/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=2)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--no-graph", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--brief", action="store_true", help="device-timed step only: no per-class brackets, stand-alone "
                    "kernels, e2e, CPU baseline or other configs (what the `configs` object of the full line runs)")
    ap.add_argument("--no-other-configs", action="store_true")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    args.warmup = max(args.warmup, 3)

    from paper_2606_19163_b200 import binding as B
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    desc = W.config(args.config)
    M = desc["microbatches"]
    data = W.draw(desc, 0)
    st = B.Stage(desc)
    st.load_params(data["params"])
    devs = [st.to_device(mb) for mb in data["microbatches"]]
    samples = desc["n"] * M
    flops_step = 3.0 * conv_flops_fwd(desc) * M
    loss = torch.zeros(1, dtype=torch.float32, device="cuda")

    def step(devs=devs):
        """One pass of the whole hot path; returns the tensors that leave the stage (what a neighbouring stage or the
        host receives: e_out, d_out, g_x_in, g_h_in of every microbatch)."""
        loss.zero_()
        if M == 1:
            r = st.step(0, devs[0], 1.0, accumulate=False, loss=loss)
            return [r[k] for k in ("e_out", "d_out", "g_x_in", "g_h_in") if r.get(k) is not None]
        fw, outs = [], []
        for m, dev in enumerate(devs):                      # wave: F0..F{M-1}
            fw.append(st.forward_temb(m, dev["x_in"], dev.get("h_in"), dev["t"]))
        for m in reversed(range(M)):                        # B{M-1}..B0
            emb, tst, e_out, d_out = fw[m]
            _, g_d = st.mse(d_out, devs[m]["target"], 1.0 / M, loss)
            g_temb = torch.zeros_like(emb)
            g_x_in, g_h_in = st.backward_temb(m, g_d, None, g_temb, tst, True, accumulate=(m != M - 1))
            outs += [t for t in (e_out, d_out, g_x_in, g_h_in) if t is not None]
        return outs

    # eager warm-up (first launches set function attributes, build tensor maps)
    for _ in range(2):
        step()
    torch.cuda.synchronize()
    l0 = st.launches()
    step()
    torch.cuda.synchronize()
    launches_per_step = st.launches() - l0 + M       # + the MSE kernel(s), which take no stage handle

    graph = None
    graph_outs = [None, None]          # the step's outputs inside each captured graph (static addresses)
    if not args.no_graph:
        try:
            graph = torch.cuda.CUDAGraph()
            with torch.cuda.graph(graph):
                graph_outs[0] = step()
        except Exception as e:      # keep measuring eagerly, say so
            graph = None
            sys.stderr.write(f"bench: CUDA graph capture failed ({e}); timing eager launches\n")
            torch.cuda.synchronize()
    run = graph.replay if graph is not None else step

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        run()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    e0.record()
    for _ in range(args.steps):
        run()
    e1.record()
    barrier()
    t1 = time.perf_counter()
    ms = max_over_ranks(e0.elapsed_time(e1), dist)
    clocks = sampler.stop(t0, t1) if rank == 0 else None
    ms_per_step = ms / args.steps
    value = job_throughput(samples, world, ms_per_step * 1e-3)

    tflops = world * flops_step / (ms_per_step * 1e-3) / 1e12
    if args.brief:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        if rank == 0:
            print(json.dumps({"metric": METRIC, "value": value, "unit": "samples/s", "n_gpus": world, "steps": args.steps,
                              "warmup": args.warmup, "ms_per_step": ms_per_step, "tflops": tflops,
                              "frac_of_bf16_peak_nominal_2250": tflops / world / 2250.0, "clocks": clocks,
                              "gpu_launches": int(launches_per_step * args.steps),
                              "config": {"workload": WORKLOADS[args.config], "samples_per_step": samples, "microbatches": M,
                                         "launch": "CUDA graph replay" if graph is not None else "eager launches"},
                              "peak_skip_cache_bytes": st.cache_stats()["peak_bytes"]}))
        return

    # ---- per-kernel-class times, live, same K steps launched eagerly with event brackets -----------------
    # Eager launches are CPU-bound here (eager_ms > ms_per_step): a bracket would also count the time the GPU waits
    # for the CPU to enqueue the kernel.  So every profiled step is enqueued behind a ~5 ms device-side sleep: by the
    # time the GPU reaches the step, its launches and events are all queued and the brackets hold GPU time only.
    torch.cuda.synchronize()
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record()
    for _ in range(args.steps):
        step()
    p1.record()
    torch.cuda.synchronize()
    eager_ms = p0.elapsed_time(p1) / args.steps
    st.profile(True)
    for _ in range(args.steps):
        torch.cuda._sleep(10_000_000)
        step()
        torch.cuda.synchronize()
    prof = st.profile_read()
    st.profile(False)

    # ---- the same kernel classes inside the CUDA-graph replays (CUPTI kernel records through torch.profiler) ----
    in_graph = None
    if graph is not None and rank == 0:
        try:
            from torch.profiler import profile, ProfilerActivity
            reps = 3
            with profile(activities=[ProfilerActivity.CUDA]) as tp:
                for _ in range(reps):
                    graph.replay()
                torch.cuda.synchronize()
            in_graph = {}
            for e in tp.events():
                if e.device_type != torch.autograd.DeviceType.CUDA:
                    continue
                nm = e.name
                if "wgrad_tc" in nm: k = "wgrad_tc"
                elif "conv_tc" in nm: k = "conv_tc"
                elif "conv_simt" in nm or "wgrad_simt" in nm or "thin_" in nm: k = "conv_simt"
                elif "gn_bwd" in nm: k = "gn_bwd"
                elif "gn_apply" in nm or "chan_stats" in nm: k = "gn_fwd"
                else: k = "other"
                a = in_graph.setdefault(k, [0, 0.0])
                a[0] += 1
                a[1] += (e.time_range.end - e.time_range.start) / 1e3
            in_graph = {k: {"launches_per_step": v[0] / reps, "ms_per_step": v[1] / reps} for k, v in in_graph.items()}
        except Exception as ex:      # the event-bracket numbers above remain
            sys.stderr.write(f"bench: CUPTI kernel timing unavailable ({ex})\n")
            in_graph = None

    # ---- the dominant kernel alone: the commonest 3x3 conv shape of the config, launched back to back through the
    # C-ABI (pulse_conv2d) between two events.  This is the kernel without the event-bracket overhead of the per-class
    # numbers above; it is compared with the BURST peak (a kernel timed alone), the brackets with the sustained one.
    alone = None
    if rank == 0 and desc["dtype"] == "bf16":
        try:
            ops = [o for o in desc["enc_ops"] + desc.get("mid_ops", []) + desc["dec_ops"] if o["kind"] == "resblock"]
            c = ops[0]["cout"]
            hh, ww = devs[0]["x_in"].shape[1], devs[0]["x_in"].shape[2]
            gen = torch.Generator(device="cuda").manual_seed(1)
            xa = torch.randn((desc["n"], hh, ww, c), device="cuda", generator=gen).to(torch.bfloat16)
            wa = (torch.randn((c, 3, 3, c), device="cuda", generator=gen) * 0.02).to(torch.bfloat16)
            ba = torch.zeros(c, device="cuda", dtype=torch.bfloat16)
            for _ in range(5):
                B.conv2d(xa, wa, bias=ba)
            reps = 50
            a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            a0.record()
            for _ in range(reps):
                B.conv2d(xa, wa, bias=ba)
            a1.record()
            torch.cuda.synchronize()
            us = a0.elapsed_time(a1) * 1e3 / reps
            fl = 2.0 * desc["n"] * hh * ww * c * c * 9
            alone = {"shape": f"M={desc['n'] * hh * ww}, N={c}, K={9 * c}", "us_per_launch": us,
                     "tflops": fl / (us * 1e-6) / 1e12, "launches": reps}
        except Exception as ex:
            sys.stderr.write(f"bench: stand-alone conv timing skipped ({ex})\n")

    # ---- the GroupNorm + SiLU kernels alone (north_star "Reporting": achieved HBM GB/s of the norm kernels): the
    # config's commonest site shapes launched back to back through the C-ABI (captured in one CUDA graph per
    # measurement, so that the CPU launch rate does not bound 10 us kernels), rotating over enough buffer sets that
    # the working set exceeds the 126 MB L2 ("hbm") and on one set ("l2_hot": what the step sees, where the producer
    # has just written the tensor).  Algorithmic bytes: forward read x + write a; backward read x, g_a (+ add),
    # write g_x.
    gn_alone = None
    if rank == 0 and desc["dtype"] == "bf16":
        try:
            ops = [o for o in desc["enc_ops"] + desc.get("mid_ops", []) + desc["dec_ops"] if o["kind"] == "resblock"]
            c = ops[0]["cout"]
            n_, hh, ww = desc["n"], devs[0]["x_in"].shape[1], devs[0]["x_in"].shape[2]
            gen = torch.Generator(device="cuda").manual_seed(2)
            rnd = lambda ch: torch.randn((n_, hh, ww, ch), device="cuda", generator=gen).to(torch.bfloat16)
            gn_alone = {}
            for name, c1 in (("single", 0), ("concat", c)):
                C_ = c + c1
                elems = n_ * hh * ww * C_
                nset = max(2, int(160e6 // (elems * 2 * 3)) + 1)
                sets = []
                for _ in range(nset):
                    x0, x1, ga = rnd(c), (rnd(c1) if c1 else None), rnd(C_)
                    sets.append({"x0": x0, "x1": x1, "g_a": ga, "a": torch.empty_like(ga), "g0": torch.empty_like(x0),
                                 "g1": None if x1 is None else torch.empty_like(x1)})
                gam = torch.ones(C_, device="cuda", dtype=torch.bfloat16)
                bet = torch.zeros(C_, device="cuda", dtype=torch.bfloat16)
                scr = torch.empty(n_ * 2 * C_, device="cuda", dtype=torch.float32)
                dg, db = torch.zeros(C_, device="cuda"), torch.zeros(C_, device="cuda")
                for q in sets:
                    q["stats"] = B.groupnorm_silu(q["x0"], gam, bet, desc["groups"], desc["eps"], x1=q["x1"])[1]

                def fwd(q):
                    B.lib.pulse_groupnorm_silu(B.BF16, B._ptr(q["x0"]), c, B._ptr(q["x1"]), c1, n_, hh, ww, desc["groups"],
                                               desc["eps"], B._ptr(gam), B._ptr(bet), B._ptr(q["stats"]), 1, B._ptr(q["a"]),
                                               B._stream())

                def bwd(q):
                    B.lib.pulse_groupnorm_silu_backward(B.BF16, 0, 1, B._ptr(q["g_a"]), B._ptr(q["x0"]), c, B._ptr(q["x1"]), c1,
                                                        n_, hh, ww, desc["groups"], desc["eps"], B._ptr(gam), B._ptr(bet),
                                                        B._ptr(q["stats"]), B._ptr(scr), None, B._ptr(q["g0"]), 0,
                                                        B._ptr(q["g1"]), 0, B._ptr(dg), B._ptr(db), B._stream())

                for kind, fn, nbytes in (("fwd", fwd, 2 * 2 * elems), ("bwd", bwd, 3 * 2 * elems)):
                    row = {"shape": f"[{n_},{hh},{ww},{c}" + (f"|{c1}]" if c1 else "]"), "bytes": nbytes}
                    for mode, use in (("hbm", sets), ("l2_hot", sets[:1])):
                        reps, replays = 10 * len(sets), 5
                        for q in use:
                            fn(q)
                        torch.cuda.synchronize()
                        gg = torch.cuda.CUDAGraph()      # one graph of `reps` launches: a 10 us kernel outruns ctypes calls
                        with torch.cuda.graph(gg):
                            for i in range(reps):
                                fn(use[i % len(use)])
                        gg.replay()
                        a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                        torch.cuda.synchronize()
                        a0.record()
                        for _ in range(replays):
                            gg.replay()
                        a1.record()
                        torch.cuda.synchronize()
                        us = a0.elapsed_time(a1) * 1e3 / (reps * replays)
                        del gg
                        row[mode] = {"us_per_call": us, "gbs": nbytes / (us * 1e-6) / 1e9, "buffer_sets": len(use)}
                    gn_alone[f"{kind}_{name}"] = row
        except Exception as ex:
            sys.stderr.write(f"bench: stand-alone GroupNorm timing skipped ({ex})\n")
            gn_alone = None

    # ---- the attention core alone at the level-2 shape of configs[2] (8 images, 32 x 32 tokens, 640
    # channels = 10 heads x 64): tcgen05 forward, CUDA-core forward and backward.  FLOPs: forward 4 n T^2 C, backward 10 n T^2 C;
    # the forward's roofline is the exponential: n heads T^2 MUFU.EX2 at 16 per clock per SM
    attn_alone = None
    if rank == 0 and desc["dtype"] == "bf16":
        try:
            an, aT, aC, ah = 8, 1024, 640, 10
            gen = torch.Generator(device="cuda").manual_seed(3)
            aq = torch.randn((an, aT, 3 * aC), device="cuda", generator=gen).to(torch.bfloat16)
            ago = torch.randn((an, aT, aC), device="cuda", generator=gen).to(torch.bfloat16)
            _, ast = B.attention(aq, ah)

            def timed(fn, reps):
                fn(); torch.cuda.synchronize()
                a0, a1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                a0.record()
                for _ in range(reps):
                    fn()
                a1.record()
                torch.cuda.synchronize()
                return a0.elapsed_time(a1) * 1e3 / reps
            f_tc = timed(lambda: B.attention(aq, ah), 20)
            f_simt = timed(lambda: B.attention(aq, ah, force_simt=True), 3)
            b_tc = timed(lambda: B.attention_backward(aq, ago, ah, ast), 20)
            b_simt = timed(lambda: B.attention_backward(aq, ago, ah, ast, force_simt=True), 3)
            ffl, bfl = 4.0 * an * aT * aT * aC, 10.0 * an * aT * aT * aC
            sm_clk = 148 * 16 * 1.9e9          # MUFU lanes per second at 1.9 GHz (B200_PROFILING.md unit counts)
            attn_alone = {"shape": f"n={an}, tokens={aT}, channels={aC}, heads={ah}",
                          "fwd_tcgen05": {"us": f_tc, "tflops": ffl / (f_tc * 1e-6) / 1e12, "bound": "alu (MUFU.EX2)",
                                          "frac_of_exp_peak": an * ah * aT * aT / (f_tc * 1e-6) / sm_clk},
                          "fwd_cuda_core": {"us": f_simt, "tflops": ffl / (f_simt * 1e-6) / 1e12},
                          "bwd_tcgen05": {"us": b_tc, "tflops": bfl / (b_tc * 1e-6) / 1e12, "bound": "alu (MUFU.EX2)",
                                          "frac_of_exp_peak": 3.0 * an * ah * aT * aT / (b_tc * 1e-6) / sm_clk},
                          "bwd_cuda_core": {"us": b_simt, "tflops": bfl / (b_simt * 1e-6) / 1e12}}
        except Exception as ex:
            sys.stderr.write(f"bench: stand-alone attention timing skipped ({ex})\n")

    # ---- end to end through the public API with HOST buffers -----------------------------------------------
    host = []
    for mb in data["microbatches"]:
        h = {}
        for k, v in mb.items():
            if k == "t":
                h[k] = torch.as_tensor(v).pin_memory()
            else:       # NHWC in the stage dtype, pinned
                h[k] = torch.as_tensor(np.ascontiguousarray(np.transpose(v, (0, 2, 3, 1)))).to(st.tdtype).pin_memory()
        host.append(h)
    h2d = sum(v.numel() * v.element_size() for h in host for v in h.values())
    loss_host = torch.zeros(1, dtype=torch.float32).pin_memory()

    # Pipelined like a training input pipeline: the H2D copies of step i+1 run on a copy stream into the second of
    # two device input sets while step i computes from the first; the step is captured once per input set (two
    # graphs), so it reads the H2D destination directly; the loss of step i is read back asynchronously and consumed
    # one step later.
    copy_stream = torch.cuda.Stream()
    d2h_stream = torch.cuda.Stream()
    main = torch.cuda.current_stream()
    stg = [devs, [{k: torch.empty_like(v) for k, v in devs[m].items()} for m in range(M)]]
    for m in range(M):
        for k, v in devs[m].items():
            stg[1][m][k].copy_(v)
    runs = [run, run]
    if graph is not None:
        try:
            step(stg[1]); torch.cuda.synchronize()          # eager once: tensor maps of the second input set
            g2 = torch.cuda.CUDAGraph()
            with torch.cuda.graph(g2):
                graph_outs[1] = step(stg[1])
            runs = [graph.replay, g2.replay]
        except Exception as e:
            sys.stderr.write(f"bench: second CUDA graph failed ({e}); e2e copies into one input set\n")
            torch.cuda.synchronize()
            runs = None
    else:
        runs = [step, lambda: step(stg[1])]
    ev_ready = [torch.cuda.Event(), torch.cuda.Event()]
    ev_free = [torch.cuda.Event(), torch.cuda.Event()]
    loss_dev = [torch.zeros(1, dtype=torch.float32, device="cuda") for _ in range(2)]
    loss_pin = [torch.zeros(1, dtype=torch.float32).pin_memory() for _ in range(2)]
    ev_loss = [torch.cuda.Event(), torch.cuda.Event()]
    ev_step = [torch.cuda.Event(), torch.cuda.Event()]
    # the step's results go back to pinned host buffers every step (what leaves the stage: e_out, d_out, g_x_in, g_h_in
    # of every microbatch, and the loss); the fp32 weight gradients stay on the device for the optimizer, as in training
    shapes0 = graph_outs[0] if graph_outs[0] is not None else step()
    torch.cuda.synchronize()
    out_pin = [[torch.empty(t.shape, dtype=t.dtype).pin_memory() for t in shapes0] for _ in range(2)]
    d2h = sum(t.numel() * t.element_size() for t in shapes0) + 4

    def prefetch(i):
        b = i % 2
        with torch.cuda.stream(copy_stream):
            copy_stream.wait_event(ev_free[b])              # staging buffer b was consumed by step i-2
            for m in range(M):
                for k, v in host[m].items():
                    stg[b][m][k].copy_(v, non_blocking=True)
            ev_ready[b].record(copy_stream)

    def e2e_run(nsteps):
        losses = []
        for b in range(2):
            ev_free[b].record(main)
            ev_loss[b].record(d2h_stream)
        prefetch(0)
        for i in range(nsteps):
            b = i % 2
            if i + 1 < nsteps:
                prefetch(i + 1)
            main.wait_event(ev_ready[b])
            main.wait_event(ev_loss[b])                      # the outputs of step i - 2 (same buffers) have been read back
            if runs is None:                                 # fallback: one graph, D2D from the staging set
                if b == 1:
                    for m in range(M):
                        for k in host[m]:
                            devs[m][k].copy_(stg[1][m][k], non_blocking=True)
                outs = run() or graph_outs[0]
            else:
                outs = runs[b]() or graph_outs[b]
            ev_free[b].record(main)                          # input set b may be overwritten by the H2D of step i + 2
            loss_dev[b].copy_(loss, non_blocking=True)
            ev_step[b].record(main)
            with torch.cuda.stream(d2h_stream):              # the D2H reads do not sit in the compute stream
                d2h_stream.wait_event(ev_step[b])
                for dst, src in zip(out_pin[b], outs):
                    dst.copy_(src, non_blocking=True)
                loss_pin[b].copy_(loss_dev[b], non_blocking=True)
                ev_loss[b].record(d2h_stream)
            if i >= 1:                                       # consume the previous step's loss
                ev_loss[1 - b].synchronize()
                losses.append(float(loss_pin[1 - b][0]))
        ev_loss[(nsteps - 1) % 2].synchronize()
        losses.append(float(loss_pin[(nsteps - 1) % 2][0]))
        return losses

    e2e_run(3)
    barrier()
    w0 = time.perf_counter()
    last_loss = e2e_run(args.steps)[-1]
    barrier()
    e2e_s = (time.perf_counter() - w0) / args.steps
    e2e_s = max_over_ranks(e2e_s, dist)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    peaks = {}
    try:
        peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        pass
    # Every tensor figure of this line is a BURST measurement (a kernel or a 30 ms timed region at full clocks, not a
    # seconds-long loop under the power cap), so the denominator is the burst cuBLAS figure; the sustained figure and
    # the nominal 2250 TFLOP/s that north_star's ">= 60 %" is stated on are reported beside it.
    tf_burst = peaks.get("bf16_tflops") or 1590.0
    tf_sustained = peaks.get("bf16_tflops_sustained") or 1400.0
    hbm_peak = peaks.get("hbm_gbs") or 6650.0
    for row in (gn_alone or {}).values():
        for mode in ("hbm", "l2_hot"):
            row[mode]["frac_of_hbm_peak"] = row[mode]["gbs"] / hbm_peak
    peak_src = ("measured (MEASURED_PEAKS.json: bf16_tflops = cuBLAS burst, hbm_gbs = copy)" if peaks
                else "fallback (B200_PROFILING.md: 1.59 PFLOP/s burst, 6.65 TB/s)")
    K = args.steps
    kern = {}
    for k, v in prof.items():
        if v["launches"] == 0:
            continue
        row = {"ms_per_step": v["ms"] / K, "launches_per_step": v["launches"] / K}
        if v["flops"]:
            row["tflops"] = v["flops"] / (v["ms"] * 1e-3) / 1e12
            row["frac_of_peak"] = row["tflops"] / tf_burst
        if v["bytes"]:
            row["gbs"] = v["bytes"] / (v["ms"] * 1e-3) / 1e9
            row["frac_of_peak"] = row["gbs"] / hbm_peak
        if in_graph and k in in_graph:      # same class inside the graph replays
            g = in_graph[k]
            row["in_graph_ms_per_step"] = g["ms_per_step"]
            if v["flops"]:
                row["in_graph_tflops"] = v["flops"] / K / (g["ms_per_step"] * 1e-3) / 1e12
            if v["bytes"]:
                row["in_graph_gbs"] = v["bytes"] / K / (g["ms_per_step"] * 1e-3) / 1e9
        kern[k] = row
    traffic, traffic_src = None, None
    try:
        tj = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))
        traffic = tj.get(f"config{args.config}.conv_tc")
        traffic_src = tj.get("source", "profiles/traffic.json") + " (an ncu --set full capture of an earlier run, NOT measured by this run)"
    except Exception:
        pass
    dom = kern.get("conv_tc") or kern.get("conv_simt") or {}
    ach = dom.get("tflops") or 0.0
    roofline = {"kernel": "conv_tc2_k (tcgen05 cta_group::2 implicit-GEMM conv, fprop + dgrad)" if "conv_tc" in kern else "conv_simt_k",
                "timing": "CUDA-event brackets around every launch of the class, K eager steps on the launch stream, each step enqueued behind a device-side sleep so that the brackets hold no CPU launch time (burst clocks)",
                "bound": "tensor", "achieved": dom.get("tflops"), "peak": tf_burst, "unit": "TFLOP/s",
                "frac": ach / tf_burst, "peak_source": peak_src,
                "frac_of_nominal_2250": ach / 2250.0, "frac_of_sustained": ach / tf_sustained, "peak_sustained": tf_sustained,
                "achieved_in_graph": dom.get("in_graph_tflops"),
                "frac_in_graph": (dom.get("in_graph_tflops") or 0.0) / tf_burst,
                "traffic": traffic, "traffic_source": traffic_src,
                "alone": None if alone is None else dict(alone, peak_burst=tf_burst, frac_of_burst=alone["tflops"] / tf_burst,
                                                         frac_of_nominal_2250=alone["tflops"] / 2250.0),
                # share of the step's kernel time (same event brackets, all classes): comparable with the share in the
                # ncu launch list under profiles/
                "share_of_step": (dom.get("ms_per_step") or 0.0) / max(1e-9, sum(r["ms_per_step"] for r in kern.values()))}
    line = {"metric": METRIC, "value": value, "unit": "samples/s", "n_gpus": world, "steps": K, "warmup": args.warmup,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16" if desc["dtype"] == "bf16" else "f32", "data": "synthetic (seeded N(0,1), DESIGN.md)",
            "config": {"workload": WORKLOADS[args.config], "samples_per_step": samples, "microbatches": M,
                       "l2": f"no flush: per-step working set {(st.stash_bytes * M + st.work_bytes + st.skip_bytes * M + st.param_bytes + st.grad_bytes) / 2**20:.0f} MiB > 126 MiB L2",
                       "launch": "CUDA graph replay" if graph is not None else "eager launches",
                       "parallelism": "replicas only" if world > 1 else "single GPU"},
            "tflops": tflops,
            "frac_of_bf16_peak_nominal_2250": tflops / world / 2250.0,
            "frac_of_bf16_peak_measured": tflops / world / tf_burst, "peak_measured": tf_burst,
            "clocks": clocks, "gpu_launches": int(launches_per_step * K), "roofline": roofline,
            "kernels": kern, "gn_alone": gn_alone, "attn_alone": attn_alone, "eager_ms_per_step": eager_ms, "loss": last_loss,
            "e2e": {"value": world * samples / e2e_s, "unit": "samples/s", "h2d_bytes_per_step": h2d,
                    "d2h_bytes_per_step": d2h, "ms_per_step": e2e_s * 1e3,
                    "d2h": "e_out, d_out, g_x_in, g_h_in of every microbatch and the loss, into pinned host buffers; the fp32 weight gradients stay on the device (optimizer state)",
                    "pipelining": "H2D of step i+1 (copy stream, into the second of two device input sets, one CUDA graph per set) and the D2H of step i-1 (second copy stream) overlap the compute of step i; "
                                  "results consumed one step later"},
            "peak_skip_cache_bytes": st.cache_stats()["peak_bytes"]}
    if world == 1 and not args.no_cpu_baseline:
        d1, note = reference_sample(desc, full=True)
        line["cpu_baseline"] = {k: v for k, v in oracle_time(d1, W.draw(d1, 0), note).items() if k != "seconds"}
    # ---- the other tensor-core configs, driver-run: device-timed graph replays only (10 steps, no CPU leg), each in
    # its own process (180 GB of HBM: the parent's ~2 GB stay allocated)
    if world == 1 and args.config == 2 and not args.no_other_configs:
        torch.cuda.empty_cache()
        others = {}
        for c in (3, 4, 5, 6):
            try:
                r = subprocess.run([sys.executable, os.path.abspath(__file__), "--config", str(c), "--steps", "10", "--warmup", "3",
                                    "--brief"], capture_output=True, text=True, timeout=900)
                last = [l for l in r.stdout.splitlines() if l.startswith("{")]
                others[f"config{c}"] = json.loads(last[-1]) if last else {"error": (r.stderr or "no output")[-300:]}
            except Exception as ex:
                others[f"config{c}"] = {"error": str(ex)[:300]}
        line["configs"] = others
    print(json.dumps(line))


if __name__ == "__main__":
    main()
