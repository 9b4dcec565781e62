"""Wave runtime over D devices: the schedule, the transports
and the traffic accounting, on the CPU with a small arithmetic stand-in for the stage executor (the executor of the
product, pipeline.CudaStageExec over libpulse.so, is exercised on the GPU in tests/test_gpu_parity.py).

What is checked: the pipelined result equals the plain sequential composition (torch autograd of the same arithmetic);
every microbatch's calls arrive in the order forward_enc -> forward_dec -> backward_dec -> backward_enc; the bytes that
cross device boundaries are 2 (D-1) a per microbatch and direction and contain no skip tensor; the same programs over
torch.distributed (gloo, world size 2) give the same numbers as the in-process driver."""
import os
import socket

import pytest
import torch
import torch.multiprocessing as mp

from paper_2606_19163_b200 import pipeline as PL


class ToyExec:
    """Stand-in stage: enc e = x w + 1 (e is also the cached skip); dec d = h + v skip; innermost d = u x^2.
    Keeps the skip and its gradient locally per microbatch, like a PULSE stage."""

    def __init__(self, rank, world, log):
        self.w, self.v, self.u = 1.0 + 0.1 * rank, 0.5 - 0.05 * rank, 0.3
        self.skip, self.x, self.gskip, self.log, self.rank = {}, {}, {}, log, rank
        self.gw = self.gv = self.gu = 0.0

    def forward_enc(self, m, x, t):
        self.log.append((self.rank, "FE", m))
        self.x[m] = x
        self.skip[m] = x * self.w + 1.0 + t.sum() * 0.0
        return self.skip[m].clone()

    def forward_dec(self, m, h):
        self.log.append((self.rank, "FD", m))
        return h + self.v * self.skip[m]

    def forward(self, m, x, t):
        self.log.append((self.rank, "F", m))
        self.x[m] = x
        return self.u * x * x

    def loss(self, m, d, target, scale):
        diff = d - target
        return scale * (diff ** 2).mean(), scale * 2.0 * diff / diff.numel()

    def backward_dec(self, m, g, accumulate):
        self.log.append((self.rank, "BD", m))
        if not accumulate:
            self.gw = self.gv = 0.0
        self.gv += float((g * self.skip[m]).sum())
        self.gskip[m] = self.v * g                       # skip gradient: stays on this device until backward_enc
        return g                                         # d/dh

    def backward_enc(self, m, ge):
        self.log.append((self.rank, "BE", m))
        ge = ge + self.gskip.pop(m)
        self.gw += float((ge * self.x[m]).sum())
        del self.skip[m]
        return ge * self.w

    def backward(self, m, g, accumulate):
        self.log.append((self.rank, "B", m))
        if not accumulate:
            self.gu = 0.0
        self.gu += float((g * self.x[m] ** 2).sum())
        return g * 2.0 * self.u * self.x[m]


def _data(M, shape=(2, 3, 4, 4)):
    g = torch.Generator().manual_seed(0)
    return [{"x_in": torch.randn(shape, generator=g, dtype=torch.float64), "t": torch.tensor([3, 7]),
             "target": torch.randn(shape, generator=g, dtype=torch.float64)} for _ in range(M)]


def _sequential(world, data):
    """The same arithmetic composed in one place and differentiated by autograd."""
    M = len(data)
    ws = [torch.tensor(1.0 + 0.1 * r, dtype=torch.float64, requires_grad=True) for r in range(world - 1)]
    vs = [torch.tensor(0.5 - 0.05 * r, dtype=torch.float64, requires_grad=True) for r in range(world - 1)]
    u = torch.tensor(0.3, dtype=torch.float64, requires_grad=True)
    xs = [d["x_in"].clone().requires_grad_(True) for d in data]
    total, losses = 0.0, []
    for m, d in enumerate(data):
        x, skips = xs[m], []
        for r in range(world - 1):
            x = x * ws[r] + 1.0
            skips.append(x)
        h = u * x * x
        for r in reversed(range(world - 1)):
            h = h + vs[r] * skips[r]
        losses.append(((h - d["target"]) ** 2).mean() / M)
        total = total + losses[-1]
    total.backward()
    return losses, [x.grad for x in xs], [float(w.grad) for w in ws], [float(v.grad) for v in vs], float(u.grad)


@pytest.mark.parametrize("world,M", [(1, 2), (2, 1), (2, 4), (3, 3), (4, 2)])
def test_wave_equals_sequential_and_traffic(world, M):
    data, log = _data(M), []
    execs = [ToyExec(r, world, log) for r in range(world)]
    progs = [PL.rank_program(r, world, execs[r], M, data if r == 0 else None) for r in range(world)]
    results, traffic = PL.run_local(progs)
    losses, gx, gw, gv, gu = _sequential(world, data)
    for m in range(M):
        assert torch.allclose(results[0][m]["loss"], losses[m].detach(), atol=1e-14)
        assert torch.allclose(results[0][m]["g_x_in"], gx[m], atol=1e-14)
    for r in range(world - 1):
        assert abs(execs[r].gw - gw[r]) < 1e-12 and abs(execs[r].gv - gv[r]) < 1e-12
    assert abs(execs[-1].gu - gu) < 1e-12
    # per microbatch and rank: forward_enc -> forward_dec -> backward_dec -> backward_enc (F -> B on the last rank)
    for r in range(world):
        for m in range(M):
            seq = [ev for (rr, ev, mm) in log if rr == r and mm == m]
            assert seq == (["F", "B"] if r == world - 1 else ["FE", "FD", "BD", "BE"]), (r, m, seq)
    # 2 (D-1) a per microbatch in the forward, the same volume of gradients in the backward; the skips
    # (one per OPEN rank and microbatch here) never appear: only x, d, g_d, g_e cross
    a = data[0]["x_in"].numel() * 8
    assert traffic.bytes["act"] == 2 * (world - 1) * a * M and traffic.bytes["grad"] == 2 * (world - 1) * a * M
    assert traffic.messages["act"] == 2 * (world - 1) * M
    # the skip caches were emptied by the backward halves
    assert all(not e.skip and not e.gskip for e in execs[:-1])


def test_deadlock_is_reported():
    def waits_forever():
        yield ("recv", 1, ("x", 0))
    with pytest.raises(RuntimeError, match="deadlock"):
        PL.run_local([waits_forever(), iter(())])


def _free_port():
    s = socket.socket()
    s.bind(("127.0.0.1", 0))
    p = s.getsockname()[1]
    s.close()
    return p


def _worker(rank, world, port, M, q):
    import torch.distributed as dist
    os.environ.update(MASTER_ADDR="127.0.0.1", MASTER_PORT=str(port))
    dist.init_process_group("gloo", rank=rank, world_size=world)
    data, log = _data(M), []
    ex = ToyExec(rank, world, log)
    shape, f64 = tuple(data[0]["x_in"].shape), torch.float64
    shapes = {"t": ((2,), torch.int64), "x": (shape, f64), "d": (shape, f64), "gd": (shape, f64), "ge": (shape, f64)}
    res, traffic = PL.run_distributed(PL.rank_program(rank, world, ex, M, data if rank == 0 else None), rank, dist, shapes, "cpu")
    out = {"rank": rank, "sent_act": traffic.bytes["act"], "sent_grad": traffic.bytes["grad"], "log": log,
           "gw": ex.gw, "gv": ex.gv, "gu": ex.gu}
    if rank == 0:
        out["loss"] = [float(res[m]["loss"]) for m in range(M)]
        out["gx"] = [res[m]["g_x_in"] for m in range(M)]
    dist.barrier()
    q.put(out)
    dist.destroy_process_group()


def test_two_ranks_over_gloo_match_the_local_driver():
    world, M = 2, 3
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = _free_port()
    procs = [ctx.Process(target=_worker, args=(r, world, port, M, q)) for r in range(world)]
    for p in procs:
        p.start()
    outs = sorted((q.get(timeout=120) for _ in range(world)), key=lambda o: o["rank"])
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    data = _data(M)
    losses, gx, gw, gv, gu = _sequential(world, data)
    assert all(abs(outs[0]["loss"][m] - float(losses[m])) < 1e-14 for m in range(M))
    assert all(torch.allclose(outs[0]["gx"][m], gx[m], atol=1e-14) for m in range(M))
    assert abs(outs[0]["gw"] - gw[0]) < 1e-12 and abs(outs[0]["gv"] - gv[0]) < 1e-12 and abs(outs[1]["gu"] - gu) < 1e-12
    a = data[0]["x_in"].numel() * 8
    # each rank sends one activation and one gradient per microbatch across the single boundary: 2 (D-1) a in total
    assert outs[0]["sent_act"] + outs[1]["sent_act"] == 2 * a * M
    assert outs[0]["sent_grad"] + outs[1]["sent_grad"] == 2 * a * M
