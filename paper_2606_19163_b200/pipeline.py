"""Wave runtime over D devices.

PAPER.md:L235-L249 (sec. V-B): with P pipeline stages per direction, "stage q and 2P-q+1" are placed on one device, so the
skip tensors never leave it; what crosses a device boundary is one activation per direction and microbatch, "2(D-1)a"
per microbatch in the forward (L241) and the same volume of gradients in the backward (L259-L261, Eq. 15).  Here one
`binding.Stage` object IS such a collocated pair: rank r < D-1 holds an OPEN stage (its encoder half is pipeline stage
r+1, its decoder half stage 2D-r-1... in the paper's numbering), the last rank holds the CLOSED innermost stage.

    rank r          forward                                   backward
    r < D-1         x_in -> forward_enc -> e_out  --> r+1     g_d_out -> backward_dec -> g_h_in --> r+1
                    h_in -> forward_dec -> d_out  --> r-1     g_e_out -> backward_enc -> g_x_in --> r-1
    r = D-1         x_in -> forward     -> d_out  --> r-1     g_d_out -> backward     -> g_x_in --> r-1

Schedule: the wave of PAPER.md:L255 - all M microbatches forward, then all backward in reverse, every rank working through
its four loops (F-enc, F-dec, B-dec, B-enc) in microbatch order.  Sends are asynchronous, receives are the only waits, and
every rank receives in the order its neighbour sends, so the schedule cannot deadlock.

`rank_program` is a generator that yields a request whenever it needs a tensor from a neighbour.  Two drivers consume it:
`run_distributed` (one process per rank, torch.distributed point-to-point: NCCL over NVLink for CUDA tensors, gloo on the
CPU in the tests) and `run_local` (all ranks in one process on one device, stepped round-robin: on a single GPU the ranks'
kernels are enqueued one after another on one stream - nothing ever waits on another kernel).
"""
from __future__ import annotations

from collections import defaultdict, deque


class Traffic:
    """Bytes that crossed each rank boundary, by kind: 'act' (x / d), 'grad' (g_d / g_e), 'meta' (timesteps)."""

    def __init__(self):
        self.bytes = defaultdict(int)
        self.messages = defaultdict(int)

    def add(self, kind, tensor):
        self.bytes[kind] += tensor.numel() * tensor.element_size()
        self.messages[kind] += 1


def rank_program(rank: int, world: int, ex, microbatches: int, data=None):
    """Generator: yields ("send", dst, tag, tensor) / ("recv", src, tag) requests; a recv request is answered (via
    .send()) with the tensor.  `ex` is the stage executor of this rank (see CudaStageExec); `data[m]` = rank 0's inputs.
    Returns (via StopIteration.value) rank 0's per-microbatch results."""
    M, last = microbatches, rank == world - 1
    out, res = {}, {}
    for m in range(M):                                   # ---- F-enc
        if rank == 0:
            x, t = data[m]["x_in"], data[m]["t"]
        else:
            t = yield ("recv", rank - 1, ("t", m))
            x = yield ("recv", rank - 1, ("x", m))
        if not last:
            yield ("send", rank + 1, ("t", m), t, "meta")
        if last:
            d = ex.forward(m, x, t)
            if world == 1:
                out[m] = d
            else:
                yield ("send", rank - 1, ("d", m), d, "act")
        else:
            yield ("send", rank + 1, ("x", m), ex.forward_enc(m, x, t), "act")
    if not last:
        for m in range(M):                               # ---- F-dec
            h = yield ("recv", rank + 1, ("d", m))
            d = ex.forward_dec(m, h)
            if rank == 0:
                out[m] = d
            else:
                yield ("send", rank - 1, ("d", m), d, "act")
    for m in reversed(range(M)):                         # ---- B-dec (the whole backward on the last rank)
        if rank == 0:
            loss, g = ex.loss(m, out[m], data[m]["target"], 1.0 / M)
            res[m] = {"loss": loss, "d_out": out[m]}
        else:
            g = yield ("recv", rank - 1, ("gd", m))
        first = m == M - 1
        if last:
            gx = ex.backward(m, g, accumulate=not first)
            if world == 1:
                res[m]["g_x_in"] = gx
            else:
                yield ("send", rank - 1, ("ge", m), gx, "grad")
        else:
            yield ("send", rank + 1, ("gd", m), ex.backward_dec(m, g, accumulate=not first), "grad")
    if not last:
        for m in reversed(range(M)):                     # ---- B-enc
            ge = yield ("recv", rank + 1, ("ge", m))
            gx = ex.backward_enc(m, ge)
            if rank == 0:
                res[m]["g_x_in"] = gx
            else:
                yield ("send", rank - 1, ("ge", m), gx, "grad")
    return res


def run_local(programs):
    """All ranks in this process: step the generators round-robin; a rank blocks only on a recv whose message has not
    been sent yet.  Returns ([result per rank], Traffic)."""
    traffic = Traffic()
    box = defaultdict(deque)                      # (src, dst, tag) -> tensors
    n = len(programs)
    waiting = [None] * n                          # pending recv request per rank
    pending = [None] * n                          # value to send into the generator next
    done, results = [False] * n, [None] * n
    started = [False] * n
    while not all(done):
        progress = False
        for r, prog in enumerate(programs):
            if done[r]:
                continue
            while True:
                if waiting[r] is not None:
                    key = (waiting[r][1], r, waiting[r][2])
                    if not box[key]:
                        break                     # still nothing to receive: let the others run
                    pending[r], waiting[r] = box[key].popleft(), None
                try:
                    req = prog.send(pending[r]) if started[r] else next(prog)
                except StopIteration as stop:
                    done[r], results[r] = True, stop.value
                    progress = True
                    break
                started[r], pending[r], progress = True, None, True
                if req[0] == "send":
                    _, dst, tag, tensor, kind = req
                    traffic.add(kind, tensor)
                    box[(r, dst, tag)].append(tensor)
                else:
                    waiting[r] = req
        if not progress:
            raise RuntimeError("wave schedule deadlocked: every rank waits for a message nobody sent")
    return results, traffic


def run_distributed(program, rank, dist, shapes, device):
    """One process per rank.  shapes[tag kind] -> (shape, dtype) of what this rank receives ('t', 'x', 'd', 'gd', 'ge').
    Sends are isend (kept alive until the end), receives are blocking recv into fresh tensors."""
    import torch
    traffic = Traffic()
    inflight, pending, started = [], None, False
    while True:
        try:
            req = program.send(pending) if started else next(program)
        except StopIteration as stop:
            for w in inflight:
                w.wait()
            return stop.value, traffic
        started, pending = True, None
        if req[0] == "send":
            _, dst, tag, tensor, kind = req
            traffic.add(kind, tensor)
            tensor = tensor.contiguous()
            inflight.append(dist.isend(tensor, dst))
            inflight.append(_Keep(tensor))
        else:
            _, src, tag = req
            shape, dtype = shapes[tag[0]]
            buf = torch.empty(shape, dtype=dtype, device=device)
            dist.recv(buf, src)
            pending = buf


class _Keep:
    """Keeps a sent tensor alive until the isend that reads it has completed."""

    def __init__(self, t):
        self.t = t

    def wait(self):
        self.t = None


class CudaStageExec:
    """The stage executor of one rank on the GPU: a binding.Stage created with FLAG_SPLIT (OPEN) or plain (CLOSED)."""

    def __init__(self, stage):
        self.st = stage
        self.emb, self.tst, self.g_temb = {}, {}, {}
        self.fresh = False          # the next timestep-MLP backward is the first of the wave: it overwrites

    def _temb(self, m, t):
        import torch
        self.emb[m], self.tst[m] = self.st.temb_forward(t)
        self.g_temb[m] = torch.zeros_like(self.emb[m])

    def forward_enc(self, m, x, t):
        self._temb(m, t)
        return self.st.forward_enc(m, x, self.emb[m])

    def forward_dec(self, m, h):
        return self.st.forward_dec(m, h)

    def forward(self, m, x, t):
        self._temb(m, t)
        return self.st.forward(m, x, None, self.emb[m])[1]

    def loss(self, m, d, target, scale):
        return self.st.mse(d, target, scale)

    def backward_dec(self, m, g, accumulate):
        self.fresh = self.fresh or not accumulate
        return self.st.backward_dec(m, g, self.g_temb[m], accumulate)

    def backward_enc(self, m, ge):
        gx = self.st.backward_enc(m, ge, self.g_temb[m])
        self._temb_backward(m)
        return gx

    def backward(self, m, g, accumulate):
        self.fresh = self.fresh or not accumulate
        gx, _ = self.st.backward(m, g, None, True, self.g_temb[m], accumulate)
        self._temb_backward(m)
        return gx

    def _temb_backward(self, m):
        # the timestep-MLP gradients accumulate over the microbatches of the wave like every other weight gradient
        self.st.temb_backward(self.g_temb[m], self.tst[m], accumulate=not self.fresh)
        self.fresh = False
