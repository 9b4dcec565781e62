"""ctypes binding of libpulse.so (include/pulse.h).  Argument marshalling only: every step
of the hot path runs in the library's kernels.  PyTorch is used for device memory and
streams.  Importing this module fails loudly if the CUDA library has not been built
(`python -m paper_2606_19163_b200.build`); there is no CPU fallback.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np
import torch

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "libpulse.so")
if not os.path.exists(LIB_PATH):
    raise ImportError(f"{LIB_PATH} is missing: build it with `python -m paper_2606_19163_b200.build` "
                      "(nvcc, sm_100a). The PULSE stage has no CPU fallback.")
lib = C.CDLL(LIB_PATH)

F32, BF16 = 0, 1
OP_KIND = {"conv_in": 0, "resblock": 1, "down": 2, "up": 3, "head": 4, "attn": 5, "tblock": 6}
FLAG_FORCE_SIMT = 1
FLAG_GN_TWO_PASS = 2
FLAG_CONV_PAIR = 4
FLAG_CONV_1CTA = 8
FLAG_UP_MATERIALISED = 16
FLAG_UP_PHASE_FWD = 32
FLAG_UP_PHASE_DGRAD = 64
FLAG_SPLIT = 128


class OpDesc(C.Structure):
    _fields_ = [("kind", C.c_int), ("cin", C.c_int), ("cout", C.c_int), ("skip_channels", C.c_int),
                ("push_skip", C.c_int), ("heads", C.c_int)]


class StageDesc(C.Structure):
    _fields_ = [("dtype", C.c_int), ("n", C.c_int), ("h", C.c_int), ("w", C.c_int), ("c_in", C.c_int),
                ("groups", C.c_int), ("eps", C.c_float),
                ("temb_kind", C.c_int), ("temb_d0", C.c_int), ("temb_dim", C.c_int),
                ("link", C.c_int), ("x_in_is_skip", C.c_int),
                ("n_enc_ops", C.c_int), ("enc_ops", C.POINTER(OpDesc)),
                ("n_mid_ops", C.c_int), ("mid_ops", C.POINTER(OpDesc)),
                ("n_dec_ops", C.c_int), ("dec_ops", C.POINTER(OpDesc)),
                ("max_inflight", C.c_int), ("flags", C.c_uint)]


_vp, _sz, _i64 = C.c_void_p, C.c_size_t, C.c_int64
_SIG = {
    "pulse_stage_create": [C.POINTER(StageDesc), C.POINTER(_vp)],
    "pulse_stage_destroy": [_vp],
    "pulse_stage_param_count": [_vp, C.POINTER(C.c_int)],
    "pulse_stage_param_info": [_vp, C.c_int, C.POINTER(C.c_char_p), C.POINTER(C.c_int), C.POINTER(C.c_int * 4),
                               C.POINTER(_sz), C.POINTER(_sz)],
    "pulse_stage_param_bytes": [_vp, C.POINTER(_sz), C.POINTER(_sz)],
    "pulse_stage_bind_params": [_vp, _vp, _vp],
    "pulse_stage_workspace_bytes": [_vp, C.POINTER(_sz), C.POINTER(_sz)],
    "pulse_stage_bind_workspace": [_vp, _vp, _sz],
    "pulse_skip_cache_bytes": [_vp, C.POINTER(_sz)],
    "pulse_skip_cache_create": [_vp, _vp, _sz, C.c_int, C.POINTER(_vp)],
    "pulse_skip_cache_get": [_vp, _i64, C.c_int, C.POINTER(_vp), C.POINTER(C.c_int * 4)],
    "pulse_skip_cache_count": [_vp, C.POINTER(C.c_int)],
    "pulse_skip_cache_release": [_vp, _i64],
    "pulse_skip_cache_stats": [_vp, C.POINTER(C.c_int), C.POINTER(_sz), C.POINTER(_sz)],
    "pulse_skip_cache_destroy": [_vp],
    "pulse_stage_forward": [_vp, _vp, _i64, _vp, _vp, _vp, _vp, _vp, _vp],
    "pulse_stage_backward": [_vp, _vp, _i64, _vp, _vp, _vp, _vp, _vp, C.c_int, _vp],
    "pulse_stage_forward_enc": [_vp, _vp, _i64, _vp, _vp, _vp, _vp],
    "pulse_stage_forward_dec": [_vp, _vp, _i64, _vp, _vp, _vp],
    "pulse_stage_backward_dec": [_vp, _vp, _i64, _vp, _vp, _vp, C.c_int, _vp],
    "pulse_stage_backward_enc": [_vp, _vp, _i64, _vp, _vp, _vp, _vp],
    "pulse_stage_forward_temb": [_vp, _vp, _i64, _vp, _vp, _vp, _vp, _vp, _vp, _vp, _vp],
    "pulse_stage_backward_temb": [_vp, _vp, _i64, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int, _vp],
    "pulse_temb_stash_elems": [_vp, C.POINTER(_sz)],
    "pulse_temb_forward": [_vp, _vp, _vp, _vp, _vp],
    "pulse_temb_backward": [_vp, _vp, _vp, C.c_int, _vp],
    "pulse_mse_fwd_bwd": [C.c_int, _vp, _vp, _sz, C.c_float, _vp, _vp, _vp],
    "pulse_stage_launch_count": [_vp, C.POINTER(C.c_uint64)],
    "pulse_stage_profile": [_vp, C.c_int],
    "pulse_stage_profile_read": [_vp, C.POINTER(C.c_double * 6), C.POINTER(C.c_uint64 * 6), C.POINTER(C.c_double * 6),
                                 C.POINTER(C.c_double * 6)],
    "pulse_conv2d": [C.c_int, C.c_int, _vp, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, _vp,
                     C.c_int, _vp, _vp, _vp, _vp, _vp, _vp],
    "pulse_conv2d_dgrad": [C.c_int, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, _vp, C.c_int,
                           _vp, _vp, C.c_int, _vp],
    "pulse_conv2d_wgrad": [C.c_int, C.c_int, _vp, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int,
                           _vp, C.c_int, _vp, C.c_int, _vp],
    "pulse_upsample_conv2d": [C.c_int, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int, _vp, C.c_int, _vp, _vp, _vp, _vp, _vp],
    "pulse_upsample_conv2d_dgrad": [C.c_int, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int, _vp, C.c_int, _vp, _vp, _vp],
    "pulse_upsample_conv2d_wgrad": [C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int, _vp, C.c_int, _vp, _vp],
    "pulse_attention": [C.c_int, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int, _vp, _vp, _vp],
    "pulse_attention_backward": [C.c_int, C.c_int, _vp, _vp, C.c_int, C.c_int, C.c_int, C.c_int, _vp, _vp, _vp],
    "pulse_groupnorm_silu": [C.c_int, _vp, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int, C.c_int, C.c_float, _vp, _vp,
                             _vp, C.c_int, _vp, _vp],
    "pulse_groupnorm_silu_backward": [C.c_int, C.c_int, C.c_int, _vp, _vp, C.c_int, _vp, C.c_int, C.c_int, C.c_int, C.c_int,
                                      C.c_int, C.c_float, _vp, _vp, _vp, _vp, _vp, _vp, C.c_int, _vp, C.c_int, _vp, _vp,
                                      _vp],
}
_dp, _ip = C.POINTER(C.c_double), C.POINTER(C.c_int)
_SIG["pulse_partition"] = [C.c_int, _dp, _dp, C.c_int, _ip, _ip, C.c_int, C.c_double, C.c_double, C.c_double, _ip, _dp]
for _name, _args in _SIG.items():
    _f = getattr(lib, _name)
    _f.argtypes = _args
    _f.restype = C.c_int
lib.pulse_version.restype = C.c_int
lib.pulse_status_string.restype = C.c_char_p
lib.pulse_status_string.argtypes = [C.c_int]
lib.pulse_last_error.restype = C.c_char_p
lib.pulse_groupnorm_stats_floats.restype = _sz
lib.pulse_groupnorm_stats_floats.argtypes = [C.c_int, C.c_int, C.c_int]
lib.pulse_attention_stats_floats.restype = _sz
lib.pulse_attention_stats_floats.argtypes = [C.c_int, C.c_int, C.c_int]
EXPORTS = list(_SIG) + ["pulse_groupnorm_stats_floats", "pulse_attention_stats_floats", "pulse_version", "pulse_status_string", "pulse_last_error"]


class PulseError(RuntimeError):
    def __init__(self, status):
        self.status = status
        super().__init__(f"{lib.pulse_status_string(status).decode()} ({status}): {lib.pulse_last_error().decode()}")


def _ck(status):
    if status != 0:
        raise PulseError(status)


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def _stream():
    return C.c_void_p(torch.cuda.current_stream().cuda_stream)


def make_desc(desc: dict, max_inflight: int = 1, flags: int = 0):
    """workloads.py structure -> (StageDesc, keep-alive arrays)."""
    def ops(lst):
        arr = (OpDesc * max(1, len(lst)))()
        for i, o in enumerate(lst):
            arr[i] = OpDesc(OP_KIND[o["kind"]], o["cin"], o["cout"], o["skip"], o["push"], o.get("heads", 0))
        return arr
    e, m, d = ops(desc["enc_ops"]), ops(desc["mid_ops"]), ops(desc["dec_ops"])
    sd = StageDesc(BF16 if desc["dtype"] == "bf16" else F32, desc["n"], desc["h"], desc["w"], desc["c_in"],
                   desc["groups"], desc["eps"], 1 if desc["temb"]["kind"] == "mlp" else 0, desc["temb"]["d0"],
                   desc["temb"]["dim"], 1 if desc["link"] == "closed" else 0, desc["x_in_is_skip"],
                   len(desc["enc_ops"]), e, len(desc["mid_ops"]), m, len(desc["dec_ops"]), d, max_inflight, flags)
    return sd, (e, m, d)


def nhwc(a, dtype, device="cuda"):
    """host [N,C,H,W] array -> device NHWC tensor in `dtype` (layout marshalling)."""
    t = torch.as_tensor(np.ascontiguousarray(a))
    return t.permute(0, 2, 3, 1).contiguous().to(device=device, dtype=dtype)


def nchw(t):
    """device NHWC tensor -> host [N,C,H,W] float64 tensor."""
    return t.detach().permute(0, 3, 1, 2).to(torch.float64).cpu()


class Stage:
    """One collocated stage + its skip cache.  No device needed to construct with
    allocate=False (plan / parameter table only)."""

    def __init__(self, desc: dict, max_inflight: int | None = None, flags: int = 0, allocate: bool = True,
                 device="cuda"):
        self.desc = desc
        self.max_inflight = max_inflight or desc.get("microbatches", 1)
        self.tdtype = torch.bfloat16 if desc["dtype"] == "bf16" else torch.float32
        self.cdtype = BF16 if desc["dtype"] == "bf16" else F32
        self._sd, self._keep = make_desc(desc, self.max_inflight, flags)
        self.h = C.c_void_p()
        _ck(lib.pulse_stage_create(C.byref(self._sd), C.byref(self.h)))
        self.cache = C.c_void_p()
        self.params = self._param_table()
        pb, gb, ws, st, sb = _sz(), _sz(), _sz(), _sz(), _sz()
        _ck(lib.pulse_stage_param_bytes(self.h, C.byref(pb), C.byref(gb)))
        _ck(lib.pulse_stage_workspace_bytes(self.h, C.byref(ws), C.byref(st)))
        _ck(lib.pulse_skip_cache_bytes(self.h, C.byref(sb)))
        self.param_bytes, self.grad_bytes = pb.value, gb.value
        self.work_bytes, self.stash_bytes, self.skip_bytes = ws.value, st.value, sb.value
        self.shapes = None
        if allocate:
            self.device = torch.device(device)
            u8 = dict(dtype=torch.uint8, device=self.device)
            self.d_params = torch.zeros(max(256, self.param_bytes), **u8)
            self.d_grads = torch.zeros(max(256, self.grad_bytes), **u8)
            self.d_work = torch.empty(self.work_bytes + self.max_inflight * self.stash_bytes + 256, **u8)
            self.d_cache = torch.empty(max(256, self.max_inflight * self.skip_bytes), **u8)
            _ck(lib.pulse_stage_bind_params(self.h, _ptr(self.d_params), _ptr(self.d_grads)))
            _ck(lib.pulse_stage_bind_workspace(self.h, _ptr(self.d_work), self.d_work.numel()))
            _ck(lib.pulse_skip_cache_create(self.h, _ptr(self.d_cache), self.d_cache.numel(), self.max_inflight,
                                            C.byref(self.cache)))

    def _param_table(self):
        n = C.c_int()
        _ck(lib.pulse_stage_param_count(self.h, C.byref(n)))
        out = []
        for i in range(n.value):
            name, rank, shape, off, goff = C.c_char_p(), C.c_int(), (C.c_int * 4)(), _sz(), _sz()
            _ck(lib.pulse_stage_param_info(self.h, i, C.byref(name), C.byref(rank), C.byref(shape), C.byref(off),
                                           C.byref(goff)))
            out.append({"name": name.value.decode(), "shape": tuple(shape[:rank.value]), "off": off.value,
                        "goff": goff.value})
        return out

    def close(self):
        if self.cache:
            lib.pulse_skip_cache_destroy(self.cache)
            self.cache = C.c_void_p()
        if self.h:
            lib.pulse_stage_destroy(self.h)
            self.h = C.c_void_p()

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- parameters -------------------------------------------------------------------
    def load_params(self, params: dict):
        """Logical layouts ([Cout,Cin,kh,kw] / [out,in]) -> device layout ([Cout,kh,kw,Cin]) in the stage dtype."""
        esz = 2 if self.cdtype == BF16 else 4
        for p in self.params:
            v = torch.as_tensor(np.asarray(params[p["name"]]))
            if v.dim() == 4:
                v = v.permute(0, 2, 3, 1)
            v = v.contiguous().to(self.tdtype)
            assert tuple(v.shape) == p["shape"], (p["name"], tuple(v.shape), p["shape"])
            dst = self.d_params[p["off"]: p["off"] + v.numel() * esz].view(self.tdtype)
            dst.copy_(v.reshape(-1).to(self.device))

    def grads(self) -> dict:
        """fp32 parameter gradients in logical layouts (host, float64)."""
        out = {}
        for p in self.params:
            numel = int(np.prod(p["shape"]))
            g = self.d_grads[p["goff"]: p["goff"] + numel * 4].view(torch.float32).reshape(p["shape"])
            if g.dim() == 4:
                g = g.permute(0, 3, 1, 2)
            out[p["name"]] = g.to(torch.float64).cpu().contiguous()
        return out

    # ---- hot path ------------------------------------------------------------------------
    def _shapes(self):
        if self.shapes is None:
            from . import workloads
            s = workloads.boundary_shapes(self.desc)
            self.shapes = {k: (v[0], v[2], v[3], v[1]) for k, v in s.items()}     # NHWC
        return self.shapes

    def forward(self, mb_id: int, x_in, h_in, temb):
        sh = self._shapes()
        d_out = torch.empty(sh["d_out"], dtype=self.tdtype, device=self.device)
        e_out = torch.empty(sh["e_out"], dtype=self.tdtype, device=self.device) if "e_out" in sh else None
        _ck(lib.pulse_stage_forward(self.h, self.cache, mb_id, _ptr(x_in), _ptr(h_in), _ptr(temb), _ptr(e_out),
                                    _ptr(d_out), _stream()))
        return e_out, d_out

    def backward(self, mb_id: int, g_d_out, g_e_out=None, want_g_x_in=True, g_temb=None, accumulate=False):
        sh = self._shapes()
        g_x_in = torch.empty(sh["x_in"], dtype=self.tdtype, device=self.device) if want_g_x_in else None
        g_h_in = torch.empty(sh["h_in"], dtype=self.tdtype, device=self.device) if "h_in" in sh else None
        _ck(lib.pulse_stage_backward(self.h, self.cache, mb_id, _ptr(g_d_out), _ptr(g_e_out), _ptr(g_x_in),
                                     _ptr(g_h_in), _ptr(g_temb), int(accumulate), _stream()))
        return g_x_in, g_h_in

    # ---- the two halves of a split (pipeline) stage (FLAG_SPLIT) ----------------------
    def forward_enc(self, mb_id: int, x_in, temb):
        e_out = torch.empty(self._shapes()["e_out"], dtype=self.tdtype, device=self.device)
        _ck(lib.pulse_stage_forward_enc(self.h, self.cache, mb_id, _ptr(x_in), _ptr(temb), _ptr(e_out), _stream()))
        return e_out

    def forward_dec(self, mb_id: int, h_in):
        d_out = torch.empty(self._shapes()["d_out"], dtype=self.tdtype, device=self.device)
        _ck(lib.pulse_stage_forward_dec(self.h, self.cache, mb_id, _ptr(h_in), _ptr(d_out), _stream()))
        return d_out

    def backward_dec(self, mb_id: int, g_d_out, g_temb=None, accumulate=False):
        g_h_in = torch.empty(self._shapes()["h_in"], dtype=self.tdtype, device=self.device)
        _ck(lib.pulse_stage_backward_dec(self.h, self.cache, mb_id, _ptr(g_d_out), _ptr(g_h_in), _ptr(g_temb), int(accumulate),
                                         _stream()))
        return g_h_in

    def backward_enc(self, mb_id: int, g_e_out, g_temb=None):
        g_x_in = torch.empty(self._shapes()["x_in"], dtype=self.tdtype, device=self.device)
        _ck(lib.pulse_stage_backward_enc(self.h, self.cache, mb_id, _ptr(g_e_out), _ptr(g_x_in), _ptr(g_temb), _stream()))
        return g_x_in

    def forward_temb(self, mb_id: int, x_in, h_in, t):
        """temb_forward + forward in one call: the timestep path runs beside the stash of the boundary tensors."""
        sh = self._shapes()
        n = _sz()
        _ck(lib.pulse_temb_stash_elems(self.h, C.byref(n)))
        emb = torch.empty((self.desc["n"], self.desc["temb"]["dim"]), dtype=torch.float32, device=self.device)
        stash = torch.empty(max(1, n.value), dtype=torch.float32, device=self.device)
        d_out = torch.empty(sh["d_out"], dtype=self.tdtype, device=self.device)
        e_out = torch.empty(sh["e_out"], dtype=self.tdtype, device=self.device) if "e_out" in sh else None
        _ck(lib.pulse_stage_forward_temb(self.h, self.cache, mb_id, _ptr(x_in), _ptr(h_in), _ptr(t), _ptr(emb),
                                         _ptr(stash), _ptr(e_out), _ptr(d_out), _stream()))
        return emb, stash, e_out, d_out

    def backward_temb(self, mb_id: int, g_d_out, g_e_out, g_temb, tstash, want_g_x_in=True, accumulate=False):
        """backward + temb_backward in one call: the timestep-MLP backward runs beside the last operator."""
        sh = self._shapes()
        g_x_in = torch.empty(sh["x_in"], dtype=self.tdtype, device=self.device) if want_g_x_in else None
        g_h_in = torch.empty(sh["h_in"], dtype=self.tdtype, device=self.device) if "h_in" in sh else None
        _ck(lib.pulse_stage_backward_temb(self.h, self.cache, mb_id, _ptr(g_d_out), _ptr(g_e_out), _ptr(g_x_in),
                                          _ptr(g_h_in), _ptr(g_temb), _ptr(tstash), int(accumulate), _stream()))
        return g_x_in, g_h_in

    def temb_forward(self, t):
        n = _sz()
        _ck(lib.pulse_temb_stash_elems(self.h, C.byref(n)))
        emb = torch.empty((self.desc["n"], self.desc["temb"]["dim"]), dtype=torch.float32, device=self.device)
        stash = torch.empty(max(1, n.value), dtype=torch.float32, device=self.device)
        _ck(lib.pulse_temb_forward(self.h, _ptr(t), _ptr(emb), _ptr(stash), _stream()))
        return emb, stash

    def temb_backward(self, g_emb, stash, accumulate=False):
        _ck(lib.pulse_temb_backward(self.h, _ptr(g_emb), _ptr(stash), int(accumulate), _stream()))

    def mse(self, d, target, scale=1.0, loss=None):
        if loss is None:
            loss = torch.zeros(1, dtype=torch.float32, device=self.device)
        g = torch.empty_like(d)
        _ck(lib.pulse_mse_fwd_bwd(self.cdtype, _ptr(d), _ptr(target), d.numel(), scale, _ptr(loss), _ptr(g), _stream()))
        return loss, g

    def skip(self, mb_id: int, k: int):
        """Device view of cached skip k of a live microbatch (tests)."""
        p, shape = C.c_void_p(), (C.c_int * 4)()
        _ck(lib.pulse_skip_cache_get(self.cache, mb_id, k, C.byref(p), C.byref(shape)))
        off = p.value - self.d_cache.data_ptr()
        numel = int(np.prod(shape[:]))
        esz = 2 if self.cdtype == BF16 else 4
        return self.d_cache[off: off + numel * esz].view(self.tdtype).reshape(tuple(shape[:]))

    def skip_count(self):
        n = C.c_int()
        _ck(lib.pulse_skip_cache_count(self.cache, C.byref(n)))
        return n.value

    def cache_stats(self):
        live, lb, pk = C.c_int(), _sz(), _sz()
        _ck(lib.pulse_skip_cache_stats(self.cache, C.byref(live), C.byref(lb), C.byref(pk)))
        return {"live_slots": live.value, "live_bytes": lb.value, "peak_bytes": pk.value}

    def launches(self):
        n = C.c_uint64()
        _ck(lib.pulse_stage_launch_count(self.h, C.byref(n)))
        return n.value

    KCLASSES = ["conv_tc", "wgrad_tc", "conv_simt", "gn_fwd", "gn_bwd", "other"]

    def profile(self, enable: bool):
        _ck(lib.pulse_stage_profile(self.h, int(enable)))

    def profile_read(self) -> dict:
        ms, ln, fl, by = (C.c_double * 6)(), (C.c_uint64 * 6)(), (C.c_double * 6)(), (C.c_double * 6)()
        _ck(lib.pulse_stage_profile_read(self.h, C.byref(ms), C.byref(ln), C.byref(fl), C.byref(by)))
        return {k: {"ms": ms[i], "launches": ln[i], "flops": fl[i], "bytes": by[i]} for i, k in enumerate(self.KCLASSES)}

    # ---- one microbatch, device-resident inputs (what bench.py times) -------------------------
    def step(self, mb_id, dev, loss_scale=1.0, accumulate=False, loss=None, g_temb=None):
        """temb -> forward -> MSE -> backward -> temb backward for device-resident inputs
        `dev` = {x_in, h_in?, t, target, g_e_out?}.  Returns (outputs dict)."""
        emb, tstash, e_out, d_out = self.forward_temb(mb_id, dev["x_in"], dev.get("h_in"), dev["t"])
        loss, g_d = self.mse(d_out, dev["target"], loss_scale, loss)
        if g_temb is None:
            g_temb = torch.zeros_like(emb)
        g_x_in, g_h_in = self.backward_temb(mb_id, g_d, dev.get("g_e_out"), g_temb, tstash, True, accumulate)
        return {"loss": loss, "e_out": e_out, "d_out": d_out, "g_x_in": g_x_in, "g_h_in": g_h_in, "g_emb": g_temb,
                "emb": emb}

    def to_device(self, mb: dict) -> dict:
        """host microbatch (workloads.draw, [N,C,H,W]) -> device NHWC tensors."""
        dev = {}
        for k, v in mb.items():
            if k == "t":
                dev[k] = torch.as_tensor(v).to(self.device)
            else:
                dev[k] = nhwc(v, self.tdtype, self.device)
        return dev


# ---- single operators (NHWC device tensors) ---------------------------------------------------------
def _cd(t):
    return BF16 if t.dtype == torch.bfloat16 else F32


CONV_KERNELS = {"auto": 0, "simt": 1, "pair": 2, "1cta": 3}     # include/pulse.h PULSE_CONV_*


def conv2d(src0, w, src1=None, bias=None, pn=None, residual=None, stride=1, kernel="auto", chan_stats=None):
    """chan_stats: zeroed fp32 [n, 2, cout]; receives the sum / sum of squares per (image, channel) of the stored output."""
    n, h, wd, c0 = src0.shape
    cout, k = w.shape[0], w.shape[1]
    out = torch.empty((n, h // stride, wd // stride, cout), dtype=src0.dtype, device=src0.device)
    _ck(lib.pulse_conv2d(_cd(src0), CONV_KERNELS[kernel], _ptr(src0), c0, _ptr(src1), 0 if src1 is None else src1.shape[3],
                         n, h, wd, k, stride, _ptr(w), cout, _ptr(bias), _ptr(pn), _ptr(residual), _ptr(out),
                         _ptr(chan_stats), _stream()))
    return out


def conv2d_dgrad(g, w, in_hw, stride=1, kernel="auto", g_in=None):
    n, cout = g.shape[0], g.shape[3]
    k, cin = w.shape[1], w.shape[3]
    acc = g_in is not None
    if g_in is None:
        g_in = torch.empty((n, in_hw[0], in_hw[1], cin), dtype=g.dtype, device=g.device)
    wt = torch.empty(w.numel(), dtype=w.dtype, device=w.device)
    _ck(lib.pulse_conv2d_dgrad(_cd(g), CONV_KERNELS[kernel], _ptr(g), n, in_hw[0], in_hw[1], cin, k, stride, _ptr(w), cout,
                               _ptr(wt), _ptr(g_in), int(acc), _stream()))
    return g_in


def conv2d_wgrad(src0, g, ksize, src1=None, stride=1, force_simt=False, dw=None):
    """dw given: += into it; else a fresh gradient (written into a NaN-filled buffer: accumulate = 0 must overwrite)."""
    n, h, wd, c0 = src0.shape
    c1 = 0 if src1 is None else src1.shape[3]
    cout = g.shape[3]
    acc = dw is not None
    if dw is None:
        dw = torch.full((cout, ksize, ksize, c0 + c1), float("nan"), dtype=torch.float32, device=g.device)
    _ck(lib.pulse_conv2d_wgrad(_cd(src0), int(force_simt), _ptr(src0), c0, _ptr(src1), c1, n, h, wd, ksize, stride,
                               _ptr(g), cout, _ptr(dw), int(acc), _stream()))
    return dw


def upsample_conv2d(src, w, bias=None, kernel="auto", chan_stats=None):
    """conv3x3(upsample2(src)) in the 4-phase form (no upsampled tensor)."""
    n, h, wd, cin = src.shape
    cout = w.shape[0]
    out = torch.empty((n, 2 * h, 2 * wd, cout), dtype=src.dtype, device=src.device)
    wp = torch.empty(16 * cout * cin, dtype=src.dtype, device=src.device)
    _ck(lib.pulse_upsample_conv2d(_cd(src), CONV_KERNELS[kernel], _ptr(src), n, h, wd, cin, _ptr(w), cout, _ptr(bias),
                                  _ptr(wp), _ptr(out), _ptr(chan_stats), _stream()))
    return out


def upsample_conv2d_dgrad(g, w, kernel="auto"):
    n, h2, w2, cout = g.shape
    cin = w.shape[3]
    g_in = torch.empty((n, h2 // 2, w2 // 2, cin), dtype=g.dtype, device=g.device)
    wpt = torch.empty(16 * cout * cin, dtype=g.dtype, device=g.device)
    _ck(lib.pulse_upsample_conv2d_dgrad(_cd(g), CONV_KERNELS[kernel], _ptr(g), n, h2 // 2, w2 // 2, cin, _ptr(w), cout,
                                        _ptr(wpt), _ptr(g_in), _stream()))
    return g_in


def upsample_conv2d_wgrad(src, g):
    n, h, wd, cin = src.shape
    cout = g.shape[3]
    dw = torch.zeros((cout, 3, 3, cin), dtype=torch.float32, device=g.device)
    _ck(lib.pulse_upsample_conv2d_wgrad(_cd(src), _ptr(src), n, h, wd, cin, _ptr(g), cout, _ptr(dw), _stream()))
    return dw


def attention(qkv, heads, force_simt=False):
    """qkv [n, tokens, 3c] -> (o [n, tokens, c], stats)."""
    n, t, c3 = qkv.shape
    c = c3 // 3
    o = torch.empty((n, t, c), dtype=qkv.dtype, device=qkv.device)
    stats = torch.empty(lib.pulse_attention_stats_floats(n, heads, t), dtype=torch.float32, device=qkv.device)
    _ck(lib.pulse_attention(_cd(qkv), int(force_simt), _ptr(qkv), n, t, c, heads, _ptr(o), _ptr(stats), _stream()))
    return o, stats


def attention_backward(qkv, g_o, heads, stats, force_simt=False):
    n, t, c3 = qkv.shape
    g_qkv = torch.empty_like(qkv)
    _ck(lib.pulse_attention_backward(_cd(qkv), int(force_simt), _ptr(qkv), _ptr(g_o), n, t, c3 // 3, heads, _ptr(stats),
                                     _ptr(g_qkv), _stream()))
    return g_qkv


def groupnorm_silu(x0, gamma, beta, groups, eps=1e-5, x1=None, stats=None):
    """a = SiLU(GroupNorm(concat_C(x0, x1))); returns (a, stats).  stats from an earlier call on the same x: only the
    normalise + SiLU pass runs."""
    n, h, wd, c0 = x0.shape
    c1 = 0 if x1 is None else x1.shape[3]
    reuse = stats is not None
    if stats is None:
        stats = torch.empty(lib.pulse_groupnorm_stats_floats(n, c0 + c1, groups), dtype=torch.float32, device=x0.device)
    a = torch.empty((n, h, wd, c0 + c1), dtype=x0.dtype, device=x0.device)
    _ck(lib.pulse_groupnorm_silu(_cd(x0), _ptr(x0), c0, _ptr(x1), c1, n, h, wd, groups, eps, _ptr(gamma), _ptr(beta),
                                 _ptr(stats), int(reuse), _ptr(a), _stream()))
    return a, stats


def groupnorm_silu_backward(g_a, x0, gamma, beta, groups, stats, eps=1e-5, x1=None, add=None, two_pass=False,
                            g_x0=None, g_x1=None, scratch=None, dgamma=None, dbeta=None, fwd_data_ready=False):
    """Returns (g_x0, g_x1 or None, dgamma, dbeta); g_x0 / g_x1 given: accumulated into (+=)."""
    n, h, wd, c0 = x0.shape
    c1 = 0 if x1 is None else x1.shape[3]
    C_ = c0 + c1
    acc0, acc1 = g_x0 is not None, g_x1 is not None
    if g_x0 is None:
        g_x0 = torch.empty((n, h, wd, c0), dtype=x0.dtype, device=x0.device)
    if g_x1 is None and c1:
        g_x1 = torch.empty((n, h, wd, c1), dtype=x0.dtype, device=x0.device)
    if scratch is None:
        scratch = torch.empty(n * 2 * C_, dtype=torch.float32, device=x0.device)
    if dgamma is None:
        dgamma = torch.zeros(C_, dtype=torch.float32, device=x0.device)
        dbeta = torch.zeros(C_, dtype=torch.float32, device=x0.device)
    _ck(lib.pulse_groupnorm_silu_backward(_cd(x0), int(two_pass), int(fwd_data_ready), _ptr(g_a), _ptr(x0), c0, _ptr(x1), c1, n, h, wd, groups,
                                          eps, _ptr(gamma), _ptr(beta), _ptr(stats), _ptr(scratch), _ptr(add), _ptr(g_x0),
                                          int(acc0), _ptr(g_x1), int(acc1), _ptr(dgamma), _ptr(dbeta), _stream()))
    return g_x0, g_x1, dgamma, dbeta


# ---- skip-aware partitioning (host only) ------------------------------------------------------------
def partition(t_f, skips, p, act_bytes=None, lam=0.0, t_lat=0.0, b_inter=1.0):
    """PAPER.md sec. IV-B: returns (cuts, bottleneck); cuts[m] = 1-based last operation of stage m + 1; skips = [(src, dst)]
    1-based."""
    n = len(t_f)
    tf = (C.c_double * n)(*[float(v) for v in t_f])
    ab = None if act_bytes is None else (C.c_double * n)(*[float(v) for v in act_bytes])
    ns = len(skips)
    ss = (C.c_int * max(1, ns))(*[int(a) for a, _ in skips])
    sd = (C.c_int * max(1, ns))(*[int(b) for _, b in skips])
    cuts = (C.c_int * max(1, p - 1))()
    best = C.c_double()
    _ck(lib.pulse_partition(n, tf, ab, ns, ss, sd, p, lam, t_lat, b_inter, cuts, C.byref(best)))
    return list(cuts[:p - 1]), best.value
