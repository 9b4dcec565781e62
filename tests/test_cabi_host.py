"""Host-side checks of libpulse.so that need no GPU: the library loads, exports every
symbol include/pulse.h declares, validates descriptors, lays out parameters in the
documented order and reports the closed-form skip-cache sizes."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2606_19163_b200 import workloads as W

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_2606_19163_b200 import build
    build.build()
    from paper_2606_19163_b200 import binding
    return binding


def test_exports_every_declared_symbol(B):
    hdr = open(os.path.join(ROOT, "include", "pulse.h")).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    declared = set(re.findall(r"\b(pulse_[a-z0-9_]+)\s*\(", hdr))
    assert len(declared) >= 25
    for name in declared:
        assert hasattr(B.lib, name), f"{name} declared in pulse.h but not exported"
    assert declared == set(B.EXPORTS), declared ^ set(B.EXPORTS)
    assert B.lib.pulse_version() >= 100
    assert B.lib.pulse_status_string(5).decode().startswith("skip cache")


@pytest.mark.parametrize("i", [1, 2, 3, 4, 5])
def test_param_table_matches_recipe(B, i):
    desc = W.config(i)
    st = B.Stage(desc, allocate=False)
    specs = W.param_specs(desc)
    assert [p["name"] for p in st.params] == [s[0] for s in specs]
    esz = 4 if desc["dtype"] == "fp32" else 2
    off = goff = 0
    for p, (name, shape, kind, fan_in) in zip(st.params, specs):
        dev_shape = (shape[0], shape[2], shape[3], shape[1]) if len(shape) == 4 else shape
        assert p["shape"] == tuple(dev_shape), name
        assert p["off"] == off and p["goff"] == goff and off % 256 == 0
        numel = int(np.prod(shape))
        off = (off + numel * esz + 255) // 256 * 256
        goff = (goff + numel * 4 + 255) // 256 * 256
    assert st.param_bytes == off and st.grad_bytes == goff


def test_skip_cache_bytes_closed_forms(B):
    """64 KiB, 30 MiB, 25 MiB, 101.25 MiB, 97.5 MiB x 8 = 780 MiB."""
    want = {1: 0.0625, 2: 30, 3: 25, 4: 101.25, 5: 97.5}
    for i, mib in want.items():
        st = B.Stage(W.config(i), allocate=False)
        assert st.skip_bytes == int(mib * 2 ** 20), (i, st.skip_bytes)
    assert B.Stage(W.config(5), allocate=False).max_inflight == 8


def test_descriptor_errors(B):
    def status_of(desc, **kw):
        with pytest.raises(B.PulseError) as ei:
            B.Stage(desc, allocate=False, **kw)
        return ei.value.status
    d = W.mini("level")
    d["dec_ops"] = d["dec_ops"] + [W.rb(8, 8, skip=8)]
    assert status_of(d) == 2                       # pops more than pushed
    d = W.mini("level")
    d["dec_ops"] = d["dec_ops"][:2]
    assert status_of(d) == 2                       # cached skip never consumed
    d = W.mini("level")
    d["dec_ops"][0] = W.rb(8, 8, skip=16)
    assert status_of(d) == 2                       # skip channel mismatch
    d = W.mini("level")
    d["groups"] = 3
    assert status_of(d) == 2                       # C % groups
    d = W.mini("updown")
    d["h"] = 5
    assert status_of(d) == 2                       # odd H into a stride-2 down
    d = W.mini("unet")
    d["link"] = "open"
    assert status_of(d) == 2                       # mid ops in an OPEN stage
    d = W.mini("level")
    d["n"] = 0
    assert status_of(d) == 1
    h = C.c_void_p()
    assert B.lib.pulse_stage_create(None, C.byref(h)) == 1
    assert B.lib.pulse_last_error().decode() != ""


def test_unbound_stage_refuses_to_run(B):
    st = B.Stage(W.mini("level"), allocate=False)
    n = C.c_size_t()
    assert B.lib.pulse_stage_workspace_bytes(st.h, C.byref(n), None) == 0 and n.value > 0
    # no cache / params: forward must fail with a status, not crash
    assert B.lib.pulse_stage_forward(st.h, None, 0, None, None, None, None, None, None) == 1
    assert B.lib.pulse_stage_bind_params(st.h, C.c_void_p(1), C.c_void_p(256)) == 1   # misaligned
    assert B.lib.pulse_stage_bind_workspace(st.h, C.c_void_p(256), 8) == 4            # too small


def test_groupnorm_entry_points_validate_before_any_launch(B):
    """include/pulse.h: INVALID_ARG for null pointers / sizes, SHAPE for C % groups and channel counts off the
    16-byte vector; the scratch size is the closed form n * 2 * (C + groups)."""
    L = B.lib
    assert L.pulse_groupnorm_stats_floats(4, 640, 32) == 4 * 2 * (640 + 32)
    assert L.pulse_groupnorm_stats_floats(0, 640, 32) == 0
    p = C.c_void_p(256)      # never dereferenced: validation comes first
    fwd = lambda dt, x0, c0, x1, c1, n, g: L.pulse_groupnorm_silu(dt, x0, c0, x1, c1, n, 8, 8, g, 1e-5, p, p, p, 0, p, None)
    INVALID, SHAPE = 1, 2
    assert fwd(B.BF16, None, 64, None, 0, 2, 8) == INVALID
    assert fwd(B.BF16, p, 64, None, 32, 2, 8) == INVALID              # c1 > 0 without x1
    assert fwd(B.BF16, p, 64, None, 0, 0, 8) == INVALID
    assert fwd(7, p, 64, None, 0, 2, 8) == INVALID
    assert fwd(B.BF16, p, 64, None, 0, 2, 7) == SHAPE                 # 64 % 7
    assert fwd(B.BF16, p, 60, None, 0, 2, 4) == SHAPE                 # 60 channels: not a multiple of 8 bf16
    bwd = lambda g_a, c0, g: L.pulse_groupnorm_silu_backward(B.BF16, 0, 0, g_a, p, c0, None, 0, 2, 8, 8, g, 1e-5, p, p, p, p,
                                                             None, p, 0, None, 0, p, p, None)
    assert bwd(None, 64, 8) == INVALID
    assert bwd(p, 64, 7) == SHAPE
    assert b"divisible" in L.pulse_last_error()
