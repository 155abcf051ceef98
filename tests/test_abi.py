"""The C-ABI library loads, exports every symbol include/radt.h declares, and validates arguments on the
host (no GPU needed: no compute call is made here)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

from paper_2509_03623_b200 import binding as B
from paper_2509_03623_b200 import build as radt_build
from synth import make_config, tiny_axisym_scene, tiny_cart_scene

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lib():
    radt_build.build()
    return B.lib()


def test_exports_match_header(lib):
    hdr = open(os.path.join(ROOT, "include", "radt.h")).read()
    declared = sorted(set(re.findall(r"\b(radt_[a-z0-9_]+)\s*\(", hdr)))
    assert len(declared) >= 14
    for name in declared:
        assert hasattr(lib, name), f"{name} declared in include/radt.h but not exported"
    assert sorted(B.EXPORTS) == declared, "binding.EXPORTS must mirror include/radt.h"
    assert lib.radt_version() == 200


def test_struct_layouts_and_workspace_size(lib):
    """radt_workspace_bytes is host-only and checks struct_size: a ctypes/C layout mismatch fails here."""
    for sc in (tiny_axisym_scene(), tiny_cart_scene(), make_config(1)):
        d = B.Descriptors(sc)
        fwd = B.radt_workspace_bytes(d, B.PASS_FWD)
        bwd = B.radt_workspace_bytes(d, B.PASS_BWD)
        assert 0 < fwd < bwd
        assert bwd - fwd >= d.cells * 16          # packed float4 gradient cells
    d = B.Descriptors(make_config(2))
    assert B.radt_workspace_bytes(d, B.PASS_FWD) >= 256 * 256 * 16 + 256 * 128 * 16


@pytest.mark.parametrize("mutate,code", [
    (lambda d: setattr(d.geom[0], "struct_size", 3), -1),
    (lambda d: setattr(d.geom[0], "nstep", 0), -1),
    (lambda d: setattr(d.geom[0], "fov_x", -1.0), -1),
    (lambda d: setattr(d.line, "nchan", 257), -1),
    (lambda d: setattr(d.line, "nlev", 65), -1),
    (lambda d: setattr(d.line, "nu0", 0.0), -1),
    (lambda d: setattr(d.grid, "kind", 7), -2),
    (lambda d: setattr(d.grid, "dens_mode", 5), -2),
    (lambda d: d.grid.lo.__setitem__(0, -1.0), -1),
    (lambda d: d.grid.n.__setitem__(1, 1), -1),
])
def test_invalid_arguments_are_rejected(lib, mutate, code):
    d = B.Descriptors(tiny_axisym_scene())
    mutate(d)
    out = C.c_size_t(0)
    rc = lib.radt_workspace_bytes(d.geom, C.byref(d.line), C.byref(d.grid), d.batch, 0, C.byref(out))
    assert rc == code
    assert len(lib.radt_last_error()) > 0


def test_null_and_unsupported(lib):
    d = B.Descriptors(tiny_cart_scene())
    d.grid.mirror_z = 1
    out = C.c_size_t(0)
    assert lib.radt_workspace_bytes(d.geom, C.byref(d.line), C.byref(d.grid), 1, 0, C.byref(out)) == -2
    d = B.Descriptors(tiny_axisym_scene())
    assert lib.radt_workspace_bytes(d.geom, C.byref(d.line), C.byref(d.grid), 1, 0, None) == -1
    assert lib.radt_workspace_bytes(None, C.byref(d.line), C.byref(d.grid), 1, 0, C.byref(out)) == -1
    assert lib.radt_workspace_bytes(d.geom, C.byref(d.line), C.byref(d.grid), 0, 0, C.byref(out)) == -1
    assert lib.radt_workspace_bytes(d.geom, C.byref(d.line), C.byref(d.grid), 1, 9, C.byref(out)) == -1
    # counter read-outs refuse null pointers before touching the device
    out4, out2 = (C.c_uint64 * 4)(), (C.c_uint64 * 2)()
    assert lib.radt_read_counters(None, out4, None) == -1 and lib.radt_read_counters(C.c_void_p(16), None, None) == -1
    assert lib.radt_read_lane_counters(None, out2, None) == -1 and lib.radt_read_lane_counters(C.c_void_p(16), None, None) == -1


def test_options_struct_defaults_and_size_check(lib):
    """radt_options: per-call POD with struct_size first; NULL means the defaults radt_options_default writes."""
    o = B.make_options()
    assert (o.struct_size, o.window, o.skip_empty, o.win_path, o.zero_dens_grad, o.reuse_setup) == (C.sizeof(B.radt_options), 1, 1, 1, 1, 0)
    assert B.make_options(window=0, zero_dens_grad=0).window == 0
    with pytest.raises(KeyError):
        B.make_options(compensated=1)
    assert not hasattr(lib, "radt_set_option") and not hasattr(lib, "radt_get_option")     # no process-wide option state
    d = B.Descriptors(tiny_axisym_scene())
    bad = B.make_options()
    bad.struct_size = 8
    fake = C.c_void_p(0x1000)          # never dereferenced: the options are checked before any device work
    assert lib.radt_render(d.geom, C.byref(d.line), C.byref(d.grid), 1, C.byref(bad), fake, None, fake, 1 << 30, None) == -1
    assert b"radt_options" in lib.radt_last_error()


def test_forward_adjoint_option_mismatch_is_refused_on_the_host(lib):
    """The library remembers per cube pointer the options of the forward that wrote it; an adjoint with other options
    (or another cube_lo choice) fails with RADT_E_INVALID before any device work.  Runs where there is no GPU: the
    pointers are fakes, and every call that gets past the host checks fails with RADT_E_CUDA."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present: tests/test_gpu_parity.py covers this with real buffers")
    d = B.Descriptors(tiny_axisym_scene())
    d.with_fields(0x10000, 0x20000, 0x30000)
    cube, lo, dl, ws = (C.c_void_p(a) for a in (0x100000, 0x200000, 0x300000, 0x400000))
    args = (d.geom, C.byref(d.line), C.byref(d.grid), 1)
    o = B.make_options()
    assert lib.radt_render(*args, C.byref(o), cube, lo, ws, 1 << 30, None) == -4          # registered, then no device
    for bad in (B.make_options(window=0), B.make_options(skip_empty=0), B.make_options(win_path=0)):
        assert lib.radt_render_bwd(*args, C.byref(bad), cube, lo, dl, None, None, None, ws, 1 << 30, None) == -1
    assert lib.radt_render_bwd(*args, C.byref(o), cube, None, dl, None, None, None, ws, 1 << 30, None) == -1      # cube_lo dropped
    assert lib.radt_render_bwd(*args, C.byref(o), cube, lo, dl, None, None, None, ws, 1 << 30, None) == -4        # consistent
    r = B.make_options(reuse_setup=1)
    assert lib.radt_render(*args, C.byref(r), cube, lo, ws, 1 << 30, None) == -1                                 # adjoint-only option
    other = C.c_void_p(0x500000)
    assert lib.radt_render_bwd(*args, C.byref(r), cube, lo, dl, None, None, None, other, 1 << 30, None) == -1    # unknown workspace
    assert lib.radt_render(*args, C.byref(o), cube, lo, ws, 1 << 30, None) == -4
    assert lib.radt_render_bwd(*args, C.byref(r), cube, lo, dl, None, None, None, ws, 1 << 30, None) == -4       # same inputs: accepted
    d.geom[0].incl = 0.3
    assert lib.radt_render_bwd(*args, C.byref(r), cube, lo, dl, None, None, None, ws, 1 << 30, None) == -1       # other geometry


def test_cube_memory_ignores_batch_and_can_be_forgotten(lib):
    """What the library remembers about a cube pointer is what shapes its partial sums (window, skip_empty, kernel family,
    cube_lo, channel count), not the batch or the image size: the adjoint of the first item of a batched forward (same
    pointer, smaller batch) is accepted.  radt_forget drops the memory of a pointer whose buffer was refilled or recycled.
    No GPU: fake pointers, calls that pass the host checks end in RADT_E_CUDA (-4)."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present: fake device pointers would be dereferenced")
    scs = make_config(5, npix=8, batch=3)
    d3, d1 = B.Descriptors(scs), B.Descriptors(scs[:1])
    for d in (d3, d1):
        d.with_fields(0x10000, 0x20000, 0x30000)
    cube, lo, dl, ws = (C.c_void_p(a) for a in (0x1100000, 0x1200000, 0x1300000, 0x1400000))
    o = B.make_options()
    a3 = (d3.geom, C.byref(d3.line), C.byref(d3.grid), 3)
    a1 = (d1.geom, C.byref(d1.line), C.byref(d1.grid), 1)
    assert lib.radt_render(*a3, C.byref(o), cube, lo, ws, 1 << 30, None) == -4
    assert lib.radt_render_bwd(*a1, C.byref(o), cube, lo, dl, None, None, None, ws, 1 << 30, None) == -4        # sub-batch: fine
    bad = B.make_options(window=0)
    assert lib.radt_render_bwd(*a1, C.byref(bad), cube, lo, dl, None, None, None, ws, 1 << 30, None) == -1      # other options
    assert b"radt_forget" in lib.radt_last_error()
    assert lib.radt_forget(cube) == 0                                                                          # buffer recycled
    assert lib.radt_render_bwd(*a1, C.byref(bad), cube, lo, dl, None, None, None, ws, 1 << 30, None) == -4      # unknown origin: accepted
    assert lib.radt_forget(C.c_void_p(0x7777000)) == 0 and lib.radt_forget(None) == -1
    # a forgotten workspace no longer vouches for reuse_setup
    r = B.make_options(reuse_setup=1)
    assert lib.radt_render(*a3, C.byref(o), cube, lo, ws, 1 << 30, None) == -4
    assert lib.radt_render_bwd(*a3, C.byref(r), cube, lo, dl, None, None, None, ws, 1 << 30, None) == -4
    assert lib.radt_forget(ws) == 0
    assert lib.radt_render_bwd(*a3, C.byref(r), cube, lo, dl, None, None, None, ws, 1 << 30, None) == -1


def test_host_split_hook_takes_sizes_not_environment_variables(lib):
    assert lib.radt_debug_host_split(2, 16) == 0 and lib.radt_debug_host_split(0, 0) == 0
    assert lib.radt_debug_host_split(-1, 0) == -1
    src = open(os.path.join(ROOT, "paper_2509_03623_b200", "csrc", "radt_api.cu")).read()
    assert "getenv" not in src                                    # the shipped library reads no environment variables


def test_grad_layout(lib):
    d = B.Descriptors(make_config(1))
    off, n = B.radt_grad_layout(d)
    assert n == 4 * d.cells and off % 256 == 0
    assert off + 4 * n <= B.radt_workspace_bytes(d, B.PASS_BWD)


def test_batch_items_must_share_image_shape(lib):
    a, b = tiny_axisym_scene(npix=6), tiny_axisym_scene(npix=7)
    d = B.Descriptors([a, b])
    out = C.c_size_t(0)
    assert lib.radt_workspace_bytes(d.geom, C.byref(d.line), C.byref(d.grid), 2, 0, C.byref(out)) == -1


def test_no_cpu_fallback_without_a_device(lib):
    """On a box without a GPU the compute entry points fail loudly (RADT_E_CUDA); nothing is computed on the CPU."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    sc = tiny_axisym_scene()
    d = B.Descriptors(sc)
    h = B.stack_fields(sc)
    cube = np.full(d.cube_shape, 7.0, np.float32)
    with pytest.raises(B.RadtError, match="-4"):
        B.radt_render_host(d, *h, cube)
    with pytest.raises(B.RadtError, match="-4"):
        B.radt_render_host(d, *h, cube, B.make_options(window=0), np.zeros_like(cube))
    assert np.all(cube == 7.0)
    from paper_2509_03623_b200 import Renderer
    with pytest.raises(B.RadtError):
        Renderer(sc)
