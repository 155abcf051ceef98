"""radt_disk_fields_static: the physics pre-pass for callers that cannot allocate device memory.

Who needs it: code that runs inside a process which gave all device memory away at start-up (an application's own
memory pool, fixed partitions of a control loop), so that it can neither cudaMalloc a workspace nor ask its host for
one, and loops that cannot take the device-wide synchronisation of cudaMalloc / cudaFree.  For them the scratch of the
forward pre-pass sits in a fixed array inside libradt.so (8 MiB on every GPU that loads the library, at most
RADT_DISK_STATIC_MAX_CELLS = 262 144 cells per call) and the entry point allocates nothing.

The test compares the new entry point with radt_disk_fields (same kernels, caller-allocated workspace) on calls made
back to back: every call shares the one array, which still holds what the call before it left, so a call that relied on
zeroed scratch, or on scratch of its own size, would show here.  The file is named so that pytest collects it last: with
`pytest -x` a failure here must not hide the other tests.  It passes alone in a fresh process (then its first call is
the one that looks up the array's device address) and after the rest of the suite.
"""
import ctypes as C
import os

import numpy as np
import pytest

from oracle import disk_physics as dp
from synth import make_config

GM_SUN = 1.32712440018e26
AMU = 1.66053906660e-24


def _params(k=0):
    return dp.DiskParams(gm_star=(2.0 + 0.2 * k) * GM_SUN, m_mol=2.37 * AMU, sigma0=30.0 + 5.0 * k, r_c=150.0 - 10.0 * k,
                         gamma=1.0 - 0.1 * k, t_freeze=19.0 + k, n_dissoc=1e21)


def test_sizes_beyond_the_fixed_scratch_are_refused_on_the_host():
    """Config 5's 16 x 256 x 128 = 524 288 cells do not fit the 262 144-cell array: the call must say so (on the host,
    before any CUDA call, so this runs without a GPU) instead of writing past the array."""
    from paper_2509_03623_b200 import binding as B
    from paper_2509_03623_b200 import build as radt_build
    radt_build.build()
    L = B.lib()
    scenes = make_config(5, npix=8)
    desc = B.Descriptors(scenes)
    assert desc.batch * desc.grid.n[0] * desc.grid.n[1] > B.DISK_STATIC_MAX_CELLS
    disks = B.make_disks([_params(k) for k in range(len(scenes))])
    fake = C.c_void_p(4096)                                      # never dereferenced: the size check comes first
    rc = L.radt_disk_fields_static(disks, C.byref(desc.grid), desc.batch, fake, fake, fake, None)
    assert rc == -1 and b"exceeds the fixed scratch" in L.radt_last_error()
    root = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
    hdr = open(os.path.join(root, "include", "radt.h")).read()
    assert f"#define RADT_DISK_STATIC_MAX_CELLS {B.DISK_STATIC_MAX_CELLS}" in hdr


@pytest.mark.gpu
def test_static_scratch_pre_pass_equals_the_workspace_path_on_calls_in_a_row():
    torch = pytest.importorskip("torch")
    from paper_2509_03623_b200 import binding as B
    B.lib()
    # three shapes one after the other on the same array: a batch (8 x 256 x 128 = the full 262 144 cells), then a
    # small grid that reuses the front of what the batch left behind, then a large single grid, then the batch again
    calls = [make_config(5, npix=8, batch=8), [make_config(1)], [make_config(3, npix=8)], make_config(5, npix=8, batch=8)]
    free0 = None
    for n, scenes in enumerate(calls):
        desc = B.Descriptors(scenes)
        params = [_params(k) for k in range(len(scenes))]
        disks = B.make_disks(params)
        temp = torch.from_numpy(B.stack_fields(scenes)[1]).cuda()
        assert temp.numel() <= B.DISK_STATIC_MAX_CELLS
        ws = torch.empty(B.radt_disk_workspace_bytes(desc), dtype=torch.uint8, device="cuda")
        want_n, want_v = torch.empty_like(temp), torch.empty_like(temp)
        B.radt_disk_fields(disks, desc, temp, want_n, want_v, ws)
        got_n, got_v = torch.full_like(temp, float("nan")), torch.full_like(temp, float("nan"))
        torch.cuda.synchronize()
        if n == 1:                                               # the address look-up happened in call 0
            free0 = torch.cuda.mem_get_info()[0]
        B.radt_disk_fields_static(disks, desc, temp, got_n, got_v)
        # and once more straight after it, into the same outputs: the second call sees the first one's scratch
        B.radt_disk_fields_static(disks, desc, temp, got_n, got_v)
        torch.cuda.synchronize()
        if n == 1:
            assert torch.cuda.mem_get_info()[0] == free0, "the call changed the amount of free device memory"
        # tolerance of tests/test_gpu_disk_physics.py (the two paths run the same fp64 kernels, so in fact equal)
        np.testing.assert_allclose(got_n.cpu().numpy(), want_n.cpu().numpy(), rtol=2e-7, atol=0.0)
        np.testing.assert_allclose(got_v.cpu().numpy(), want_v.cpu().numpy(), rtol=2e-7, atol=1e-3)
        assert (want_n > 0).any() and (want_n == 0).any()
    # and against the oracle itself on the last call's first item, as the workspace path is checked
    gr = calls[-1][0].grid
    r, zeta = dp.nodes(gr.n[0], gr.n[1], gr.lo[0], gr.hi[0], gr.hi[1])
    fw = dp.forward(_params(0), temp[0].cpu().numpy(), r, zeta)
    same = (got_n[0].cpu().numpy() > 0) == fw["mask"]
    assert same.mean() > 0.999
    np.testing.assert_allclose(got_n[0].cpu().numpy()[same], fw["n_co"][same], rtol=2e-7)
    np.testing.assert_allclose(got_v[0].cpu().numpy(), fw["v_phi"], rtol=2e-7, atol=1e-3)
