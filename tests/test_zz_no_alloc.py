"""lpc_fid_sample_noalloc (include/lpc.h): Eq. 12 with the reduction's scratch in the library's static device array.

Collected last on purpose (the suite runs with ``pytest -x``).  Needs nothing from the other tests: it passes alone in a
fresh process and after them.  The existing path it is compared with is the lattice's own FID series: G[0] from the
reduction behind lpc_set_site_params / lpc_set_state (block partials in the caller's workspace) and G[n] from the sweep's
fused reduction, within the FID tolerance of the parity tests (1e-9 of sum |g|).
"""
import importlib.util
import os

import numpy as np
import pytest

import lpc_inputs

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def lpc():
    import torch

    assert torch.cuda.is_available(), "this test needs the B200"
    spec = importlib.util.spec_from_file_location("_lpc_build", os.path.join(ROOT, "paper_2603_22553_b200", "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.build()
    import paper_2603_22553_b200 as m

    return m


def _sample(lpc, g_host):
    """One call of the new entry point on a host array of complex numbers; returns (G, the device tensors kept alive)."""
    import torch

    g_dev = torch.from_numpy(np.ascontiguousarray(g_host, dtype=np.complex128).reshape(-1)).cuda()
    out = torch.full((2,), float("nan"), dtype=torch.float64, device="cuda")
    lpc.lpc_fid_sample_noalloc(g_dev.data_ptr(), g_dev.numel(), out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    return complex(o[0], o[1])


def test_no_alloc_fid_sample_matches_the_lattice_series(lpc):
    import torch

    n = 24
    # 64 x 48 x 100 = 307200 sites: ten block partials, the last one ragged
    lat = lpc_inputs.random_small((64, 48, 100), bc=(0, 1, 0), p_block=0.25, alpha=0.9, seed=17, n_steps=n, n_moments=0)
    rng = np.random.default_rng(4)
    g0 = (rng.standard_normal(lat.shape) + 1j * rng.standard_normal(lat.shape)) * (lat.blocked == 0)
    gpu = lpc.Lattice.from_inputs(lat, max_steps=n, g0=g0)

    # first call: the initial state against G[0] of the existing reduction
    G0 = gpu.fid()[0]
    got0 = _sample(lpc, g0)
    assert abs(got0 - G0) <= 1e-9 * np.abs(g0).sum()
    assert abs(got0 - g0.sum()) <= 1e-12 * np.abs(g0).sum()

    # second call, right after: the state n steps on against G[n] of the sweep's fused reduction; the scratch array still
    # holds the first call's partials
    gpu.step(n)
    g_n = gpu.field(lpc.LPC_FIELD_G)
    Gn = gpu.fid()[n]
    got_n = _sample(lpc, g_n)
    assert abs(got_n - Gn) <= 1e-9 * np.abs(g_n).sum()

    # third and fourth call: a smaller array (one partial: the nine stale ones must not be read), then the first one again,
    # bit for bit what the first call gave
    small = g_n[:3, :5, :7]
    got_s = _sample(lpc, small)
    assert abs(got_s - small.sum()) <= 1e-12 * max(np.abs(small).sum(), 1e-300)
    again = _sample(lpc, g0)
    assert again == got0

    # the same input through a device-resident read-out (lpc_read_field to a device pointer), no host copy in between
    dev = torch.empty(2 * lat.n_sites, dtype=torch.float64, device="cuda")
    lpc.lpc_read_field(gpu.handle, lpc.LPC_FIELD_G, dev)
    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    lpc.lpc_fid_sample_noalloc(dev.data_ptr(), lat.n_sites, out.data_ptr(), torch.cuda.current_stream().cuda_stream)
    torch.cuda.synchronize()
    o = out.cpu().numpy()
    assert complex(o[0], o[1]) == got_n
    gpu.close()


def test_no_alloc_fid_sample_limits_and_errors(lpc):
    import torch

    out = torch.zeros(2, dtype=torch.float64, device="cuda")
    g = torch.zeros(8, dtype=torch.float64, device="cuda")
    # beyond what the static array covers: refused before anything is touched
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_fid_sample_noalloc(g.data_ptr(), lpc.LPC_NOALLOC_MAX_SITES + 1, out.data_ptr())
    assert e.value.code == lpc.LPC_EINVAL and "LPC_NOALLOC_MAX_SITES" in str(e.value)
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_fid_sample_noalloc(g.data_ptr(), -1, out.data_ptr())
    assert e.value.code == lpc.LPC_EINVAL
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_fid_sample_noalloc(0, 4, out.data_ptr())
    assert e.value.code == lpc.LPC_EINVAL
    host = np.zeros(8)
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_fid_sample_noalloc(host.ctypes.data, 4, out.data_ptr())
    assert e.value.code == lpc.LPC_EINVAL
    # no sites: the sum is zero
    out.fill_(7.0)
    lpc.lpc_fid_sample_noalloc(g.data_ptr(), 0, out.data_ptr())
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [0.0, 0.0]
    # and a good call after the refused ones
    g.copy_(torch.arange(8, dtype=torch.float64))
    lpc.lpc_fid_sample_noalloc(g.data_ptr(), 4, out.data_ptr())
    torch.cuda.synchronize()
    assert out.cpu().tolist() == [0.0 + 2 + 4 + 6, 1.0 + 3 + 5 + 7]
