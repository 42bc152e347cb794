"""Parity of the CUDA library (through the C ABI) against the CPU oracle, on a B200.

Tolerances, fp64:
  per site   |g_gpu - g_orc|_i  <= 1e-10 * pi_i            (|g_i(n)| <= pi_i for all n)
  FID        |G_gpu - G_orc|[n] <= 1e-9 * sum_i |g_i(n)|   (the sum's own scale, <= G[0] = 1)
  moments    |P_gpu - P_orc|_i  <= 1e-10 * a * pi_i,  |Z_gpu - Z_orc|[m] <= 1e-9 * Z[1],
             |D_gpu - D_orc|    <= 1e-9 * Z[1] / (2 dt)
fp32 mode: the same with 1e-5, checked at n <= 200.
"""
import importlib.util
import os

import numpy as np
import pytest

import lpc_inputs

pytestmark = pytest.mark.gpu

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
FULL = os.environ.get("LPC_FULL", "0") == "1"


@pytest.fixture(scope="module")
def lpc():
    import torch

    assert torch.cuda.is_available(), "these tests need the B200"
    spec = importlib.util.spec_from_file_location("_lpc_build", os.path.join(ROOT, "paper_2603_22553_b200", "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.build()
    import paper_2603_22553_b200 as m

    return m


def _check(lpc, lat, gpu, orc, n, tol_site=1e-10, tol_sum=1e-9, what=""):
    pi = orc.pi()
    G_o, sabs = orc.fid(with_scale=True)
    G_g = gpu.fid()
    assert G_g.shape == G_o.shape == (n + 1,)
    err_G = np.abs(G_g - G_o) / sabs
    assert err_G.max() <= tol_sum, f"{what} FID: max scaled error {err_G.max():.3e} at n={err_G.argmax()}"
    g_o, g_g = orc.g(), gpu.field(lpc.LPC_FIELD_G)
    opn = lat.blocked == 0
    assert np.all(g_g[~opn] == 0)
    err_g = np.abs(g_g - g_o)[opn] / pi[opn]
    assert err_g.max() <= tol_site, f"{what} g: max scaled per-site error {err_g.max():.3e}"
    out = {"err_G": float(err_G.max()), "err_g": float(err_g.max())}
    if gpu.cfg.n_moments == 3:
        v_o, D_o = orc.moments()
        v_g, D_g = gpu.moments()
        z1 = np.abs(v_o[:, :1])
        z1 = np.where(z1 > 0, z1, z1.max())   # an axis of one site between walls has Z_d = 0: scale by the other axes
        err_Z = np.abs(v_g - v_o) / z1
        assert err_Z.max() <= tol_sum, f"{what} VACF: max scaled error {err_Z.max():.3e}"
        err_D = np.abs(D_g - D_o) / (z1[:, 0] / (2 * lat.dt))
        assert err_D.max() <= tol_sum, f"{what} D: scaled error {err_D.max():.3e}"
        for d in range(3):
            P_o, P_g = orc.P(d), gpu.field(lpc.LPC_FIELD_PX + d)
            err_P = np.abs(P_g - P_o)[opn] / (lat.a * pi[opn])
            assert err_P.max() <= tol_site, f"{what} P^{d}: max scaled per-site error {err_P.max():.3e}"
        out.update(err_Z=float(err_Z.max()), err_D=float(err_D.max()))
    return out


def _pair(lpc, oracle_mod, lat, n, kernel, n_moments=None, n_density=0, precision=0, g0=None):
    nm = lat.n_moments if n_moments is None else n_moments
    gpu = lpc.Lattice.from_inputs(lat, precision=precision, n_moments=nm, n_density=n_density, max_steps=n, g0=g0)
    gpu.set_kernel(kernel)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=nm, max_steps=n)
    if g0 is not None:
        orc.set_g(g0)
    return gpu, orc


KERNELS = [1, 2, 3]  # LPC_KERNEL_DIRECT, LPC_KERNEL_TMA, LPC_KERNEL_PERSIST


# ---------------------------------------------------------------------------------------------
# precompute (S0) against oracle O1-O4, O7
# ---------------------------------------------------------------------------------------------
def test_precompute_matches_oracle(lpc, oracle_mod):
    lat = lpc_inputs.random_small((20, 13, 37), bc=(1, 0, 0), p_block=0.3, alpha=0.8, seed=21, n_moments=3)
    gpu, orc = _pair(lpc, oracle_mod, lat, 0, 1)
    pi_o, pi_g = orc.pi(), gpu.field(lpc.LPC_FIELD_PI)
    opn = lat.blocked == 0
    assert np.all(pi_g[~opn] == 0)
    assert np.max(np.abs(pi_g - pi_o)[opn] / pi_o[opn]) < 5e-15
    assert abs(gpu.fid()[0] - 1.0) < 1e-14
    g = gpu.field(lpc.LPC_FIELD_G)
    assert np.max(np.abs(g - pi_o)[opn] / pi_o[opn]) < 5e-15
    v_o, _ = orc.moments(1)
    v_g, _ = gpu.moments(1)
    assert np.max(np.abs(v_g - v_o) / v_o) < 1e-13
    for d in range(3):
        P_o, P_g = orc.P(d), gpu.field(lpc.LPC_FIELD_PX + d)
        assert np.max(np.abs(P_g - P_o)[opn] / (lat.a * pi_o[opn])) < 1e-14


# ---------------------------------------------------------------------------------------------
# BASELINE configs[0]: 32^3, 2000 steps, G(t) and density
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", KERNELS)
def test_config0_full(lpc, oracle_mod, kernel):
    lat = lpc_inputs.config0()
    n = lat.n_steps
    gpu, orc = _pair(lpc, oracle_mod, lat, n, kernel, n_density=1)
    gpu.step(n)
    orc.step(n)
    _check(lpc, lat, gpu, orc, n, what=f"config0 kernel={kernel}")
    # "output G(t) and density": the density started at pi stays at pi (stationarity)
    rho = gpu.field(lpc.LPC_FIELD_RHO)
    pi = orc.pi()
    opn = lat.blocked == 0
    assert np.max(np.abs(rho - pi)[opn] / pi[opn]) <= 1e-10


# ---------------------------------------------------------------------------------------------
# several tiles + ragged tails, mixed boundary conditions, moments fused in
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", KERNELS)
@pytest.mark.parametrize("shape,bc,alpha", [
    ((70, 19, 133), (1, 0, 0), 0.8),    # ragged in y and z, 3 z-tiles, 3 y-tiles, 2+ x-chunks, reflective x
    ((33, 40, 64), (0, 1, 1), 1.0),     # exact z tile, reflective y and z
    ((9, 8, 200), (0, 0, 0), 0.5),      # short x, 4 z-tiles
    ((5, 3, 7), (0, 0, 0), 1.0),        # odd nz, smaller than one tile
    ((2, 1, 3), (0, 0, 0), 0.9),        # degenerate axes (Q17)
    ((1, 1, 1), (0, 0, 0), 1.0),        # a single site
    ((4, 4, 4), (1, 1, 1), 1.0),        # closed box
])
def test_shapes_and_boundaries(lpc, oracle_mod, kernel, shape, bc, alpha):
    lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.3 if np.prod(shape) > 8 else 0.0, alpha=alpha, seed=22, n_moments=3)
    lat.dt = 2.0e-5
    n = 60
    gpu, orc = _pair(lpc, oracle_mod, lat, n, kernel, n_density=1)
    gpu.step(n)
    orc.step(n)
    _check(lpc, lat, gpu, orc, n, what=f"{shape} {bc} kernel={kernel}")
    rho, pi = gpu.field(lpc.LPC_FIELD_RHO), orc.pi()
    opn = lat.blocked == 0
    assert np.max(np.abs(rho - pi)[opn] / pi[opn]) <= 1e-10


@pytest.mark.parametrize("nm,nd", [(0, 0), (0, 1), (3, 0), (3, 1)])
def test_channel_combinations_tma(lpc, oracle_mod, nm, nd):
    lat = lpc_inputs.random_small((40, 24, 96), bc=(0, 0, 1), p_block=0.2, alpha=0.9, seed=23)
    n = 40
    gpu, orc = _pair(lpc, oracle_mod, lat, n, 2, n_moments=nm, n_density=nd)
    gpu.step(17)
    gpu.step(n - 17)     # series append across calls
    orc.step(n)
    _check(lpc, lat, gpu, orc, n, what=f"nm={nm} nd={nd}")


def test_kernels_agree_bitwise_on_state_and_are_deterministic(lpc):
    lat = lpc_inputs.random_small((48, 20, 130), bc=(1, 0, 0), p_block=0.25, seed=24, n_moments=3)
    res = []
    for kernel in (1, 2, 2, 3, 3):
        gpu = lpc.Lattice.from_inputs(lat, max_steps=31)
        gpu.set_kernel(kernel)
        gpu.step(30)
        res.append((gpu.field(lpc.LPC_FIELD_G), gpu.fid(), gpu.moments()[0]))
    # same per-site arithmetic in both kernels: the fields agree bit for bit; the sums differ only by order
    assert np.array_equal(res[0][0], res[1][0])
    assert np.max(np.abs(res[0][1] - res[1][1])) < 1e-14
    # repeated runs of one kernel are bitwise reproducible (fixed-order reduction, no atomics on data)
    assert np.array_equal(res[1][0], res[2][0])
    assert np.array_equal(res[1][1], res[2][1])
    assert np.array_equal(res[1][2], res[2][2])
    # the persistent kernel (30 steps in one launch): same state bits, reproducible series
    assert np.array_equal(res[0][0], res[3][0])
    assert np.max(np.abs(res[0][1] - res[3][1])) < 1e-14
    assert np.max(np.abs(res[0][2] - res[3][2])) < 1e-14 * np.abs(res[0][2][:, :1]).max()
    assert np.array_equal(res[3][1], res[4][1]) and np.array_equal(res[3][2], res[4][2])
    # odd step counts, repeated calls and a single step (which takes the per-step path) keep the buffers straight
    a, b = lpc.Lattice.from_inputs(lat, max_steps=31), lpc.Lattice.from_inputs(lat, max_steps=31)
    a.set_kernel(3)
    b.set_kernel(1)
    for n in (7, 1, 2, 21):
        a.step(n)
        b.step(n)
    assert a.steps_done == b.steps_done == 31 and a.launch_count < b.launch_count
    assert np.array_equal(a.field(lpc.LPC_FIELD_G), b.field(lpc.LPC_FIELD_G))
    assert np.max(np.abs(a.fid() - b.fid())) < 1e-14


# ---------------------------------------------------------------------------------------------
# the two-step sweep (temporal blocking, lpc_step2.cuh): same per-site arithmetic as the one-step sweeps, so the state
# agrees bit for bit; G[n] of every step is still recorded; against the oracle like everything else
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("shape,bc,alpha", [
    ((70, 19, 133), (1, 0, 0), 0.8),    # ragged in y and z, 3 z-tiles, 3 y-tiles, reflective x
    ((33, 40, 64), (0, 1, 1), 1.0),     # exact z tile, reflective y and z, periodic x with an odd length
    ((9, 8, 200), (0, 0, 0), 0.5),      # short x, 4 z-tiles, periodic everywhere
    ((20, 13, 37), (0, 0, 0), 0.9),     # odd ny and nz: the last group of a row is ragged
    ((4, 4, 4), (0, 0, 0), 1.0),        # every site lies within two of every periodic face
    ((6, 5, 7), (0, 0, 1), 0.7),
    ((130, 12, 70), (0, 0, 0), 1.0),    # several x chunks
])
def test_two_step_sweep_matches_one_step_sweep_and_oracle(lpc, oracle_mod, shape, bc, alpha, precision):
    lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.3, alpha=alpha, seed=61, n_moments=0)
    lat.dt = 2.0e-5
    n = 41                               # odd: twenty two-step sweeps and one one-step sweep
    rng = np.random.default_rng(12)
    g0 = (rng.standard_normal(shape) + 1j * rng.standard_normal(shape)) * (lat.blocked == 0)
    two, orc = _pair(lpc, oracle_mod, lat, n, 2, precision=precision, g0=g0)
    two.set_option(lpc.LPC_OPT_TIME_BLOCK, 2)
    one = lpc.Lattice.from_inputs(lat, precision=precision, max_steps=n, g0=g0)
    one.set_kernel(2)
    one.set_option(lpc.LPC_OPT_TIME_BLOCK, 1)
    l2, l1 = two.launch_count, one.launch_count
    for k in (6, 1, 3, 20, 11):          # even and odd calls in turn: the sweeps alternate, the ghost shell is refilled when needed
        two.step(k)
        one.step(k)
    assert one.launch_count - l1 == n
    assert two.launch_count - l2 < n     # two steps per launch wherever a call had two left
    assert two.steps_done == one.steps_done == n
    assert np.array_equal(two.field(lpc.LPC_FIELD_G), one.field(lpc.LPC_FIELD_G))
    scale = np.abs(g0).sum()
    assert np.max(np.abs(two.fid() - one.fid())) <= (1e-6 if precision else 1e-14) * scale
    orc.step(n)
    G_o, sabs = orc.fid(with_scale=True)
    tol_site, tol_sum = (1e-5, 1e-5) if precision else (1e-10, 1e-9)
    assert np.max(np.abs(two.fid() - G_o) / sabs) <= tol_sum
    pi, opn = orc.pi(), lat.blocked == 0
    hmax = np.max(np.abs(g0)[opn] / pi[opn])
    assert np.max(np.abs(two.field(lpc.LPC_FIELD_G) - orc.g())[opn] / pi[opn]) <= tol_site * hmax
    # x chunks of other lengths give the same state bits (the chunk seams carry no arithmetic)
    for xc in (5, 16):
        alt = lpc.Lattice.from_inputs(lat, precision=precision, max_steps=n, g0=g0)
        alt.set_option(lpc.LPC_OPT_X_CHUNK2, xc)
        alt.step(n - 1)
        alt.step(1)
        assert np.array_equal(alt.field(lpc.LPC_FIELD_G), one.field(lpc.LPC_FIELD_G)), xc


@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("shape,bc,alpha", [((70, 19, 133), (1, 0, 0), 0.8), ((33, 40, 64), (0, 1, 1), 1.0), ((20, 13, 37), (0, 0, 0), 0.9),
                                            ((6, 5, 7), (0, 0, 1), 0.7)])
def test_two_step_sweep_with_moment_fields(lpc, oracle_mod, shape, bc, alpha, precision):
    """The moment fields take two steps per sweep as well (a sweep of their own before the magnetisation's): Z_d[m] of every
    step, P^d bit for bit as from the one-step sweeps, everything against the oracle."""
    lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.3, alpha=alpha, seed=63, n_moments=3)
    lat.dt = 2.0e-5
    n = 31
    two, orc = _pair(lpc, oracle_mod, lat, n, 2, precision=precision)
    two.set_option(lpc.LPC_OPT_TIME_BLOCK, 2)
    one = lpc.Lattice.from_inputs(lat, precision=precision, max_steps=n)
    one.set_kernel(2)
    one.set_option(lpc.LPC_OPT_TIME_BLOCK, 1)
    l2 = two.launch_count
    for k in (4, 1, 7, 19):
        two.step(k)
        one.step(k)
    assert two.launch_count - l2 < 2 * n
    for w in (lpc.LPC_FIELD_G, lpc.LPC_FIELD_PX, lpc.LPC_FIELD_PY, lpc.LPC_FIELD_PZ):
        assert np.array_equal(two.field(w), one.field(w)), w
    Z2, D2 = two.moments()
    Z1, D1 = one.moments()
    z1 = np.abs(Z1[:, :1]).max()
    assert np.max(np.abs(Z2 - Z1)) <= (1e-6 if precision else 1e-14) * z1
    assert np.max(np.abs(two.fid() - one.fid())) <= (1e-6 if precision else 1e-14)
    orc.step(n)
    tol_site, tol_sum = (1e-5, 1e-5) if precision else (1e-10, 1e-9)
    _check(lpc, lat, two, orc, n, tol_site=tol_site, tol_sum=tol_sum, what=f"two-step moments {shape} p{precision}")


@pytest.mark.parametrize("precision", [0, 1])
def test_two_step_sweep_on_several_waves_of_ctas(lpc, precision):
    """The hand-over between the two groups of warps under load: a lattice of several waves of CTAs (one CTA per SM), 30 steps,
    bit for bit the one-step sweeps and bitwise reproducible."""
    n = 30
    lat = lpc_inputs.sweep(128, n_steps=n)
    shape = (130, 200, 384)                                   # 25 y-tiles x 6 (3 in fp32) z-tiles x 2 or 3 x chunks
    rng = np.random.default_rng(2)
    dF = -3.0 * rng.random(shape)
    blocked = (rng.random(shape) < 0.2).astype(np.uint8)
    omega = -12000.0 * rng.random(shape)
    outs = []
    for tb in (1, 2, 2):
        gpu = lpc.Lattice(shape, bc=(0, 0, 0), precision=precision, dt=lat.dt, max_steps=n)
        gpu.set_kernel(2)
        gpu.set_option(lpc.LPC_OPT_TIME_BLOCK, tb)
        gpu.set_site_params(dF, blocked, omega)
        gpu.step(n)
        outs.append((gpu.field(lpc.LPC_FIELD_G), gpu.fid()))
        gpu.close()
    assert np.array_equal(outs[0][0], outs[1][0])             # the state: same arithmetic per site
    assert np.array_equal(outs[1][0], outs[2][0]) and np.array_equal(outs[1][1], outs[2][1])
    scale = 1e-5 if precision else 1e-12                      # the series: another summation order
    assert np.max(np.abs(outs[0][1] - outs[1][1])) <= scale


def test_two_step_sweep_default_and_eligibility(lpc, oracle_mod):
    lat = lpc_inputs.random_small((24, 16, 70), bc=(0, 0, 0), p_block=0.2, seed=62, n_moments=0)
    n = 10
    # the default is one step per sweep; on request a lattice that carries the magnetisation alone takes two
    gpu, orc = _pair(lpc, oracle_mod, lat, n, 2)
    assert gpu.time_block_steps == 1
    gpu.set_option(lpc.LPC_OPT_TIME_BLOCK, 2)
    assert gpu.time_block_steps == 2
    l0 = gpu.launch_count
    gpu.step(n)
    assert gpu.launch_count - l0 == n // 2
    orc.step(n)
    _check(lpc, lat, gpu, orc, n, what="two-step default")
    # the series is bitwise reproducible
    again = lpc.Lattice.from_inputs(lat, max_steps=n)
    again.set_kernel(2)
    again.set_option(lpc.LPC_OPT_TIME_BLOCK, 2)
    again.step(n)
    assert np.array_equal(again.fid(), gpu.fid())
    # lattices that cannot: a density channel, a periodic axis shorter than four
    for kw, shape in ((dict(n_density=1), lat.shape), (dict(n_moments=3, n_density=1), lat.shape), (dict(), (24, 3, 70))):
        m = lpc.Lattice(shape, max_steps=4, **kw)
        with pytest.raises(lpc.LpcError) as e:
            m.set_option(lpc.LPC_OPT_TIME_BLOCK, 2)
        assert e.value.code == lpc.LPC_EINVAL
    with pytest.raises(lpc.LpcError) as e:
        gpu.set_option(99, 1)
    assert e.value.code == lpc.LPC_EINVAL


@pytest.mark.parametrize("bc,n_slabs,precision", [((0, 0, 0), 2, 0), ((1, 0, 0), 3, 0), ((0, 1, 0), 1, 0), ((0, 0, 1), 4, 1)])
def test_two_step_sweep_on_slabs(lpc, oracle_mod, bc, n_slabs, precision):
    """Slabs that carry the magnetisation alone take two steps per sweep and exchange two planes per face (include/lpc.h
    "Slabs"): against the oracle and, bit for bit, against the unsplit lattice."""
    from paper_2603_22553_b200 import slab

    n = 31
    lat = lpc_inputs.random_small((46, 18, 70), bc=bc, p_block=0.25, alpha=0.9, seed=83, n_steps=n, n_moments=0)
    rng = np.random.default_rng(5)
    g0 = (rng.random(lat.shape) + 1j * rng.random(lat.shape)) * (lat.blocked == 0)
    ss = slab.SlabSet(lat.shape, bc=lat.bc, slabs_per_rank=n_slabs, precision=precision, dt=lat.dt, a=lat.a, alpha=lat.alpha, max_steps=n, time_block=2)
    assert ss.two_step
    ss.set_site_params(lat.dF, lat.blocked, lat.omega, g0)
    l0 = sum(m.launch_count for m in ss.lat.values())
    ss.step(n)                  # fifteen two-step sweeps and one one-step sweep per slab (plus one ghost refill)
    assert sum(m.launch_count for m in ss.lat.values()) - l0 <= n_slabs * (n // 2 + 3)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=0, max_steps=n)
    orc.set_g(g0)
    orc.step(n)
    G_o, sabs = orc.fid(with_scale=True)
    tol_site, tol_sum = (1e-5, 1e-5) if precision else (1e-10, 1e-9)
    assert np.max(np.abs(ss.fid() - G_o) / sabs) <= tol_sum
    pi, opn = orc.pi(), lat.blocked == 0
    hmax = np.max(np.abs(g0)[opn] / pi[opn])
    g = ss.gather_field(lpc.LPC_FIELD_G, dtype=np.complex128)
    assert np.max(np.abs(g - orc.g())[opn] / pi[opn]) <= tol_site * hmax
    # more steps after an odd count: the one-step sweep left the shells to be refilled before the next exchange
    ss2 = slab.SlabSet(lat.shape, bc=lat.bc, slabs_per_rank=n_slabs, precision=precision, dt=lat.dt, a=lat.a, alpha=lat.alpha, max_steps=n, time_block=2)
    ss2.set_site_params(lat.dF, lat.blocked, lat.omega, g0)
    for k in (3, 1, 8, 19):
        ss2.step(k)
    assert np.array_equal(ss2.gather_field(lpc.LPC_FIELD_G, dtype=np.complex128), g)
    if precision == 0:
        whole = lpc.Lattice.from_inputs(lat, max_steps=n, g0=g0)
        whole.step(n)
        assert np.max(np.abs(g - whole.field(lpc.LPC_FIELD_G))[opn] / pi[opn]) <= 1e-12 * hmax


def test_two_step_slabs_agree_on_the_phase_factors(lpc, oracle_mod):
    """One wide phase angle on a boundary plane of one slab: the neighbour slab rotates that site in its first step too, so
    every slab has to read cos and sin (lpc_reads_sin_alone); against the oracle and against the unsplit lattice."""
    from paper_2603_22553_b200 import slab

    n = 20
    lat = lpc_inputs.random_small((40, 18, 70), bc=(0, 0, 0), p_block=0.2, alpha=0.9, seed=84, n_steps=n, n_moments=0)
    lat.blocked[19, 5, 7] = 0
    lat.omega[19, 5, 7] = 2.0 / lat.dt                        # cos = -0.42, on the last plane of slab 0 of 2
    ss = slab.SlabSet(lat.shape, bc=lat.bc, slabs_per_rank=2, dt=lat.dt, a=lat.a, alpha=lat.alpha, max_steps=n, time_block=2)
    assert ss.two_step
    ss.set_site_params(lat.dF, lat.blocked, lat.omega)
    assert not any(m.reads_sin_alone for m in ss.lat.values())
    ss.step(n)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=0, max_steps=n)
    orc.step(n)
    G_o, sabs = orc.fid(with_scale=True)
    assert np.max(np.abs(ss.fid() - G_o) / sabs) <= 1e-9
    pi, opn = orc.pi(), lat.blocked == 0
    g = ss.gather_field(lpc.LPC_FIELD_G, dtype=np.complex128)
    assert np.max(np.abs(g - orc.g())[opn] / pi[opn]) <= 1e-10
    whole = lpc.Lattice.from_inputs(lat, max_steps=n)
    whole.set_kernel(2)
    whole.step(n)
    # (the slabs add their partition sums in another order than the unsplit lattice: pi may differ in the last bit)
    assert np.max(np.abs(g - whole.field(lpc.LPC_FIELD_G))[opn] / pi[opn]) <= 1e-12


@pytest.mark.parametrize("precision", [0, 1])
def test_sweeps_that_read_sin_alone(lpc, oracle_mod, precision):
    """Lattices whose phase angles are all small (cos(omega dt) >= 1/2) store cos as sqrt(1 - sin^2) and the plain
    magnetisation sweeps read sin alone (48 instead of 56 bytes per site update in fp64): same state bit for
    bit as the sweeps that read both, parity with the oracle (which takes cos and sin from libm); a lattice with one wide
    angle reads cos and sin everywhere."""
    n = 60
    sT = 4 if precision else 8
    tol_site, tol_sum = (1e-5, 1e-5) if precision else (1e-10, 1e-9)
    lat = lpc_inputs.random_small((40, 19, 150), bc=(0, 1, 0), p_block=0.25, alpha=0.9, seed=71, n_steps=n, n_moments=0)
    lat.dt = 4.0e-5                                           # |omega dt| up to 1.0: cos >= 0.54
    assert np.cos(lat.omega * lat.dt).min() >= 0.5
    out = {}
    for full in (0, 1):
        for tb in (1, 2):
            gpu, orc = _pair(lpc, oracle_mod, lat, n, 2, precision=precision)
            gpu.set_option(lpc.LPC_OPT_FULL_PHASE, full)
            gpu.set_option(lpc.LPC_OPT_TIME_BLOCK, tb)
            assert gpu.bytes_per_site_step == sT * (7 if full else 6)
            gpu.step(n)
            orc.step(n)
            _check(lpc, lat, gpu, orc, n, tol_site=tol_site, tol_sum=tol_sum, what=f"sin alone full={full} tb={tb} p{precision}")
            out[full, tb] = (gpu.field(lpc.LPC_FIELD_G), gpu.fid())
    for tb in (1, 2):
        assert np.array_equal(out[0, tb][0], out[1, tb][0])
    assert np.array_equal(out[0, 1][1], out[1, 1][1])
    # one site beyond the limit: the whole lattice reads cos and sin, whatever the option says
    wide = lpc_inputs.random_small((40, 19, 150), bc=(0, 1, 0), p_block=0.25, alpha=0.9, seed=71, n_steps=n, n_moments=0)
    wide.dt = 4.0e-5
    i = tuple(np.argwhere(wide.blocked == 0)[5])
    wide.omega[i] = 2.0 / wide.dt                             # cos = -0.42
    for tb in (1, 2):
        gpu, orc = _pair(lpc, oracle_mod, wide, n, 2, precision=precision)
        gpu.set_option(lpc.LPC_OPT_TIME_BLOCK, tb)
        assert gpu.bytes_per_site_step == sT * 7
        gpu.step(n)
        orc.step(n)
        _check(lpc, wide, gpu, orc, n, tol_site=tol_site, tol_sum=tol_sum, what=f"wide angle tb={tb} p{precision}")


@pytest.mark.parametrize("kernel,nm,precision", [(2, 0, 0), (2, 3, 0), (1, 0, 0), (2, 0, 1)])
def test_step_n_under_cuda_graph_capture(lpc, oracle_mod, kernel, nm, precision):
    """lpc_step_n only enqueues launches: captured into a CUDA graph and replayed it appends to the series like direct calls
    (include/lpc.h "CUDA graphs"); lpc_sync_steps brings the host's count up to date.  Against the oracle and, bit for bit,
    against a lattice stepped without a graph."""
    import torch

    k, reps = 6, 4
    n = 3 + k * reps + 2
    lat = lpc_inputs.random_small((40, 24, 100), bc=(0, 1, 0), p_block=0.25, alpha=0.9, seed=88, n_steps=n, n_moments=nm)
    tol_site, tol_sum = (1e-5, 1e-5) if precision else (1e-10, 1e-9)
    st = torch.cuda.Stream()
    with torch.cuda.stream(st):
        gpu, orc = _pair(lpc, oracle_mod, lat, n, kernel, precision=precision)
        gpu.step(3)                                     # odd: the graph starts from buffer 1
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph, stream=st):
            gpu.step(k)
        assert gpu.steps_done == 3 + k                  # the host counted the capture, the device has not run it
        assert gpu.sync_steps() == 3
        for _ in range(reps):
            graph.replay()
        assert gpu.sync_steps() == 3 + k * reps
        gpu.step(2)                                     # and on without the graph
        assert gpu.steps_done == n
        plain = lpc.Lattice.from_inputs(lat, precision=precision, n_moments=nm, max_steps=n)
        plain.set_kernel(kernel)
        plain.step(n)
        orc.step(n)
        _check(lpc, lat, gpu, orc, n, tol_site=tol_site, tol_sum=tol_sum, what=f"graph k{kernel} m{nm} p{precision}")
        assert np.array_equal(gpu.fid(), plain.fid())
        assert np.array_equal(gpu.field(lpc.LPC_FIELD_G), plain.field(lpc.LPC_FIELD_G))
        if nm:
            assert np.array_equal(gpu.moments()[0], plain.moments()[0])
        # replays beyond the series' capacity are the caller's to avoid; what sync_steps can still tell is that it happened
        small = lpc.Lattice.from_inputs(lat, precision=precision, n_moments=0, max_steps=k + 1)
        small.set_kernel(kernel)
        g2 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g2, stream=st):
            small.step(k)
        small.sync_steps()
        g2.replay()
        assert small.sync_steps() == k
        small.close()
        plain.close()
        gpu.close()


# ---------------------------------------------------------------------------------------------
# states set from outside, device-resident inputs
# ---------------------------------------------------------------------------------------------
def test_arbitrary_initial_magnetisation_and_relaxation(lpc, oracle_mod):
    lat = lpc_inputs.random_small((16, 12, 34), bc=(0, 0, 0), p_block=0.2, alpha=0.7, seed=25)
    rng = np.random.default_rng(3)
    g0 = (rng.standard_normal(lat.shape) + 1j * rng.standard_normal(lat.shape))
    n = 50
    gpu, orc = _pair(lpc, oracle_mod, lat, n, 2, n_density=1, g0=g0)
    pi = orc.pi()
    G0 = gpu.fid()[0]
    assert abs(G0 - g0[lat.blocked == 0].sum()) < 1e-12 * np.abs(g0).sum()
    gpu.step(n)
    orc.step(n)
    G_o, G_g = orc.fid(), gpu.fid()
    scale = np.abs(g0[lat.blocked == 0]).sum()
    assert np.max(np.abs(G_g - G_o)) <= 1e-9 * scale
    g_o, g_g = orc.g(), gpu.field(lpc.LPC_FIELD_G)
    assert np.max(np.abs(g_g - g_o)) <= 1e-10 * np.abs(g0).max()
    # relaxation of an arbitrary density towards exp(-dF) through lpc_set_state
    rho0 = rng.random(lat.shape) * (lat.blocked == 0)
    gpu2 = lpc.Lattice.from_inputs(lat, n_density=1, max_steps=400)
    gpu2.set_state(lpc.LPC_FIELD_RHO, rho0)
    gpu2.step(400)
    want = orc.propagate_real(rho0, 400)
    got = gpu2.field(lpc.LPC_FIELD_RHO)
    assert np.max(np.abs(got - want)) <= 1e-10 * rho0.max()
    assert abs(got.sum() - rho0.sum()) <= 1e-12 * rho0.sum()   # conservation of total density
    assert np.abs(got / got.sum() - pi).max() < np.abs(rho0 / rho0.sum() - pi).max() * 0.5


# ---------------------------------------------------------------------------------------------
# equilibration loop against oracle O9
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("shape,bc,precision", [((24, 20, 70), (1, 0, 0), 0), ((17, 9, 33), (0, 0, 0), 0),
                                                ((24, 20, 70), (0, 1, 0), 1)])
def test_equilibration_loop_matches_oracle(lpc, oracle_mod, shape, bc, precision):
    lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.25, alpha=0.9, seed=31)
    tol = 1e-5 if precision else 1e-10
    rng = np.random.default_rng(4)
    opn = lat.blocked == 0
    rho0 = rng.random(lat.shape) * opn
    rho0 /= rho0.sum()
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=0, max_steps=8)
    pi = orc.pi()
    # a threshold the loop crosses after a few dozen sweeps, placed mid-way between two oracle deltas so
    # that rounding cannot move the stopping iteration (both sides decide in fp64 on an fp64 delta)
    _, _, dl = orc.equilibrate(rho0, 0.0, 60)
    k_stop = 41
    thr = float(np.sqrt(dl[k_stop - 1] * dl[k_stop - 2]))
    assert dl[k_stop - 1] < thr < dl[k_stop - 2] and np.all(dl[: k_stop - 1] > thr)
    rho_o, it_o, deltas = orc.equilibrate(rho0, thr, 5000)
    assert it_o == k_stop

    gpu = lpc.Lattice.from_inputs(lat, precision=precision, n_density=1, max_steps=8)
    gpu.set_state(lpc.LPC_FIELD_RHO, rho0)
    it_g, d_g = gpu.equilibrate(thr, 5000, 1)
    if precision == 0:
        assert it_g == it_o
        assert abs(d_g - deltas[-1]) <= tol * rho0.max()
        assert np.max(np.abs(gpu.field(lpc.LPC_FIELD_RHO) - rho_o)) <= tol * rho0.max()
    else:
        # fp32 storage: the per-sweep delta is resolved to about 1e-7 rho, compare the state at equal sweeps
        want = orc.propagate_real(rho0, it_g)
        assert np.max(np.abs(gpu.field(lpc.LPC_FIELD_RHO) - want)) <= tol * rho0.max()
    assert abs(gpu.field(lpc.LPC_FIELD_RHO).sum() - 1.0) <= (1e-5 if precision else 1e-12)
    # the magnetisation and its series are untouched
    assert gpu.steps_done == 0 and abs(gpu.fid()[0] - 1.0) < (1e-5 if precision else 1e-13)
    assert np.max(np.abs(gpu.field(lpc.LPC_FIELD_G) - pi)[opn] / pi[opn]) < (1e-5 if precision else 1e-13)

    # host checks every 7 sweeps: stops at the first multiple of 7 at or after the paper's stopping sweep
    gpu.set_state(lpc.LPC_FIELD_RHO, rho0)
    it7, d7 = gpu.equilibrate(thr, 5000, 7)
    if precision == 0:
        assert it7 == 7 * ((it_o + 6) // 7)
    want = orc.propagate_real(rho0, it7)
    assert np.max(np.abs(gpu.field(lpc.LPC_FIELD_RHO) - want)) <= tol * rho0.max()
    # iteration cap, even and odd (the density ends in either ping-pong buffer)
    for cap in (3, 4):
        gpu.set_state(lpc.LPC_FIELD_RHO, rho0)
        itc, dc = gpu.equilibrate(0.0, cap, 1)
        assert itc == cap
        assert abs(dc - dl[cap - 1]) <= tol * rho0.max()
        assert np.max(np.abs(gpu.field(lpc.LPC_FIELD_RHO) - orc.propagate_real(rho0, cap))) <= tol * rho0.max()
    assert gpu.equilibrate(1.0, 0, 1)[0] == 0

    # Fig. 3: the equilibrated density starts the propagation loop
    gpu.set_state(lpc.LPC_FIELD_RHO, rho0)
    it_g, _ = gpu.equilibrate(thr, 5000, 1)
    rho_g = gpu.field(lpc.LPC_FIELD_RHO)
    gpu.seed_from_density()
    assert abs(gpu.fid()[0] - rho_g.sum()) <= 1e-12
    gpu.step(8)
    orc.set_g(rho_g.astype(np.complex128))
    orc.step(8)
    G_o, sabs = orc.fid(with_scale=True)
    assert np.max(np.abs(gpu.fid() - G_o) / sabs) <= (1e-5 if precision else 1e-9)
    assert np.max(np.abs(gpu.field(lpc.LPC_FIELD_G) - orc.g())) <= tol * rho0.max()


def test_equilibration_errors(lpc):
    lat = lpc_inputs.random_small((8, 8, 8), seed=32)
    gpu = lpc.Lattice.from_inputs(lat, n_density=0, max_steps=2)
    with pytest.raises(lpc.LpcError) as e:
        gpu.equilibrate(1e-9, 10)
    assert e.value.code == lpc.LPC_ESTATE
    with pytest.raises(lpc.LpcError) as e:
        gpu.seed_from_density()
    assert e.value.code == lpc.LPC_ESTATE
    gpu = lpc.Lattice.from_inputs(lat, n_density=1, max_steps=2)
    for bad in ((1e-9, -1, 1), (1e-9, 10, 0), (float("nan"), 10, 1)):
        with pytest.raises(lpc.LpcError) as e:
            gpu.equilibrate(*bad)
        assert e.value.code == lpc.LPC_EINVAL


# ---------------------------------------------------------------------------------------------
# region-resolved FID and spectrum (Eq. 9 :115)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel,precision", [(1, 0), (2, 0), (2, 1)])
def test_regional_fid_and_spectrum_match_oracle(lpc, oracle_mod, kernel, precision):
    import torch

    lat = lpc_inputs.supercap(96, 24, 70, n_steps=120)        # electrodes | bulk | electrodes along x
    n, nreg = 120, 3
    tol = 1e-5 if precision else 1e-9
    x = np.arange(lat.nx)[:, None, None] * np.ones(lat.shape, dtype=int)
    region = np.where(x < lat.nx * 3 // 8, 0, np.where(x < lat.nx * 5 // 8, 1, 2)).astype(np.uint8)
    region[:, 0, 0] = 200                                     # a few sites in no region
    gpu = lpc.Lattice.from_inputs(lat, precision=precision, max_steps=n, n_regions=nreg)
    gpu.set_kernel(kernel)
    gpu.set_regions(region)
    # the TMA sweep reads the labels itself (+1 B); the direct kernel is followed by a pass over h, pi and the labels
    assert gpu.bytes_per_site_step == (4 if precision else 8) * (6 if kernel == 2 else 10) + 1
    gpu.step(n)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=0, max_steps=n)
    Gr_o = orc.step_with_regions(region, nreg, n)
    _, sabs = orc.fid(with_scale=True)
    for r in range(nreg):
        Gr_g = gpu.fid_region(r)
        assert Gr_g.shape == (n + 1,)
        assert np.max(np.abs(Gr_g - Gr_o[r]) / sabs) <= tol, f"region {r}"
    # the whole-lattice FID is what it is without regions, and the regions never exceed it
    assert np.max(np.abs(gpu.fid() - orc.fid()) / sabs) <= tol
    # spectra: whole lattice and one region, with and without line broadening, against Eq. 9 written out
    f0, df, nf = -4500.0, 37.5, 161
    freqs = f0 + df * np.arange(nf)
    for reg, series in ((-1, orc.fid()), (0, Gr_o[0]), (2, Gr_o[2])):
        for lb in (0.0, 200.0):
            want = oracle_mod.spectrum(series, lat.dt, freqs, lb)
            got = gpu.spectrum(f0, df, nf, lb, region=reg)
            scale = lat.dt * np.abs(series).sum()
            assert np.max(np.abs(got - want)) <= tol * scale, f"spectrum region {reg} lb {lb}"
    # a shorter record, device-resident labels, and a restart of both series from a new initial state
    want = oracle_mod.spectrum(orc.fid()[:50], lat.dt, freqs[:7], 0.0)
    assert np.max(np.abs(gpu.spectrum(f0, df, 7, 0.0, count=50) - want)) <= tol * lat.dt * 50
    gpu.set_regions(torch.from_numpy(region).cuda())
    assert np.max(np.abs(gpu.fid_region(1, first=n, count=1) - Gr_o[1][n:]) / sabs[n:]) <= tol
    with pytest.raises(lpc.LpcError) as e:
        gpu.fid_region(1, first=0, count=5)                   # recorded from step n only now
    assert e.value.code == lpc.LPC_EINVAL
    with pytest.raises(lpc.LpcError) as e:
        gpu.spectrum(f0, df, 3, region=1)
    assert e.value.code == lpc.LPC_ESTATE
    g0 = orc.g()
    gpu.set_state(lpc.LPC_FIELD_G, g0)
    assert gpu.steps_done == 0
    for r in range(nreg):
        assert abs(gpu.fid_region(r, 0, 1)[0] - Gr_o[r][n]) <= tol * sabs[n]


@pytest.mark.parametrize("kernel,precision", [(1, 0), (2, 0), (2, 1)])
def test_regional_vacf_and_diffusion_match_oracle(lpc, oracle_mod, kernel, precision):
    """Regional D (Table 1) on a small supercapacitor-shaped lattice."""
    n, nreg = 80, 3
    lat = lpc_inputs.supercap(64, 16, 70, n_steps=n, n_moments=3)
    tol = 1e-5 if precision else 1e-9
    x = np.arange(lat.nx)[:, None, None] * np.ones(lat.shape, dtype=int)
    region = np.where(x < lat.nx * 3 // 8, 0, np.where(x < lat.nx * 5 // 8, 1, 2)).astype(np.uint8)
    gpu = lpc.Lattice.from_inputs(lat, precision=precision, max_steps=n, n_regions=nreg)
    gpu.set_kernel(kernel)
    gpu.set_regions(region)
    gpu.step(n)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=3, max_steps=n)
    Zr_o, w = orc.step_with_regional_moments(region, nreg, n)
    Zall_g, D_all = gpu.moments()
    acc = np.zeros_like(Zall_g)
    for r in range(nreg):
        Z_g, D_g = gpu.moments_region(r)
        assert Z_g.shape == (3, n + 1)
        z1 = np.abs(Zr_o[r][:, :1])
        assert np.max(np.abs(Z_g - Zr_o[r]) / z1) <= tol, f"region {r}"
        D_o = Zr_o[r][:, 0] / (2 * lat.dt) + Zr_o[r][:, 1:].sum(axis=1) / lat.dt
        assert np.max(np.abs(D_g - D_o) / (z1[:, 0] / (2 * lat.dt))) <= tol
        acc += w[r] * Z_g
        # a shorter record
        Z_s, D_s = gpu.moments_region(r, count=10)
        assert np.array_equal(Z_s, Z_g[:, :10])
    # the regions tile the lattice: population-weighted, they add up to the whole-lattice VACF
    assert np.max(np.abs(acc - Zall_g) / np.abs(Zall_g[:, :1])) <= tol
    # the bulk region (dF = 0, no carbon) is faster than the electrodes in the transverse directions
    assert gpu.moments_region(1)[1][1] > gpu.moments_region(0)[1][1]
    # labels that arrive after the first step cannot give the series
    late = lpc.Lattice.from_inputs(lat, max_steps=4, n_regions=nreg)
    late.step(1)
    late.set_regions(region)
    late.step(2)
    with pytest.raises(lpc.LpcError) as e:
        late.moments_region(0)
    assert e.value.code == lpc.LPC_ESTATE
    assert late.fid_region(0, first=1).shape == (3,)


# ---------------------------------------------------------------------------------------------
# f3: per-link mobility factors alpha_ij (oracle O10)
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel,precision,bc", [(0, 0, (1, 0, 0)), (1, 0, (0, 0, 0)), (3, 0, (0, 1, 0)), (1, 1, (1, 0, 0)), (2, 0, (0, 0, 1)),
                                                 (2, 0, (0, 0, 0)), (2, 1, (0, 1, 0))])
def test_link_mobility_matches_oracle(lpc, oracle_mod, kernel, precision, bc):
    n = 80
    lat = lpc_inputs.random_small((22, 18, 70), bc=bc, p_block=0.25, alpha=0.9, seed=71, n_steps=n, n_moments=3)
    link = lpc_inputs.random_links(lat.shape, seed=3, lo=0.0)
    link[:, 5:9, 3:6, 10:20] = 0.0   # a pocket of dead links
    tol_site, tol_sum = (1e-5, 1e-5) if precision else (1e-10, 1e-9)
    gpu = lpc.Lattice.from_inputs(lat, precision=precision, n_moments=3, n_density=1, max_steps=n, link=link)
    gpu.set_kernel(kernel)
    # (the TMA path takes the moment channels in a sweep of their own, which stages pi a second time)
    assert gpu.bytes_per_site_step == (4 if precision else 8) * (2 * 6 + 3 + 3 + (1 if kernel == 2 else 0))
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=3, max_steps=n, link=link)
    # the precompute: Z_d[1] and P^d(1) of the scaled hop probabilities
    v_o, _ = orc.moments(1)
    v_g, _ = gpu.moments(1)
    assert np.max(np.abs(v_g - v_o) / v_o) < (1e-5 if precision else 1e-13)
    gpu.step(n)
    orc.step(n)
    print(_check(lpc, lat, gpu, orc, n, tol_site=tol_site, tol_sum=tol_sum, what="links"))
    # the density channel started at pi and stays there (the factors keep Eq. 2 stationary)
    pi = orc.pi()
    opn = lat.blocked == 0
    assert np.max(np.abs(gpu.field(lpc.LPC_FIELD_RHO) - pi)[opn] / pi[opn]) < (1e-4 if precision else 1e-12)
    # and the result differs from the run without factors by far more than the tolerance
    plain = lpc.Lattice.from_inputs(lat, precision=precision, n_moments=3, n_density=1, max_steps=n)
    plain.step(n)
    assert np.max(np.abs(plain.fid() - gpu.fid())) > 1e-3


def test_link_mobility_kernels_agree_bitwise(lpc):
    lat = lpc_inputs.random_small((40, 21, 131), bc=(0, 1, 0), p_block=0.25, seed=73, n_moments=3)
    link = lpc_inputs.random_links(lat.shape, seed=4, lo=0.0)
    res = []
    for kernel, prec in ((1, 0), (2, 0), (3, 0), (1, 1), (2, 1)):
        gpu = lpc.Lattice.from_inputs(lat, precision=prec, n_density=1, max_steps=25, link=link)
        gpu.set_kernel(kernel)
        gpu.step(25)
        res.append([gpu.field(w) for w in (lpc.LPC_FIELD_G, lpc.LPC_FIELD_PX, lpc.LPC_FIELD_PY, lpc.LPC_FIELD_PZ, lpc.LPC_FIELD_RHO)])
    for k in (1, 2):
        assert all(np.array_equal(x, y) for x, y in zip(res[0], res[k])), f"fp64 kernel {k}"
    assert all(np.array_equal(x, y) for x, y in zip(res[3], res[4])), "fp32"


def test_link_mobility_regions_equilibration_and_errors(lpc, oracle_mod):
    n, nreg = 40, 2
    lat = lpc_inputs.random_small((20, 16, 40), bc=(1, 0, 0), p_block=0.2, alpha=0.8, seed=72, n_steps=n, n_moments=3)
    confined = np.zeros(lat.shape, dtype=np.uint8)
    confined[:10] = 1
    link = lpc_inputs.confined_links(confined, 0.25)
    region = (1 - confined).astype(np.uint8)
    gpu = lpc.Lattice.from_inputs(lat, n_moments=3, n_density=1, max_steps=n, n_regions=nreg, link=link)
    gpu.set_regions(region)
    gpu.step(n)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=3, max_steps=n, link=link)
    Zr_o, w = orc.step_with_regional_moments(region, nreg, n)
    for r in range(nreg):
        Z_g, D_g = gpu.moments_region(r)
        assert np.max(np.abs(Z_g - Zr_o[r]) / np.abs(Zr_o[r][:, :1])) <= 1e-9
    # the confined half diffuses more slowly along y and z
    assert gpu.moments_region(0)[1][1] < 0.5 * gpu.moments_region(1)[1][1]
    # equilibration loop with the scaled hop probabilities
    rng = np.random.default_rng(8)
    rho0 = rng.random(lat.shape) * (lat.blocked == 0)
    rho0 /= rho0.sum()
    eq = lpc.Lattice.from_inputs(lat, n_moments=0, n_density=1, max_steps=4, link=link)
    eq.set_state(lpc.LPC_FIELD_RHO, rho0)
    it_g, d_g = eq.equilibrate(0.0, 25, 5)
    orc2 = oracle_mod.Oracle.from_lattice(lat, n_moments=0, max_steps=4, link=link)
    rho_o, it_o, dl = orc2.equilibrate(rho0, 0.0, 25)
    assert it_g == it_o == 25 and abs(d_g - dl[-1]) <= 1e-10 * rho0.max()
    assert np.max(np.abs(eq.field(lpc.LPC_FIELD_RHO) - rho_o)) <= 1e-10 * rho0.max()
    # NULL removes the factors: bit-identical to a lattice that never had them
    eq2 = lpc.Lattice.from_inputs(lat, n_moments=3, max_steps=6, link=link)
    eq2.set_link_mobility(None)
    assert eq2.bytes_per_site_step == 8 * (2 * 5 + 3)
    ref = lpc.Lattice.from_inputs(lat, n_moments=3, max_steps=6)
    eq2.set_kernel(1); ref.set_kernel(1)
    eq2.step(6); ref.step(6)
    assert np.array_equal(eq2.fid(), ref.fid()) and np.array_equal(eq2.field(lpc.LPC_FIELD_G), ref.field(lpc.LPC_FIELD_G))
    assert np.array_equal(eq2.moments()[0], ref.moments()[0])
    # errors: no room reserved, after the first step, factor out of range
    with pytest.raises(lpc.LpcError) as e:
        ref.set_link_mobility(link)
    assert e.value.code == lpc.LPC_ESTATE
    with pytest.raises(lpc.LpcError) as e:
        eq2.set_link_mobility(link)
    assert e.value.code == lpc.LPC_ESTATE
    bad = link.copy()
    bad[2, 3, 3, 3] = 1.0000001
    with pytest.raises(lpc.LpcError) as e:
        lpc.Lattice.from_inputs(lat, n_moments=0, max_steps=2, link=bad)
    assert e.value.code == lpc.LPC_EINVAL
    # device-resident factors
    import torch
    dev = lpc.Lattice.from_inputs(lat, n_moments=3, n_density=1, max_steps=n, n_regions=nreg, link=torch.from_numpy(link).cuda())
    dev.set_regions(region)   # same launch sequence as `gpu`, hence the same summation order
    dev.step(n)
    assert np.array_equal(dev.fid(), gpu.fid())


# ---------------------------------------------------------------------------------------------
# f4: the film-electrode cell of PAPER.md:236-248 (100 x 100 x 300, no periodic boundary in z)
# ---------------------------------------------------------------------------------------------
def test_film_electrode_cell(lpc, oracle_mod):
    n = 2000 if FULL else 150
    lat = lpc_inputs.film(n_steps=n, n_moments=3)
    assert lat.shape == (100, 100, 300) and lat.bc == (0, 0, 1) and abs(lat.notes["fraction"] - 0.38) < 0.01
    label = lat.notes["particle"]
    region = np.where(label > 0, 0, np.where((np.arange(300) >= 100) & (np.arange(300) < 200), 1, 2))[...].astype(np.uint8)
    gpu = lpc.Lattice.from_inputs(lat, n_moments=3, max_steps=n, n_regions=3)
    gpu.set_regions(region)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=3, max_steps=n)
    gpu.step(n)
    orc.step(n)
    print(_check(lpc, lat, gpu, orc, n, what="film"))
    # in-particle + bulk between the electrodes + bulk between the particles make up the whole signal
    G = gpu.fid()
    assert np.max(np.abs(sum(gpu.fid_region(r) for r in range(3)) - G)) < 1e-12
    # the bulk gap between the electrodes keeps its line at delta = 0: a real, slowly shrinking signal
    G1 = gpu.fid_region(1)
    assert np.all(np.abs(G1.imag) < 0.02 * np.abs(G1.real)) and G1.real[-1] > 0.8 * G1.real[0]


def test_regional_fid_large_spectrum_batches_and_errors(lpc):
    lat = lpc_inputs.random_small((12, 10, 20), seed=43, p_block=0.1)
    lat.omega[...] = -2 * np.pi * 2500.0
    n = 64
    gpu = lpc.Lattice.from_inputs(lat, max_steps=n, n_regions=0)
    with pytest.raises(lpc.LpcError) as e:
        gpu.set_regions(np.zeros(lat.shape, dtype=np.uint8))
    assert e.value.code == lpc.LPC_ESTATE
    gpu.step(n)
    # uniform shift: G[n] = exp(i w n dt) (Eq. 8), whose spectrum is the geometric sum in closed form;
    # 9000 frequencies span three launches of the spectrum kernel
    nf, f0, df = 9000, -5000.0, 1.0
    f = f0 + df * np.arange(nf)
    q = np.exp(1j * (-2 * np.pi * 2500.0 - 2 * np.pi * f) * lat.dt)
    with np.errstate(invalid="ignore", divide="ignore"):
        want = lat.dt * np.where(np.abs(1 - q) < 1e-14, n + 1, (1 - q ** (n + 1)) / (1 - q))
    got = gpu.spectrum(f0, df, nf)
    assert np.max(np.abs(got - want)) <= 1e-9 * lat.dt * (n + 1)
    assert abs(f[np.argmax(got.real)] + 2500.0) <= df
    for bad in (dict(n_freq=-1), dict(lb_hz=-1.0), dict(count=n + 2), dict(count=0), dict(region=0)):
        kw = dict(f0_hz=0.0, df_hz=1.0, n_freq=4)
        kw.update(bad)
        with pytest.raises(lpc.LpcError):
            gpu.spectrum(**kw)
    with pytest.raises(lpc.LpcError) as e:
        lpc.make_config(8, 8, 8, n_regions=9) and lpc.lpc_workspace_bytes(lpc.make_config(8, 8, 8, n_regions=9))
    assert e.value.code == lpc.LPC_EINVAL


def test_device_resident_inputs_give_the_same_result(lpc):
    import torch

    lat = lpc_inputs.random_small((24, 16, 70), p_block=0.3, seed=26)
    a = lpc.Lattice.from_inputs(lat, max_steps=10)
    b = lpc.Lattice(lat.shape, bc=lat.bc, dt=lat.dt, a=lat.a, alpha=lat.alpha, max_steps=10)
    dev = [torch.from_numpy(x).cuda() for x in (lat.dF, lat.blocked, lat.omega)]
    b.set_site_params(*dev)
    a.step(10)
    b.step(10)
    assert np.array_equal(a.fid(), b.fid())
    out = torch.empty(lat.shape, dtype=torch.complex128, device="cuda")
    lpc.lpc_read_field(b.handle, lpc.LPC_FIELD_G, out)
    assert np.array_equal(out.cpu().numpy(), a.field(lpc.LPC_FIELD_G))


# ---------------------------------------------------------------------------------------------
# fp32 mode
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kernel", KERNELS)
def test_fp32_mode(lpc, oracle_mod, kernel):
    lat = lpc_inputs.random_small((40, 24, 100), bc=(1, 0, 0), p_block=0.2, alpha=0.9, seed=27, n_moments=3)
    n = 200
    gpu, orc = _pair(lpc, oracle_mod, lat, n, kernel, precision=1)
    gpu.step(n)
    orc.step(n)
    _check(lpc, lat, gpu, orc, n, tol_site=1e-5, tol_sum=1e-5, what=f"fp32 kernel={kernel}")


# ---------------------------------------------------------------------------------------------
# BASELINE configs[1..3]: the stated lattices in the default run (config 1 for 2000 steps, config 2 at 256^3 with the
# moment fields for 200, config 3 at 2048 x 256 x 256 for 20), their full lengths (20000 / 20000 / 10000 steps) with
# LPC_FULL=1 (profiles/r2_full_parity.md), and small copies of configs 2 and 3 that run longer per site
# ---------------------------------------------------------------------------------------------
def _report(name, res):
    """One line per full-size case, also appended to gpurun_out/parity_full.log when that directory exists."""
    line = f"PARITY {name}: " + ", ".join(f"{k}={v:.2e}" for k, v in res.items())
    print(line)
    out = os.path.join(ROOT, "gpurun_out")
    if os.path.isdir(out):
        with open(os.path.join(out, "parity_full.log"), "a") as f:
            f.write(line + "\n")


def test_config1_particle(lpc, oracle_mod):
    n = 20000 if FULL else 2000
    lat = lpc_inputs.particle(n_steps=n)
    assert lat.shape == (128, 128, 128)
    gpu, orc = _pair(lpc, oracle_mod, lat, n, 0)
    gpu.step(n)
    orc.step(n)
    _report(f"config1 128^3 {n} steps", _check(lpc, lat, gpu, orc, n, what="config1"))


def test_config2_monolith_scaled(lpc, oracle_mod):
    L, n = 96, 200
    lat = lpc_inputs.monolith(L=L, n_steps=n)
    gpu, orc = _pair(lpc, oracle_mod, lat, n, 0)
    gpu.step(n)
    orc.step(n)
    print(_check(lpc, lat, gpu, orc, n, what="config2 scaled"))


def test_config2_monolith_full_size(lpc, oracle_mod):
    n = 20000 if FULL else 200
    lat = lpc_inputs.monolith(n_steps=n)
    assert lat.shape == (256, 256, 256) and lat.n_moments == 3
    gpu, orc = _pair(lpc, oracle_mod, lat, n, 0)
    gpu.step(n)
    orc.step(n)
    _report(f"config2 256^3 + 3 moment fields {n} steps", _check(lpc, lat, gpu, orc, n, what="config2"))


def test_config3_supercap_scaled(lpc, oracle_mod):
    shape, n = (256, 32, 64), 200
    lat = lpc_inputs.supercap(*shape, n_steps=n)
    gpu, orc = _pair(lpc, oracle_mod, lat, n, 0)
    gpu.step(n)
    orc.step(n)
    print(_check(lpc, lat, gpu, orc, n, what="config3 scaled"))
    # reflective x: nothing leaks through the walls -- total magnetisation magnitude is bounded by 1
    assert np.abs(gpu.fid()).max() <= 1 + 1e-12


def test_config3_supercap_full_size(lpc, oracle_mod):
    import torch

    # (the full length is 10000 steps; LPC_FULL_C3_STEPS shortens it where the oracle's 55 minutes do not fit one GPU lease)
    n = int(os.environ.get("LPC_FULL_C3_STEPS", "10000")) if FULL else 20
    lat = lpc_inputs.supercap(n_steps=n)
    assert lat.shape == (2048, 256, 256) and lat.bc == (1, 0, 0)
    gpu, orc = _pair(lpc, oracle_mod, lat, n, 0)
    gpu.step(n)
    orc.step(n)
    _report(f"config3 2048x256x256 {n} steps", _check(lpc, lat, gpu, orc, n, what="config3"))
    assert np.abs(gpu.fid()).max() <= 1 + 1e-12
    del gpu, orc
    torch.cuda.empty_cache()


# ---------------------------------------------------------------------------------------------
# BASELINE configs[4]: every sweep size, both precisions, 50 steps against the oracle (SURVEY 8(d) "Parity runs"), in the
# launch configuration bench.py times (kernel AUTO).  64^3 .. 256^3 element by element; 512^3 on sampled sites below.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("precision", [0, 1])
@pytest.mark.parametrize("L,nm", [(64, 0), (128, 0), (128, 3), (256, 0)])
def test_sweep_sizes_50_steps(lpc, oracle_mod, L, nm, precision):
    n = 50
    lat = lpc_inputs.sweep(L, n_moments=nm, n_steps=n)
    gpu, orc = _pair(lpc, oracle_mod, lat, n, 0, precision=precision)
    gpu.step(n)
    orc.step(n)
    tol_site, tol_sum = (1e-5, 1e-5) if precision else (1e-10, 1e-9)
    _report(f"sweep {L}^3 m{nm} {'fp32' if precision else 'fp64'} {n} steps",
            _check(lpc, lat, gpu, orc, n, tol_site=tol_site, tol_sum=tol_sum, what=f"sweep {L} p{precision}"))


# ---------------------------------------------------------------------------------------------
# properties that hold at any size, on the bench configuration (512^3 NMR kernel)
# ---------------------------------------------------------------------------------------------
def test_bench_size_properties(lpc):
    import torch

    L = 512
    n_sites = L ** 3
    # uniform shift on a heterogeneous lattice: G[n] = exp(i omega n dt) exactly (Eq. 8)
    rng = np.random.default_rng(5)
    dF = -3.0 * rng.random((L, L, L))
    blocked = (rng.random((L, L, L)) < 0.2).astype(np.uint8)
    omega = np.full((L, L, L), -12000.0)
    gpu = lpc.Lattice((L, L, L), dt=5e-6, max_steps=20)
    gpu.set_site_params(dF, blocked, omega)
    gpu.step(20)
    G = gpu.fid()
    k = np.arange(21)
    assert np.max(np.abs(G - np.exp(1j * -12000.0 * 5e-6 * k))) < 1e-12
    # the reduction agrees with an independent fp64 sum of the field read back
    g = gpu.field(lpc.LPC_FIELD_G)
    assert abs(g.sum() - G[-1]) < 1e-12
    del gpu, g
    torch.cuda.empty_cache()


_SWEEP512 = {}


def _sweep512():
    """The bench lattice, generated once per test session (the 512^3 pore field takes a while)."""
    if "lat" not in _SWEEP512:
        _SWEEP512["lat"] = lpc_inputs.sweep(512)
    return _SWEEP512["lat"]


@pytest.mark.parametrize("precision", [0, 1])
def test_bench_workload_sampled_sites_against_oracle(lpc, oracle_mod, precision):
    """The bench workload itself (512^3 sweep lattice, launch configuration of bench.py, fp64 and fp32), sampled outputs
    after 50 steps.

    g_i(n) depends only on the sites within n hops of i (Eq. 13, is a nearest-neighbour
    recurrence) and on dF one site further (Eq. 1).  The oracle therefore reproduces g_i(n) exactly on a
    (2n+5)^3 box cut around i (walls n+2 sites away cannot reach the centre in n steps); only the
    normalisation of Eq. 2 differs, by the known factor Z_box / Z_lattice.
    """
    import torch

    L, n = 512, 50
    tol = 1e-5 if precision else 1e-10
    lat = _sweep512()
    gpu = lpc.Lattice.from_inputs(lat, precision=precision, max_steps=n)
    gpu.step(n)
    g_gpu = gpu.field(lpc.LPC_FIELD_G)
    G_gpu = gpu.fid()
    del gpu
    torch.cuda.empty_cache()
    # the reduction agrees with an independent fp64 sum of the field read back
    assert abs(g_gpu.sum() - G_gpu[-1]) < (1e-6 if precision else 1e-12)
    opn = lat.blocked == 0
    z_full = np.exp(-lat.dF[opn]).sum()
    r = n + 2
    rng = np.random.default_rng(77)
    sites = [(0, 0, 0), (L - 1, L - 1, L - 1), (0, 255, L - 1), (L - 1, 0, 256), (63, 64, 65), (7, 8, 63), (300, 7, 64), (31, 15, 127), (32, 16, 128)]
    sites += [tuple(int(v) for v in rng.integers(0, L, 3)) for _ in range(7)]
    worst = 0.0
    for c in sites:
        # nearest open site along z so that the sample carries a value
        while lat.blocked[c]:
            c = (c[0], c[1], (c[2] + 1) % L)
        ix = [(c[d] + np.arange(-r, r + 1)) % L for d in range(3)]
        sub = np.ix_(*ix)
        dF, blk, om = (np.ascontiguousarray(a[sub]) for a in (lat.dF, lat.blocked, lat.omega))
        orc = oracle_mod.Oracle(dF.shape, (1, 1, 1), lat.dt, lat.a, lat.alpha, dF, blk, om, n_moments=0, max_steps=n)
        orc.step(n)
        z_box = np.exp(-dF[blk == 0]).sum()
        want = orc.g()[r, r, r] * (z_box / z_full)
        pi_c = np.exp(-lat.dF[c]) / z_full
        err = abs(g_gpu[c] - want) / pi_c
        assert err <= tol, f"site {c}: scaled error {err:.3e}"
        assert abs(want) > 0
        worst = max(worst, err)
    _report(f"sweep 512^3 {'fp32' if precision else 'fp64'} {n} steps, {len(sites)} sampled sites", {"err_g": worst})


# ---------------------------------------------------------------------------------------------
# the features next to the step (regional FID inside the sweep, equilibration sweep, x-slabs) on a lattice of several
# waves of CTAs (192 x 256 x 512: 1536 tiles-by-chunks on 296 resident CTAs), against the oracle
# ---------------------------------------------------------------------------------------------
def test_features_at_several_waves_against_oracle(lpc, oracle_mod):
    from paper_2603_22553_b200 import slab

    n, nreg = 12, 3
    shape = (192, 256, 512)
    lat = lpc_inputs.supercap(*shape, n_steps=n)          # reflective x, electrodes | bulk | electrodes
    x = np.arange(lat.nx)[:, None, None] * np.ones(lat.shape, dtype=np.int64)
    region = np.where(x < lat.nx * 3 // 8, 0, np.where(x < lat.nx * 5 // 8, 1, 2)).astype(np.uint8)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=0, max_steps=n)
    Gr_o = orc.step_with_regions(region, nreg, n)
    G_o, sabs = orc.fid(with_scale=True)
    g_o, pi = orc.g(), orc.pi()
    opn = lat.blocked == 0
    for precision, tol_sum, tol_site in ((0, 1e-9, 1e-10), (1, 1e-5, 1e-5)):
        gpu = lpc.Lattice.from_inputs(lat, precision=precision, max_steps=n, n_regions=nreg)
        gpu.set_regions(region)
        assert gpu.bytes_per_site_step == (4 if precision else 8) * 6 + 1      # the labels ride on the sweep (which reads sin alone)
        gpu.step(n)
        for r in range(nreg):
            assert np.max(np.abs(gpu.fid_region(r) - Gr_o[r]) / sabs) <= tol_sum, f"region {r} p{precision}"
        assert np.max(np.abs(gpu.fid() - G_o) / sabs) <= tol_sum
        assert np.max(np.abs(gpu.field(lpc.LPC_FIELD_G) - g_o)[opn] / pi[opn]) <= tol_site
        gpu.close()
    # the same lattice as three x-slabs (plane exchange after every step), sums of the slabs' series
    ss = slab.SlabSet(lat.shape, bc=lat.bc, slabs_per_rank=3, dt=lat.dt, a=lat.a, alpha=lat.alpha, max_steps=n)
    ss.set_site_params(lat.dF, lat.blocked, lat.omega)
    ss.step(n)
    assert np.max(np.abs(ss.fid() - G_o) / sabs) <= 1e-9
    assert np.max(np.abs(ss.gather_field(lpc.LPC_FIELD_G, dtype=np.complex128) - g_o)[opn] / pi[opn]) <= 1e-10
    del ss
    # five sweeps of the equilibration loop from a random density, delta of every sweep
    rng = np.random.default_rng(6)
    rho0 = rng.random(lat.shape) * opn
    rho0 /= rho0.sum()
    rho_o, it_o, deltas = orc.equilibrate(rho0, 0.0, 5)
    eq = lpc.Lattice.from_inputs(lat, n_density=1, max_steps=2)
    eq.set_state(lpc.LPC_FIELD_RHO, rho0)
    for k in range(5):
        it, d = eq.equilibrate(0.0, 1, 1)
        assert it == 1 and abs(d - deltas[k]) <= 1e-10 * rho0.max(), k
    assert np.max(np.abs(eq.field(lpc.LPC_FIELD_RHO) - rho_o)) <= 1e-10 * rho0.max()


# ---------------------------------------------------------------------------------------------
# error behaviour through the ABI
# ---------------------------------------------------------------------------------------------
def test_error_codes(lpc):
    import torch

    lat = lpc_inputs.random_small((8, 8, 8), seed=28)
    cfg = lpc.make_config(8, 8, 8, max_steps=3)
    ws = torch.empty(lpc.lpc_workspace_bytes(cfg), dtype=torch.uint8, device="cuda")
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_create_lattice(cfg, ws[: ws.numel() // 2])
    assert e.value.code == lpc.LPC_ENOMEM
    h = lpc.lpc_create_lattice(cfg, ws)
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_step_n(h, 1)
    assert e.value.code == lpc.LPC_ESTATE
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_set_site_params(h, lat.dF, np.ones_like(lat.blocked), lat.omega)
    assert e.value.code == lpc.LPC_EINVAL and "blocked" in str(e.value)
    wide = lat.dF.copy()
    wide[0, 0, 0] = 2000.0
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_set_site_params(h, wide, np.zeros_like(lat.blocked), lat.omega)
    assert e.value.code == lpc.LPC_EINVAL
    lpc.lpc_set_site_params(h, lat.dF, lat.blocked, lat.omega)
    lpc.lpc_step_n(h, 3)
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_step_n(h, 1)
    assert e.value.code == lpc.LPC_EINVAL
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_read_fid(h, 2, 5)
    assert e.value.code == lpc.LPC_EINVAL
    with pytest.raises(lpc.LpcError) as e:
        lpc.lpc_moments(h, 1)
    assert e.value.code == lpc.LPC_ESTATE
    assert lpc.lpc_read_fid(h).shape == (4,)
    assert lpc.lpc_steps_done(h) == 3 and lpc.lpc_launch_count(h) > 3
    lpc.lpc_destroy(h)


# ---------------------------------------------------------------------------------------------
# x-slab decomposition.  All slabs live on the one GPU here; the plane exchange is a device copy,
# the driver code (paper_2603_22553_b200/slab.py) is the one a multi-GPU run executes.
# ---------------------------------------------------------------------------------------------
@pytest.mark.parametrize("bc,n_slabs,kernel,precision,direct", [
    ((0, 0, 0), 2, 2, 0, False), ((1, 0, 0), 3, 2, 0, False), ((0, 1, 0), 1, 1, 0, False), ((1, 0, 1), 4, 0, 0, False),
    ((0, 0, 0), 3, 2, 1, False), ((0, 0, 0), 2, 2, 0, True), ((1, 0, 0), 3, 0, 0, True), ((0, 1, 0), 1, 2, 0, True), ((0, 0, 1), 4, 2, 1, True)])
def test_slabs_match_unsplit_lattice_and_oracle(lpc, oracle_mod, bc, n_slabs, kernel, precision, direct):
    from paper_2603_22553_b200 import slab

    n = 40
    lat = lpc_inputs.random_small((50, 18, 70), bc=bc, p_block=0.25, alpha=0.9, seed=81, n_steps=n, n_moments=3)
    rng = np.random.default_rng(3)
    g0 = (rng.random(lat.shape) + 1j * rng.random(lat.shape)) * (lat.blocked == 0)
    tol_site, tol_sum = (1e-5, 1e-5) if precision else (1e-10, 1e-9)

    def factory(shape, bc, **cfg):
        m = lpc.Lattice(shape, bc=bc, **cfg)
        m.set_kernel(kernel)
        return m

    ss = slab.SlabSet(lat.shape, bc=lat.bc, slabs_per_rank=n_slabs, lattice_factory=factory, precision=precision, n_moments=3,
                      n_density=1, dt=lat.dt, a=lat.a, alpha=lat.alpha, max_steps=n)
    assert sorted(ss.lat) == list(range(n_slabs)) and sum(hi - lo for lo, hi in ss.ranges.values()) == lat.nx
    ss.set_site_params(lat.dF, lat.blocked, lat.omega, g0)
    if direct:
        # the sweeps store their outermost planes into the neighbours' ghost planes themselves: nothing is copied
        assert ss.enable_direct_stores() == len(slab.messages(n_slabs, lat.bc[0] == 0))
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=3, max_steps=n)
    orc.set_g(g0)
    assert abs(ss.fid()[0] - orc.fid()[0]) <= tol_sum * np.abs(g0).sum()
    before = dict(ss.stats)
    ss.step(n)
    if direct:
        assert ss.stats == before      # the unpatched driver found nothing left to copy after any step
    else:
        assert ss.stats["copies"] - before["copies"] == n * len(slab.messages(n_slabs, lat.bc[0] == 0))
    orc.step(n)
    pi = orc.pi()
    opn = lat.blocked == 0
    G_o, sabs = orc.fid(with_scale=True)
    assert np.max(np.abs(ss.fid() - G_o) / sabs) <= tol_sum
    g = ss.gather_field(lpc.LPC_FIELD_G, dtype=np.complex128)
    hmax = np.max(np.abs(g0)[opn] / pi[opn])   # |g_i(n)| <= max_j |g_j(0)| / pi_j * pi_i (detailed balance), the scale of Q13
    assert np.max(np.abs(g - orc.g())[opn] / pi[opn]) <= tol_site * hmax
    Z_o, D_o = orc.moments()
    Z_g, D_g = ss.moments()
    assert np.max(np.abs(Z_g - Z_o) / np.abs(Z_o[:, :1])) <= tol_sum
    assert np.max(np.abs(D_g - D_o) / (np.abs(Z_o[:, 0]) / (2 * lat.dt))) <= tol_sum
    for d in range(3):
        P = ss.gather_field(lpc.LPC_FIELD_PX + d)
        assert np.max(np.abs(P - orc.P(d))[opn] / (lat.a * pi[opn])) <= tol_site
    # the density channel started at pi and stays there across the slab faces
    rho = ss.gather_field(lpc.LPC_FIELD_RHO)
    assert np.max(np.abs(rho - pi)[opn] / pi[opn]) <= (1e-4 if precision else 1e-12)
    if precision == 0:
        # against the unsplit lattice on the same kernel: same arithmetic per site, pi differs only through the
        # order in which the partition sum was added up
        whole = lpc.Lattice.from_inputs(lat, n_moments=3, n_density=1, max_steps=n, g0=g0)
        whole.set_kernel(kernel)
        whole.step(n)
        assert np.max(np.abs(g - whole.field(lpc.LPC_FIELD_G))[opn] / pi[opn]) <= 1e-12 * hmax
        assert np.max(np.abs(ss.fid() - whole.fid())) <= 1e-12 * np.abs(g0).sum()


def test_slab_mode_errors(lpc):
    lat = lpc_inputs.random_small((12, 10, 20), seed=82)
    m = lpc.Lattice((12, 10, 20), bc=(lpc.LPC_BC_HALO, 0, 0), n_density=1, max_steps=5)
    assert m.partition_sum(lat.dF, lat.blocked) == pytest.approx(np.exp(-lat.dF)[lat.blocked == 0].sum(), rel=1e-13)
    m.set_site_params(lat.dF, lat.blocked, lat.omega)
    with pytest.raises(lpc.LpcError) as e:
        m.step(1)                      # lpc_slab_finish first
    assert e.value.code == lpc.LPC_ESTATE
    m.slab_finish()
    m.step(1)
    assert m.equilibrate(0.0, 1, 1)[0] == 1          # one sweep at a time is what the slab driver runs
    for bad in (lambda: m.step(2), lambda: m.equilibrate(1e-3, 5)):
        with pytest.raises(lpc.LpcError) as e:
            bad()
        assert e.value.code == lpc.LPC_ESTATE
    with pytest.raises(lpc.LpcError) as e:
        lpc.Lattice((12, 10, 20), bc=(0, lpc.LPC_BC_HALO, 0))
    assert e.value.code == lpc.LPC_EINVAL
    plain = lpc.Lattice.from_inputs(lat, max_steps=2)
    with pytest.raises(lpc.LpcError) as e:
        plain.slab_finish()
    assert e.value.code == lpc.LPC_ESTATE
    # the plane views address the workspace: shape [channels, (ny+2) * padded nz]
    v = plain.halo_planes(lpc.LPC_HALO_STATE, 0, lpc.LPC_HALO_SEND)
    assert v.shape[0] == 2 + lat.n_moments and v.shape[1] % 14 == 0 and float(v[0].max()) == 1.0   # ny + 4 padded rows


def test_regional_fid_fused_sweep_matches_separate_pass(lpc, oracle_mod):
    """The TMA sweep accumulates G_r itself (per-thread slots, label changes inside a thread's column, ragged tiles,
    labels outside 0..n_regions-1); the separate reduction pass gives the same series up to summation order."""
    n, nreg = 30, 5
    lat = lpc_inputs.random_small((37, 21, 131), bc=(0, 1, 0), p_block=0.2, alpha=0.9, seed=91, n_steps=n, n_moments=0)
    rng = np.random.default_rng(9)
    region = rng.integers(0, 7, size=lat.shape).astype(np.uint8)          # iid labels 0..6: 5 and 6 are in no region
    region[:, :, 40:90] = 2                                                # and a blob
    link = lpc_inputs.random_links(lat.shape, seed=5)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=0, max_steps=n)
    Gr_o = orc.step_with_regions(region, nreg, n)
    _, sabs = orc.fid(with_scale=True)
    for precision, tol in ((0, 1e-9), (1, 1e-5)):
        out = {}
        for fused in (True, False):
            gpu = lpc.Lattice.from_inputs(lat, precision=precision, max_steps=n, n_regions=nreg)
            gpu.set_kernel(2)
            if not fused:
                gpu.set_option(lpc.LPC_OPT_REGION_FUSION, 1)      # the separate reduction pass after every sweep
            gpu.set_regions(region)
            # (the sweep next to a separate pass reads sin alone: this lattice's phase angles are all small)
            assert gpu.bytes_per_site_step == (4 if precision else 8) * 6 + (1 if fused else (4 if precision else 8) * 3 + 1)
            l0 = gpu.launch_count
            gpu.step(n)
            assert gpu.launch_count - l0 == (n if fused else 2 * n)
            out[fused] = np.array([gpu.fid_region(r) for r in range(nreg)])
        assert np.max(np.abs(out[True] - Gr_o) / sabs) <= tol
        assert np.max(np.abs(out[True] - out[False]) / sabs) <= (1e-5 if precision else 1e-13)
    # with stored link weights the fused sweep is the links kernel
    gpu = lpc.Lattice.from_inputs(lat, max_steps=n, n_regions=nreg, link=link)
    gpu.set_regions(region)
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=0, max_steps=n, link=link)
    Gr_o = orc.step_with_regions(region, nreg, n)
    _, sabs = orc.fid(with_scale=True)
    gpu.step(n)
    assert np.max(np.abs(np.array([gpu.fid_region(r) for r in range(nreg)]) - Gr_o) / sabs) <= 1e-9


@pytest.mark.parametrize("precision", [0, 1])
def test_equilibration_tma_sweep_agrees_bitwise_with_direct_sweep(lpc, precision):
    """The equilibration sweep runs on the TMA march (density channel alone) or, with LPC_KERNEL_DIRECT, on the
    per-pair kernel: same per-site arithmetic, and a maximum does not depend on the order it is taken in."""
    lat = lpc_inputs.random_small((37, 21, 131), bc=(0, 1, 0), p_block=0.2, alpha=0.9, seed=92, n_moments=3)
    rng = np.random.default_rng(10)
    rho0 = rng.random(lat.shape) * (lat.blocked == 0)
    rho0 /= rho0.sum()
    link = lpc_inputs.random_links(lat.shape, seed=6)
    for lk in (None, link):
        res = []
        for kernel in (0, 1):
            gpu = lpc.Lattice.from_inputs(lat, precision=precision, n_moments=3, n_density=1, max_steps=4, link=lk)
            gpu.set_kernel(kernel)
            gpu.set_state(lpc.LPC_FIELD_RHO, rho0)
            its, delta = gpu.equilibrate(0.0, 17, 17)
            res.append((its, delta, gpu.field(lpc.LPC_FIELD_RHO), gpu.field(lpc.LPC_FIELD_G), gpu.field(lpc.LPC_FIELD_PX)))
        assert res[0][0] == res[1][0] == 17 and res[0][1] == res[1][1] > 0
        assert all(np.array_equal(x, y) for x, y in zip(res[0][2:], res[1][2:]))


@pytest.mark.parametrize("bc,n_slabs", [((0, 0, 0), 2), ((1, 0, 0), 3)])
def test_slab_equilibration_loop_matches_oracle(lpc, oracle_mod, bc, n_slabs):
    from paper_2603_22553_b200 import slab

    lat = lpc_inputs.random_small((30, 12, 40), bc=bc, p_block=0.25, alpha=0.9, seed=83)
    rng = np.random.default_rng(12)
    rho0 = rng.random(lat.shape) * (lat.blocked == 0)
    rho0 /= rho0.sum()
    orc = oracle_mod.Oracle.from_lattice(lat, n_moments=0, max_steps=4)
    _, _, dl = orc.equilibrate(rho0, 0.0, 40)
    k_stop = 27
    thr = float(np.sqrt(dl[k_stop - 1] * dl[k_stop - 2]))
    rho_o, it_o, deltas = orc.equilibrate(rho0, thr, 500)
    assert it_o == k_stop
    ss = slab.SlabSet(lat.shape, bc=lat.bc, slabs_per_rank=n_slabs, n_density=1, dt=lat.dt, a=lat.a, alpha=lat.alpha, max_steps=4)
    ss.set_site_params(lat.dF, lat.blocked, lat.omega)
    ss.set_state(lpc.LPC_FIELD_RHO, rho0)
    it_g, d_g = ss.equilibrate(thr, 500)
    assert it_g == it_o and abs(d_g - deltas[-1]) <= 1e-10 * rho0.max()
    assert np.max(np.abs(ss.gather_field(lpc.LPC_FIELD_RHO) - rho_o)) <= 1e-10 * rho0.max()


@pytest.mark.parametrize("seed", [7, 11])
def test_random_shapes_and_features_tma_against_direct(lpc, seed):
    """Seeded random lattices (1..120 x 1..70 x 1..300 and tiny ones), boundary conditions, precision, channels, link
    weights and region labels: the TMA march and the per-pair kernel must agree bit for bit on every field and to
    rounding on every series (the sums are taken in a different order)."""
    rng = np.random.default_rng(seed)
    for case in range(60):
        shape = tuple(int(rng.integers(1, hi)) for hi in ((120, 70, 300) if case % 2 else (12, 12, 20)))
        bc = tuple(int(v) for v in rng.integers(0, 2, size=3))
        prec, nm, nd = int(rng.integers(0, 2)), int(rng.choice([0, 3])), int(rng.integers(0, 2))
        use_link, nreg, n = bool(rng.integers(0, 2)), int(rng.choice([0, 3])), int(rng.integers(1, 12))
        lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.25 if np.prod(shape) > 8 else 0.0, alpha=0.9, seed=1000 + case, n_moments=nm)
        link = lpc_inputs.random_links(shape, seed=case, lo=0.0) if use_link else None
        region = rng.integers(0, 4, size=shape).astype(np.uint8)
        out = []
        for kernel in (1, 2):
            g = lpc.Lattice.from_inputs(lat, precision=prec, n_moments=nm, n_density=nd, max_steps=n + 1, n_regions=nreg, link=link)
            g.set_kernel(kernel)
            if nreg:
                g.set_regions(region)
            g.step(n)
            fields = [g.field(lpc.LPC_FIELD_G)] + ([g.field(lpc.LPC_FIELD_PX + d) for d in range(3)] if nm else [])
            fields += [g.field(lpc.LPC_FIELD_RHO)] if nd else []
            series = [g.fid()] + ([g.moments()[0]] if nm else [])
            series += [np.array([g.fid_region(r) for r in range(nreg)])] if nreg else []
            series += [np.array([g.moments_region(r)[0] for r in range(nreg)])] if nreg and nm else []
            out.append((fields, series))
            g.close()
        what = f"case {case}: {shape} bc={bc} prec={prec} nm={nm} nd={nd} link={use_link} nreg={nreg} n={n}"
        assert all(np.array_equal(a, b) for a, b in zip(out[0][0], out[1][0])), what
        tol = 2e-5 if prec else 1e-12
        for a, b in zip(out[0][1], out[1][1]):
            assert np.all(np.abs(a - b) <= tol * max(np.abs(a).max(), 1e-300)), what


def test_random_lattices_against_oracle(lpc, oracle_mod):
    """Seeded random lattices against the oracle at the stated tolerances: shapes, boundaries, alpha, precision, moment
    fields, link factors, kernel selector."""
    rng = np.random.default_rng(5)
    for case in range(40):
        shape = tuple(int(rng.integers(1, hi)) for hi in (50, 30, 140))
        bc = tuple(int(v) for v in rng.integers(0, 2, size=3))
        prec, nm, kernel = int(rng.integers(0, 2)), int(rng.choice([0, 3])), int(rng.choice([0, 1, 2, 3]))
        use_link, n = bool(rng.integers(0, 2)), int(rng.integers(2, 40))
        lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.25 if np.prod(shape) > 8 else 0.0, alpha=float(rng.uniform(0.3, 1.0)),
                                      seed=3000 + case, n_steps=n, n_moments=nm)
        lat.dt = 2.0e-5
        link = lpc_inputs.random_links(shape, seed=100 + case, lo=0.0) if use_link else None
        gpu = lpc.Lattice.from_inputs(lat, precision=prec, n_moments=nm, max_steps=n, link=link)
        gpu.set_kernel(kernel)
        orc = oracle_mod.Oracle.from_lattice(lat, n_moments=nm, max_steps=n, link=link)
        gpu.step(n)
        orc.step(n)
        tol_site, tol_sum = (1e-5, 1e-5) if prec else (1e-10, 1e-9)
        _check(lpc, lat, gpu, orc, n, tol_site=tol_site, tol_sum=tol_sum,
               what=f"case {case}: {shape} bc={bc} prec={prec} nm={nm} kernel={kernel} link={use_link} n={n}")
        gpu.close()


@pytest.mark.parametrize("precision,nm,nd,nreg,use_link,bc", [(0, 3, 1, 3, True, (0, 0, 0)), (1, 3, 1, 3, True, (1, 0, 1)), (0, 0, 0, 0, False, (0, 1, 0)),
                                                              (1, 0, 0, 2, False, (0, 0, 0)), (0, 3, 0, 0, False, (2, 0, 0)), (1, 3, 0, 0, False, (0, 0, 0))])
def test_nothing_is_written_outside_the_workspace(lpc, precision, nm, nd, nreg, use_link, bc):
    """Guard bytes before and after the workspace stay untouched through the precompute, every step kernel, the
    equilibration sweeps, the regional passes and the read-outs (a bounds check of our own: the sanitizer is not
    available on the GPU pool)."""
    import torch

    shape = (21, 19, 133)   # ragged against every tile shape
    lat = lpc_inputs.random_small(shape, bc=tuple(b if b != 2 else 1 for b in bc), p_block=0.25, alpha=0.9, seed=95, n_moments=nm)
    cfg = lpc.make_config(*shape, bc=bc, precision=precision, n_moments=nm, n_density=nd, dt=lat.dt, a=lat.a, alpha=lat.alpha,
                          max_steps=40, stream=torch.cuda.current_stream().cuda_stream, n_regions=nreg,
                          link_mobility=1 if use_link and bc[0] != 2 else 0)
    nbytes = lpc.lpc_workspace_bytes(cfg)
    guard = 1 << 20
    buf = torch.full((nbytes + 2 * guard,), 0xAB, dtype=torch.uint8, device="cuda:0")
    assert buf.data_ptr() % 256 == 0
    handle = lpc.lpc_create_lattice(cfg, buf.data_ptr() + guard, nbytes)
    try:
        rng = np.random.default_rng(1)
        for kernel in (1, 2, 3):
            lpc.lpc_set_kernel(handle, kernel)
            lpc.lpc_set_site_params(handle, lat.dF, lat.blocked, lat.omega)
            if use_link and bc[0] != 2:
                lpc.lpc_set_link_mobility(handle, lpc_inputs.random_links(shape, seed=9))
            if bc[0] == 2:
                lpc.lpc_slab_finish(handle)
            if nreg:
                lpc.lpc_set_regions(handle, rng.integers(0, 4, size=shape).astype(np.uint8))
            if bc[0] == 2:
                for _ in range(7):
                    lpc.lpc_step_n(handle, 1)
            else:
                lpc.lpc_step_n(handle, 7)
                lpc.lpc_step_n(handle, 1)
            if nd and bc[0] != 2:
                lpc.lpc_equilibrate(handle, 0.0, 5, 2)
            lpc.lpc_read_fid(handle)
            if nm:
                lpc.lpc_moments(handle)
            if nreg:
                lpc.lpc_read_fid_region(handle, 0)
        # the two-step sweep (own tiles, two ghost layers, ghost images of the face sites) where the lattice can run it, and the
        # sweeps that read cos and sin
        if nd == 0 and nreg == 0 and bc[0] != 2:
            lpc.lpc_set_kernel(handle, 2)
            lpc.lpc_set_site_params(handle, lat.dF, lat.blocked, lat.omega)
            lpc.lpc_set_option(handle, lpc.LPC_OPT_TIME_BLOCK, 2)
            assert lpc.lpc_time_block_steps(handle) == 2
            lpc.lpc_step_n(handle, 6)
            lpc.lpc_set_option(handle, lpc.LPC_OPT_FULL_PHASE, 1)
            lpc.lpc_step_n(handle, 5)
            lpc.lpc_read_fid(handle)
        torch.cuda.synchronize()
        assert bool((buf[:guard] == 0xAB).all()) and bool((buf[guard + nbytes:] == 0xAB).all())
    finally:
        lpc.lpc_destroy(handle)
