"""Pins of the CPU oracle against what the paper and the mathematics fix.

Nothing here touches the CUDA library.  Each test names the passage of
/root/reference/PAPER.md (or the SURVEY.md section 8(c) pin) it follows.  The
brute-force tests enumerate trajectories from the *definitions* (Eq. 8/11 for
G, <dx_1 dx_n> for the VACF) and never call the recursion they check.
"""
import itertools
import os
import subprocess
import sys

import numpy as np
import pytest

import lpc_inputs

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
GOLD = os.path.join(ROOT, "tests", "golden")


def _mk(oracle_mod, lat, **kw):
    return oracle_mod.Oracle.from_lattice(lat, **kw)


def _uniform(shape, bc=(0, 0, 0), alpha=1.0, dt=1.0, a=1.0, omega=0.0):
    lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.0, alpha=alpha, seed=0)
    lat.dF[...] = 0.0
    lat.omega[...] = omega
    lat.dt = dt
    lat.a = a
    return lat


# --------------------------------------------------------------------------
# helpers that restate the *model*, not the oracle's recursion
# --------------------------------------------------------------------------
def _metropolis(dFi, dFj):
    """Eq. 1."""
    return np.exp(-(dFj - dFi)) if dFj > dFi else 1.0


def _moves(lat, link=None):
    """For every site: list of (target, probability, displacement vector) incl. staying.

    link: optional [3, nx, ny, nz] factors alpha_ij of PAPER.md:105; link[d][i] belongs to the link between i and
    its +d neighbour and multiplies the hop probability in both directions.

    Lattice-gas rule of PAPER.md:51-55: one of z = 6 neighbours is tried with
    probability alpha/6 (alpha: :101); the hop is accepted with Eq. 1; a move
    into an obstacle or through a wall leaves the particle where it is.
    """
    shape = lat.shape
    moves = {}
    for idx in itertools.product(*[range(n) for n in shape]):
        if lat.blocked[idx]:
            continue
        lst, stay = [], 1.0
        for d in range(3):
            for s in (-1, 1):
                tgt = list(idx)
                tgt[d] += s
                if tgt[d] < 0 or tgt[d] >= shape[d]:
                    if lat.bc[d]:
                        continue
                    tgt[d] %= shape[d]
                tgt = tuple(tgt)
                if lat.blocked[tgt]:
                    continue
                p = lat.alpha / 6.0 * _metropolis(lat.dF[idx], lat.dF[tgt])
                if link is not None:
                    p *= link[d][idx] if s > 0 else link[d][tgt]
                disp = np.zeros(3)
                disp[d] = s * lat.a
                lst.append((tgt, p, disp))
                stay -= p
        lst.append((idx, stay, np.zeros(3)))
        moves[idx] = lst
    return moves


def _boltzmann(lat):
    """Eq. 2 with <rho> = 1/N so that the densities sum to one."""
    e = np.where(lat.blocked != 0, 0.0, np.exp(-lat.dF))
    return e / e.sum()


def _enumerate(lat, n, link=None):
    """All n-step trajectories: returns G[0..n] (Eq. 8/11) and C[d, m] = <dx_1 dx_m>, m = 1..n."""
    moves = _moves(lat, link)
    pi = _boltzmann(lat)
    G = np.zeros(n + 1, dtype=complex)
    Cm = np.zeros((3, n + 1))

    def walk(site, prob, phase, depth, dx1):
        # phase = dt * sum of omega over the sites visited at steps 1..depth (Eq. 11)
        G[depth] += prob * np.exp(1j * phase)
        if depth == n:
            return
        for tgt, p, disp in moves[site]:
            if p == 0.0:
                continue
            first = disp if depth == 0 else dx1
            Cm[:, depth + 1] += prob * p * first * disp
            walk(tgt, prob * p, phase + lat.dt * lat.omega[tgt], depth + 1, first)

    for site in moves:
        walk(site, pi[site], 0.0, 0, None)
    return G, Cm


# --------------------------------------------------------------------------
# P1 conservation / P2 detailed balance / P3 stationarity
# --------------------------------------------------------------------------
@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 0, 0), (1, 1, 1)])
def test_p1_total_density_is_conserved(oracle_mod, bc):
    lat = lpc_inputs.random_small((6, 5, 7), bc=bc, p_block=0.3, alpha=0.8, seed=1)
    o = _mk(oracle_mod, lat)
    rng = np.random.default_rng(5)
    rho = rng.random(lat.shape) * (lat.blocked == 0)
    out = o.propagate_real(rho, 50)
    assert abs(out.sum() - rho.sum()) <= 1e-13 * rho.sum()
    assert np.all(out[lat.blocked != 0] == 0.0)
    assert out.min() >= 0.0


def test_p1_delta_source_keeps_unit_mass(oracle_mod):
    lat = lpc_inputs.random_small((5, 5, 5), bc=(0, 1, 0), p_block=0.2, seed=2)
    o = _mk(oracle_mod, lat)
    open_sites = np.argwhere(lat.blocked == 0)
    for k in (0, len(open_sites) // 2, len(open_sites) - 1):
        rho = np.zeros(lat.shape)
        rho[tuple(open_sites[k])] = 1.0
        for n in (1, 2, 9):
            assert abs(o.propagate_real(rho, n).sum() - 1.0) < 1e-14


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 0, 1)])
def test_p2_detailed_balance(oracle_mod, bc):
    """pi_i p(i->j) = pi_j p(j->i) = (alpha/6) min(pi_i, pi_j)."""
    lat = lpc_inputs.random_small((4, 5, 3), bc=bc, p_block=0.25, alpha=0.7, seed=3)
    o = _mk(oracle_mod, lat)
    pi = o.pi().reshape(-1)
    blk = lat.blocked.reshape(-1)
    for i in range(lat.n_sites):
        for d in range(3):
            for s in (-1, 1):
                j = oracle_mod.neighbor(lat.shape, bc, i, d, s)
                if j < 0:
                    continue
                pij = oracle_mod.hop(lat.shape, bc, lat.alpha, lat.dF, lat.blocked, i, j)
                pji = oracle_mod.hop(lat.shape, bc, lat.alpha, lat.dF, lat.blocked, j, i)
                if blk[i] or blk[j]:
                    assert pij == 0.0 and pji == 0.0
                    continue
                want = lat.alpha / 6.0 * min(pi[i], pi[j])
                assert abs(pi[i] * pij - want) <= 2e-15 * want
                assert abs(pi[j] * pji - want) <= 2e-15 * want


def test_o1_boltzmann_density(oracle_mod):
    """Eq. 2: rho_i proportional to exp(-dF_i), zero on carbon, normalised."""
    lat = lpc_inputs.config0(L=8, n_steps=0)
    o = _mk(oracle_mod, lat)
    pi = o.pi()
    assert abs(pi.sum() - 1.0) < 1e-14
    assert np.all(pi[lat.blocked != 0] == 0.0)
    opn = np.argwhere(lat.blocked == 0)
    i, j = tuple(opn[0]), tuple(opn[-1])
    assert np.isclose(np.log(pi[i] / pi[j]), -(lat.dF[i] - lat.dF[j]), rtol=0, atol=1e-14)
    assert np.isclose(o.partition_sum, np.exp(-lat.dF[lat.blocked == 0]).sum(), rtol=1e-14)


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 0, 0)])
def test_p3_boltzmann_is_stationary(oracle_mod, bc):
    lat = lpc_inputs.random_small((6, 6, 6), bc=bc, p_block=0.3, seed=4)
    o = _mk(oracle_mod, lat)
    pi = o.pi()
    out = o.propagate_real(pi, 200)
    assert np.max(np.abs(out - pi)) <= 1e-13 * pi.max()


def test_p3_magnetisation_without_shift_stays_at_pi(oracle_mod):
    lat = lpc_inputs.random_small((5, 4, 6), p_block=0.3, seed=6)
    lat.omega[...] = 0.0
    o = _mk(oracle_mod, lat, max_steps=100)
    o.step(100)
    assert np.max(np.abs(o.g() - o.pi())) <= 1e-13 * o.pi().max()
    assert np.allclose(o.fid(), 1.0, rtol=0, atol=1e-13)


# --------------------------------------------------------------------------
# P4 relaxation to exp(-dF) within each connected cluster
# --------------------------------------------------------------------------
def _clusters(lat):
    shape = lat.shape
    label = -np.ones(shape, dtype=int)
    nlab = 0
    for start in itertools.product(*[range(n) for n in shape]):
        if lat.blocked[start] or label[start] >= 0:
            continue
        stack = [start]
        label[start] = nlab
        while stack:
            cur = stack.pop()
            for d in range(3):
                for s in (-1, 1):
                    t = list(cur)
                    t[d] += s
                    if t[d] < 0 or t[d] >= shape[d]:
                        if lat.bc[d]:
                            continue
                        t[d] %= shape[d]
                    t = tuple(t)
                    if not lat.blocked[t] and label[t] < 0:
                        label[t] = nlab
                        stack.append(t)
        nlab += 1
    return label, nlab


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 0, 0)])
def test_p4_relaxes_to_boltzmann_per_cluster(oracle_mod, bc):
    lat = lpc_inputs.random_small((8, 8, 8), bc=bc, p_block=0.3, alpha=0.9, seed=7, dF_span=2.0)
    # carve two pockets cut off from the main pore network: a single site and a pair
    for cell, keep in (((2, 2, 2), [(2, 2, 2)]), ((5, 5, 5), [(5, 5, 5), (5, 5, 6)])):
        for k in keep:
            for d in range(3):
                for s in (-1, 1):
                    t = list(k)
                    t[d] += s
                    lat.blocked[tuple(t)] = 1
        for k in keep:
            lat.blocked[k] = 0
    o = _mk(oracle_mod, lat)
    pi = o.pi()
    rng = np.random.default_rng(11)
    rho0 = rng.random(lat.shape) * (lat.blocked == 0)
    out = o.propagate_real(rho0, 6000)
    label, nlab = _clusters(lat)
    assert nlab >= 3  # isolated pockets: the per-cluster statement matters
    for c in range(nlab):
        m = label == c
        mass = rho0[m].sum()
        assert abs(out[m].sum() - mass) <= 1e-12 * max(mass, 1e-300)
        want = mass * pi[m] / pi[m].sum()
        assert np.max(np.abs(out[m] - want)) <= 1e-9 * want.max()


def test_p4_bipartite_lattice_never_relaxes_at_alpha_one(oracle_mod):
    """SURVEY P4 caveat: alpha = 1 on a homogeneous even lattice has stay = 0 (period 2)."""
    lat = _uniform((4, 4, 4), alpha=1.0)
    o = _mk(oracle_mod, lat)
    assert np.all(np.abs(o.stay()) <= 2.3e-16)  # 1 - 6 * (1/6) up to rounding
    rho = np.zeros(lat.shape)
    rho[0, 0, 0] = 1.0
    out = o.propagate_real(rho, 1001)
    parity = np.indices(lat.shape).sum(axis=0) % 2
    assert out[parity == 0].sum() <= 1e-12  # an equilibrated lattice would hold one half here
    assert abs(out[parity == 1].sum() - 1.0) <= 1e-12


# --------------------------------------------------------------------------
# P13 equilibration loop (O9): closed-form iteration count and deltas on a single Fourier mode
# --------------------------------------------------------------------------
@pytest.mark.parametrize("alpha,L,thr", [(0.6, 12, 1e-9), (0.9, 8, 3e-7), (0.3, 16, 1e-6)])
def test_p13_equilibration_loop_single_mode_closed_form(oracle_mod, alpha, L, thr):
    """Homogeneous periodic lattice, rho(0) = 1/N + eps cos(2 pi x / L): the cosine is an eigenvector of W
    with eigenvalue lam = 1 - (alpha/3)(1 - cos(2 pi / L)) (one hop in +-x with probability alpha/6 each),
    so delta(k) = max_i |rho_i(k) - rho_i(k-1)| = eps (1 - lam) lam^(k-1) exactly, and the loop of
    PAPER.md:190-194 stops at the first k with delta(k) < threshold."""
    lat = _uniform((L, 4, 4), alpha=alpha)
    o = _mk(oracle_mod, lat)
    N, eps = L * 16, 1e-3
    x = np.arange(L)[:, None, None]
    rho0 = 1.0 / N + eps / N * np.cos(2 * np.pi * x / L) * np.ones(lat.shape)
    lam = 1.0 - (alpha / 3.0) * (1.0 - np.cos(2 * np.pi / L))
    k = np.arange(1, 5000)
    want_delta = eps / N * (1.0 - lam) * lam ** (k - 1)
    want_iters = int(k[np.argmax(want_delta < thr / N)])
    rho, iters, deltas = o.equilibrate(rho0, thr / N, 5000)
    assert iters == want_iters and 3 < iters < 4000
    # delta is a difference of nearly equal densities: it is exact to a few spacings of rho, not of delta
    assert np.max(np.abs(deltas - want_delta[:iters])) < 8 * np.spacing(rho0.max())
    assert abs(rho.sum() - rho0.sum()) < 1e-12
    want_rho = 1.0 / N + eps / N * lam ** iters * np.cos(2 * np.pi * x / L) * np.ones(lat.shape)
    assert np.max(np.abs(rho - want_rho)) < 1e-13 / N
    # the iteration cap is honoured and reported
    _, it2, d2 = o.equilibrate(rho0, 0.0, 7)
    assert it2 == 7 and d2.shape == (7,)
    _, it0, _ = o.equilibrate(rho0, 1.0, 0)
    assert it0 == 0


def test_p13_equilibration_reaches_boltzmann(oracle_mod):
    """From a flat density the loop ends at the Boltzmann density of Eq. 2 on a connected lattice."""
    lat = lpc_inputs.random_small((6, 6, 6), p_block=0.0, alpha=0.9, seed=5, dF_span=2.0)
    o = _mk(oracle_mod, lat)
    rho0 = np.full(lat.shape, 1.0 / lat.n_sites)
    rho, iters, deltas = o.equilibrate(rho0, 1e-15, 100000)
    assert 10 < iters < 100000 and deltas[-1] < 1e-15 and np.all(deltas[:-1] >= 1e-15)
    want = np.exp(-lat.dF)
    want /= want.sum()
    assert np.max(np.abs(rho - want) / want) < 1e-9


# --------------------------------------------------------------------------
# P14 spectrum (Eq. 9) and P15 region-resolved FID
# --------------------------------------------------------------------------
def test_p14_spectrum_single_line_closed_form_and_fft(oracle_mod):
    """G[n] = exp((i w0 - 1/T2) n dt) sums to a geometric series: F(f) = dt (1 - q^M)/(1 - q),
    q = exp((i (w0 - 2 pi f) - 1/T2 - pi lb) dt); on the grid f_k = k/(M dt) the sum is numpy's FFT."""
    dt, M, w0, T2 = 5e-6, 400, -2 * np.pi * 3200.0, 4e-4
    n = np.arange(M)
    G = np.exp((1j * w0 - 1.0 / T2) * n * dt)
    f = np.array([-3200.0, -3000.0, 0.0, 1234.5, 99000.0])
    for lb in (0.0, 150.0):
        q = np.exp((1j * (w0 - 2 * np.pi * f) - 1.0 / T2 - np.pi * lb) * dt)
        want = dt * (1 - q ** M) / (1 - q)
        got = oracle_mod.spectrum(G, dt, f, lb)
        assert np.max(np.abs(got - want)) < 1e-12 * np.abs(want).max()
    # the line sits at f = w0 / 2 pi, and the broadening lowers and widens it (Lorentzian: height ~ 1/(1/T2 + pi lb))
    grid = np.linspace(-6400.0, 0.0, 257)
    s0, s1 = oracle_mod.spectrum(G, dt, grid, 0.0), oracle_mod.spectrum(G, dt, grid, 800.0)
    assert grid[np.argmax(s0.real)] == -3200.0 and grid[np.argmax(s1.real)] == -3200.0
    assert s1.real.max() < 0.6 * s0.real.max()
    fk = np.arange(M) / (M * dt)
    assert np.max(np.abs(oracle_mod.spectrum(G, dt, fk) - dt * np.fft.fft(G))) < 1e-12 * M * dt


def test_p15_regional_fid_closed_form_on_sealed_pockets(oracle_mod):
    """Two pore pockets sealed from each other by carbon, each with its own uniform shift: nothing crosses
    the wall, so G_r[n] = (sum_{i in r} pi_i) exp(i w_r n dt) whatever dF is inside (Eq. 8 on each pocket),
    and the regions add up to G."""
    lat = lpc_inputs.random_small((10, 6, 6), bc=(1, 0, 0), p_block=0.2, alpha=0.8, seed=41, dF_span=2.0)
    lat.blocked[4:6] = 1                      # the wall
    region = np.zeros(lat.shape, dtype=np.uint8)
    region[5:] = 1
    w = (-9000.0, 4000.0)
    lat.omega[:5], lat.omega[5:] = w
    n = 60
    o = _mk(oracle_mod, lat, max_steps=n)
    pi = o.pi()
    Gr = o.step_with_regions(region, 2, n)
    k = np.arange(n + 1)
    for r in range(2):
        mass = pi[region == r].sum()
        assert 0.2 < mass < 0.8
        assert np.max(np.abs(Gr[r] - mass * np.exp(1j * w[r] * lat.dt * k))) < 1e-13
    assert np.max(np.abs(Gr.sum(axis=0) - o.fid())) < 1e-14
    # a label outside 0..n_regions-1 belongs to no region
    region[0] = 7
    o2 = _mk(oracle_mod, lat, max_steps=3)
    Gr2 = o2.step_with_regions(region, 2, 3)
    assert np.max(np.abs(Gr2[1] - Gr[1][:4])) < 1e-15 and np.all(np.abs(Gr2[0]) < np.abs(Gr[0][:4]))


# --------------------------------------------------------------------------
# P16 regional VACF / D
# --------------------------------------------------------------------------
def test_p16_regional_vacf_adds_up_and_matches_closed_forms(oracle_mod):
    """(i) sum_r w_r Z^r_d[m] = Z_d[m] of the whole lattice; (ii) on a homogeneous lattice every region has the
    free-diffusion values of Eq. 7, Z_d[1] = alpha a^2 / 3 and Z_d[m >= 2] = 0, hence D_r = alpha a^2 / (6 dt);
    (iii) a sealed pocket has the regional series of the pocket run on its own."""
    n = 25
    lat = lpc_inputs.random_small((9, 7, 8), bc=(1, 0, 0), p_block=0.25, alpha=0.8, seed=51, dF_span=2.0, n_moments=3)
    region = (np.indices(lat.shape)[1] % 3).astype(np.uint8)
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=n)
    Zr, w = o.step_with_regional_moments(region, 3, n)
    Zall, _ = o.moments()
    assert abs(w.sum() - 1.0) < 1e-14
    assert np.max(np.abs(np.einsum("r,rdm->dm", w, Zr) - Zall)) < 1e-15
    assert np.all(np.abs(Zr[:, :, 2:]) > 0)   # a heterogeneous lattice has memory

    a, alpha = 1.7, 0.6
    lat = _uniform((8, 6, 6), alpha=alpha, a=a)
    region = (np.indices(lat.shape)[0] >= 4).astype(np.uint8)
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=6)
    Zr, w = o.step_with_regional_moments(region, 2, 6)
    assert np.allclose(w, 0.5, atol=1e-15)
    assert np.max(np.abs(Zr[:, :, 0] - alpha * a * a / 3.0)) < 1e-15 and np.max(np.abs(Zr[:, :, 1:])) < 1e-16

    # sealed pocket: x < 4 is cut off from the rest by a carbon wall at x = 4 (reflective x closes the other side)
    lat = lpc_inputs.random_small((9, 5, 5), bc=(1, 0, 0), p_block=0.15, alpha=0.9, seed=52, dF_span=1.5, n_moments=3)
    lat.blocked[4] = 1
    region = (np.indices(lat.shape)[0] > 4).astype(np.uint8)
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=n)
    Zr, w = o.step_with_regional_moments(region, 2, n)
    import copy
    sub = copy.copy(lat)
    sub.nx = 4
    sub.dF, sub.blocked, sub.omega = (np.ascontiguousarray(v[:4]) for v in (lat.dF, lat.blocked, lat.omega))
    o_sub = _mk(oracle_mod, sub, n_moments=3, max_steps=n)
    o_sub.step(n)
    Zsub, _ = o_sub.moments()
    assert np.max(np.abs(Zr[0] - Zsub)) < 1e-14


# --------------------------------------------------------------------------
# P17 per-link mobility factors alpha_ij (O10)
# --------------------------------------------------------------------------
@pytest.mark.parametrize("shape,bc,n", [((3, 3, 4), (0, 0, 0), 3), ((3, 2, 4), (1, 0, 1), 4)])
def test_p17_links_trajectory_enumeration(oracle_mod, shape, bc, n):
    """Eq. 8/11 and <dx_1 dx_m> over every trajectory of the lattice gas whose hops carry alpha_ij."""
    lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.2, alpha=0.9, seed=61, n_steps=n)
    lat.dt = 2.0e-5
    link = lpc_inputs.random_links(shape, seed=1, lo=0.0)
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=n, link=link)
    o.step(n)
    G_def, C_def = _enumerate(lat, n, link)
    assert np.max(np.abs(o.fid() - G_def)) < 1e-12
    vacf, D = o.moments(n)
    assert np.max(np.abs(vacf - C_def[:, 1:])) < 1e-13
    # the factors matter: without them the answer is different
    G0, _ = _enumerate(lat, n)
    assert np.max(np.abs(G0 - G_def)) > 1e-6


def test_p17_links_keep_detailed_balance_and_boltzmann(oracle_mod):
    """":105: the same factor both ways, so that the equilibrium stays Eq. 2": pi_i p(i->j) = pi_j p(j->i) =
    alpha_ij (alpha/6) min(pi_i, pi_j), W pi = pi, mass conserved."""
    shape, bc = (6, 5, 7), (0, 1, 0)
    lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.25, alpha=0.8, seed=62)
    link = lpc_inputs.random_links(shape, seed=2)
    o = _mk(oracle_mod, lat, n_moments=0, max_steps=30, link=link)
    pi = _boltzmann(lat)
    assert np.max(np.abs(o.pi() - pi)) < 1e-16
    for d in range(3):
        # p_in(2d+1)[i] = p(i + e_d -> i), p_in(2d)[i] = p(i - e_d -> i)
        flow_back = pi * 0 + np.roll(pi, -1, axis=d) * o.p_in(2 * d + 1)          # pi_j p(j -> i), j = i + e_d
        flow_fwd = np.roll(np.roll(pi, 1, axis=d) * o.p_in(2 * d), -1, axis=d)    # pi_i p(i -> j) read at j, moved back to i
        want = link[d] * (lat.alpha / 6.0) * np.minimum(pi, np.roll(pi, -1, axis=d))
        if bc[d]:
            idx = [slice(None)] * 3
            idx[d] = -1
            want[tuple(idx)] = 0.0
        assert np.max(np.abs(flow_back - want)) < 1e-17 and np.max(np.abs(flow_fwd - want)) < 1e-17
    rho = o.propagate_real(pi, 30)
    assert np.max(np.abs(rho - pi) / np.where(pi > 0, pi, 1)) < 1e-13
    rng = np.random.default_rng(5)
    r0 = rng.random(shape) * (lat.blocked == 0)
    assert abs(o.propagate_real(r0, 30).sum() - r0.sum()) < 1e-12 * r0.sum()
    # the stay probability is what the moves leave over
    assert np.all(o.stay() >= 1.0 - lat.alpha - 1e-15) and np.all(o.stay() <= 1.0)


def test_p17_links_special_cases(oracle_mod):
    """(i) all factors 1 = no factors, bit for bit; (ii) anisotropic uniform factors on a homogeneous lattice: Eq. 7
    per axis, D_d = alpha alpha_d a^2 / (6 dt), Z_d[1] = alpha alpha_d a^2 / 3, Z_d[m >= 2] = 0; (iii) factor 0 on
    the links that close a periodic axis = a reflective wall there."""
    n = 20
    lat = lpc_inputs.random_small((5, 6, 4), p_block=0.2, alpha=0.9, seed=63, n_steps=n)
    a = _mk(oracle_mod, lat, n_moments=3, max_steps=n)
    b = _mk(oracle_mod, lat, n_moments=3, max_steps=n, link=np.ones((3,) + lat.shape))
    a.step(n); b.step(n)
    assert np.array_equal(a.fid(), b.fid()) and np.array_equal(a.moments()[0], b.moments()[0]) and np.array_equal(a.g(), b.g())

    alpha, aa, dt = 0.7, 1.3, 2.0
    ad = np.array([1.0, 0.5, 0.125])
    lat = _uniform((6, 6, 8), alpha=alpha, a=aa, dt=dt)
    link = np.ones((3,) + lat.shape) * ad[:, None, None, None]
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=8, link=link)
    o.step(8)
    Z, D = o.moments()
    assert np.max(np.abs(Z[:, 0] - alpha * ad * aa * aa / 3.0)) < 1e-15 and np.max(np.abs(Z[:, 1:])) < 1e-16
    assert np.max(np.abs(D - alpha * ad * aa * aa / (6.0 * dt))) < 1e-15
    # mean-square displacement of a delta source along each axis: n alpha alpha_d a^2 / 3 (n < L/2)
    src = np.zeros(lat.shape); src[3, 3, 4] = 1.0
    rho = o.propagate_real(src, 2)
    for d, L in enumerate(lat.shape):
        x = (np.arange(L) - (3, 3, 4)[d]) * aa
        msd = (rho.sum(axis=tuple(k for k in range(3) if k != d)) * x * x).sum()
        assert abs(msd - 2 * alpha * ad[d] * aa * aa / 3.0) < 1e-14

    lat = lpc_inputs.random_small((6, 4, 5), bc=(0, 0, 0), p_block=0.2, alpha=1.0, seed=64, n_steps=n)
    link = np.ones((3,) + lat.shape)
    link[0][-1] = 0.0   # the links between x = nx-1 and x = 0
    cut = _mk(oracle_mod, lat, n_moments=3, max_steps=n, link=link)
    import copy
    wall = copy.copy(lat); wall.bc = (1, 0, 0)
    ref = _mk(oracle_mod, wall, n_moments=3, max_steps=n)
    cut.step(n); ref.step(n)
    assert np.max(np.abs(cut.fid() - ref.fid())) < 1e-15 and np.max(np.abs(cut.moments()[0] - ref.moments()[0])) < 1e-16
    # factors outside [0, 1] are rejected
    bad = np.ones((3,) + lat.shape); bad[1, 0, 0, 0] = 1.5
    with pytest.raises(ValueError):
        _mk(oracle_mod, lat, link=bad)


# --------------------------------------------------------------------------
# P5 free diffusion closed form (Eq. 6, Eq. 7) -- golden values
# --------------------------------------------------------------------------
def _golden(name):
    rows = []
    with open(os.path.join(GOLD, name)) as fh:
        for line in fh:
            if line.strip() and not line.startswith("#"):
                rows.append([float(v) for v in line.split()])
    return rows


@pytest.mark.parametrize("row", _golden("free_diffusion.txt"))
def test_p5_free_diffusion(oracle_mod, row):
    alpha, a, dt, D_want, Z1_want = row
    L = 12
    lat = _uniform((L, L, L), alpha=alpha, dt=dt, a=a)
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=8)
    o.step(8)
    vacf, D = o.moments()
    assert np.allclose(vacf[:, 0], Z1_want, rtol=1e-14)
    assert np.max(np.abs(vacf[:, 1:])) <= 1e-17  # uncorrelated successive jumps
    assert np.allclose(D, D_want, rtol=1e-13)
    # MSD(n) = n alpha a^2 from a delta start, while the cloud has not met its image (n < L/2)
    rho = np.zeros(lat.shape)
    rho[0, 0, 0] = 1.0
    ax = np.minimum(np.arange(L), L - np.arange(L)) * a
    r2 = ax[:, None, None] ** 2 + ax[None, :, None] ** 2 + ax[None, None, :] ** 2
    for n in (1, 3, 5):
        out = o.propagate_real(rho, n)
        assert np.isclose((out * r2).sum(), n * alpha * a * a, rtol=1e-13)


# --------------------------------------------------------------------------
# P6 uniform shift -> one line at omega (Eq. 8) -- golden values
# --------------------------------------------------------------------------
@pytest.mark.parametrize("row", _golden("uniform_shift.txt"))
def test_p6_uniform_shift_single_line(oracle_mod, row):
    omega, dt, n, re, im = row
    n = int(n)
    lat = lpc_inputs.random_small((5, 6, 4), bc=(0, 1, 0), p_block=0.3, alpha=0.6, seed=8)
    lat.omega[...] = omega
    lat.dt = dt
    o = _mk(oracle_mod, lat, max_steps=n)
    o.step(n)
    G = o.fid()
    assert abs(G[n] - complex(re, im)) < 1e-12
    k = np.arange(n + 1)
    assert np.max(np.abs(G - np.exp(1j * omega * dt * k))) < 1e-12
    assert np.max(np.abs(np.abs(G) - 1.0)) < 1e-12


# --------------------------------------------------------------------------
# P7 brute force: every trajectory, from the definitions
# --------------------------------------------------------------------------
@pytest.mark.parametrize("shape,bc,n,alpha", [
    ((4, 4, 4), (0, 0, 0), 3, 1.0),
    ((3, 2, 4), (1, 0, 1), 4, 0.7),
    ((2, 1, 3), (0, 0, 0), 5, 0.9),   # degenerate axes: neighbours coincide / are the site itself (Q17)
])
def test_p7_trajectory_enumeration(oracle_mod, shape, bc, n, alpha):
    lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.25, alpha=alpha, seed=9, n_steps=n)
    lat.dt = 2.0e-5  # larger phase steps than the default so that the test has teeth
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=n)
    o.step(n)
    G_def, C_def = _enumerate(lat, n)
    G = o.fid()
    assert np.max(np.abs(G - G_def)) < 1e-12   # the enumeration adds ~1e5 terms uncompensated
    vacf, D = o.moments(n)
    for d in range(3):
        assert np.max(np.abs(vacf[d] - C_def[d, 1:])) < 1e-13
    D_def = C_def[:, 1] / (2 * lat.dt) + C_def[:, 2:].sum(axis=1) / lat.dt   # Eq. 4
    assert np.allclose(D, D_def, rtol=1e-10, atol=1e-10 * abs(D_def).max())


def _dense_step_matrices(lat):
    """The one-step matrices on a tiny lattice, entry by entry from the move table: W[j, i] = P(i -> j) (Eq. 1 with the
    rest term) and Phi = diag(exp(i omega_i dt)) (Eq. 13 prefactor, :144).  Blocked sites have no moves:
    their rows and columns are zero."""
    moves = _moves(lat)
    N = lat.n_sites
    flat = lambda idx: (idx[0] * lat.ny + idx[1]) * lat.nz + idx[2]
    W = np.zeros((N, N))
    for src, lst in moves.items():
        for tgt, p, _ in lst:
            W[flat(tgt), flat(src)] += p
    Phi = np.diag(np.exp(1j * lat.omega.reshape(-1) * lat.dt))
    return W, Phi


def test_p7_dense_matrix_power_4cubed(oracle_mod):
    """4^3: G[n] = 1^T (Phi W)^n pi with W built entry by entry from the move table."""
    lat = lpc_inputs.config0(L=4, n_steps=50)
    W, Phi = _dense_step_matrices(lat)
    v = _boltzmann(lat).reshape(-1).astype(complex)
    o = _mk(oracle_mod, lat)
    o.step(50)
    G = o.fid()
    for n in range(51):
        assert abs(G[n] - v.sum()) < 1e-13
        v = Phi @ (W @ v)
    assert np.max(np.abs(o.g().reshape(-1) - np.linalg.matrix_power(Phi @ W, 50) @ _boltzmann(lat).reshape(-1))) < 1e-15


@pytest.mark.parametrize("shape,bc", [((4, 4, 4), (0, 0, 0)), ((3, 2, 4), (1, 0, 1))])
def test_p18_set_g_against_dense_power(oracle_mod, shape, bc):
    """lpco_set_g (an arbitrary initial magnetisation): Eq. 13 is linear, so from any complex g(0) the
    state is (Phi W)^n g(0) and G[n] = 1^T (Phi W)^n g(0) (Eq. 12, :137).  g(0) has unrelated real and imaginary parts
    (a re/im swap fails), non-zero values on blocked sites (they must be dropped: carbon holds no fluid, :47-55) and the
    series must restart (G[0] = sum of g(0) over open sites, steps = 0) although steps were taken before."""
    n = 12
    lat = lpc_inputs.random_small(shape, bc=bc, p_block=0.25, alpha=0.8, seed=13, n_steps=n)
    lat.dt = 2.0e-5
    assert lat.blocked.any()
    W, Phi = _dense_step_matrices(lat)
    rng = np.random.default_rng(4)
    g0 = rng.standard_normal(shape) * np.array(3.0) + 1j * (0.25 + rng.random(shape))   # |re| and im of different size and sign pattern
    o = _mk(oracle_mod, lat, max_steps=n)
    o.step(5)                                   # a series that set_g has to discard
    o.set_g(g0)
    assert o.steps == 0
    opn = (lat.blocked == 0).reshape(-1)
    v = np.where(opn, g0.reshape(-1), 0.0)
    assert np.array_equal(o.g().reshape(-1), v)          # blocked sites zeroed, open ones taken as they are
    G, sabs = o.fid(with_scale=True)
    assert G.shape == (1,) and abs(G[0] - v.sum()) < 1e-14 * np.abs(v).sum()
    assert abs(sabs[0] - np.abs(v).sum()) < 1e-14 * np.abs(v).sum()
    o.step(n)
    G, sabs = o.fid(with_scale=True)
    scale = np.abs(v).sum()
    for k in range(n + 1):
        assert abs(G[k] - v.sum()) < 1e-14 * scale, k
        assert abs(sabs[k] - np.abs(v).sum()) < 1e-14 * scale, k
        if k == n:
            assert np.max(np.abs(o.g().reshape(-1) - v)) < 1e-14 * np.abs(g0).max()
            assert np.all(o.g().reshape(-1)[~opn] == 0)
        v = Phi @ (W @ v)


def test_p19_tolerance_scale_series_against_dense_power(oracle_mod):
    """The sum_i |g_i(n)| series of the oracle is the denominator of every FID tolerance (SURVEY
    Q12): it must be exactly sum_i |((Phi W)^n pi)_i|, not an upper bound of it.  Dense power on 4^3 with the chemical
    shifts of configs[0] stretched so that the sites dephase and the series falls well below 1 (an oracle that returned
    |G|, sum |Re g| + |Im g|, or the constant 1 fails)."""
    lat = lpc_inputs.config0(L=4, n_steps=60)
    lat.dt = 2.0e-5
    W, Phi = _dense_step_matrices(lat)
    v = _boltzmann(lat).reshape(-1).astype(complex)
    o = _mk(oracle_mod, lat)
    o.step(60)
    G, sabs = o.fid(with_scale=True)
    for n in range(61):
        assert abs(sabs[n] - np.abs(v).sum()) < 1e-14, n
        if n < 60:
            v = Phi @ (W @ v)
    # the case separates the candidates: each plausible wrong series is far outside the 1e-14 the right one meets
    assert sabs[60] < 0.98
    assert abs(G[60]) < 0.95 * sabs[60]
    assert np.abs(v.real).sum() + np.abs(v.imag).sum() > 1.05 * sabs[60]


# --------------------------------------------------------------------------
# P8 bounds
# --------------------------------------------------------------------------
def test_p8_bounds(oracle_mod):
    lat = lpc_inputs.config0(L=8, n_steps=300)
    o = _mk(oracle_mod, lat)
    pi = o.pi()
    prev = 1.0
    for _ in range(30):
        o.step(10)
        assert np.all(np.abs(o.g()) <= pi * (1 + 1e-12))
        G, sabs = o.fid(with_scale=True)
        assert sabs[-1] <= prev * (1 + 1e-14)
        prev = sabs[-1]
        assert abs(G[-1]) <= sabs[-1] + 1e-15
    assert abs(G[0] - 1.0) < 1e-14 and abs(sabs[0] - 1.0) < 1e-14


# --------------------------------------------------------------------------
# P9 bounded system: D_x -> 0     P10 Lorentz gas first lag
# --------------------------------------------------------------------------
def test_p9_reflective_box_sum_rule(oracle_mod):
    lat = lpc_inputs.random_small((6, 3, 3), bc=(1, 0, 0), p_block=0.0, alpha=0.8, seed=10, dF_span=1.5)
    lat.dt = 1.0
    n = 4000
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=n)
    o.step(n)
    vacf, D = o.moments()
    assert abs(D[0]) < 1e-13          # confined along x: no long-time diffusion
    assert D[1] > 1e-2 and D[2] > 1e-2  # free along the periodic axes


def test_p10_lorentz_gas_first_lag(oracle_mod):
    lat = lpc_inputs.random_small((10, 10, 10), p_block=0.3, alpha=0.8, seed=12)
    lat.dF[...] = 0.0
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=1)
    o.step(1)
    vacf, _ = o.moments(2)
    opn = (lat.blocked == 0).astype(float)
    n_open = opn.sum()
    for d in range(3):
        diff = np.roll(opn, -1, axis=d) - np.roll(opn, 1, axis=d)
        want2 = -(lat.alpha ** 2 * lat.a ** 2 / (36.0 * n_open)) * (opn * diff * diff).sum()
        want1 = (lat.alpha * lat.a ** 2 / (6.0 * n_open)) * (opn * (np.roll(opn, -1, axis=d) + np.roll(opn, 1, axis=d))).sum()
        assert np.isclose(vacf[d, 1], want2, rtol=1e-12)
        assert np.isclose(vacf[d, 0], want1, rtol=1e-12)


# --------------------------------------------------------------------------
# P11 two-site exchange (Bloch-McConnell in discrete time), exact 2x2 form
# --------------------------------------------------------------------------
def test_p11_two_site_exchange(oracle_mod):
    lat = lpc_inputs.random_small((2, 1, 1), p_block=0.0, alpha=0.6, seed=13)
    lat.dF[:, 0, 0] = [0.0, 1.2]
    lat.omega[:, 0, 0] = [0.0, -9000.0]
    lat.dt = 2.0e-5
    n = 200
    o = _mk(oracle_mod, lat, max_steps=n)
    o.step(n)
    # site A <-> B through the two x links (both lead to the other site); y, z links lead back home
    kAB = 2 * lat.alpha / 6 * np.exp(-1.2)
    kBA = 2 * lat.alpha / 6
    W = np.array([[1 - kAB, kBA], [kAB, 1 - kBA]])
    Phi = np.diag(np.exp(1j * lat.omega[:, 0, 0] * lat.dt))
    p = np.array([1.0, np.exp(-1.2)])
    v = (p / p.sum()).astype(complex)
    want = []
    for _ in range(n + 1):
        want.append(v.sum())
        v = Phi @ (W @ v)
    assert np.max(np.abs(o.fid() - np.array(want))) < 1e-14


# --------------------------------------------------------------------------
# P12 symmetries
# --------------------------------------------------------------------------
def test_p12_axis_permutation_and_translation(oracle_mod):
    lat = lpc_inputs.random_small((5, 6, 7), bc=(1, 0, 0), p_block=0.25, alpha=0.9, seed=14)
    n = 25
    o = _mk(oracle_mod, lat, n_moments=3, max_steps=n)
    o.step(n)
    G, (vacf, D) = o.fid(), o.moments()
    # permute axes (x,y,z) -> (z,x,y)
    perm = (2, 0, 1)
    lat2 = lpc_inputs.random_small((7, 5, 6), bc=tuple(lat.bc[p] for p in perm), alpha=0.9, seed=14)
    lat2.dF = np.ascontiguousarray(lat.dF.transpose(perm))
    lat2.blocked = np.ascontiguousarray(lat.blocked.transpose(perm))
    lat2.omega = np.ascontiguousarray(lat.omega.transpose(perm))
    o2 = _mk(oracle_mod, lat2, n_moments=3, max_steps=n)
    o2.step(n)
    assert np.max(np.abs(o2.fid() - G)) < 1e-14
    vacf2, D2 = o2.moments()
    for new_axis, old_axis in enumerate(perm):
        assert np.allclose(vacf2[new_axis], vacf[old_axis], rtol=1e-11, atol=1e-16)
        assert np.isclose(D2[new_axis], D[old_axis], rtol=1e-9)
    assert np.max(np.abs(o2.g() - o.g().transpose(perm))) < 1e-16
    # translate along the periodic axes
    lat3 = lpc_inputs.random_small((5, 6, 7), bc=(1, 0, 0), alpha=0.9, seed=14)
    for name in ("dF", "blocked", "omega"):
        setattr(lat3, name, np.ascontiguousarray(np.roll(getattr(lat, name), (2, -3), axis=(1, 2))))
    o3 = _mk(oracle_mod, lat3, max_steps=n)
    o3.step(n)
    assert np.max(np.abs(o3.fid() - G)) < 1e-14


# --------------------------------------------------------------------------
# Q16 isolated site, API guards, thread-count independence
# --------------------------------------------------------------------------
def test_q16_isolated_open_site_only_rotates(oracle_mod):
    lat = lpc_inputs.random_small((4, 4, 4), p_block=0.0, seed=15)
    lat.blocked[...] = 0
    c = (2, 2, 2)
    for d in range(3):
        for s in (-1, 1):
            t = list(c)
            t[d] += s
            lat.blocked[tuple(t)] = 1
    o = _mk(oracle_mod, lat, max_steps=7)
    o.step(7)
    assert o.stay()[c] == 1.0
    want = o.pi()[c] * np.exp(1j * lat.omega[c] * lat.dt * 7)
    assert abs(o.g()[c] - want) < 1e-15 * abs(want) * 10


def test_rejects_bad_inputs(oracle_mod):
    lat = lpc_inputs.random_small((3, 3, 3), seed=16)
    with pytest.raises(ValueError):
        oracle_mod.Oracle(lat.shape, lat.bc, lat.dt, lat.a, 0.0, lat.dF, lat.blocked, lat.omega)
    with pytest.raises(ValueError):
        oracle_mod.Oracle(lat.shape, lat.bc, lat.dt, lat.a, 1.0, lat.dF, np.ones_like(lat.blocked), lat.omega)
    o = _mk(oracle_mod, lat, max_steps=2)
    with pytest.raises(ValueError):
        o.step(3)


def test_result_does_not_depend_on_thread_count():
    code = (
        "import sys; sys.path.insert(0, %r); import importlib.util, numpy as np, lpc_inputs;"
        "s = importlib.util.spec_from_file_location('o', %r); m = importlib.util.module_from_spec(s); s.loader.exec_module(m);"
        "lat = lpc_inputs.config0(L=12, n_steps=20, n_moments=3); o = m.Oracle.from_lattice(lat); o.step(20);"
        "v, D = o.moments(); sys.stdout.write(o.fid().tobytes().hex() + v.tobytes().hex())"
    ) % (ROOT, os.path.join(ROOT, "oracle", "lpc_oracle.py"))
    outs = []
    for nt in ("1", "3", "8"):
        env = dict(os.environ, OMP_NUM_THREADS=nt)
        outs.append(subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, check=True).stdout)
    assert outs[0] == outs[1] == outs[2] and len(outs[0]) > 100


def test_oracle_is_clean_under_asan_and_ubsan(tmp_path):
    """the oracle built with -fsanitize=address,undefined (no OpenMP, so that every access is the
    calling thread's) and driven through all its entry points by tests/c_client/oracle_sanitize.c."""
    exe = str(tmp_path / "oracle_sanitize")
    subprocess.check_call(["gcc", "-std=gnu11", "-O1", "-g", "-fno-omit-frame-pointer", "-ffp-contract=off", "-fsanitize=address,undefined",
                           "-fno-sanitize-recover=all", "-Wall", "-Wextra", "-Wno-unknown-pragmas",
                           os.path.join(ROOT, "oracle", "lpc_oracle.c"), os.path.join(ROOT, "tests", "c_client", "oracle_sanitize.c"),
                           "-o", exe, "-lm"])
    out = subprocess.run([exe], capture_output=True, text=True, timeout=300,
                         env=dict(os.environ, ASAN_OPTIONS="detect_leaks=1:abort_on_error=0", UBSAN_OPTIONS="print_stacktrace=1"))
    assert out.returncode == 0, out.stdout + out.stderr
    assert out.stdout.strip() == "CLEAN" and "runtime error" not in out.stderr and "AddressSanitizer" not in out.stderr
