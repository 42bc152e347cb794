"""Seeded synthetic lattices for the LPC3D hot path (inputs only).

This module is the ONE thing the CPU oracle (``oracle/``) and the CUDA library
(``paper_2603_22553_b200/``) share: it produces the per-site input arrays
(free energy dF in kT, blocked mask, resonance frequency omega in rad/s) and
the scalar parameters of a run. It holds none of the method's arithmetic: no
hop weights, no Boltzmann factors, no propagation.

The recipes stand in for the paper's single-particle, monolith and
supercapacitor systems; the paper's MD/DFT parametrisation
and the YP50F pore-size distribution are not available, so every array here is
seeded noise with the shapes, value ranges and structure BASELINE.json's
``configs`` describe.  DESIGN.md ("Input recipe") lists each choice.

Seeds follow SURVEY.md section 8(d): ``seed = 2603225530 + 10*config + k`` with
k = 0 for the mask, 1 for the pore field, 2 for the config-0 uniforms.
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

SEED_BASE = 2603225530
LARMOR_MHZ = 400.0  # BASELINE.json configs[0]: omega = 2 pi delta * 400 MHz * 1e-6
DT_DEFAULT = 5.0e-6  # s


@dataclass
class Lattice:
    """Inputs of one run, as both implementations receive them."""

    name: str
    nx: int
    ny: int
    nz: int
    bc: tuple  # per axis: 0 periodic, 1 reflective
    dt: float
    a: float
    alpha: float
    n_steps: int
    n_moments: int
    dF: np.ndarray  # float64 [nx,ny,nz], kT
    blocked: np.ndarray  # uint8   [nx,ny,nz]
    omega: np.ndarray  # float64 [nx,ny,nz], rad/s
    notes: dict = field(default_factory=dict)

    @property
    def n_sites(self) -> int:
        return self.nx * self.ny * self.nz

    @property
    def shape(self) -> tuple:
        return (self.nx, self.ny, self.nz)


def _rng(config: int, k: int) -> np.random.Generator:
    return np.random.Generator(np.random.PCG64(SEED_BASE + 10 * config + k))


def ppm_to_omega(delta_ppm: np.ndarray) -> np.ndarray:
    """Chemical shift in ppm -> angular frequency offset in rad/s at 400 MHz."""
    return 2.0 * np.pi * delta_ppm * LARMOR_MHZ


def gaussian_field(shape, ell: float, rng: np.random.Generator) -> np.ndarray:
    """Standardised periodic Gaussian random field with C(r) ~ exp(-r^2 / 2 ell^2).

    White N(0,1) noise, filtered in Fourier space by exp(-|k|^2 ell^2 / 4),
    then shifted and scaled to zero mean and unit variance.
    """
    try:
        from scipy import fft as _fft

        kw = {"workers": -1}
    except Exception:  # pragma: no cover - scipy is in the image
        _fft = np.fft
        kw = {}
    white = rng.standard_normal(size=shape)
    spec = _fft.rfftn(white, **kw)
    del white
    kx = 2.0 * np.pi * np.fft.fftfreq(shape[0])
    ky = 2.0 * np.pi * np.fft.fftfreq(shape[1])
    kz = 2.0 * np.pi * np.fft.rfftfreq(shape[2])
    c = ell * ell / 4.0
    spec *= np.exp(-c * kx * kx)[:, None, None]
    spec *= np.exp(-c * ky * ky)[None, :, None]
    spec *= np.exp(-c * kz * kz)[None, None, :]
    xi = _fft.irfftn(spec, s=shape, **kw)
    del spec
    xi -= xi.mean()
    xi /= xi.std()
    return xi


def pore_width_nm(xi: np.ndarray) -> np.ndarray:
    """Pore width from the standardised field, clipped to 0.5-2 nm."""
    return np.clip(1.0 + 0.35 * xi, 0.5, 2.0)


def pore_site_fields(w: np.ndarray):
    """dF (kT) and delta (ppm) of a pore of width w nm (BASELINE.json configs[1])."""
    dF = -4.0 * np.exp(-(w - 0.5) / 0.4)
    delta = -8.0 * np.exp(-(w - 0.5) / 0.5)
    return dF, delta


def _finish(name, shape, bc, n_steps, n_moments, dF, blocked, delta, alpha=1.0, notes=None, larmor_mhz=LARMOR_MHZ):
    blocked = np.ascontiguousarray(blocked, dtype=np.uint8)
    dF = np.ascontiguousarray(dF, dtype=np.float64)
    omega = np.ascontiguousarray(ppm_to_omega(np.asarray(delta, dtype=np.float64)) * (larmor_mhz / LARMOR_MHZ))
    return Lattice(
        name=name, nx=shape[0], ny=shape[1], nz=shape[2], bc=tuple(bc), dt=DT_DEFAULT,
        a=1.0, alpha=alpha, n_steps=n_steps, n_moments=n_moments,
        dF=dF, blocked=blocked, omega=omega, notes=notes or {},
    )


def config0(L: int = 32, n_steps: int = 2000, n_moments: int = 0) -> Lattice:
    """BASELINE.json configs[0]: 32^3 periodic, 30% blocked iid, uniform dF and delta."""
    shape = (L, L, L)
    blocked = _rng(0, 0).random(shape) < 0.3
    u = _rng(0, 2)
    dF = -3.0 * u.random(shape)  # U(-3, 0]
    delta = -10.0 * u.random(shape)  # U(-10, 0] ppm
    return _finish("config0_uniform", shape, (0, 0, 0), n_steps, n_moments, dF, blocked, delta)


def particle(L: int = 128, radius: float = 48.0, ell: float = 4.0, n_steps: int = 20000,
             n_moments: int = 0) -> Lattice:
    """BASELINE.json configs[1]: one porous carbon particle in bulk electrolyte."""
    shape = (L, L, L)
    xi = gaussian_field(shape, ell, _rng(1, 1))
    dF, delta = pore_site_fields(pore_width_nm(xi))
    ax = np.arange(L, dtype=np.float64) - L / 2.0
    r2 = ax[:, None, None] ** 2 + ax[None, :, None] ** 2 + ax[None, None, :] ** 2
    inside = r2 < radius * radius
    blocked = (_rng(1, 0).random(shape) < 0.1) & inside
    dF = np.where(inside, dF, 0.0)
    delta = np.where(inside, delta, 0.0)
    return _finish("config1_particle", shape, (0, 0, 0), n_steps, n_moments, dF, blocked, delta,
                   notes={"radius": radius, "ell": ell})


def monolith(L: int = 256, ell: float = 8.0, p_block: float = 0.2, n_steps: int = 20000,
             n_moments: int = 3, config: int = 2, shape=None) -> Lattice:
    """BASELINE.json configs[2] (and the configs[4] sweep statistics): porous everywhere."""
    shape = tuple(shape) if shape is not None else (L, L, L)
    xi = gaussian_field(shape, ell, _rng(config, 1))
    dF, delta = pore_site_fields(pore_width_nm(xi))
    del xi
    blocked = _rng(config, 0).random(shape) < p_block
    return _finish("config2_monolith", shape, (0, 0, 0), n_steps, n_moments, dF, blocked, delta,
                   notes={"ell": ell, "p_block": p_block})


def supercap(nx: int = 2048, ny: int = 256, nz: int = 256, ell: float = 8.0,
             p_block: float = 0.2, n_steps: int = 10000, n_moments: int = 0) -> Lattice:
    """BASELINE.json configs[3]: two film electrodes, bulk in the middle, reflective x.

    x in [0, 3nx/8) is the positive electrode (dF + 0.5 kT), x in [5nx/8, nx) the
    negative one (dF - 0.5 kT), the middle quarter bulk electrolyte.
    At nx = 2048 those are the 768 / 512 / 768 planes BASELINE.json names.
    """
    shape = (nx, ny, nz)
    xi = gaussian_field(shape, ell, _rng(3, 1))
    dF, delta = pore_site_fields(pore_width_nm(xi))
    del xi
    x = np.arange(nx)
    pos = (x < (3 * nx) // 8)[:, None, None]
    neg = (x >= (5 * nx) // 8)[:, None, None]
    electrode = pos | neg
    blocked = (_rng(3, 0).random(shape) < p_block) & electrode
    dF = np.where(pos, dF + 0.5, np.where(neg, dF - 0.5, 0.0))
    delta = np.where(electrode, delta, 0.0)
    return _finish("config3_supercap", shape, (1, 0, 0), n_steps, n_moments, dF, blocked, delta,
                   notes={"ell": ell, "p_block": p_block})


def sweep(L: int, n_moments: int = 0, n_steps: int = 1000) -> Lattice:
    """BASELINE.json configs[4]: L^3 with monolith statistics."""
    lat = monolith(L=L, ell=8.0, p_block=0.2, n_steps=n_steps, n_moments=n_moments, config=4)
    lat.name = f"config4_sweep_{L}"
    return lat


def random_small(shape, bc=(0, 0, 0), p_block=0.3, alpha=1.0, seed=0, n_steps=10,
                 n_moments=3, dF_span=3.0, ppm_span=10.0) -> Lattice:
    """Small iid lattice for unit tests (config-0 statistics on any shape)."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 1000 + seed))
    blocked = rng.random(shape) < p_block
    dF = -dF_span * rng.random(shape)
    delta = -ppm_span * rng.random(shape)
    lat = _finish("random_small", tuple(shape), bc, n_steps, n_moments, dF, blocked, delta, alpha)
    return lat


def film(nx: int = 100, ny: int = 100, nz: int = 300, radius: float = 9.0, spacing: int = 20, ell: float = 4.0,
         p_block: float = 0.1, alpha: float = 0.025, n_steps: int = 50000, n_moments: int = 0) -> Lattice:
    """Film-electrode supercapacitor of PAPER.md:236-248: a 100 x 100 x 300 lattice, no periodic
    boundary in z, two electrodes made of monodisperse porous carbon particles of radius 9 sites that fill 38% of
    the electrode volume, bulk electrolyte between the particles and between the electrodes.

    Stand-in recipe (the paper's particle positions are not given): the electrodes are z < nz/3 and z >= 2nz/3;
    particle centres sit on a simple-cubic grid of `spacing` sites (20: (4/3) pi 9^3 / 20^3 = 0.382) with a seeded
    jitter of -1..1 sites per axis; inside the particles the pore field of configs[1] (ell = 4, 10% blocked), the
    positive / negative electrode shifted by +-0.5 kT as in configs[3]; everything else is bulk (dF = delta = 0,
    open).  alpha = dt / tau = 5 us / 0.2 ms, 19F at 282 MHz (:248).  notes["particle"] is the particle
    mask (1 positive-electrode particle, 2 negative, 0 bulk).
    """
    shape = (nx, ny, nz)
    rng = _rng(5, 0)
    label = np.zeros(shape, dtype=np.uint8)
    zel = nz // 3
    R = int(np.ceil(radius)) + 1
    off = np.arange(-R, R + 1)
    ball = (off[:, None, None] ** 2 + off[None, :, None] ** 2 + off[None, None, :] ** 2) <= radius * radius
    half = spacing // 2
    for zlo, lab in ((0, 1), (nz - zel, 2)):
        for cx in range(half, nx - half + 1, spacing):
            for cy in range(half, ny - half + 1, spacing):
                for cz in range(zlo + half, zlo + zel - half + 1, spacing):
                    j = rng.integers(-1, 2, size=3)
                    c = np.array([cx, cy, cz]) + j
                    c[2] = min(max(c[2], zlo + R), zlo + zel - R - 1) if zel > 2 * R + 1 else c[2]
                    ix = (c[0] + off) % nx
                    iy = (c[1] + off) % ny
                    iz = np.clip(c[2] + off, 0, nz - 1)
                    sub = label[np.ix_(ix, iy, iz)]
                    sub[ball] = lab
                    label[np.ix_(ix, iy, iz)] = sub
    inside = label > 0
    xi = gaussian_field(shape, ell, _rng(5, 1))
    dF, delta = pore_site_fields(pore_width_nm(xi))
    del xi
    blocked = (rng.random(shape) < p_block) & inside
    dF = np.where(label == 1, dF + 0.5, np.where(label == 2, dF - 0.5, 0.0))
    delta = np.where(inside, delta, 0.0)
    return _finish("film_supercap", shape, (0, 0, 1), n_steps, n_moments, dF, blocked, delta, alpha=alpha,
                   notes={"radius": radius, "spacing": spacing, "particle": label, "fraction": float(inside[:, :, :zel].mean())},
                   larmor_mhz=282.0)


def random_links(shape, seed=0, lo=0.1) -> np.ndarray:
    """Seeded iid per-link mobility factors alpha_ij ~ U[lo, 1]: [3, nx, ny, nz], entry [d, i] belongs to
    the link between site i and its +d neighbour."""
    rng = np.random.Generator(np.random.PCG64(SEED_BASE + 2000 + seed))
    return lo + (1.0 - lo) * rng.random((3,) + tuple(shape))


def confined_links(confined: np.ndarray, mu: float) -> np.ndarray:
    """Link factors for "mobility decreased due to confinement": a link has factor mu when either of
    its two ends lies in the confined region (a particle or an electrode) and 1 between two bulk sites."""
    c = np.asarray(confined) != 0
    out = np.ones((3,) + c.shape)
    for d in range(3):
        out[d][c | np.roll(c, -1, axis=d)] = mu
    return out
