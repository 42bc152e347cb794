"""ctypes front end of the CPU oracle (oracle/lpc_oracle.c).  TEST INFRASTRUCTURE.

Only tests/, ``__graft_entry__.smoke()`` and bench.py's cpu_baseline /
``--impl reference`` legs may import this.  It does not import, and is not
imported by, ``paper_2603_22553_b200``.  The propagation itself (O1-O10) lives in
the C file and this module marshals numpy arrays for it; three read-outs that
are plain sums over the oracle's own fields are written out here in numpy:
``step_with_regions`` (Eq. 12 per region, pin P15), ``step_with_regional_moments``
(Eq. 4 per region, pin P16) and ``spectrum`` (Eq. 9, pin P14).
"""
from __future__ import annotations

import ctypes as C
import importlib.util
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))


def _load():
    spec = importlib.util.spec_from_file_location("_lpc_oracle_build", os.path.join(_HERE, "build.py"))
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    return C.CDLL(mod.build())


class _Cfg(C.Structure):
    _fields_ = [("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("bc", C.c_int32 * 3),
                ("dt", C.c_double), ("a", C.c_double), ("alpha", C.c_double)]


_lib = _load()
_dp = C.POINTER(C.c_double)
_u8p = C.POINTER(C.c_uint8)
_lib.lpco_create.restype = C.c_void_p
_lib.lpco_create.argtypes = [C.POINTER(_Cfg), _dp, _u8p, _dp, C.c_int, C.c_int64]
_lib.lpco_create_links.restype = C.c_void_p
_lib.lpco_create_links.argtypes = [C.POINTER(_Cfg), _dp, _u8p, _dp, _dp, C.c_int, C.c_int64]
_lib.lpco_destroy.argtypes = [C.c_void_p]
_lib.lpco_step.argtypes = [C.c_void_p, C.c_int64]
_lib.lpco_set_g.argtypes = [C.c_void_p, _dp]
_lib.lpco_propagate_real.argtypes = [C.c_void_p, _dp, _dp, C.c_int64]
_lib.lpco_equilibrate.restype = C.c_int64
_lib.lpco_equilibrate.argtypes = [C.c_void_p, _dp, C.c_double, C.c_int64, _dp]
_lib.lpco_steps.restype = C.c_int64
_lib.lpco_steps.argtypes = [C.c_void_p]
_lib.lpco_partition_sum.restype = C.c_double
_lib.lpco_partition_sum.argtypes = [C.c_void_p]
for _n in ("lpco_get_pi", "lpco_get_stay", "lpco_get_g"):
    getattr(_lib, _n).argtypes = [C.c_void_p, _dp]
    getattr(_lib, _n).restype = None
_lib.lpco_get_p_in.argtypes = [C.c_void_p, C.c_int, _dp]
_lib.lpco_get_p_in.restype = None
_lib.lpco_get_P.argtypes = [C.c_void_p, C.c_int, _dp]
_lib.lpco_get_u.argtypes = [C.c_void_p, C.c_int, _dp]
_lib.lpco_get_fid.argtypes = [C.c_void_p, C.c_int64, C.c_int64, _dp, _dp]
_lib.lpco_get_moments.argtypes = [C.c_void_p, C.c_int64, _dp, _dp]
_lib.lpco_neighbor.restype = C.c_int64
_lib.lpco_neighbor.argtypes = [C.POINTER(_Cfg), C.c_int64, C.c_int, C.c_int]
_lib.lpco_hop.restype = C.c_double
_lib.lpco_hop.argtypes = [C.POINTER(_Cfg), _dp, _u8p, C.c_int64, C.c_int64]


def _d(a):
    return a.ctypes.data_as(_dp)


def _cfg(shape, bc, dt, a, alpha):
    return _Cfg(int(shape[0]), int(shape[1]), int(shape[2]), (C.c_int32 * 3)(*[int(b) for b in bc]),
                float(dt), float(a), float(alpha))


def neighbor(shape, bc, i, d, s):
    """O2: index of the neighbour of site i along axis d, direction s; -1 if none."""
    cfg = _cfg(shape, bc, 1.0, 1.0, 1.0)
    return int(_lib.lpco_neighbor(C.byref(cfg), int(i), int(d), int(s)))


def hop(shape, bc, alpha, dF, blocked, i, j):
    """O3: p(i->j)."""
    cfg = _cfg(shape, bc, 1.0, 1.0, alpha)
    dF = np.ascontiguousarray(dF, dtype=np.float64)
    blocked = np.ascontiguousarray(blocked, dtype=np.uint8)
    return float(_lib.lpco_hop(C.byref(cfg), _d(dF), blocked.ctypes.data_as(_u8p), int(i), int(j)))


class Oracle:
    """One oracle run: create from the site arrays, step, read series and fields."""

    def __init__(self, shape, bc, dt, a, alpha, dF, blocked, omega, n_moments=0, max_steps=0, link=None):
        """link: None, or 3 x shape factors alpha_ij in [0, 1] (O10): link[d][i] belongs to the
        link between site i and its +d neighbour and scales the hop both ways."""
        self.shape = tuple(int(v) for v in shape)
        self.n = int(np.prod(self.shape))
        self.n_moments = int(n_moments)
        self.bc = tuple(int(b) for b in bc)
        self.a = float(a)
        self.cfg = _cfg(shape, bc, dt, a, alpha)
        dF = np.ascontiguousarray(dF, dtype=np.float64).reshape(-1)
        blocked = np.ascontiguousarray(blocked, dtype=np.uint8).reshape(-1)
        omega = np.ascontiguousarray(omega, dtype=np.float64).reshape(-1)
        assert dF.size == self.n and blocked.size == self.n and omega.size == self.n
        if link is None:
            self._h = _lib.lpco_create(C.byref(self.cfg), _d(dF), blocked.ctypes.data_as(_u8p), _d(omega),
                                       self.n_moments, int(max_steps))
        else:
            link = np.ascontiguousarray(link, dtype=np.float64).reshape(-1)
            assert link.size == 3 * self.n
            self._h = _lib.lpco_create_links(C.byref(self.cfg), _d(dF), blocked.ctypes.data_as(_u8p), _d(omega), _d(link),
                                             self.n_moments, int(max_steps))
        if not self._h:
            raise ValueError("lpco_create rejected the inputs")

    @classmethod
    def from_lattice(cls, lat, n_moments=None, max_steps=None, link=None):
        return cls(lat.shape, lat.bc, lat.dt, lat.a, lat.alpha, lat.dF, lat.blocked, lat.omega,
                   lat.n_moments if n_moments is None else n_moments,
                   lat.n_steps if max_steps is None else max_steps, link=link)

    def close(self):
        if getattr(self, "_h", None):
            _lib.lpco_destroy(self._h)
            self._h = None

    __del__ = close

    def step(self, n=1):
        if _lib.lpco_step(self._h, int(n)) != 0:
            raise ValueError("lpco_step: over capacity")

    @property
    def steps(self):
        return int(_lib.lpco_steps(self._h))

    @property
    def partition_sum(self):
        return float(_lib.lpco_partition_sum(self._h))

    def set_g(self, g):
        g = np.ascontiguousarray(g, dtype=np.complex128).reshape(-1)
        assert g.size == self.n
        _lib.lpco_set_g(self._h, g.view(np.float64).ctypes.data_as(_dp))

    def propagate_real(self, rho, n_steps):
        rho = np.ascontiguousarray(rho, dtype=np.float64).reshape(-1)
        out = np.empty_like(rho)
        _lib.lpco_propagate_real(self._h, _d(rho), _d(out), int(n_steps))
        return out.reshape(self.shape)

    def equilibrate(self, rho, threshold, max_iters):
        """The paper's equilibration loop: returns (rho, iterations, deltas[1..iterations])."""
        rho = np.array(rho, dtype=np.float64).reshape(-1)
        deltas = np.zeros(max(int(max_iters), 1), dtype=np.float64)
        it = int(_lib.lpco_equilibrate(self._h, _d(rho), float(threshold), int(max_iters), _d(deltas)))
        assert it >= 0
        return rho.reshape(self.shape), it, deltas[:it]

    def step_with_regions(self, region, n_regions, n_steps):
        """Region-resolved FID (PAPER.md:180 blocks, Fig. 9 :275-281): Eq. 12 (:137) restricted to each
        region, G_r[k] = sum_{i in r} g_i(k), for k = current step .. current step + n_steps, taken from the
        site values after every single step.  Returns an array [n_regions, n_steps + 1]."""
        region = np.asarray(region).reshape(self.shape)
        out = np.zeros((n_regions, n_steps + 1), dtype=np.complex128)
        for k in range(n_steps + 1):
            if k:
                self.step(1)
            g = self.g()
            for r in range(n_regions):
                out[r, k] = g[region == r].sum()
        return out

    def step_with_regional_moments(self, region, n_regions, n_steps):
        """Regional VACF (the regional D of Table 1; reading Q27): the sum of
        Eq. 4 (:79) over the sites of region r only -- the site a particle occupies when the later
        displacement starts -- divided by the region's equilibrium population w_r = sum_{i in r} pi_i:
            Z^r_d[1] = sum_{i in r} pi_i sum_s p(i -> i + s e_d) a^2 / w_r            (Eq. 5, :92)
            Z^r_d[m] = sum_{i in r} P^d_i(m-1) u^d_i / w_r,  m = 2 .. n_steps + 1     (O8)
        Must be called at step 0.  Returns (Z[n_regions, 3, n_steps + 1] with Z[r, d, m-1], w[n_regions])."""
        assert self.n_moments == 3 and self.steps == 0
        region = np.asarray(region).reshape(self.shape)
        pi = self.pi()
        w = np.array([pi[region == r].sum() for r in range(n_regions)])
        Z = np.zeros((n_regions, 3, n_steps + 1))
        for d in range(3):
            # p(i -> i + e_d) is the probability with which i + e_d receives from its -d neighbour, and likewise for -e_d
            out_plus = np.roll(self.p_in(2 * d), -1, axis=d)
            out_minus = np.roll(self.p_in(2 * d + 1), +1, axis=d)
            if self.bc[d]:  # reflective: no neighbour beyond the wall
                idx = [slice(None)] * 3
                idx[d] = -1
                out_plus[tuple(idx)] = 0.0
                idx[d] = 0
                out_minus[tuple(idx)] = 0.0
            z1 = pi * (out_plus + out_minus) * self.a ** 2
            for r in range(n_regions):
                Z[r, d, 0] = z1[region == r].sum() / w[r]
        u = [self.u(d) for d in range(3)]
        for m in range(1, n_steps + 1):
            for d in range(3):
                prod = self.P(d) * u[d]
                for r in range(n_regions):
                    Z[r, d, m] = prod[region == r].sum() / w[r]
            self.step(1)
        return Z, w

    def _get(self, fn, *a):
        out = np.empty(self.n, dtype=np.float64)
        fn(self._h, *a, _d(out))
        return out.reshape(self.shape)

    def pi(self):
        return self._get(_lib.lpco_get_pi)

    def stay(self):
        return self._get(_lib.lpco_get_stay)

    def p_in(self, k):
        """p(nb_k(i) -> i) with k = 2*d + (s > 0)."""
        return self._get(_lib.lpco_get_p_in, int(k))

    def g(self):
        out = np.empty(self.n, dtype=np.complex128)
        _lib.lpco_get_g(self._h, out.view(np.float64).ctypes.data_as(_dp))
        return out.reshape(self.shape)

    def P(self, d):
        return self._get(_lib.lpco_get_P, int(d))

    def u(self, d):
        return self._get(_lib.lpco_get_u, int(d))

    def fid(self, first=0, count=None, with_scale=False):
        count = self.steps + 1 - first if count is None else count
        out = np.empty(count, dtype=np.complex128)
        sabs = np.empty(count, dtype=np.float64)
        rc = _lib.lpco_get_fid(self._h, int(first), int(count), out.view(np.float64).ctypes.data_as(_dp), _d(sabs))
        if rc != 0:
            raise ValueError("lpco_get_fid: range")
        return (out, sabs) if with_scale else out

    def moments(self, count=None):
        """(vacf[3, count] = Z_d[1..count], D[3])."""
        count = self.steps + 1 if count is None else count
        vacf = np.empty((3, count), dtype=np.float64)
        D = np.empty(3, dtype=np.float64)
        if _lib.lpco_get_moments(self._h, int(count), _d(vacf), _d(D)) != 0:
            raise ValueError("lpco_get_moments: range or no moments")
        return vacf, D


def spectrum(G, dt, freqs_hz, lb_hz=0.0):
    """Eq. 9, F(f) = int G(t) exp(-2 i pi f t) dt, as the plain sum over the samples
    (reading Q23): F(f) = dt * sum_n G[n] exp(-pi lb n dt) exp(-2 pi i f n dt).  lb_hz is an
    optional Lorentzian line broadening (0 = none).  One frequency at a time, written out."""
    G = np.asarray(G, dtype=np.complex128)
    t = np.arange(G.size) * float(dt)
    w = np.exp(-np.pi * float(lb_hz) * t)
    out = np.empty(len(freqs_hz), dtype=np.complex128)
    for k, f in enumerate(np.asarray(freqs_hz, dtype=np.float64)):
        out[k] = float(dt) * np.sum(G * w * np.exp(-2j * np.pi * f * t))
    return out
