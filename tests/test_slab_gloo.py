"""Routing of the x-slab decomposition (paper_2603_22553_b200/slab.py) with world_size 2 on gloo.

The slab driver is written against a small lattice interface; here a stand-in with CPU tensors takes the place of
the CUDA lattice (a weighted three-point exchange along x whose weights need the neighbour's pi plane, so both the
PARAMS and the STATE exchange matter) and the result is compared with the same recurrence on the whole array.
The CUDA lattice itself runs through the same driver in tests/test_gpu_parity.py (all slabs on one GPU).
"""
import os
import sys

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)

from paper_2603_22553_b200 import slab  # noqa: E402


class FakeLattice:
    """nx owned planes + 2 ghost planes of ny*nz values; channels: 1 (PARAMS: pi) and 2 (STATE: f, 2 f)."""

    def __init__(self, shape, bc, max_steps=0, **_):
        assert bc[0] == slab.LPC_BC_HALO
        self.nx, self.m = shape[0], shape[1] * shape[2]
        self.shape = shape
        self.pi = torch.zeros(1, self.nx + 2, self.m, dtype=torch.float64)
        self.f = torch.zeros(2, self.nx + 2, self.m, dtype=torch.float64)
        self.Z = None
        self.series = []

    def partition_sum(self, dF, blocked):
        return float(np.exp(-dF)[blocked == 0].sum())

    def set_partition_sum(self, Z):
        self.Z = Z

    def set_site_params(self, dF, blocked, omega):
        e = np.where(blocked == 0, np.exp(-dF), 0.0) / self.Z
        self.pi[0, 1:-1] = torch.from_numpy(e.reshape(self.nx, self.m))

    def halo_planes(self, which, side, role):
        t = self.pi if which == slab.HALO_PARAMS else self.f
        x = (1 if role == slab.SEND else 0) if side == 0 else (self.nx if role == slab.SEND else self.nx + 1)
        return t[:, x]

    def slab_finish(self):
        self.f.zero_()
        self.f[0, 1:-1] = 1.0
        self.f[1, 1:-1] = 2.0
        self.series = [self._sum()]

    def set_state(self, which, arr):
        a = torch.from_numpy(np.real(arr).reshape(self.nx, self.m).copy())
        self.f[0, 1:-1] = a
        self.f[1, 1:-1] = 2 * a
        self.series = [self._sum()]

    def _sum(self):
        return complex(float((self.pi[0, 1:-1] * self.f[0, 1:-1]).sum()), 0.0)

    def step(self, n):
        assert n == 1
        p, f = self.pi[0], self.f
        wl = torch.minimum(p[1:-1], p[:-2])
        wh = torch.minimum(p[1:-1], p[2:])
        new = f.clone()
        new[:, 1:-1] = f[:, 1:-1] + 0.25 * (wl * (f[:, :-2] - f[:, 1:-1]) + wh * (f[:, 2:] - f[:, 1:-1])) / p[1:-1].clamp_min(1e-300)
        self.f = new
        self.series.append(self._sum())

    def fid(self):
        return np.array(self.series, dtype=np.complex128)

    def moments(self):
        z = np.tile(np.real(self.fid())[None, :], (3, 1))
        return z, z.sum(axis=1)

    def field(self, which):
        return self.f[0, 1:-1].numpy().reshape(self.shape).copy()


def _reference(dF, blocked, g0, periodic, n):
    e = np.where(blocked == 0, np.exp(-dF), 0.0)
    p = e / e.sum()
    f = g0.copy()
    G = [(p * f).sum()]
    for _ in range(n):
        pl, ph, fl, fh = np.roll(p, 1, 0), np.roll(p, -1, 0), np.roll(f, 1, 0), np.roll(f, -1, 0)
        if not periodic:
            pl[0] = 0.0
            ph[-1] = 0.0
        f = f + 0.25 * (np.minimum(p, pl) * (fl - f) + np.minimum(p, ph) * (fh - f)) / np.maximum(p, 1e-300)
        G.append((p * f).sum())
    return f, np.array(G)


def _inputs(shape):
    rng = np.random.default_rng(11)
    return -2.0 * rng.random(shape), (rng.random(shape) < 0.2).astype(np.uint8), rng.random(shape)


def _run(shape, bc, spr, n):
    dF, blocked, g0 = _inputs(shape)
    g0 = g0 * (blocked == 0)
    ss = slab.SlabSet(shape, bc=bc, slabs_per_rank=spr, lattice_factory=FakeLattice, max_steps=n)
    Z = ss.set_site_params(dF, blocked, np.zeros(shape), g0.astype(np.complex128))
    ss.step(n)
    f_ref, G_ref = _reference(dF, blocked, g0, bc[0] == 0, n)
    assert abs(Z - np.exp(-dF)[blocked == 0].sum()) < 1e-9
    assert np.max(np.abs(ss.fid().real - G_ref)) < 1e-13
    assert np.max(np.abs(ss.gather_field(0) - f_ref)) < 1e-12
    z, d = ss.moments()
    assert z.shape == (3, n + 1) and np.max(np.abs(z[0] - G_ref)) < 1e-13 and abs(d[0] - G_ref.sum()) < 1e-11
    return ss


def _run_local(shape, bc, spr, n):
    """Every rank hands in its own planes only (local=True), as bench.py does for the weak-scaling run."""
    dF, blocked, g0 = _inputs(shape)
    g0 = g0 * (blocked == 0)
    ss = slab.SlabSet(shape, bc=bc, slabs_per_rank=spr, lattice_factory=FakeLattice, max_steps=n)
    lo, hi = ss.rank_range()
    Z = ss.set_site_params(dF[lo:hi], blocked[lo:hi], np.zeros(shape)[lo:hi], g0[lo:hi].astype(np.complex128), local=True)
    ss.step(n)
    f_ref, G_ref = _reference(dF, blocked, g0, bc[0] == 0, n)
    assert abs(Z - np.exp(-dF)[blocked == 0].sum()) < 1e-9        # Eq. 2 normalises over the whole lattice
    assert np.max(np.abs(ss.fid().real - G_ref)) < 1e-13
    assert np.max(np.abs(ss.gather_field(0) - f_ref)) < 1e-12
    with pytest.raises(ValueError):
        ss.set_site_params(dF, blocked, np.zeros(shape), local=True) if ss.world > 1 else ss.local_part(dF[:-1], ss.owned[0])
    return ss


def _worker(rank, world, port, q):
    import torch.distributed as dist

    dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
    try:
        for bc in ((0, 0, 0), (1, 0, 0)):
            for spr in (1, 2):
                ss = _run((11, 3, 4), bc, spr, 9)
                assert ss.world == 2 and ss.n_slabs == 2 * spr and ss.owned == list(range(rank * spr, (rank + 1) * spr))
                _run_local((11, 3, 4), bc, spr, 9)
        q.put((rank, "ok"))
    except Exception as exc:  # report instead of hanging the other rank
        q.put((rank, repr(exc)))
    dist.barrier()
    dist.destroy_process_group()


def test_two_ranks_exchange_planes_and_add_series():
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 31500 + os.getpid() % 2000
    procs = [ctx.Process(target=_worker, args=(r, 2, port, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=180) for _ in procs)
    for p in procs:
        p.join(60)
        assert p.exitcode == 0
    assert got == [(0, "ok"), (1, "ok")], got


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 0, 0)])
@pytest.mark.parametrize("spr", [1, 2, 5])
def test_single_process_slabs(bc, spr):
    _run((11, 3, 4), bc, spr, 9)
    _run_local((11, 3, 4), bc, spr, 9)


def test_ranges_neighbours_and_message_order():
    assert [slab.slab_range(10, 4, s) for s in range(4)] == [(0, 3), (3, 6), (6, 8), (8, 10)]
    assert slab.neighbour(4, 0, 0, True) == 3 and slab.neighbour(4, 0, 0, False) is None
    assert slab.neighbour(4, 3, 1, True) == 0 and slab.neighbour(4, 3, 1, False) is None
    assert slab.neighbour(1, 0, 0, True) == 0   # one periodic slab is its own neighbour
    msgs = slab.messages(2, True)
    # a periodic ring of two: each slab's two planes go to the other one, to opposite ghosts
    assert msgs == [(0, 0, 1, 1), (0, 1, 1, 0), (1, 0, 0, 1), (1, 1, 0, 0)]
    assert slab.messages(3, False) == [(0, 1, 1, 0), (1, 0, 0, 1), (1, 1, 2, 0), (2, 0, 1, 1)]
    with pytest.raises(ValueError):
        slab.SlabSet((2, 3, 3), slabs_per_rank=3, lattice_factory=FakeLattice)
