"""Slab decomposition across PROCESSES with direct halo stores (paper_2603_22553_b200/slab.py):
two ranks (gloo for the handshake) each own half of the lattice; every rank maps the other's workspace through a CUDA
IPC handle and its step kernel stores its outermost planes straight into the other rank's ghost planes.  The box has
one GPU, so both ranks use cuda:0 -- the kernels of the two ranks never wait on one another (the per-step fence is a
host barrier), this checks the plumbing and the result, not a speed."""
import os
import sys

import numpy as np
import pytest
import torch.multiprocessing as mp

pytestmark = pytest.mark.gpu
ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _worker(rank, world, port, bc, q):
    try:
        import importlib.util

        import torch
        import torch.distributed as dist

        sys.path.insert(0, ROOT)
        import lpc_inputs
        import paper_2603_22553_b200 as lpc
        from paper_2603_22553_b200 import slab

        torch.cuda.set_device(0)
        dist.init_process_group("gloo", init_method=f"tcp://127.0.0.1:{port}", rank=rank, world_size=world)
        n = 25
        lat = lpc_inputs.random_small((26, 18, 70), bc=bc, p_block=0.25, alpha=0.9, seed=85, n_steps=n, n_moments=3)
        ss = slab.SlabSet(lat.shape, bc=lat.bc, slabs_per_rank=1, n_moments=3, dt=lat.dt, a=lat.a, alpha=lat.alpha, max_steps=n)
        ss.set_site_params(lat.dF, lat.blocked, lat.omega)
        n_direct = ss.enable_direct_stores(remote=True)
        before = dict(ss.stats)
        ss.step(n)            # the real driver: sweep, exchange (which must find nothing left to do), fence
        posted = sum(ss.stats[k] - before[k] for k in before)
        G = ss.fid()
        g = ss.gather_field(lpc.LPC_FIELD_G, dtype=np.complex128)
        Z, D = ss.moments()
        if rank == 0:
            spec = importlib.util.spec_from_file_location("lpc_oracle", os.path.join(ROOT, "oracle", "lpc_oracle.py"))
            orc_mod = importlib.util.module_from_spec(spec)
            spec.loader.exec_module(orc_mod)
            orc = orc_mod.Oracle.from_lattice(lat, n_moments=3, max_steps=n)
            orc.step(n)
            G_o, sabs = orc.fid(with_scale=True)
            pi, opn = orc.pi(), lat.blocked == 0
            Z_o, _ = orc.moments()
            q.put((rank, n_direct, posted, float(np.max(np.abs(G - G_o) / sabs)), float(np.max(np.abs(g - orc.g())[opn] / pi[opn])),
                   float(np.max(np.abs(Z - Z_o) / np.abs(Z_o[:, :1])))))
        else:
            q.put((rank, n_direct, posted, 0.0, 0.0, 0.0))
        dist.barrier()
        dist.destroy_process_group()
    except Exception as exc:  # report instead of hanging the other rank
        import traceback

        q.put((rank, -1, -1, repr(exc) + traceback.format_exc(), 0.0, 0.0))


@pytest.mark.parametrize("bc", [(0, 0, 0), (1, 0, 0)])
def test_two_processes_store_into_each_others_ghost_planes(bc):
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    port = 33500 + os.getpid() % 2000 + (7 if bc[0] else 0)
    procs = [ctx.Process(target=_worker, args=(r, 2, port, bc, q)) for r in range(2)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=300) for _ in procs)
    for p in procs:
        p.join(120)
    for rank, n_direct, n_sent, eG, eg, eZ in got:
        assert n_direct >= 0, eG
        # a periodic ring of two: both faces of a rank's slab face the other rank; with walls only one does
        assert n_direct == (2 if bc[0] == 0 else 1)
        assert n_sent == 0           # the unpatched step() posted no copy, send or receive after any of the 25 steps
        assert eG <= 1e-9 and eg <= 1e-10 and eZ <= 1e-9
