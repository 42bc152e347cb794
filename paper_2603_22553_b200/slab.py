"""One lattice split into x-slabs over several GPUs (include/lpc.h "Slabs").

The lattice is cut along x into ``n_slabs = world * slabs_per_rank`` contiguous ranges; slab ``s`` lives on rank
``s // slabs_per_rank``.  Every slab is an ordinary ``liblpc`` lattice created with ``bc[0] = LPC_BC_HALO``: the
library leaves its two x ghost planes alone and this module fills them after every step with the neighbour's
outermost owned plane -- a device copy when the neighbour lives in the same process, ``torch.distributed``
send/recv (NCCL over NVLink between GPUs) otherwise.  That plane exchange is the only data-path communication per
step.  G[n] and Z_d[m] stay per-slab partial series and are added once, when they are read.

This module holds routing only; every number is computed by the kernels behind the C ABI.  The same driver code
runs with all slabs in one process (how the GPU tests check it against the unsplit lattice on one B200) and with
one process per GPU.
"""
from __future__ import annotations

import numpy as np

LPC_BC_HALO = 2
HALO_PARAMS, HALO_STATE = 0, 1
HALO_STATE2, HALO_PARAMS2, HALO_PHASE2 = 4, 5, 6   # two planes per face: slabs that take two time steps per sweep
SEND, RECV = 0, 1


def slab_range(nx: int, n_slabs: int, s: int):
    """Planes [lo, hi) of slab s: contiguous, sizes differ by at most one."""
    base, rem = divmod(int(nx), int(n_slabs))
    lo = s * base + min(s, rem)
    return lo, lo + base + (1 if s < rem else 0)


def neighbour(n_slabs: int, s: int, side: int, periodic: bool):
    """Slab beyond the low (side 0) or high (side 1) face of slab s; None at a wall of the whole lattice."""
    t = s - 1 if side == 0 else s + 1
    if 0 <= t < n_slabs:
        return t
    return (t % n_slabs) if periodic else None


def messages(n_slabs: int, periodic: bool):
    """Every plane transfer of one exchange as (src_slab, src_side, dst_slab, dst_side), in the one global order
    both ends of a pair of ranks use to match their sends and receives."""
    out = []
    for s in range(n_slabs):
        for side in (0, 1):
            t = neighbour(n_slabs, s, side, periodic)
            if t is not None:
                out.append((s, side, t, 1 - side))   # my low plane is the neighbour's high ghost and vice versa
    return out


class SlabSet:
    """The slabs this process owns, and the routing between all of them.

    lattice_factory(shape, bc, **cfg) builds one slab (default: ``paper_2603_22553_b200.Lattice``); it must offer
    partition_sum / set_partition_sum / set_site_params / halo_planes / slab_finish / step / fid / moments /
    field / set_state.  ``group`` is a torch.distributed process group (None: the default group if
    torch.distributed is initialised, else a single process).
    """

    def __init__(self, global_shape, bc=(0, 0, 0), slabs_per_rank=1, lattice_factory=None, group=None, time_block=0, **cfg):
        self.dist = None
        self.rank, self.world = 0, 1
        try:
            import torch.distributed as dist

            if dist.is_available() and dist.is_initialized():
                self.dist = dist
                self.group = group
                self.rank, self.world = dist.get_rank(group), dist.get_world_size(group)
        except ImportError:  # pragma: no cover
            pass
        self.global_shape = tuple(int(v) for v in global_shape)
        self.bc = tuple(int(b) for b in bc)
        if self.bc[0] not in (0, 1):
            raise ValueError("bc[0] of the whole lattice must be 0 (periodic) or 1 (reflective)")
        self.spr = int(slabs_per_rank)
        self.n_slabs = self.world * self.spr
        if self.n_slabs > self.global_shape[0]:
            raise ValueError("more slabs than x planes")
        self.periodic = self.bc[0] == 0
        self.owned = list(range(self.rank * self.spr, (self.rank + 1) * self.spr))
        if lattice_factory is None:
            from . import Lattice as lattice_factory
        self.ranges = {s: slab_range(self.global_shape[0], self.n_slabs, s) for s in range(self.n_slabs)}
        self.lat = {}
        for s in self.owned:
            lo, hi = self.ranges[s]
            self.lat[s] = lattice_factory((hi - lo,) + self.global_shape[1:], bc=(LPC_BC_HALO, self.bc[1], self.bc[2]), **cfg)
        self.steps = 0
        # two time steps per sweep (include/lpc.h "Slabs"; on request, time_block=2 -> LPC_OPT_TIME_BLOCK): every slab of
        # every rank must be able to, because all slabs exchange two planes per face then
        if time_block:
            for m in self.lat.values():
                if hasattr(m, "set_option"):
                    try:
                        m.set_option(1, int(time_block))   # LPC_OPT_TIME_BLOCK
                    except Exception:
                        pass                               # a slab that cannot: `can` below turns out False
        can = all(getattr(m, "time_block_steps", 1) == 2 for m in self.lat.values())
        self.two_step = bool(self._allreduce_min(1.0 if can else 0.0) > 0.5)
        self.direct = set()   # (src slab, src side) of OWNED slabs whose plane the step kernel stores into the neighbour itself
        self.direct_all = set()   # the same over the slabs of all ranks: what both ends of a message skip after a step
        self.remote_direct = False
        self.stats = {"copies": 0, "sends": 0, "recvs": 0}   # plane transfers `exchange` has issued so far
        self._peer_maps = {}       # IPC handle -> base address here of another rank's workspace allocation
        self._fence = None         # the one-element tensor of the per-step fence

    def enable_direct_stores(self, remote=False):
        """Let the step kernel write a slab's outermost planes straight into the neighbours' ghost planes -- the
        transfer rides on the sweep's own stores and `exchange` has nothing left to do for those faces.  Neighbours in
        this process: plain device addresses.  remote=True: neighbours on other ranks of the SAME NODE as well -- every
        rank exports its workspace allocation as a CUDA IPC handle (lpc_ipc_export), the ranks swap handles and
        ghost-plane offsets once (all_gather_object) and map each other's workspaces (lpc_ipc_open); after every step a
        fence (`_step_fence`) makes sure all ranks' sweeps have finished before any rank starts the next one.  Faces
        that are not direct keep the copy / send-recv.  Call after set_site_params.  Returns the direct faces here."""
        self.direct = set()
        self._close_peers()
        self.two_step = False   # the direct stores ride on the one-step sweep
        remote = bool(remote) and self.dist is not None and self.world > 1
        table = {}
        if remote:
            # CUDA IPC handles open on the same node only, and the fence and the plane copies are ordered by torch's current
            # stream: every rank must sit on one host and every slab must run on that stream, else the faces between ranks
            # keep their send / recv
            import socket

            ok = all(self._on_current_stream(m) for m in self.lat.values())
            names = [None] * self.world
            self.dist.all_gather_object(names, (socket.gethostname(), ok), group=self.group)
            remote = len({n for n, _ in names}) == 1 and all(o for _, o in names)
        if remote:
            # every rank publishes, per owned slab, the CUDA IPC handle of its workspace allocation and where the ghost
            # planes lie in it (lpc_ipc_export behind the C ABI); a rank maps each remote allocation once (lpc_ipc_open)
            mine = {s: self.lat[s].ipc_export() for s in self.owned}
            gathered = [None] * self.world
            self.dist.all_gather_object(gathered, mine, group=self.group)
            for part in gathered:
                table.update(part)
        for s in self.owned:
            peers = [None, None]
            for side in (0, 1):
                t = neighbour(self.n_slabs, s, side, self.periodic)
                if t is None:
                    continue
                if self.owner(t) == self.rank:
                    if hasattr(self.lat[t], "ghost_plane_addresses"):
                        peers[side] = self.lat[t].ghost_plane_addresses(1 - side)
                        self.direct.add((s, side))
                elif remote:
                    handle, ws_off, ghosts = table[t]
                    if handle not in self._peer_maps:
                        self._peer_maps[handle] = self._ipc_open(handle)      # maps the other rank's allocation here
                    base = self._peer_maps[handle] + ws_off
                    off0, off1, stride = ghosts[1 - side]
                    peers[side] = (base + off0, base + off1, stride)
                    self.direct.add((s, side))
            self.lat[s].set_halo_peers(lo=peers[0], hi=peers[1])
        self.remote_direct = remote
        # the receiving end of a direct face must skip its receive as well: every rank learns all ranks' direct faces
        self.direct_all = set(self.direct)
        if self.dist is not None and self.world > 1:
            gathered = [None] * self.world
            self.dist.all_gather_object(gathered, sorted(self.direct), group=self.group)
            for part in gathered:
                self.direct_all.update(tuple(f) for f in part)
        return len(self.direct)

    @staticmethod
    def _on_current_stream(m):
        """True if the slab's sweeps are ordered with torch's current stream (what the copies and the fence use)."""
        st = getattr(m, "stream", None)
        if st is None or not hasattr(st, "cuda_stream"):
            return True
        import torch

        return st.cuda_stream == torch.cuda.current_stream(getattr(m, "device", None)).cuda_stream

    def _ipc_open(self, handle):
        from . import lpc_ipc_open

        return lpc_ipc_open(handle)

    def _close_peers(self):
        if self._peer_maps:
            from . import lpc_ipc_close

            for base in self._peer_maps.values():
                lpc_ipc_close(base)
        self._peer_maps = {}

    def _step_fence(self):
        """All ranks' sweeps of this step have finished (their direct stores have landed) before anyone goes on."""
        import torch

        if self.dist.get_backend(self.group) == "nccl":
            # a one-element all-reduce on the compute stream orders the ranks' streams without stopping the host
            # (the slabs run on torch's current stream: checked when the direct stores were enabled)
            if self._fence is None:
                self._fence = torch.zeros(1, device="cuda")
            self.dist.all_reduce(self._fence, group=self.group)
        else:
            torch.cuda.synchronize()
            self.dist.barrier(group=self.group)

    def owner(self, s: int) -> int:
        return s // self.spr

    def rank_range(self):
        """Planes [lo, hi) of the whole lattice that this rank's slabs cover (they are contiguous)."""
        return self.ranges[self.owned[0]][0], self.ranges[self.owned[-1]][1]

    def local_part(self, arr, s, local=False):
        """The planes of slab s of an array over the whole lattice -- or, with local=True, of an array that holds this
        rank's planes only (`rank_range`); leading axes before x are kept."""
        lo, hi = self.ranges[s]
        a = np.asarray(arr)
        if local:
            r0, r1 = self.rank_range()
            if a.shape[-3] != r1 - r0:
                raise ValueError(f"a local array must hold this rank's {r1 - r0} planes, got {a.shape[-3]}")
            lo, hi = lo - r0, hi - r0
        elif a.shape[-3] != self.global_shape[0]:
            raise ValueError(f"a global array must hold all {self.global_shape[0]} planes, got {a.shape[-3]}")
        lead = a.ndim - 3
        return np.ascontiguousarray(a[(slice(None),) * lead + (slice(lo, hi),)])

    # ---- reductions over all slabs -------------------------------------------------------------
    def _allreduce(self, x: np.ndarray) -> np.ndarray:
        """Sum over ranks of a float64 / complex128 host array (plumbing: the series are added once per read)."""
        if self.dist is None or self.world == 1:
            return x
        import torch

        t = torch.from_numpy(np.ascontiguousarray(x).view(np.float64).copy())
        if self.dist.get_backend(self.group) == "nccl":
            t = t.cuda()
        self.dist.all_reduce(t, op=self.dist.ReduceOp.SUM, group=self.group)
        return t.cpu().numpy().view(x.dtype).reshape(x.shape)

    # ---- the plane exchange -------------------------------------------------------------------
    def exchange(self, which, after_step=False):
        """Fill every x ghost plane of `which` (HALO_PARAMS or HALO_STATE) from the neighbour's outermost owned
        plane.  Same process: one device copy per plane.  Other rank: one send / recv per channel plane, all of one
        exchange batched into a single group; both ends enumerate `messages()` in the same order, which is what
        matches the two planes a pair of ranks swaps in each direction on a periodic ring of two."""
        ops, keep, landed = [], [], []
        for src, sside, dst, dside in messages(self.n_slabs, self.periodic):
            so, do = self.owner(src), self.owner(dst)
            if so != self.rank and do != self.rank:
                continue
            if after_step and (src, sside) in self.direct_all:
                continue   # the sweep stored this plane into the neighbour's ghost plane already (both ends skip it)
            if so == self.rank and do == self.rank:
                self.lat[dst].halo_planes(which, dside, RECV).copy_(self.lat[src].halo_planes(which, sside, SEND))
                self.stats["copies"] += 1
                continue
            # gloo cannot send device tensors: stage them through the host (tests; NCCL sends the planes in place)
            via_host = self.dist.get_backend(self.group) != "nccl"
            if so == self.rank:
                planes = self.lat[src].halo_planes(which, sside, SEND)
                wire = planes.cpu() if via_host and planes.is_cuda else planes
                for c in range(planes.shape[0]):
                    ops.append(self.dist.P2POp(self.dist.isend, wire[c], self._global_rank(do), group=self.group))
                self.stats["sends"] += 1
            else:
                planes = self.lat[dst].halo_planes(which, dside, RECV)
                wire = planes.cpu() if via_host and planes.is_cuda else planes
                for c in range(planes.shape[0]):
                    ops.append(self.dist.P2POp(self.dist.irecv, wire[c], self._global_rank(so), group=self.group))
                self.stats["recvs"] += 1
                if wire is not planes:
                    landed.append((planes, wire))
            keep.append(wire)
        if ops:
            for req in self.dist.batch_isend_irecv(ops):
                req.wait()
        for planes, wire in landed:
            planes.copy_(wire)

    def _global_rank(self, r):
        return r if self.group is None else self.dist.get_global_rank(self.group, r)

    # ---- the call sequence of include/lpc.h "Slabs" ---------------------------------------------
    def set_site_params(self, dF, blocked, omega, g0=None, local=False):
        """dF, blocked, omega (and g0): host arrays over the WHOLE lattice, of which every rank cuts out its planes, or
        (local=True) over this rank's own planes only (`rank_range`) -- nothing of the other ranks' input is needed here:
        Eq. 2's normalisation travels as one scalar, the neighbours' pi as one plane."""
        parts = {s: (self.local_part(dF, s, local), self.local_part(blocked, s, local).astype(np.uint8), self.local_part(omega, s, local))
                 for s in self.owned}
        z_local = np.array([sum(self.lat[s].partition_sum(parts[s][0], parts[s][1]) for s in self.owned)], dtype=np.float64)
        Z = float(self._allreduce(z_local)[0])
        for s in self.owned:
            self.lat[s].set_partition_sum(Z)
            self.lat[s].set_site_params(*parts[s])
        # slabs that take two steps per sweep rotate their neighbours' boundary sites too: all slabs read the phase factors the
        # same way (sin alone only if every slab of every rank may, include/lpc.h lpc_reads_sin_alone)
        if self.two_step:
            mine = all(getattr(self.lat[s], "reads_sin_alone", True) for s in self.owned)
            if self._allreduce_min(1.0 if mine else 0.0) < 0.5:
                for s in self.owned:
                    if hasattr(self.lat[s], "set_option"):
                        self.lat[s].set_option(6, 1)   # LPC_OPT_FULL_PHASE
        if self.two_step:
            self.exchange(HALO_PARAMS2)
            self.exchange(HALO_PHASE2)     # the two-step sweep rotates the ring of neighbour sites as well
        else:
            self.exchange(HALO_PARAMS)
        for s in self.owned:
            self.lat[s].slab_finish()
        if g0 is not None:
            for s in self.owned:
                self.lat[s].set_state(0, self.local_part(g0, s, local))
        self.exchange(self.state_set)
        self.steps = 0
        return Z

    @property
    def state_set(self):
        """Which planes of the state an exchange moves: two per face for slabs that take two steps per sweep."""
        return HALO_STATE2 if self.two_step else HALO_STATE

    def step(self, n=1):
        """n time steps: per sweep (one step, or two on slabs that can) one launch per slab, then the plane exchange."""
        n = int(n)
        while n > 0:
            k = 2 if (self.two_step and n >= 2) else 1
            for s in self.owned:
                self.lat[s].step(k)
            self.exchange(self.state_set, after_step=True)
            if self.remote_direct:
                self._step_fence()
            self.steps += k
            n -= k

    def _allreduce_min(self, v: float) -> float:
        return -self._allreduce_max(-v)

    def _allreduce_max(self, v: float) -> float:
        if self.dist is None or self.world == 1:
            return v
        import torch

        t = torch.tensor([v], dtype=torch.float64)
        if self.dist.get_backend(self.group) == "nccl":
            t = t.cuda()
        self.dist.all_reduce(t, op=self.dist.ReduceOp.MAX, group=self.group)
        return float(t.item())

    def set_state(self, which, arr):
        """arr over the WHOLE lattice (e.g. an initial density for the equilibration loop)."""
        for s in self.owned:
            self.lat[s].set_state(which, self.local_part(arr, s))
        self.exchange(self.state_set)

    def equilibrate(self, threshold, max_iters):
        """The equilibration loop over all slabs: one sweep per slab, the plane exchange, and the
        largest per-site change of all slabs compared with the threshold.  Returns (sweeps done, last delta)."""
        done, delta = 0, 0.0
        while done < max_iters:
            delta = 0.0
            for s in self.owned:
                _, d = self.lat[s].equilibrate(0.0, 1, 1)
                delta = max(delta, d)
            self.exchange(self.state_set)
            delta = self._allreduce_max(delta)
            done += 1
            if delta < threshold:
                break
        return done, delta

    def fid(self):
        """G[0..steps] of the whole lattice: the slabs' partial series added in slab order, then over ranks."""
        part = sum(self.lat[s].fid() for s in self.owned)
        return self._allreduce(np.asarray(part, dtype=np.complex128))

    def moments(self):
        """(Z_d[1..steps+1], D_d) of the whole lattice; both are linear in the per-slab sums."""
        zs, ds = zip(*(self.lat[s].moments() for s in self.owned))
        z = self._allreduce(np.asarray(sum(zs), dtype=np.float64))
        d = self._allreduce(np.asarray(sum(ds), dtype=np.float64))
        return z, d

    def field(self, which):
        """Owned planes of a field, as {slab: array}; use ``gather_field`` for the whole lattice on every rank."""
        return {s: self.lat[s].field(which) for s in self.owned}

    def gather_field(self, which, dtype=np.float64):
        out = np.zeros(self.global_shape, dtype=dtype)
        for s, a in self.field(which).items():
            lo, hi = self.ranges[s]
            out[lo:hi] = a
        return self._allreduce(out)
