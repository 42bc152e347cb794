"""paper_2603_22553_b200 -- thin Python binding of liblpc.so (include/lpc.h).

Argument marshalling only: every step of the LPC3D hot path (site-parameter
precompute, fused propagate + phase-rotate + FID reduce, moment propagation)
runs in the CUDA kernels of ``csrc/`` behind the C ABI.  PyTorch is used for
device memory (the workspace) and streams, nothing else.

There is no CPU fallback.  If ``liblpc.so`` has not been built
(``python -m paper_2603_22553_b200.build``) the first call raises ImportError.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.path.join(_HERE, "liblpc.so")

LPC_OK, LPC_EINVAL, LPC_ESTATE, LPC_ENOMEM, LPC_ECUDA = 0, -1, -2, -3, -4
LPC_FIELD_G, LPC_FIELD_PI, LPC_FIELD_PX, LPC_FIELD_PY, LPC_FIELD_PZ, LPC_FIELD_RHO = range(6)
LPC_BC_HALO = 2
LPC_HALO_PARAMS, LPC_HALO_STATE, LPC_HALO_STATE0, LPC_HALO_STATE1 = 0, 1, 2, 3
LPC_HALO_STATE2, LPC_HALO_PARAMS2, LPC_HALO_PHASE2 = 4, 5, 6
LPC_HALO_SEND, LPC_HALO_RECV = 0, 1
LPC_KERNEL_AUTO, LPC_KERNEL_DIRECT, LPC_KERNEL_TMA, LPC_KERNEL_PERSIST = range(4)
LPC_OPT_TIME_BLOCK, LPC_OPT_X_CHUNK, LPC_OPT_X_CHUNK2, LPC_OPT_PERSIST_MAX_MB, LPC_OPT_REGION_FUSION, LPC_OPT_FULL_PHASE, LPC_OPT_SERIAL_LAUNCH = 1, 2, 3, 4, 5, 6, 7

EXPORTS = (
    "lpc_workspace_bytes", "lpc_create_lattice", "lpc_set_site_params", "lpc_set_link_mobility", "lpc_step_n", "lpc_read_fid",
    "lpc_moments", "lpc_read_field", "lpc_set_state", "lpc_equilibrate", "lpc_seed_from_density", "lpc_set_regions", "lpc_read_fid_region", "lpc_moments_region", "lpc_spectrum", "lpc_set_kernel",
    "lpc_set_option", "lpc_time_block_steps", "lpc_reads_sin_alone", "lpc_ipc_export", "lpc_ipc_open", "lpc_ipc_close", "lpc_steps_done", "lpc_partition_sum", "lpc_set_partition_sum", "lpc_halo_view", "lpc_set_halo_peers", "lpc_slab_finish",
    "lpc_launch_count", "lpc_bytes_per_site_step", "lpc_fid_sample_noalloc", "lpc_sync_steps", "lpc_destroy", "lpc_last_error",
)


class LpcError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"liblpc error {code}: {msg}")
        self.code = code


class lpc_config(C.Structure):
    _fields_ = [
        ("nx", C.c_int32), ("ny", C.c_int32), ("nz", C.c_int32), ("bc", C.c_int32 * 3),
        ("precision", C.c_int32), ("n_moments", C.c_int32), ("n_density", C.c_int32), ("n_regions", C.c_int32),
        ("link_mobility", C.c_int32),
        ("dt", C.c_double), ("a", C.c_double), ("alpha", C.c_double),
        ("max_steps", C.c_int64), ("stream", C.c_void_p),
    ]


_lib_handle = None


def _load():
    """Load liblpc.so on first use; there is no fallback if it is missing."""
    global _lib_handle
    if _lib_handle is not None:
        return _lib_handle
    if not os.path.exists(LIB_PATH):
        raise ImportError(
            f"{LIB_PATH} is missing: build the CUDA library with `python -m paper_2603_22553_b200.build` "
            "(there is no CPU fallback)")
    lib = C.CDLL(LIB_PATH)
    lib.lpc_workspace_bytes.argtypes = [C.POINTER(lpc_config), C.POINTER(C.c_size_t)]
    lib.lpc_create_lattice.argtypes = [C.POINTER(lpc_config), C.c_void_p, C.c_size_t, C.POINTER(C.c_void_p)]
    lib.lpc_set_site_params.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    lib.lpc_set_link_mobility.argtypes = [C.c_void_p, C.c_void_p]
    lib.lpc_partition_sum.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.POINTER(C.c_double)]
    lib.lpc_set_partition_sum.argtypes = [C.c_void_p, C.c_double]
    lib.lpc_halo_view.argtypes = [C.c_void_p, C.c_int32, C.c_int32, C.c_int32, C.POINTER(C.c_void_p), C.POINTER(C.c_size_t),
                                  C.POINTER(C.c_size_t), C.POINTER(C.c_int32)]
    lib.lpc_slab_finish.argtypes = [C.c_void_p]
    lib.lpc_ipc_export.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_size_t)]
    lib.lpc_ipc_open.argtypes = [C.c_void_p, C.POINTER(C.c_void_p)]
    lib.lpc_ipc_close.argtypes = [C.c_void_p]
    lib.lpc_set_halo_peers.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_size_t, C.c_void_p, C.c_void_p, C.c_size_t]
    lib.lpc_step_n.argtypes = [C.c_void_p, C.c_int64]
    lib.lpc_read_fid.argtypes = [C.c_void_p, C.c_int64, C.c_int64, C.c_void_p]
    lib.lpc_moments.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    lib.lpc_read_field.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    lib.lpc_set_state.argtypes = [C.c_void_p, C.c_int32, C.c_void_p]
    lib.lpc_set_kernel.argtypes = [C.c_void_p, C.c_int32]
    lib.lpc_set_option.argtypes = [C.c_void_p, C.c_int32, C.c_int64]
    lib.lpc_equilibrate.argtypes = [C.c_void_p, C.c_double, C.c_int64, C.c_int64, C.POINTER(C.c_int64), C.POINTER(C.c_double)]
    lib.lpc_seed_from_density.argtypes = [C.c_void_p]
    lib.lpc_set_regions.argtypes = [C.c_void_p, C.c_void_p]
    lib.lpc_read_fid_region.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_int64, C.c_void_p]
    lib.lpc_moments_region.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_void_p, C.c_void_p]
    lib.lpc_spectrum.argtypes = [C.c_void_p, C.c_int32, C.c_int64, C.c_double, C.c_double, C.c_int64, C.c_double, C.c_void_p]
    lib.lpc_sync_steps.argtypes = [C.c_void_p, C.POINTER(C.c_int64)]
    lib.lpc_fid_sample_noalloc.argtypes = [C.c_void_p, C.c_int64, C.c_void_p, C.c_void_p]
    lib.lpc_time_block_steps.argtypes = [C.c_void_p]
    lib.lpc_time_block_steps.restype = C.c_int32
    lib.lpc_reads_sin_alone.argtypes = [C.c_void_p]
    lib.lpc_reads_sin_alone.restype = C.c_int32
    lib.lpc_steps_done.argtypes = [C.c_void_p]
    lib.lpc_steps_done.restype = C.c_int64
    lib.lpc_launch_count.argtypes = [C.c_void_p]
    lib.lpc_launch_count.restype = C.c_int64
    lib.lpc_bytes_per_site_step.argtypes = [C.c_void_p]
    lib.lpc_bytes_per_site_step.restype = C.c_double
    lib.lpc_destroy.argtypes = [C.c_void_p]
    lib.lpc_destroy.restype = None
    lib.lpc_last_error.restype = C.c_char_p
    _lib_handle = lib
    return lib


class _LazyLib:
    def __getattr__(self, name):
        return getattr(_load(), name)


_lib = _LazyLib()


def lpc_last_error() -> str:
    return _lib.lpc_last_error().decode()


def _check(rc):
    if rc != LPC_OK:
        raise LpcError(rc, lpc_last_error())


def _ptr(x, dtype=None, count=None):
    """Address of a numpy array (host) or torch tensor (host or device); keeps nothing alive."""
    if x is None:
        return None
    if isinstance(x, np.ndarray):
        if dtype is not None and x.dtype != dtype:
            raise TypeError(f"expected {dtype}, got {x.dtype}")
        if not x.flags.c_contiguous:
            raise ValueError("array must be C-contiguous")
        if count is not None and x.size != count:
            raise ValueError(f"expected {count} elements, got {x.size}")
        return C.c_void_p(x.ctypes.data)
    if hasattr(x, "data_ptr"):
        if not x.is_contiguous():
            raise ValueError("tensor must be contiguous")
        if count is not None and x.numel() != count:
            raise ValueError(f"expected {count} elements, got {x.numel()}")
        return C.c_void_p(x.data_ptr())
    raise TypeError(f"cannot take the address of {type(x)}")


def make_config(nx, ny, nz, bc=(0, 0, 0), precision=0, n_moments=0, n_density=0, dt=5e-6, a=1.0, alpha=1.0,
                max_steps=0, stream=None, n_regions=0, link_mobility=0) -> lpc_config:
    return lpc_config(int(nx), int(ny), int(nz), (C.c_int32 * 3)(*[int(b) for b in bc]), int(precision),
                      int(n_moments), int(n_density), int(n_regions), int(link_mobility), float(dt), float(a), float(alpha), int(max_steps),
                      C.c_void_p(stream) if stream else None)


def lpc_workspace_bytes(cfg: lpc_config) -> int:
    out = C.c_size_t(0)
    _check(_lib.lpc_workspace_bytes(C.byref(cfg), C.byref(out)))
    return int(out.value)


def lpc_create_lattice(cfg: lpc_config, workspace, nbytes=None):
    """workspace: torch uint8 CUDA tensor (or a raw device address with nbytes)."""
    handle = C.c_void_p()
    if hasattr(workspace, "data_ptr"):
        addr, nbytes = workspace.data_ptr(), workspace.numel() * workspace.element_size()
    else:
        addr = int(workspace)
    _check(_lib.lpc_create_lattice(C.byref(cfg), C.c_void_p(addr), C.c_size_t(int(nbytes)), C.byref(handle)))
    return handle


def lpc_set_site_params(handle, dF, blocked, omega, g0=None):
    _check(_lib.lpc_set_site_params(handle, _ptr(dF), _ptr(blocked), _ptr(omega), _ptr(g0)))


def lpc_set_link_mobility(handle, alpha_link):
    """alpha_link: [3, nx, ny, nz] float64 (host numpy or CUDA tensor), or None to remove the factors."""
    _check(_lib.lpc_set_link_mobility(handle, _ptr(alpha_link)))


def lpc_partition_sum(handle, dF, blocked) -> float:
    out = C.c_double(0.0)
    _check(_lib.lpc_partition_sum(handle, _ptr(dF), _ptr(blocked), C.byref(out)))
    return float(out.value)


def lpc_set_partition_sum(handle, Z):
    _check(_lib.lpc_set_partition_sum(handle, float(Z)))


def lpc_halo_view(handle, which, side, role):
    """(device address of channel 0's plane, bytes per plane, byte stride between channels, channels)."""
    ptr, nb, st, nc = C.c_void_p(), C.c_size_t(), C.c_size_t(), C.c_int32()
    _check(_lib.lpc_halo_view(handle, int(which), int(side), int(role), C.byref(ptr), C.byref(nb), C.byref(st), C.byref(nc)))
    return int(ptr.value), int(nb.value), int(st.value), int(nc.value)


def lpc_set_halo_peers(handle, lo=None, hi=None):
    """lo / hi: None or (address in buffer 0, address in buffer 1, channel stride in bytes) of the neighbour's ghost plane."""
    lo = lo or (None, None, 0)
    hi = hi or (None, None, 0)
    _check(_lib.lpc_set_halo_peers(handle, C.c_void_p(lo[0]), C.c_void_p(lo[1]), C.c_size_t(lo[2]), C.c_void_p(hi[0]), C.c_void_p(hi[1]),
                                   C.c_size_t(hi[2])))


def lpc_ipc_export(handle):
    """(64-byte CUDA IPC handle of the allocation the workspace lies in, byte offset of the workspace inside it)."""
    buf = C.create_string_buffer(64)
    off = C.c_size_t()
    _check(_lib.lpc_ipc_export(handle, buf, C.byref(off)))
    return bytes(buf.raw), int(off.value)


def lpc_ipc_open(handle_bytes) -> int:
    """Map an exported allocation into this process; returns its base device address here."""
    buf = C.create_string_buffer(bytes(handle_bytes), 64)
    base = C.c_void_p()
    _check(_lib.lpc_ipc_open(buf, C.byref(base)))
    return int(base.value)


def lpc_ipc_close(base):
    _check(_lib.lpc_ipc_close(C.c_void_p(int(base))))


def lpc_slab_finish(handle):
    _check(_lib.lpc_slab_finish(handle))


def lpc_step_n(handle, n):
    _check(_lib.lpc_step_n(handle, int(n)))


def lpc_read_fid(handle, first=0, count=None):
    if count is None:
        count = int(_lib.lpc_steps_done(handle)) + 1 - first
    out = np.empty(count, dtype=np.complex128)
    _check(_lib.lpc_read_fid(handle, int(first), int(count), C.c_void_p(out.ctypes.data)))
    return out


def lpc_moments(handle, count=None):
    """(vacf[3, count] with vacf[d, m-1] = Z_d[m], D[3])."""
    if count is None:
        count = int(_lib.lpc_steps_done(handle)) + 1
    vacf = np.empty((3, count), dtype=np.float64)
    D = np.empty(3, dtype=np.float64)
    _check(_lib.lpc_moments(handle, int(count), C.c_void_p(vacf.ctypes.data), C.c_void_p(D.ctypes.data)))
    return vacf, D


def lpc_read_field(handle, which, out):
    _check(_lib.lpc_read_field(handle, int(which), _ptr(out)))
    return out


def lpc_set_state(handle, which, arr):
    _check(_lib.lpc_set_state(handle, int(which), _ptr(arr)))


def lpc_equilibrate(handle, threshold, max_iters, check_every=1):
    """(iterations done, delta of the last sweep)."""
    iters, delta = C.c_int64(0), C.c_double(0.0)
    _check(_lib.lpc_equilibrate(handle, float(threshold), int(max_iters), int(check_every), C.byref(iters), C.byref(delta)))
    return int(iters.value), float(delta.value)


def lpc_seed_from_density(handle):
    _check(_lib.lpc_seed_from_density(handle))


def lpc_set_regions(handle, region):
    _check(_lib.lpc_set_regions(handle, _ptr(region)))


def lpc_read_fid_region(handle, region, first=0, count=None):
    if count is None:
        count = int(_lib.lpc_steps_done(handle)) + 1 - first
    out = np.empty(count, dtype=np.complex128)
    _check(_lib.lpc_read_fid_region(handle, int(region), int(first), int(count), C.c_void_p(out.ctypes.data)))
    return out


def lpc_moments_region(handle, region, count=None):
    """(vacf[3, count], D[3]) of one region."""
    if count is None:
        count = int(_lib.lpc_steps_done(handle)) + 1
    vacf = np.empty((3, max(count, 0)), dtype=np.float64)
    D = np.empty(3, dtype=np.float64)
    _check(_lib.lpc_moments_region(handle, int(region), int(count), C.c_void_p(vacf.ctypes.data), C.c_void_p(D.ctypes.data)))
    return vacf, D


def lpc_spectrum(handle, f0_hz, df_hz, n_freq, lb_hz=0.0, region=-1, count=None):
    """F(f0 + k df), k = 0..n_freq-1, of G[0..count) (Eq. 9); region = -1 takes the whole lattice."""
    if count is None:
        count = int(_lib.lpc_steps_done(handle)) + 1
    out = np.empty(max(int(n_freq), 0), dtype=np.complex128)
    _check(_lib.lpc_spectrum(handle, int(region), int(count), float(f0_hz), float(df_hz), int(n_freq), float(lb_hz),
                             C.c_void_p(out.ctypes.data)))
    return out


def lpc_set_kernel(handle, which):
    _check(_lib.lpc_set_kernel(handle, int(which)))


def lpc_set_option(handle, key, value):
    _check(_lib.lpc_set_option(handle, int(key), int(value)))


LPC_NOALLOC_MAX_SITES = 1 << 28


def lpc_sync_steps(handle) -> int:
    """Read the device's step count back after CUDA graph replays of lpc_step_n (include/lpc.h "CUDA graphs")."""
    n = C.c_int64(0)
    _check(_lib.lpc_sync_steps(handle, C.byref(n)))
    return int(n.value)


def lpc_fid_sample_noalloc(g_dev_ptr, n_sites, out_dev_ptr, stream=None):
    """G = sum of n_sites complex numbers at the DEVICE address g_dev_ptr into the 2 doubles at the DEVICE address
    out_dev_ptr (Eq. 12); scratch in the library's static device array, nothing is allocated (include/lpc.h)."""
    _check(_lib.lpc_fid_sample_noalloc(C.c_void_p(int(g_dev_ptr)), int(n_sites), C.c_void_p(int(out_dev_ptr)),
                                       C.c_void_p(int(stream)) if stream else None))


def lpc_time_block_steps(handle) -> int:
    return int(_lib.lpc_time_block_steps(handle))


def lpc_reads_sin_alone(handle) -> int:
    return int(_lib.lpc_reads_sin_alone(handle))


def lpc_steps_done(handle) -> int:
    return int(_lib.lpc_steps_done(handle))


def lpc_launch_count(handle) -> int:
    return int(_lib.lpc_launch_count(handle))


def lpc_bytes_per_site_step(handle) -> float:
    return float(_lib.lpc_bytes_per_site_step(handle))


def lpc_destroy(handle):
    _lib.lpc_destroy(handle)


class Lattice:
    """Owns the torch workspace and the handle; methods forward to the C calls one to one."""

    def __init__(self, shape, bc=(0, 0, 0), precision=0, n_moments=0, n_density=0, dt=5e-6, a=1.0, alpha=1.0,
                 max_steps=0, device="cuda:0", stream=None, n_regions=0, link_mobility=0):
        import torch

        self.shape = tuple(int(v) for v in shape)
        self.n = int(np.prod(self.shape))
        self.device = torch.device(device)
        if stream is None:
            stream = torch.cuda.current_stream(self.device)
        self.stream = stream
        self.cfg = make_config(*self.shape, bc=bc, precision=precision, n_moments=n_moments, n_density=n_density,
                               dt=dt, a=a, alpha=alpha, max_steps=max_steps, stream=stream.cuda_stream, n_regions=n_regions,
                               link_mobility=link_mobility)
        self.workspace_bytes = lpc_workspace_bytes(self.cfg)
        with torch.cuda.device(self.device):
            self.workspace = torch.empty(self.workspace_bytes, dtype=torch.uint8, device=self.device)
            self.handle = lpc_create_lattice(self.cfg, self.workspace)

    @classmethod
    def from_inputs(cls, lat, precision=0, n_moments=None, n_density=0, max_steps=None, device="cuda:0", g0=None,
                    n_regions=0, link=None):
        """Build from an ``lpc_inputs.Lattice`` (host arrays) and run the precompute."""
        self = cls(lat.shape, bc=lat.bc, precision=precision,
                   n_moments=lat.n_moments if n_moments is None else n_moments, n_density=n_density,
                   dt=lat.dt, a=lat.a, alpha=lat.alpha,
                   max_steps=lat.n_steps if max_steps is None else max_steps, device=device, n_regions=n_regions,
                   link_mobility=0 if link is None else 1)
        self.set_site_params(lat.dF, lat.blocked, lat.omega, None if link is not None else g0)
        if link is not None:
            self.set_link_mobility(link)
            if g0 is not None:
                self.set_state(LPC_FIELD_G, g0)
        return self

    def close(self):
        if getattr(self, "handle", None):
            lpc_destroy(self.handle)
            self.handle = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_site_params(self, dF, blocked, omega, g0=None):
        if isinstance(dF, np.ndarray):
            dF = np.ascontiguousarray(dF, dtype=np.float64)
            blocked = np.ascontiguousarray(blocked, dtype=np.uint8)
            omega = np.ascontiguousarray(omega, dtype=np.float64)
        if isinstance(g0, np.ndarray):
            g0 = np.ascontiguousarray(g0, dtype=np.complex128)
        lpc_set_site_params(self.handle, dF, blocked, omega, g0)

    def set_link_mobility(self, alpha_link):
        if isinstance(alpha_link, np.ndarray):
            alpha_link = np.ascontiguousarray(alpha_link, dtype=np.float64)
        lpc_set_link_mobility(self.handle, alpha_link)

    def partition_sum(self, dF, blocked):
        return lpc_partition_sum(self.handle, np.ascontiguousarray(dF, dtype=np.float64), np.ascontiguousarray(blocked, dtype=np.uint8))

    def set_partition_sum(self, Z):
        lpc_set_partition_sum(self.handle, Z)

    def slab_finish(self):
        lpc_slab_finish(self.handle)

    def ghost_plane_addresses(self, side):
        """(address in state buffer 0, in buffer 1, channel stride in bytes) of this lattice's x ghost plane on `side`."""
        p0, _, st, _ = lpc_halo_view(self.handle, LPC_HALO_STATE0, side, LPC_HALO_RECV)
        p1, _, _, _ = lpc_halo_view(self.handle, LPC_HALO_STATE1, side, LPC_HALO_RECV)
        return p0, p1, st

    def ipc_export(self):
        """What another process needs to store into this lattice's ghost planes: the IPC handle of the workspace's
        allocation, the workspace's offset in it, and per side the ghost-plane offsets (buffer 0, buffer 1) inside the
        workspace plus the channel stride."""
        handle, off = lpc_ipc_export(self.handle)
        base = self.workspace.data_ptr()
        ghosts = []
        for side in (0, 1):
            p0, p1, st = self.ghost_plane_addresses(side)
            ghosts.append((p0 - base, p1 - base, st))
        return handle, off, ghosts

    def set_halo_peers(self, lo=None, hi=None):
        lpc_set_halo_peers(self.handle, lo, hi)

    def halo_planes(self, which, side, role):
        """The halo plane(s) as a [channels, plane_elements] strided view of the workspace tensor (no copy)."""
        import torch

        ptr, nb, st, nc = lpc_halo_view(self.handle, which, side, role)
        off = ptr - self.workspace.data_ptr()
        esz = 4 if self.cfg.precision else 8
        flat = self.workspace.view(torch.float32 if self.cfg.precision else torch.float64)
        return flat.as_strided((nc, nb // esz), (st // esz, 1), off // esz)

    def step(self, n=1):
        lpc_step_n(self.handle, n)

    def fid(self, first=0, count=None):
        return lpc_read_fid(self.handle, first, count)

    def moments(self, count=None):
        return lpc_moments(self.handle, count)

    def field(self, which):
        out = np.empty(self.shape, dtype=np.complex128 if which == LPC_FIELD_G else np.float64)
        return lpc_read_field(self.handle, which, out)

    def set_state(self, which, arr):
        arr = np.ascontiguousarray(arr, dtype=np.complex128 if which == LPC_FIELD_G else np.float64)
        lpc_set_state(self.handle, which, arr)

    def equilibrate(self, threshold, max_iters, check_every=1):
        return lpc_equilibrate(self.handle, threshold, max_iters, check_every)

    def seed_from_density(self):
        lpc_seed_from_density(self.handle)

    def set_regions(self, region):
        if isinstance(region, np.ndarray):
            region = np.ascontiguousarray(region, dtype=np.uint8)
        lpc_set_regions(self.handle, region)

    def fid_region(self, region, first=0, count=None):
        return lpc_read_fid_region(self.handle, region, first, count)

    def moments_region(self, region, count=None):
        return lpc_moments_region(self.handle, region, count)

    def spectrum(self, f0_hz, df_hz, n_freq, lb_hz=0.0, region=-1, count=None):
        return lpc_spectrum(self.handle, f0_hz, df_hz, n_freq, lb_hz, region, count)

    def set_kernel(self, which):
        lpc_set_kernel(self.handle, which)

    def set_option(self, key, value):
        lpc_set_option(self.handle, key, value)

    def sync_steps(self):
        """After CUDA graph replays of ``step``: take the device's step count (include/lpc.h "CUDA graphs")."""
        return lpc_sync_steps(self.handle)

    @property
    def time_block_steps(self):
        return lpc_time_block_steps(self.handle)

    @property
    def reads_sin_alone(self):
        return bool(lpc_reads_sin_alone(self.handle))

    @property
    def steps_done(self):
        return lpc_steps_done(self.handle)

    @property
    def launch_count(self):
        return lpc_launch_count(self.handle)

    @property
    def bytes_per_site_step(self):
        return lpc_bytes_per_site_step(self.handle)
