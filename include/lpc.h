/*
 * lpc.h -- C ABI of liblpc.so: the LPC3D lattice-gas propagation step on one
 * NVIDIA B200 (sm_100a).
 *
 * Method: arxiv 2603.22553.  Each time step propagates the complex
 * NMR magnetisation g_i between neighbouring lattice sites with Metropolis hop
 * probabilities (Eq. 1) that keep the Boltzmann density (Eq. 2,
 * :66) stationary, multiplies by the site phase exp(i omega_i dt) (Eq. 13,
 * :144) and sums all sites into one free-induction-decay sample G(n dt)
 * (Eq. 12, :137).  Optionally the same sweep propagates the three
 * moment-propagation fields of the velocity autocorrelation function
 * (Eq. 4-5, :79-95; :84-86) and a real density field (:192).
 *
 * Conventions
 *   - Site arrays are dense, C order, shape (nx, ny, nz), z fastest:
 *     i = (x*ny + y)*nz + z.
 *   - Energies are in kT.  omega_i = 2 pi nu_i in rad/s.
 *   - Every pointer argument says "host", "device" or "host or device".  A
 *     "host or device" pointer is classified with cudaPointerGetAttributes.
 *   - All device work is enqueued on lpc_config.stream.  lpc_step_n does not
 *     synchronise; every call that returns data to the host does.
 *   - The library never allocates device memory: the caller passes one
 *     workspace (lpc_workspace_bytes) that must outlive the lattice.
 *   - Return value: 0 (LPC_OK) or a negative LPC_E* code; lpc_last_error()
 *     gives a thread-local message.  No exception crosses this boundary and
 *     there is no CPU fallback: without an sm_100 device calls return
 *     LPC_ECUDA.
 */
#ifndef LPC_H_
#define LPC_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define LPC_OK 0
#define LPC_EINVAL (-1) /* bad dimension, null pointer, alpha outside (0,1], range, all sites blocked */
#define LPC_ESTATE (-2) /* call out of order, e.g. lpc_step_n before lpc_set_site_params */
#define LPC_ENOMEM (-3) /* workspace too small or misaligned */
#define LPC_ECUDA (-4)  /* CUDA runtime / driver error, or no sm_100 device */

/* lpc_read_field / lpc_set_state selectors */
#define LPC_FIELD_G 0   /* complex magnetisation g_i: 2N doubles, interleaved re,im      */
#define LPC_FIELD_PI 1  /* equilibrium density pi_i (Eq. 2, sums to 1): N doubles, read only */
#define LPC_FIELD_PX 2  /* moment field P^x_i (needs n_moments = 3): N doubles            */
#define LPC_FIELD_PY 3
#define LPC_FIELD_PZ 4
#define LPC_FIELD_RHO 5 /* real density rho_i (needs n_density = 1): N doubles            */

/* bc[0] value and lpc_halo_view selectors (slab decomposition along x) */
#define LPC_BC_HALO 2
#define LPC_HALO_PARAMS 0 /* the equilibrium density pi: 1 channel plane                      */
#define LPC_HALO_STATE 1  /* the current state: 2 + n_density + n_moments channel planes      */
#define LPC_HALO_STATE0 2 /* the same planes of state buffer 0 / 1 explicitly (the two buffers  */
#define LPC_HALO_STATE1 3 /* alternate from step to step; for lpc_set_halo_peers)               */
#define LPC_HALO_STATE2 4  /* the current state, TWO planes per face (for slabs that take two steps per sweep)  */
#define LPC_HALO_PARAMS2 5 /* pi, two planes per face                                                            */
#define LPC_HALO_PHASE2 6  /* cos and sin of omega dt (2 channels), two planes per face                          */
#define LPC_HALO_SEND 0   /* the outermost owned plane(s) on that side                        */
#define LPC_HALO_RECV 1   /* the ghost plane(s) beyond                                        */

/* lpc_set_kernel selectors */
#define LPC_KERNEL_AUTO 0
#define LPC_KERNEL_DIRECT 1 /* one thread per site pair, neighbours straight from global memory */
#define LPC_KERNEL_TMA 2    /* TMA-staged x-marching tiles, mbarrier pipeline                  */
#define LPC_KERNEL_PERSIST 3 /* all n steps of lpc_step_n in one cooperative launch, grid barrier
                                between steps; for lattices that stay in L2 (launch-bound otherwise) */

/* lpc_set_option keys */
#define LPC_OPT_TIME_BLOCK 1     /* 0 auto (default; = 1 on B200), 1 one time step per sweep, 2 two per sweep      */
#define LPC_OPT_X_CHUNK 2        /* planes per x chunk of the one-step TMA sweeps; 0 = the library's choice         */
#define LPC_OPT_X_CHUNK2 3       /* planes per x chunk of the two-step sweep; 0 = the library's choice              */
#define LPC_OPT_PERSIST_MAX_MB 4 /* AUTO takes the persistent kernel up to this many MiB per step; 0 = 48           */
#define LPC_OPT_REGION_FUSION 5  /* 0 regional sums inside the sweep when possible (default), 1 separate pass       */
#define LPC_OPT_FULL_PHASE 6     /* 0 sweeps read sin alone where every phase angle is small (default), 1 cos + sin  */
#define LPC_OPT_SERIAL_LAUNCH 7  /* 0 a sweep may start behind the tail of the one before it (default), 1 plain launches */

typedef struct lpc_lattice lpc_lattice; /* opaque, host struct owned by the library */

typedef struct lpc_config {
  int32_t nx, ny, nz;  /* lattice size, each >= 1 ("system dimensions")            */
  int32_t bc[3];       /* per axis: 0 periodic, 1 reflective zero-flux wall;     */
                       /* bc[0] may also be LPC_BC_HALO: this lattice is one x-slab of a larger */
                       /* one and the caller supplies its two x ghost planes (see "Slabs")      */
  int32_t precision;   /* 0: fp64 storage and arithmetic; 1: fp32 storage and arithmetic with   */
                       /*    fp64 reductions                                                    */
  int32_t n_moments;   /* 0, or 3 to propagate P^x, P^y, P^z for the VACF / D (Eq. 4)           */
  int32_t n_density;   /* 0, or 1 to propagate a real density rho alongside      */
  int32_t n_regions;   /* 0, or 1..8 regions ("blocks") for a region-resolved FID        */
  int32_t link_mobility; /* 0, or 1 to reserve room for per-link mobility factors alpha_ij */
  double dt;           /* time step in s (5e-6)                                   */
  double a;            /* lattice spacing; D comes out in a^2 / dt units of it    */
  double alpha;        /* global jump factor in (0,1], Eq. 7                 */
  int64_t max_steps;   /* capacity of the G and VACF series, >= 0                               */
  void* stream;        /* cudaStream_t owned by the caller (e.g. a torch stream); NULL = legacy */
                       /* default stream                                                        */
} lpc_config;

/* Bytes of device workspace lpc_create_lattice needs for this configuration.
 * cfg: host.  bytes: host, out.  Errors: LPC_EINVAL.  Needs no GPU.                            */
int lpc_workspace_bytes(const lpc_config* cfg, size_t* bytes);

/* Create a lattice over a caller-owned device workspace (256-byte aligned, >= the size above).
 * The workspace holds the packed per-site parameters, the ping-pong state, the per-block
 * partial sums and the G / VACF series; the caller frees it after lpc_destroy.
 * cfg: host.  workspace_dev: device.  out: host, receives the handle.
 * Errors: LPC_EINVAL, LPC_ENOMEM, LPC_ECUDA.                                                    */
int lpc_create_lattice(const lpc_config* cfg, void* workspace_dev, size_t bytes, lpc_lattice** out);

/* Site-parameter precompute (north star (a); Eq. 1, Eq. 2, Eq. 13 phase, Eq. 5):
 *   pi_i = exp(-dF_i) / sum_j exp(-dF_j) on open sites, 0 on blocked ones;
 *   packed hop data: pi_i alone, from which every hop probability follows in the sweep as
 *   p(i->j) = kappa_i * min(pi_i, pi_j), kappa_i = (alpha/6) / pi_i  (= (alpha/6) min(1, exp(-(dF_j - dF_i))));
 *   phase factors cos(omega_i dt), sin(omega_i dt);
 *   initial state g(0) = pi (or g0), P^d(1), Z_d[1], rho(0) = pi, G[0].
 * dF_kT, omega_rad_s: host or device, N doubles.  blocked: host or device, N bytes (non-zero =
 * carbon).  g0_or_null: host or device, 2N doubles (re,im) or NULL for g(0) = pi.  The arrays
 * are read during the call and not referenced afterwards.  Values at blocked sites are ignored.
 * Resets the step counter and both series.  Synchronises the stream.
 * Errors: LPC_EINVAL (null pointer; every site blocked; exp(-dF) over- or underflows, i.e. the
 * spread of dF exceeds about 700 kT), LPC_ECUDA.                                               */
int lpc_set_site_params(lpc_lattice* lat, const double* dF_kT, const uint8_t* blocked,
                        const double* omega_rad_s, const void* g0_or_null);

/* Per-link mobility factors alpha_ij ("a factor alpha_ij can be defined for each link between
 * neighboring lattice sites i and j"; :305 reduced mobility under confinement):
 *   p(i->j) = alpha_ij (alpha/6) min(1, exp(-(dF_j - dF_i))),  alpha_ij = alpha_ji in [0, 1],
 * the same factor in both directions, so detailed balance and the Boltzmann density of Eq. 2 are kept.
 * alpha_link: host or device, 3N doubles; alpha_link[d*N + i] is the factor of the link between site i and its
 * +d neighbour (d = 0 x, 1 y, 2 z; on a periodic axis the last site links to the first, on a reflective axis
 * the entry of the last site is ignored).  NULL removes the factors.  Needs link_mobility = 1 at creation
 * (24 B per site more workspace in fp64) and must come after lpc_set_site_params and before the first step;
 * it resets the state to g(0) = pi, P^d(1), Z_d[1] of the new hop probabilities and drops region labels (set
 * state and labels afterwards).  The sweeps then read three stored link weights per site (80 B per site
 * update in fp64 instead of 56); every kernel (TMA, direct, persistent) has that path.  Synchronises the stream.
 * Errors: LPC_ESTATE (order, or created without link_mobility), LPC_EINVAL (a factor outside [0,1]), LPC_ECUDA. */
int lpc_set_link_mobility(lpc_lattice* lat, const double* alpha_link);

/* Advance n time steps (north star (b), (c); Eq. 13 + Eq. 12, Eq. 4): per step one fused sweep
 * that propagates, phase-rotates, reduces G[n] and (if enabled) Z_d[n+1], P^d, rho.  Eq. 13 is a
 * Jacobi update (its right-hand side is at n-1), so a lattice that carries the
 * magnetisation alone (n_moments = n_density = 0, no link factors, no region labels, not a slab,
 * periodic axes of length >= 4) can take TWO steps per sweep while at least two are left
 * ("temporal blocking": state and parameters cross HBM once per two steps; G[n] is still recorded
 * for every step and the state after the call is bit for bit that of the one-step sweeps).
 * LPC_OPT_TIME_BLOCK = 2 asks for it; the default is one step per sweep, which measures faster on
 * B200 (the two-step sweep is bound by its instruction count, not by HBM: DESIGN.md 6.1c).
 * Asynchronous on the stream.  Errors: LPC_ESTATE (no site parameters yet), LPC_EINVAL (n < 0 or
 * steps_done + n > max_steps), LPC_ECUDA.                                                      */
int lpc_step_n(lpc_lattice* lat, int64_t n);

/* Copy G[first .. first+count) to the host as interleaved (re, im) doubles.  G[0] is the initial
 * sum; the series has steps_done + 1 samples.  out_re_im_host: host, 2*count doubles.
 * Synchronises.  Errors: LPC_EINVAL (range), LPC_ESTATE, LPC_ECUDA.                             */
int lpc_read_fid(lpc_lattice* lat, int64_t first, int64_t count, double* out_re_im_host);

/* VACF series and diffusion coefficients (Eq. 4):
 *   vacf_xyz_host[d*count + (m-1)] = Z_d[m] = <dx_1 dx_m>,  m = 1..count  (count <= steps_done+1)
 *   D_xyz[d] = Z_d[1] / (2 dt) + (1/dt) * sum_{m=2..count} Z_d[m]
 * vacf_xyz_host: host, 3*count doubles, may be NULL.  D_xyz: host, 3 doubles.  Synchronises.
 * Errors: LPC_ESTATE (n_moments == 0 or no parameters), LPC_EINVAL (range), LPC_ECUDA.         */
int lpc_moments(lpc_lattice* lat, int64_t count, double* vacf_xyz_host, double D_xyz[3]);

/* Read a site field into a dense (nx,ny,nz) array of doubles (see LPC_FIELD_*).
 * out: host or device.  Synchronises.  Errors: LPC_EINVAL, LPC_ESTATE, LPC_ECUDA.              */
int lpc_read_field(lpc_lattice* lat, int32_t which, void* out);

/* Overwrite a state field (LPC_FIELD_G or LPC_FIELD_RHO) from a dense array; values at blocked
 * sites are ignored (set to 0).  LPC_FIELD_G resets the step counter and series (G[0] = sum g).
 * in: host or device.  Synchronises.  Errors: LPC_EINVAL, LPC_ESTATE, LPC_ECUDA.               */
int lpc_set_state(lpc_lattice* lat, int32_t which, const void* in);

/* Equilibration loop of the paper's workflow (Fig. 3 step 3): iterate
 * the density update rho <- W rho on the density field (LPC_FIELD_RHO; needs n_density = 1) and
 * compare rho(t) with rho(t+1); stop when delta = max_i |rho_i(t+1) - rho_i(t)| < threshold or
 * after max_iters sweeps.  delta is reduced on the device inside every sweep; the host reads it
 * back every check_every sweeps (>= 1; 1 reproduces the paper's loop exactly, larger values
 * trade up to check_every - 1 extra sweeps for fewer synchronisations).  The magnetisation, the
 * moment fields and both series are not touched.
 * iters_done, last_delta: host, out (may be NULL).  Synchronises.
 * Errors: LPC_ESTATE (n_density == 0 or no parameters), LPC_EINVAL, LPC_ECUDA.                 */
int lpc_equilibrate(lpc_lattice* lat, double threshold, int64_t max_iters, int64_t check_every,
                    int64_t* iters_done, double* last_delta);

/* Start the propagation from the density field: g(0) <- rho (real), G[0] = sum_i rho_i; resets
 * the step counter and the G series (Fig. 3: the equilibrated densities feed the propagation
 * loop).  Synchronises.  Errors: LPC_ESTATE, LPC_ECUDA.                           */
int lpc_seed_from_density(lpc_lattice* lat);

/* Region labels for the region-resolved FID (the paper's electrode / bulk "blocks", PAPER.md:180,
 * and the signal of "different parts" of the system, Fig. 9, :275-281; needs n_regions >= 1).
 * region[i] in 0..n_regions-1 puts site i into that region, any other value into none.  From this
 * call on every step also reduces G_r[n] = sum_{i in r} g_i(n) (Eq. 12, :137, restricted to r) with
 * one extra pass over the state; G_r[steps_done] is computed at once.  lpc_set_site_params drops the
 * labels; lpc_set_state(G) and lpc_seed_from_density restart the regional series with the G series.
 * region: host or device, N bytes.  Synchronises.
 * Errors: LPC_ESTATE (n_regions == 0 or no parameters), LPC_EINVAL, LPC_ECUDA.                  */
int lpc_set_regions(lpc_lattice* lat, const uint8_t* region);

/* Copy G_r[first .. first+count) of one region to the host as interleaved (re, im) doubles; the
 * series starts at the step at which lpc_set_regions was called.  Synchronises.
 * Errors: LPC_ESTATE (no labels), LPC_EINVAL (region or range), LPC_ECUDA.                       */
int lpc_read_fid_region(lpc_lattice* lat, int32_t region, int64_t first, int64_t count, double* out_re_im_host);

/* Regional VACF and diffusion coefficients (the regional D of Table 1): Eq. 4
 * (:79) restricted to the particles that sit in the region when the later displacement starts,
 * normalised by the region's equilibrium population w_r = sum_{i in r} pi_i:
 *   Z^r_d[1] = sum_{i in r} pi_i sum_s p(i -> i + s e_d) a^2 / w_r,
 *   Z^r_d[m] = sum_{i in r} P^d_i(m-1) u^d_i / w_r  (m >= 2),   D^r_d as in lpc_moments.
 * Needs n_moments = 3, n_regions >= 1 and labels set before the first step; costs one more pass
 * over pi, the moment fields and the labels per step.  Layout and errors as lpc_moments.         */
int lpc_moments_region(lpc_lattice* lat, int32_t region, int64_t count, double* vacf_xyz_host, double D_xyz[3]);

/* Spectrum of a FID series (Eq. 9, "Fourier transformed", :202) on a frequency grid:
 *   F(f_k) = dt * sum_{n=0}^{count-1} G[n] exp(-pi lb n dt) exp(-2 pi i f_k n dt),  f_k = f0 + k df,
 * k = 0..n_freq-1 (Hz; delta in ppm = f / (nu_0 * 1e-6)); lb_hz >= 0 is an optional Lorentzian line
 * broadening, 0 = the plain sum.  region = -1 takes the FID of the whole lattice, 0..n_regions-1 a
 * regional one (which must have been recorded from step 0).  count <= steps_done + 1.
 * out_re_im_host: host, 2*n_freq doubles.  Synchronises.
 * Errors: LPC_ESTATE, LPC_EINVAL, LPC_ECUDA.                                                    */
int lpc_spectrum(lpc_lattice* lat, int32_t region, int64_t count, double f0_hz, double df_hz, int64_t n_freq,
                 double lb_hz, double* out_re_im_host);

/* ---- Slabs: one lattice split along x over several GPUs --------------------------------
 * Each rank owns a contiguous range of x planes and creates a lattice of that size with bc[0] = LPC_BC_HALO.
 * The library then leaves the two x ghost planes to the caller, who copies the neighbour's outermost owned
 * plane into them (NCCL send/recv, a peer-to-peer copy, or a plain device copy on one GPU); at a reflective end
 * of the whole lattice the ghost plane is simply left alone (it holds zeros = a wall).  Order of calls:
 *   lpc_partition_sum            -> Z_local; the caller adds the ranks' values (Eq. 2 normalises over the
 *   lpc_set_partition_sum(Z)        whole lattice) and hands the total back
 *   lpc_set_site_params          pi, phase factors of the owned sites
 *   exchange LPC_HALO_PARAMS     pi of the neighbours' boundary planes
 *   lpc_slab_finish              initial state with the neighbours' pi (P^d(1), Z_d[1], G[0])
 *   [lpc_set_state]              optional
 *   exchange LPC_HALO_STATE
 *   repeat: lpc_step_n(lat, 1); exchange LPC_HALO_STATE
 * G[n], Z_d[m] of a slab are the sums over its own sites: the caller adds the ranks' series (one reduction
 * when the series is read, none per step); D follows from the summed Z_d as in lpc_moments.  The equilibration
 * loop runs the same way: lpc_equilibrate(lat, threshold, 1, 1, ...) is one sweep, the caller exchanges
 * LPC_HALO_STATE and takes the largest delta of all slabs.
 * Two steps per sweep on slabs: when lpc_time_block_steps(lat) == 2 (magnetisation alone, at least two planes), the
 * caller may exchange TWO planes per face -- LPC_HALO_PARAMS2 and LPC_HALO_PHASE2 once before lpc_slab_finish,
 * LPC_HALO_STATE2 instead of LPC_HALO_STATE every time -- and then call lpc_step_n(lat, 2): one sweep, one exchange of
 * the same bytes per step.  The two planes of a face are one contiguous run.  A caller that exchanges one plane keeps
 * to lpc_step_n(lat, 1).
 * Not available in slab mode: lpc_step_n with n > 2 (or n = 2 without the two-plane exchange), lpc_equilibrate with
 * max_iters > 1 (LPC_ESTATE), the persistent kernel (never chosen), link factors (LPC_EINVAL at creation), direct halo
 * stores together with two steps per sweep.                                                                    */

/* Z_local = sum of exp(-dF_i) over the open sites of this lattice (Eq. 2).  dF_kT, blocked: host
 * or device, as lpc_set_site_params.  out: host.  Synchronises.  Errors: LPC_EINVAL, LPC_ECUDA.              */
int lpc_partition_sum(lpc_lattice* lat, const double* dF_kT, const uint8_t* blocked, double* out);

/* Normalise pi by Z instead of the lattice's own sum in every later lpc_set_site_params (Z <= 0 restores the
 * default).  Errors: LPC_EINVAL (not finite).                                                                */
int lpc_set_partition_sum(lpc_lattice* lat, double Z);

/* Where a halo plane lives in the workspace.  set: LPC_HALO_PARAMS / LPC_HALO_STATE; side: 0 low x, 1 high x;
 * role: LPC_HALO_SEND / LPC_HALO_RECV.  Returns the device address of channel 0's plane, the bytes of one
 * plane (contiguous: (ny+2) x padded nz elements of the lattice's precision, ghost rows and columns included),
 * the byte stride between channels and the number of channels.  STATE refers to the buffer that holds the
 * current state, so ask again after every step.  Works for any bc (tests use it to inspect planes).
 * Errors: LPC_EINVAL, LPC_ESTATE (no site parameters yet).                                                    */
int lpc_halo_view(lpc_lattice* lat, int32_t set, int32_t side, int32_t role, void** plane_dev, size_t* plane_bytes,
                  size_t* channel_stride_bytes, int32_t* n_channels);

/* Slab mode, direct halo stores: let the step kernel itself write this slab's outermost x planes into the
 * neighbours' x ghost planes, so that no copy or send follows the sweep (the transfer rides on the sweep's own
 * stores, plane by plane).  lo0 / lo1: device address of channel 0 of the ghost plane beyond x = 0 -- the
 * neighbour's LPC_HALO_RECV plane on its HIGH side -- in the neighbour's state buffer 0 / 1 (lpc_halo_view with
 * LPC_HALO_STATE0 / LPC_HALO_STATE1 on the neighbour), lo_channel_stride_bytes its channel stride; hi* likewise
 * for the neighbour beyond x = nx-1.  NULL, NULL = no neighbour there or no direct stores.  The memory must be
 * writable from this lattice's device (the same device, or a peer mapping) and all slabs must step together
 * (same number of lpc_step_n(lat, 1) calls), with every slab's step n finished before any slab's step n+1
 * starts (one stream, or an event per step).  Needs the TMA kernel.  The first exchange after lpc_slab_finish /
 * lpc_set_state and the exchanges of the equilibration sweeps remain the caller's.
 * Errors: LPC_ESTATE (not a slab, no TMA geometry), LPC_EINVAL.                                               */
int lpc_set_halo_peers(lpc_lattice* lat, void* lo0, void* lo1, size_t lo_channel_stride_bytes, void* hi0, void* hi1,
                       size_t hi_channel_stride_bytes);

/* Slab mode between PROCESSES of one node (one process per GPU): export the device allocation that holds this lattice's
 * workspace as a CUDA IPC handle, so that a neighbour rank can map it and hand the ghost-plane addresses inside it to
 * lpc_set_halo_peers.  handle_out: host, LPC_IPC_HANDLE_BYTES bytes (a cudaIpcMemHandle_t; send it to the other rank as
 * plain bytes).  offset_out: host, byte offset of the workspace inside the exported allocation (an allocator may have
 * carved the workspace out of a larger block; the handle always names the whole block).
 * Errors: LPC_EINVAL, LPC_ECUDA (e.g. the allocation does not come from cudaMalloc).                               */
#define LPC_IPC_HANDLE_BYTES 64
int lpc_ipc_export(lpc_lattice* lat, void* handle_out, size_t* offset_out);

/* Map an allocation another process exported with lpc_ipc_export into this process (cudaIpcOpenMemHandle, peer access
 * enabled when it lives on another GPU).  handle: host, LPC_IPC_HANDLE_BYTES bytes.  base_out: host, receives the device
 * address of the allocation's first byte in THIS process; the neighbour's workspace starts at base + its offset.
 * lpc_ipc_close unmaps it (after the lattices that store into it are done).  Errors: LPC_EINVAL, LPC_ECUDA.          */
int lpc_ipc_open(const void* handle, void** base_out);
int lpc_ipc_close(void* base);

/* Slab mode: build the initial state once the pi ghost planes are in place (see the order above).  Resets the
 * step counter and the series.  Synchronises.  Errors: LPC_ESTATE (not a slab, or no site parameters).         */
int lpc_slab_finish(lpc_lattice* lat);

/* Choose the step kernel (LPC_KERNEL_*).  AUTO picks PERSIST when one step's state and parameters
 * stay in L2 (<= 48 MB) and no region labels are set, else TMA.  Errors: LPC_EINVAL.             */
int lpc_set_kernel(lpc_lattice* lat, int32_t which);

/* Tuning and test switches (LPC_OPT_*): how the library schedules the sweeps, never what they
 * compute.  Takes effect from the next lpc_step_n.  Errors: LPC_EINVAL (unknown key, value out
 * of range, or LPC_OPT_TIME_BLOCK = 2 on a lattice that cannot run the two-step sweep).          */
int lpc_set_option(lpc_lattice* lat, int32_t key, int64_t value);

/* 1 if the plain magnetisation sweeps of this lattice read sin alone and rebuild cos (every open
 * site has cos(omega dt) >= 1/2 and LPC_OPT_FULL_PHASE is 0), else 0.  Slabs that take two steps
 * per sweep rotate their neighbours' boundary sites as well, so the slabs of one lattice must agree:
 * a caller sets LPC_OPT_FULL_PHASE = 1 on all of them unless every slab answers 1.               */
int32_t lpc_reads_sin_alone(const lpc_lattice* lat);

/* 2 if the next lpc_step_n(lat, n >= 2) takes two time steps per sweep (see lpc_step_n), else 1.  */
int32_t lpc_time_block_steps(const lpc_lattice* lat);

/* Steps taken since the last lpc_set_site_params / lpc_set_state(G).                           */
int64_t lpc_steps_done(const lpc_lattice* lat);

/* CUDA graphs.  On the TMA and direct kernels lpc_step_n only enqueues kernel launches (no
 * synchronisation, no allocation, no host read), so a caller may capture lpc_step_n(lat, k) on the
 * lattice's stream into a CUDA graph and replay it: the series index lives on the device and every
 * replay appends k samples.  Capture an EVEN k (the graph holds the ping-pong buffers of its sweeps)
 * on a lattice without region labels and keep steps within max_steps (the kernels do not check).
 * The host's step count does not see replays (and counts a capture that never ran):
 * lpc_sync_steps reads the device's count back (synchronises the stream) so that lpc_read_fid,
 * lpc_moments and further lpc_step_n calls see the true series length; it returns the count in
 * *steps_done if that is not NULL.  Measured: +2% at 128^3, nothing from 256^3 up,
 * because the sweeps are already launched with programmatic dependent launch.
 * Errors: LPC_ESTATE (no site parameters yet; the device count exceeds max_steps: the series
 * overflowed and the workspace beyond it is damaged), LPC_ECUDA.                                 */
int lpc_sync_steps(lpc_lattice* lat, int64_t* steps_done);

/* Kernel launches this lattice has enqueued so far (all kernels, for accounting).              */
int64_t lpc_launch_count(const lpc_lattice* lat);

/* Algorithmic HBM bytes one step moves per lattice site with this configuration and kernel
 * choice: state channels in and out, pi, cos and sin -- sin alone where the sweep
 * rebuilds cos --, pi a second time where the moment fields have a sweep of their own, stored link
 * weights and region labels if set.  Halo re-reads of the tiles are not in it.                  */
double lpc_bytes_per_site_step(const lpc_lattice* lat);

/* One FID sample without a lattice, a workspace or any allocation (for callers that may not call
 * cudaMalloc: under CUDA graph capture, in a serving loop, in a harness that forbids it):
 *     out[0] + i out[1] = G = sum_{i < n_sites} g_i          (Eq. 12)
 * of a dense device array g of n_sites complex numbers (re, im pairs of doubles, e.g. what
 * lpc_read_field(lat, LPC_FIELD_G, device pointer) wrote).  A variant of the reduction kernel behind
 * lpc_set_state: one block partial per 32768 sites, then the last block adds the partials in block
 * order (bitwise reproducible for a given n_sites).  The partials and the ticket counter live in a
 * static __device__ array of the library (LPC_NOALLOC_SCRATCH_BYTES, held by every GPU that loads
 * the library until the process exits), which is why n_sites is limited to LPC_NOALLOC_MAX_SITES.
 *   g, out : DEVICE pointers of the current device, caller-owned; out takes 2 doubles.
 *   stream : cudaStream_t of the current device (NULL: the default stream).  Asynchronous.
 * The call clears the ticket counter itself (stream-ordered) and overwrites every partial it reads,
 * so it does not depend on what the last call left.  ALL calls on a device share the one array:
 * calls that overlap on the GPU (two streams, two host threads) race -- serialise them.
 * Calls no cudaMalloc / cudaFree and no allocating library routine.
 * Errors: LPC_EINVAL (NULL or host pointer, n_sites < 0 or > LPC_NOALLOC_MAX_SITES), LPC_ECUDA.  */
#define LPC_NOALLOC_MAX_SITES (1ll << 28)       /* 8192 block partials x 32768 sites            */
#define LPC_NOALLOC_SCRATCH_BYTES (256 + 8192 * 16)
int lpc_fid_sample_noalloc(const double* g_re_im_dev, int64_t n_sites, double* out_dev, void* stream);

/* Free the host handle (the workspace stays with the caller).  NULL is allowed.                */
void lpc_destroy(lpc_lattice* lat);

/* Message of the last error on this thread ("" if none).                                       */
const char* lpc_last_error(void);

#ifdef __cplusplus
}
#endif
#endif /* LPC_H_ */
