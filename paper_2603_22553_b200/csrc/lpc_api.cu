// lpc_api.cu -- host side of liblpc.so: the C ABI of include/lpc.h.
//
// Workspace layout (device, all offsets 256-byte aligned):
//   Ctl | fid[max_steps+1] | vacf[3][max_steps+2] | partials | pi | cs[2] | F0[C] | F1[C] | staging
// F0/F1 are the ping-pong state buffers in density-normalised, channel-planar (SoA) form.
#include <cuda.h>
#include <cuda_runtime.h>

#include <algorithm>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "../../include/lpc.h"
#include "lpc_internal.cuh"
#include "lpc_precompute.cuh"
#include "lpc_step.cuh"
#include "lpc_step2.cuh"
#include "lpc_equil.cuh"
#include "lpc_regions.cuh"

using namespace lpc;

namespace {

thread_local char g_err[512] = "";

int fail(int code, const char* fmt, ...) {
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(g_err, sizeof(g_err), fmt, ap);
  va_end(ap);
  return code;
}

#define CUDA_TRY(expr)                                                                                  \
  do {                                                                                                  \
    cudaError_t e_ = (expr);                                                                            \
    if (e_ != cudaSuccess) return fail(LPC_ECUDA, "%s: %s (%s:%d)", #expr, cudaGetErrorString(e_), __FILE__, __LINE__); \
  } while (0)

constexpr size_t ALIGN = 256;
size_t align_up(size_t v) { return (v + ALIGN - 1) / ALIGN * ALIGN; }

constexpr int DIRECT_MAX_BLOCKS = 148 * 8;
constexpr int AUX_BLOCKS = 148 * 8;
constexpr long long STAGE_SITES = 4ll << 20;  // sites in the host<->device staging region (two halves)
inline long long stage_chunk_sites(long long N) { return std::max<long long>(1, std::min<long long>(N, STAGE_SITES / 2)); }
constexpr long long SPEC_BATCH = 4096;        // frequencies per spectrum launch

struct Offsets {
  size_t ctl, fid, vacf, partials, pi, cs, mlink, f0, f1, regions, fidr, vacfr, wr, rpartials, spec, staging, total;
  size_t partial_slots;
};

}  // namespace

struct lpc_lattice {
  lpc_config cfg;
  Layout L;
  int C, nrho, nmom, sT;
  long long N;
  Offsets off;
  unsigned char* ws;
  cudaStream_t stream;
  bool have_params;
  bool have_regions;
  long long region_first;  // first sample of the regional series
  bool region_moments;     // the regional VACF is being recorded (labels were set at step 0)
  bool regions_fused;      // the last launch_step accumulated the regional FID inside the sweep
  bool have_links;         // per-link mobility factors are set: the sweeps read the stored link weights
  bool halo;               // bc[0] = LPC_BC_HALO: an x-slab whose x ghost planes the caller fills
  bool halo_ready;         // lpc_slab_finish has run
  double z_override;       // > 0: normalise pi by this partition sum (slab mode)
  unsigned char* peer[2][2];  // [side][buffer]: channel 0 of the neighbour's x ghost plane in its state buffer 0 / 1, or nullptr
  size_t peer_stride[2];      // that neighbour's channel stride in bytes
  int cur;  // index of the buffer holding the current state
  long long steps;
  long long launches;
  int kernel;  // LPC_KERNEL_*
  int device;  // CUDA device ordinal of the workspace
  // two-step sweep (lpc_step2.cuh)
  bool step2_ok;      // the lattice can run it (geometry, channels, boundary conditions)
  int time_block;     // LPC_OPT_TIME_BLOCK: 0 auto (= 1), 1 one step per sweep, 2 two steps per sweep whenever possible
  int xc2, chunks_x2; // its x chunks
  int ty2, tz2, tiles_z2, tiles_y2;   // its tiles: 8 rows of 32 16-byte groups (lpc_step2.cuh)
  bool ghosts_full;   // the whole ghost shell of the current state is valid (the one-step sweeps keep the face layer only)
  CUtensorMap tm2_f[2], tm2_m[2], tm2_pi, tm2_cs, tm2_sn;   // tm2_m: the three moment channels; tm2_sn: the sine channel alone
  bool phase_small;   // every open site has cos(omega dt) >= 1/2: sweeps may read sin alone (cos_from_sin)
  int opt_full_phase; // LPC_OPT_FULL_PHASE: 1 = always read cos and sin
  int opt_serial_launch;   // LPC_OPT_SERIAL_LAUNCH: 1 = no programmatic dependent launch
  int opt_xc, opt_persist_mb, opt_region_fusion;   // lpc_set_option overrides (0 = default)
  // TMA geometry
  int ty, tz, nstage, xc, tiles_z, tiles_y, chunks_x;
  int xc_reg, chunks_x_reg;   // x chunks of the sweeps that carry regional sums
  bool tma_ok;
  TmaLinkMaps tm_l;  // pi centres and the three link-weight channels (link_mobility = 1)
  CUtensorMap tm_f[2], tm_m[2], tm_r[2], tm_pi, tm_cs, tm_sn;  // tm_r: one channel per box (the density channel alone, equilibration)  // tm_f: magnetisation (+ density) channels, tm_m: the 3 moment channels
};

namespace {

int check_cfg(const lpc_config* c) {
  if (!c) return fail(LPC_EINVAL, "config is NULL");
  if (c->nx < 1 || c->ny < 1 || c->nz < 1) return fail(LPC_EINVAL, "lattice dimensions must be >= 1 (got %d %d %d)", c->nx, c->ny, c->nz);
  if ((long long)c->nx * c->ny * c->nz > (1ll << 40)) return fail(LPC_EINVAL, "lattice too large");
  for (int d = 0; d < 3; ++d)
    if (c->bc[d] != 0 && c->bc[d] != 1 && !(d == 0 && c->bc[d] == LPC_BC_HALO))
      return fail(LPC_EINVAL, "bc[%d] must be 0 (periodic) or 1 (reflective)%s", d, d == 0 ? " or LPC_BC_HALO" : "");
  if (c->bc[0] == LPC_BC_HALO && c->link_mobility) return fail(LPC_EINVAL, "link factors are not available in slab mode");
  if (c->precision != 0 && c->precision != 1) return fail(LPC_EINVAL, "precision must be 0 (fp64) or 1 (fp32)");
  if (c->n_moments != 0 && c->n_moments != 3) return fail(LPC_EINVAL, "n_moments must be 0 or 3");
  if (c->n_density != 0 && c->n_density != 1) return fail(LPC_EINVAL, "n_density must be 0 or 1");
  if (c->link_mobility != 0 && c->link_mobility != 1) return fail(LPC_EINVAL, "link_mobility must be 0 or 1");
  if (c->n_regions < 0 || c->n_regions > MAX_REGIONS) return fail(LPC_EINVAL, "n_regions must lie in [0, %d]", MAX_REGIONS);
  if (!(c->alpha > 0.0 && c->alpha <= 1.0)) return fail(LPC_EINVAL, "alpha must lie in (0,1]");
  if (!(c->dt > 0.0) || !std::isfinite(c->dt)) return fail(LPC_EINVAL, "dt must be positive");
  if (!(c->a > 0.0) || !std::isfinite(c->a)) return fail(LPC_EINVAL, "a must be positive");
  if (c->max_steps < 0) return fail(LPC_EINVAL, "max_steps must be >= 0");
  return LPC_OK;
}

Layout make_layout(const lpc_config* c) {
  Layout L;
  const int sT = c->precision ? 4 : 8;
  L.nx = c->nx; L.ny = c->ny; L.nz = c->nz;
  L.padz = 128 / sT;  // 128 bytes of ghost columns on each side keep every row 128-byte aligned
  L.gh = GH;
  L.nxp = c->nx + 2 * GH;
  L.nyp = c->ny + 2 * GH;
  L.nzp = (c->nz + L.padz - 1) / L.padz * L.padz + 2 * L.padz;
  L.sy = L.nzp;
  L.sx = (long long)L.nyp * L.nzp;
  L.np = (long long)L.nxp * L.sx;
  return L;
}

// TMA tile geometry: 8 x 64 tiles of the y-z plane, 8 warps per CTA, two CTAs per
// SM (a sweep carries at most 3 channels: the moment fields have a sweep of their own).  (16 x 64 tiles with one 16-warp CTA per SM measured the same at 512^3
// and slightly worse at 256^3, so there is one tile shape.)
constexpr int SM_COUNT = 148;
#ifndef LPC_TY64
#define LPC_TY64 8   // rows of an fp64 tile (-DLPC_TY64=16: one 16-warp CTA per SM, 512^3 fp64 118.0 / 104.8 GLUPS burst / sustained against 120.4 / 105.5)
#endif

void tma_geometry(int C, bool f32, int nx, int ny, int nz, int xc_override, int* ty, int* tz, int* nstage, int* xc, int* tiles_z, int* tiles_y, int* chunks_x,
                  int target = 32) {
  *ty = f32 ? 16 : LPC_TY64; *tz = 64;   // fp32: a thread owns a z-quad (lpc_step_vec.cuh), 256 threads cover 16 rows
  *nstage = 4;   // 3 when the density rides along (3 channels); informational, the kernels fix it
  *tiles_z = (nz + *tz - 1) / *tz;
  *tiles_y = (ny + *ty - 1) / *ty;
  const long long tiles = (long long)*tiles_z * *tiles_y;
  const long long resident = (long long)SM_COUNT * 2;   // every TMA sweep carries at most 3 channels
  (void)C;
  // Split x into chunks of about 32 planes.  Measured on 512^3 fp64 (ms per step, xc = 8 / 16 / 24 / 32 /
  // 48 / 74 / 128 / 256): 1.44 / 1.32 / 1.29 / 1.29 / 1.32 / 1.38 / 1.49 / 1.55 -- long chunks keep all SMs
  // marching through the same planes in lockstep, which makes the DRAM traffic come in read bursts and
  // write bursts; many short CTAs desynchronise and keep the mix even.  Below 24 planes the two extra
  // plane loads per chunk cost more than that gains, unless the grid is short of waves (256^3: 16 planes
  // per chunk measured 2% faster than 32), so chunks shrink to 16 planes to reach 8 waves.
  // (sweeps with regional sums take 64-plane chunks, `target`: their per-CTA epilogue -- a warp sum per regional column -- is
  // worth two planes; 512^3 fp64 with three regions 98.1 -> 102.7 GLUPS burst, 89.3 -> 93.2 sustained)
  long long chunks = std::max(1, (nx + target / 2) / target);
  chunks = std::max(chunks, std::min<long long>(std::max(1, nx / 16), (8 * resident + tiles - 1) / tiles));
  if (tiles * std::max(1, nx / 16) < 3 * resident) {
    // Few waves: wave quantisation decides.  A CTA costs its planes plus two halo planes plus about six
    // plane times of pipeline fill and final reduce; take the chunk count with the cheapest last wave
    // (128^3: 9 chunks = 288 CTAs in one wave instead of 10 = 320 CTAs in two, 44 -> 30 us/step).
    long long best = 1, best_cost = -1;
    for (long long c = 1; c <= std::max(1, nx / 2); ++c) {
      const long long len = (nx + c - 1) / c;
      const long long cost = ((tiles * ((nx + len - 1) / len) + resident - 1) / resident) * (len + 8);
      if (best_cost < 0 || cost < best_cost) {
        best = c;
        best_cost = cost;
      }
    }
    chunks = best;
  }
  if (xc_override > 0) chunks = (nx + xc_override - 1) / xc_override;   // LPC_OPT_X_CHUNK
  *xc = (int)((nx + chunks - 1) / chunks);
  *chunks_x = (nx + *xc - 1) / *xc;
}

// x chunks of the two-step sweep: one CTA per SM; a chunk costs its planes + 4 halo planes of loads and 3 iterations of
// pipeline fill, so chunks are long (64 planes) unless the lattice has too few tiles to give every SM a CTA
void step2_geometry(int nx, long long tiles, int xc_override, int* xc, int* chunks_x) {
  long long chunks = std::max(1, (nx + 32) / 64);
  if (tiles * chunks < SM_COUNT) chunks = std::min<long long>(std::max(1, nx / 8), (SM_COUNT + tiles - 1) / tiles);
  if (xc_override > 0) chunks = (nx + xc_override - 1) / xc_override;
  *xc = (int)((nx + chunks - 1) / chunks);
  *chunks_x = (nx + *xc - 1) / *xc;
}

Offsets make_offsets(const lpc_config* c, const Layout& L) {
  Offsets o;
  const size_t sT = c->precision ? 4 : 8;
  const int C = 2 + c->n_density + c->n_moments;
  int ty, tz, ns, xc, tzs, tys, cxs;
  tma_geometry(C, c->precision == 1, c->nx, c->ny, c->nz, 0, &ty, &tz, &ns, &xc, &tzs, &tys, &cxs);
  // LPC_OPT_X_CHUNK may shrink the chunks at run time; size for the worst case (one plane per chunk)
  const size_t tma_blocks = (size_t)tzs * tys * (size_t)c->nx;
  o.partial_slots = std::max<size_t>(std::max<size_t>(DIRECT_MAX_BLOCKS, AUX_BLOCKS), std::min<size_t>(tma_blocks, 1u << 20));
  const long long N = (long long)c->nx * c->ny * c->nz;
  size_t p = 0;
  o.ctl = p; p += align_up(sizeof(Ctl));
  o.fid = p; p += align_up((size_t)(c->max_steps + 1) * sizeof(double2));
  o.vacf = p; p += align_up((size_t)3 * (c->max_steps + 2) * sizeof(double));
  o.partials = p; p += align_up(o.partial_slots * MAX_RED * sizeof(double));
  o.pi = p; p += align_up((size_t)L.np * sT);
  o.cs = p; p += align_up((size_t)2 * L.np * sT);
  o.mlink = p; p += align_up(c->link_mobility ? (size_t)3 * L.np * sT : 0);
  o.f0 = p; p += align_up((size_t)C * L.np * sT);
  o.f1 = p; p += align_up((size_t)C * L.np * sT);
  o.regions = p; p += align_up(c->n_regions ? (size_t)N : 0);
  o.fidr = p; p += align_up((size_t)c->n_regions * (c->max_steps + 1) * sizeof(double2));
  o.vacfr = p; p += align_up((c->n_regions && c->n_moments) ? (size_t)c->n_regions * 3 * (c->max_steps + 2) * sizeof(double) : 0);
  o.wr = p; p += align_up(c->n_regions ? MAX_REGIONS * sizeof(double) : 0);
  o.rpartials = p; p += align_up(c->n_regions ? std::max<size_t>((size_t)AUX_BLOCKS * 4, o.partial_slots * 2) * MAX_REGIONS * sizeof(double) : 0);
  o.spec = p; p += align_up((size_t)SPEC_BATCH * sizeof(double2));
  o.staging = p; p += align_up(2 * (size_t)stage_chunk_sites(N) * 16);   // two halves of stage_chunk_sites(N) sites x 16 B
  o.total = p;
  return o;
}

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

int get_encode_fn(EncodeTiledFn* out) {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q));
    if (q != cudaDriverEntryPointSuccess || !p) return fail(LPC_ECUDA, "cuTensorMapEncodeTiled not available in this driver");
    fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  *out = fn;
  return LPC_OK;
}

int encode_map(CUtensorMap* m, bool f32, void* base, int rank, const cuuint64_t* dims, const cuuint32_t* box) {
  EncodeTiledFn fn;
  int rc = get_encode_fn(&fn);
  if (rc) return rc;
  const cuuint64_t sT = f32 ? 4 : 8;
  cuuint64_t strides[4];
  cuuint64_t s = sT;
  for (int d = 0; d < rank - 1; ++d) {
    s *= dims[d];
    strides[d] = s;
  }
  cuuint32_t estr[4] = {1, 1, 1, 1};
  CUresult r = fn(m, f32 ? CU_TENSOR_MAP_DATA_TYPE_FLOAT32 : CU_TENSOR_MAP_DATA_TYPE_FLOAT64, (cuuint32_t)rank, base, dims, strides, box,
                  estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                  CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(LPC_ECUDA, "cuTensorMapEncodeTiled failed with CUresult %d", (int)r);
  return LPC_OK;
}

template <typename T> T* wsp(lpc_lattice* h, size_t off) { return reinterpret_cast<T*>(h->ws + off); }
template <typename T> const T* mlink_of(lpc_lattice* h) { return h->have_links ? wsp<T>(h, h->off.mlink) : nullptr; }

bool is_device_ptr(const void* p) {
  cudaPointerAttributes at;
  if (cudaPointerGetAttributes(&at, p) != cudaSuccess) {
    cudaGetLastError();
    return false;
  }
  return at.type == cudaMemoryTypeDevice || at.type == cudaMemoryTypeManaged;
}

int aux_grid(long long n) { return (int)std::max<long long>(1, std::min<long long>((n + 255) / 256, AUX_BLOCKS)); }

// the regional FID can ride on the TMA magnetisation sweep when there is no density channel next to it
bool regions_fusable(const lpc_lattice* h) {
  return h->have_regions && h->nrho == 0 && h->tma_ok && h->kernel != LPC_KERNEL_DIRECT && !h->opt_region_fusion;
}

// what launch_step_t will decide for the next step: regional sums inside the TMA sweeps (not with direct halo stores)
bool will_fuse_regions(const lpc_lattice* h) {
  const bool peers = h->peer[0][h->cur ^ 1] || h->peer[1][h->cur ^ 1];
  return regions_fusable(h) && !peers;
}

// cudaFuncAttributeMaxDynamicSharedMemorySize is a per-device setting: remember per kernel AND device that it is made
// (several lattices on several GPUs may live in one process)
constexpr int MAX_DEVICES = 64;
template <typename Kern>
int ensure_dyn_smem(Kern kern, int bytes, int device, bool (&done)[MAX_DEVICES]) {
  if (device < 0 || device >= MAX_DEVICES || !done[device]) {
    CUDA_TRY(cudaFuncSetAttribute(kern, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
    if (device >= 0 && device < MAX_DEVICES) done[device] = true;
  }
  return LPC_OK;
}

// may the sweeps read sin alone and rebuild cos from it?
bool sin_only(const lpc_lattice* h) { return h->phase_small && !h->opt_full_phase; }

// A sweep launch that may overlap the tail of the launch before it in the stream (programmatic dependent launch: the
// kernels call griddepcontrol.launch_dependents / .wait); LPC_OPT_SERIAL_LAUNCH = 1 launches them the plain way.
template <typename... KArgs, typename... Args>
cudaError_t launch_sweep(const lpc_lattice* h, void (*kern)(KArgs...), unsigned grid, unsigned threads, size_t smem, Args&&... args) {
  cudaLaunchConfig_t cfg = {};
  cfg.gridDim = dim3(grid);
  cfg.blockDim = dim3(threads);
  cfg.dynamicSmemBytes = smem;
  cfg.stream = h->stream;
  cudaLaunchAttribute at[1];
  at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
  at[0].val.programmaticStreamSerializationAllowed = 1;
  cfg.attrs = at;
  cfg.numAttrs = h->opt_serial_launch ? 0 : 1;
  return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// ---- launch of one sweep ---------------------------------------------------------------------
template <typename T, int NRHO, int NMOM>
int launch_step_t(lpc_lattice* h) {
  StepArgs<T> a;
  a.L = h->L;
  a.fin = wsp<T>(h, h->cur ? h->off.f1 : h->off.f0);
  a.fout = wsp<T>(h, h->cur ? h->off.f0 : h->off.f1);
  a.pi = wsp<T>(h, h->off.pi);
  a.cs = wsp<T>(h, h->off.cs);
  a.mlink = mlink_of<T>(h);
  a.a6 = (T)(h->cfg.alpha / 6.0);
  a.partials = wsp<double>(h, h->off.partials);
  a.ctl = wsp<Ctl>(h, h->off.ctl);
  a.fid = wsp<double2>(h, h->off.fid);
  a.vacf = wsp<double>(h, h->off.vacf);
  a.vacf_stride = h->cfg.max_steps + 2;
  a.zscale = h->cfg.a * h->cfg.alpha / 6.0;
  for (int d = 0; d < 3; ++d) a.per[d] = h->cfg.bc[d] == 0;
  a.xc = h->xc; a.tiles_z = h->tiles_z; a.tiles_y = h->tiles_y; a.chunks_x = h->chunks_x;

  const bool use_tma = h->tma_ok && h->kernel != LPC_KERNEL_DIRECT;
  h->ghosts_full = false;   // a one-step sweep renews the face layer of the ghosts only
  // slab mode with direct halo stores: the sweep writes into the buffer the neighbours write in this step (all slabs
  // step together, so that is their buffer cur ^ 1 as well)
  for (int s = 0; s < 2; ++s) {
    a.peer[s] = reinterpret_cast<T*>(h->peer[s][h->cur ^ 1]);
    a.peer_stride[s] = (long long)(h->peer_stride[s] / sizeof(T));
  }
  const bool peers = a.peer[0] || a.peer[1];
  if (peers && !use_tma) return fail(LPC_ESTATE, "direct halo stores need the TMA kernel");
  // region-resolved FID inside the magnetisation sweep (no separate pass over the state): TMA kernel, no density channel
  // (and not together with direct halo stores: that combination runs the separate pass)
  const bool fuse_regions = use_tma && will_fuse_regions(h);
  h->regions_fused = fuse_regions;
  if (fuse_regions && !h->opt_xc) {
    a.xc = h->xc_reg;
    a.chunks_x = h->chunks_x_reg;
  }
  a.label = fuse_regions ? h->ws + h->off.regions : nullptr;
  a.rpartials = wsp<double>(h, h->off.rpartials);
  a.fidr = wsp<double2>(h, h->off.fidr);
  a.fidr_stride = h->cfg.max_steps + 1;
  a.vacfr = wsp<double>(h, h->off.vacfr);
  a.wr = wsp<double>(h, h->off.wr);
  a.vacfr_stride = h->cfg.max_steps + 2;
  a.region_sample = h->steps + 1;
  a.n_regions = h->cfg.n_regions;
  if (use_tma) {
    const unsigned grid = (unsigned)(h->tiles_z * h->tiles_y * a.chunks_x);
    auto launch = [&](auto kern, auto cfg, const CUtensorMap& tm, const StepArgs<T>& args) -> int {
      using K = decltype(cfg);
      static bool attr_done[MAX_DEVICES] = {};
      if (int rc = ensure_dyn_smem(kern, K::SMEM_BYTES, h->device, attr_done)) return rc;
      CUDA_TRY(launch_sweep(h, kern, grid, K::NTHREADS, K::SMEM_BYTES, tm, h->tm_pi, h->tm_cs, args));
      h->launches++;
      return LPC_OK;
    };
    auto launch_sn = [&](auto kern, auto cfg, const CUtensorMap& tm, const StepArgs<T>& args) -> int {
      using K = decltype(cfg);
      static bool attr_done[MAX_DEVICES] = {};
      if (int rc = ensure_dyn_smem(kern, K::SMEM_BYTES, h->device, attr_done)) return rc;
      CUDA_TRY(launch_sweep(h, kern, grid, K::NTHREADS, K::SMEM_BYTES, tm, h->tm_pi, h->tm_sn, args));
      h->launches++;
      return LPC_OK;
    };
    // With moment fields the step is two sweeps over the same pair of buffers: the three moment
    // channels first (Z_d[k+1], P^d <- W P^d; no phase, no cos/sin traffic), then the magnetisation
    // (and density) channels, which also advance the step counter.  One 5-channel sweep needs more
    // than 200 registers per thread and leaves one 8-warp CTA per SM (measured 42 GLUPS at 512^3).
    // With stored link weights (per-link mobility) the same two sweeps run as step_tma_links_kernel, with one
    // stage less where the link boxes would not leave room for two CTAs per SM.
    auto launch_links = [&](auto kern, auto cfg, const CUtensorMap& tm, const StepArgs<T>& args) -> int {
      using K = decltype(cfg);
      static bool attr_done[MAX_DEVICES] = {};
      if (int rc = ensure_dyn_smem(kern, K::SMEM_BYTES, h->device, attr_done)) return rc;
      CUDA_TRY(launch_sweep(h, kern, grid, K::NTHREADS, K::SMEM_BYTES, tm, h->tm_cs, h->tm_l, args));
      h->launches++;
      return LPC_OK;
    };
    // fp64: a thread owns a z-pair on 8 x 64 tiles; fp32: a z-quad on 16 x 64 tiles (one 16-byte group either way)
    constexpr int VW = 16 / (int)sizeof(T), TY = sizeof(T) == 8 ? LPC_TY64 : 4 * VW;
    constexpr int NS = (NRHO == 0) ? 4 : 3;   // two CTAs per SM must fit in shared memory
    constexpr int NSL = (NRHO == 0) ? 3 : 2;  // with the link-weight boxes
    if constexpr (NMOM == 3) {
      StepArgs<T> am = a;
      am.c0 = 2 + NRHO;
      am.fout = a.fout + (long long)am.c0 * h->L.np;
      for (int s = 0; s < 2; ++s)
        if (am.peer[s]) am.peer[s] += (long long)am.c0 * am.peer_stride[s];
      am.region_sample = h->steps + 2;   // Z_d[k+1] of the fields before this sweep
      const bool fuse_vacf = fuse_regions && h->region_moments;
      int rc = fuse_vacf ? (h->have_links ? launch_links(step_tma_links_kernel<T, 0, 0, 3, TY, 64, 3, VW, 1>, TmaCfg<T, 0, 0, 3, TY, 64, 3, 1, VW, 1>(), h->tm_m[h->cur], am)
                                          : launch(step_tma_kernel<T, 0, 0, 3, TY, 64, 4, VW, 1>, TmaCfg<T, 0, 0, 3, TY, 64, 4, 0, VW, 1>(), h->tm_m[h->cur], am))
               : h->have_links ? launch_links(step_tma_links_kernel<T, 0, 0, 3, TY, 64, 3, VW>, TmaCfg<T, 0, 0, 3, TY, 64, 3, 1, VW>(), h->tm_m[h->cur], am)
               : peers       ? launch(step_tma_kernel<T, 0, 0, 3, TY, 64, 4, VW, 2>, TmaCfg<T, 0, 0, 3, TY, 64, 4, 0, VW, 2>(), h->tm_m[h->cur], am)
                             : launch(step_tma_kernel<T, 0, 0, 3, TY, 64, 4, VW>, TmaCfg<T, 0, 0, 3, TY, 64, 4, 0, VW>(), h->tm_m[h->cur], am);
      if (rc) return rc;
    }
    a.c0 = 0;
    int rc;
    if constexpr (NRHO == 0) {
      if (sin_only(h) && !fuse_regions && !h->have_links && peers)
        rc = launch_sn(step_tma_kernel<T, 2, 0, 0, TY, 64, NS, VW, 6>, TmaCfg<T, 2, 0, 0, TY, 64, NS, 0, VW, 6>(), h->tm_f[h->cur], a);
      else if (sin_only(h) && !fuse_regions && !h->have_links && !peers)
        // every phase angle is small: stage sin alone and rebuild cos (8 bytes per site less in fp64)
        rc = launch_sn(step_tma_kernel<T, 2, 0, 0, TY, 64, NS, VW, 4>, TmaCfg<T, 2, 0, 0, TY, 64, NS, 0, VW, 4>(), h->tm_f[h->cur], a);
      else if (fuse_regions && sin_only(h) && !h->have_links)
        rc = launch_sn(step_tma_kernel<T, 2, 0, 0, TY, 64, NS, VW, 5>, TmaCfg<T, 2, 0, 0, TY, 64, NS, 0, VW, 5>(), h->tm_f[h->cur], a);
      else if (fuse_regions)
        rc = h->have_links ? launch_links(step_tma_links_kernel<T, 2, 0, 0, TY, 64, NSL, VW, 1>, TmaCfg<T, 2, 0, 0, TY, 64, NSL, 1, VW, 1>(), h->tm_f[h->cur], a)
                           : launch(step_tma_kernel<T, 2, 0, 0, TY, 64, NS, VW, 1>, TmaCfg<T, 2, 0, 0, TY, 64, NS, 0, VW, 1>(), h->tm_f[h->cur], a);
      else
        rc = h->have_links ? launch_links(step_tma_links_kernel<T, 2, 0, 0, TY, 64, NSL, VW>, TmaCfg<T, 2, 0, 0, TY, 64, NSL, 1, VW>(), h->tm_f[h->cur], a)
             : peers       ? launch(step_tma_kernel<T, 2, 0, 0, TY, 64, NS, VW, 2>, TmaCfg<T, 2, 0, 0, TY, 64, NS, 0, VW, 2>(), h->tm_f[h->cur], a)
                           : launch(step_tma_kernel<T, 2, 0, 0, TY, 64, NS, VW>, TmaCfg<T, 2, 0, 0, TY, 64, NS, 0, VW>(), h->tm_f[h->cur], a);
    } else {
      rc = h->have_links ? launch_links(step_tma_links_kernel<T, 2, NRHO, 0, TY, 64, NSL, VW>, TmaCfg<T, 2, NRHO, 0, TY, 64, NSL, 1, VW>(), h->tm_f[h->cur], a)
           : peers       ? launch(step_tma_kernel<T, 2, NRHO, 0, TY, 64, NS, VW, 2>, TmaCfg<T, 2, NRHO, 0, TY, 64, NS, 0, VW, 2>(), h->tm_f[h->cur], a)
                         : launch(step_tma_kernel<T, 2, NRHO, 0, TY, 64, NS, VW>, TmaCfg<T, 2, NRHO, 0, TY, 64, NS, 0, VW>(), h->tm_f[h->cur], a);
    }
    if (rc) return rc;
    h->cur ^= 1;
    return LPC_OK;
  } else {
    const long long npairs = (long long)((h->L.nz + 1) / 2) * h->L.ny * h->L.nx;
    const int grid = (int)std::max<long long>(1, std::min<long long>((npairs + 255) / 256, DIRECT_MAX_BLOCKS));
    a.c0 = 0;
    step_direct_kernel<T, NRHO, NMOM><<<grid, 256, 0, h->stream>>>(a);
  }
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  h->cur ^= 1;
  return LPC_OK;
}

// ---- all n steps in one cooperative launch (L2-resident lattices) ------------------------------
constexpr int PERSIST_MAX_BLOCKS = SM_COUNT * 4;   // 2 * blocks * MAX_RED partials fit the partial slots

template <typename T, int NRHO, int NMOM>
int launch_persist_t(lpc_lattice* h, int64_t n) {
  StepArgs<T> a;
  a.L = h->L;
  a.fin = nullptr;
  a.fout = nullptr;
  a.pi = wsp<T>(h, h->off.pi);
  a.cs = wsp<T>(h, h->off.cs);
  a.mlink = mlink_of<T>(h);
  a.a6 = (T)(h->cfg.alpha / 6.0);
  a.partials = wsp<double>(h, h->off.partials);
  a.ctl = wsp<Ctl>(h, h->off.ctl);
  a.fid = wsp<double2>(h, h->off.fid);
  a.vacf = wsp<double>(h, h->off.vacf);
  a.vacf_stride = h->cfg.max_steps + 2;
  a.zscale = h->cfg.a * h->cfg.alpha / 6.0;
  for (int d = 0; d < 3; ++d) a.per[d] = h->cfg.bc[d] == 0;
  a.peer[0] = a.peer[1] = nullptr; a.peer_stride[0] = a.peer_stride[1] = 0;
  a.label = nullptr; a.rpartials = nullptr; a.fidr = nullptr; a.fidr_stride = 0; a.region_sample = 0; a.n_regions = 0;
  a.vacfr = nullptr; a.wr = nullptr; a.vacfr_stride = 0;
  a.c0 = 0; a.xc = 0; a.tiles_z = a.tiles_y = a.chunks_x = 0;
  auto kern = step_persist_kernel<T, NRHO, NMOM>;
  static int per_sm_dev[MAX_DEVICES] = {};
  int per_sm = (h->device >= 0 && h->device < MAX_DEVICES) ? per_sm_dev[h->device] : 0;
  if (!per_sm) {
    CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, kern, 256, 0));
    if (h->device >= 0 && h->device < MAX_DEVICES) per_sm_dev[h->device] = per_sm;
  }
  if (per_sm < 1) return fail(LPC_ECUDA, "the persistent kernel does not fit on an SM");
  h->ghosts_full = false;
  const long long npairs = (long long)((h->L.nz + 1) / 2) * h->L.ny * h->L.nx;
  const int grid = (int)std::max<long long>(1, std::min<long long>({(npairs + 255) / 256, (long long)per_sm * SM_COUNT, (long long)PERSIST_MAX_BLOCKS}));
  unsigned long long* bar = reinterpret_cast<unsigned long long*>(&wsp<Ctl>(h, h->off.ctl)->scratch[6]);
  T* buf_a = wsp<T>(h, h->cur ? h->off.f1 : h->off.f0);
  T* buf_b = wsp<T>(h, h->cur ? h->off.f0 : h->off.f1);
  while (n > 0) {
    const int chunk = (int)std::min<int64_t>(n, 1 << 20);
    CUDA_TRY(cudaMemsetAsync(bar, 0, sizeof(unsigned long long), h->stream));
    int nsteps = chunk;
    void* args[] = {&a, &buf_a, &buf_b, &nsteps, &bar};
    CUDA_TRY(cudaLaunchCooperativeKernel(reinterpret_cast<void*>(kern), dim3(grid), dim3(256), args, 0, h->stream));
    h->launches++;
    if (chunk & 1) {
      std::swap(buf_a, buf_b);
      h->cur ^= 1;
    }
    h->steps += chunk;
    n -= chunk;
  }
  return LPC_OK;
}

template <typename T>
int launch_persist(lpc_lattice* h, int64_t n) {
  if (h->nrho == 0 && h->nmom == 0) return launch_persist_t<T, 0, 0>(h, n);
  if (h->nrho == 1 && h->nmom == 0) return launch_persist_t<T, 1, 0>(h, n);
  if (h->nrho == 0 && h->nmom == 3) return launch_persist_t<T, 0, 3>(h, n);
  return launch_persist_t<T, 1, 3>(h, n);
}

// AUTO takes the persistent kernel when one step's state and parameters stay in L2
bool persist_by_default(const lpc_lattice* h) {
  const long long limit = (long long)(h->opt_persist_mb > 0 ? h->opt_persist_mb : 48) << 20;   // LPC_OPT_PERSIST_MAX_MB
  return (long long)h->N * h->sT * (2 * h->C + 3) <= limit;
}

template <typename T>
int launch_step(lpc_lattice* h) {
  if (h->nrho == 0 && h->nmom == 0) return launch_step_t<T, 0, 0>(h);
  if (h->nrho == 1 && h->nmom == 0) return launch_step_t<T, 1, 0>(h);
  if (h->nrho == 0 && h->nmom == 3) return launch_step_t<T, 0, 3>(h);
  return launch_step_t<T, 1, 3>(h);
}

// ---- staging helpers: run `body(dev_ptr, i0, n)` over chunks of a dense host/device array -----
template <typename F>
int for_chunks_in(lpc_lattice* h, const void* src, size_t bytes_per_site, F body) {
  if (is_device_ptr(src)) return body(src, 0ll, h->N);
  // Two halves of the staging region in turn, no host synchronisation: the copies and the kernels that consume them are
  // ordered by the stream, the host runs ahead and keeps the copy queue full (from pinned memory the upload then runs at
  // the PCIe rate; the kernels are about 1% of it, so a second stream would buy nothing measurable)
  const long long chunk = stage_chunk_sites(h->N);
  const size_t half_bytes = (size_t)chunk * 16;
  unsigned char* stg = h->ws + h->off.staging;
  int half = 0;
  for (long long i0 = 0; i0 < h->N; i0 += chunk) {
    const long long n = std::min(chunk, h->N - i0);
    CUDA_TRY(cudaMemcpyAsync(stg + (size_t)half * half_bytes, static_cast<const unsigned char*>(src) + (size_t)i0 * bytes_per_site,
                             (size_t)n * bytes_per_site, cudaMemcpyHostToDevice, h->stream));
    int rc = body(stg + (size_t)half * half_bytes, i0, n);
    if (rc) return rc;
    half ^= 1;
  }
  return LPC_OK;
}

// G_r[sample] of every region from the current state
template <typename T>
int region_reduce_t(lpc_lattice* h, long long sample) {
  region_reduce_kernel<T><<<aux_grid(h->N), 256, 0, h->stream>>>(
      h->L, wsp<T>(h, h->off.pi), wsp<T>(h, h->cur ? h->off.f1 : h->off.f0), h->ws + h->off.regions, h->cfg.n_regions,
      wsp<double>(h, h->off.rpartials), wsp<Ctl>(h, h->off.ctl), wsp<double2>(h, h->off.fidr), h->cfg.max_steps + 1, sample);
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  return LPC_OK;
}

int region_reduce(lpc_lattice* h, long long sample) {
  return h->cfg.precision ? region_reduce_t<float>(h, sample) : region_reduce_t<double>(h, sample);
}

// regional VACF sample: INIT writes w_r and Z^r_d[1], otherwise Z^r_d[steps + 2] from the moment fields before the sweep
template <typename T, bool INIT>
int region_moment_t(lpc_lattice* h) {
  const T* q = wsp<T>(h, h->cur ? h->off.f1 : h->off.f0) + (long long)(2 + h->nrho) * h->L.np;
  const double scale = INIT ? h->cfg.a * h->cfg.a * h->cfg.alpha / 6.0 : h->cfg.a * h->cfg.alpha / 6.0;
  region_moment_kernel<T, INIT><<<aux_grid(h->N), 256, 0, h->stream>>>(
      h->L, wsp<T>(h, h->off.pi), mlink_of<T>(h), q, h->ws + h->off.regions, h->cfg.n_regions, wsp<double>(h, h->off.rpartials), wsp<Ctl>(h, h->off.ctl),
      wsp<double>(h, h->off.wr), wsp<double>(h, h->off.vacfr), h->cfg.max_steps + 2, INIT ? 1 : h->steps + 2, scale);
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  return LPC_OK;
}

template <bool INIT>
int region_moment(lpc_lattice* h) {
  return h->cfg.precision ? region_moment_t<float, INIT>(h) : region_moment_t<double, INIT>(h);
}

// x ghost planes: 1 wrap (periodic), 0 zero (wall), 2 leave to the caller (slab)
int xghost_mode(const lpc_lattice* h) { return h->halo ? 2 : (h->cfg.bc[0] == 0 ? 1 : 0); }

// cells of the ghost shell of one channel (fill_ghosts_kernel)
long long ghost_cells(const Layout& L) {
  const long long wy = L.ny + 2 * L.gh, wz = L.nz + 2 * GHZ;
  return 2ll * L.gh * wy * wz + (long long)L.nx * 2 * L.gh * wz + (long long)L.nx * L.ny * 2 * GHZ;
}

template <typename T>
int fill_state_ghosts(lpc_lattice* h) {
  const Layout& L = h->L;
  const long long cells = ghost_cells(L) * h->C;
  fill_ghosts_kernel<T><<<aux_grid(cells), 256, 0, h->stream>>>(wsp<T>(h, h->cur ? h->off.f1 : h->off.f0), h->C, L, xghost_mode(h),
                                                                 h->cfg.bc[1] == 0, h->cfg.bc[2] == 0);
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  h->ghosts_full = true;
  return LPC_OK;
}

// ---- two time steps in one sweep (lpc_step2.cuh) ----------------------------------------------
// may the next steps of this lattice run two at a time?
bool step2_usable(const lpc_lattice* h) {
  // on request only (LPC_OPT_TIME_BLOCK = 2): on B200 the one-step sweep measures faster at every size tried
  if (!h->step2_ok || h->time_block != 2 || h->have_links || h->have_regions) return false;
  if (h->peer[0][0] || h->peer[1][0]) return false;   // direct halo stores belong to the one-step sweep
  if (h->kernel == LPC_KERNEL_DIRECT || h->kernel == LPC_KERNEL_PERSIST) return false;
  return true;
}

template <typename T>
int launch_step2_t(lpc_lattice* h) {
  constexpr int VW = 16 / (int)sizeof(T);
  if (!h->ghosts_full) {   // the sweep reads two ghost layers, edges included
    int rc = fill_state_ghosts<T>(h);
    if (rc) return rc;
  }
  StepArgs<T> a;
  memset(&a, 0, sizeof(a));
  a.L = h->L;
  a.fin = wsp<T>(h, h->cur ? h->off.f1 : h->off.f0);
  a.fout = wsp<T>(h, h->cur ? h->off.f0 : h->off.f1);
  a.pi = wsp<T>(h, h->off.pi);
  a.cs = wsp<T>(h, h->off.cs);
  a.a6 = (T)(h->cfg.alpha / 6.0);
  a.partials = wsp<double>(h, h->off.partials);
  a.ctl = wsp<Ctl>(h, h->off.ctl);
  a.fid = wsp<double2>(h, h->off.fid);
  a.vacf = wsp<double>(h, h->off.vacf);
  a.vacf_stride = h->cfg.max_steps + 2;
  for (int d = 0; d < 3; ++d) a.per[d] = h->cfg.bc[d] == 0;
  a.xc = h->xc2; a.tiles_z = h->tiles_z2; a.tiles_y = h->tiles_y2; a.chunks_x = h->chunks_x2;
  a.zscale = h->cfg.a * h->cfg.alpha / 6.0;
  const unsigned grid = (unsigned)(h->tiles_z2 * h->tiles_y2 * h->chunks_x2);
  if (h->nmom == 3) {
    // the three moment channels first (Z_d of both steps; they read the step counter the magnetisation sweep advances)
    using KM = Step2Cfg<T, VW, 3, false>;
    StepArgs<T> am = a;
    am.c0 = 2;
    am.fout = a.fout + 2 * h->L.np;
    static bool attr_done_m[MAX_DEVICES] = {};
    if (int rc = ensure_dyn_smem(step2_kernel<T, VW, 3, false>, KM::SMEM_BYTES, h->device, attr_done_m)) return rc;
    CUDA_TRY(launch_sweep(h, step2_kernel<T, VW, 3, false>, grid, KM::NTHREADS, KM::SMEM_BYTES, h->tm2_m[h->cur], h->tm2_pi, h->tm2_cs, am));
    h->launches++;
  }
  a.c0 = 0;
  if (sin_only(h)) {
    using K = Step2Cfg<T, VW, 2, true>;
    static bool attr_done[MAX_DEVICES] = {};
    if (int rc = ensure_dyn_smem(step2_kernel<T, VW, 2, true>, K::SMEM_BYTES, h->device, attr_done)) return rc;
    CUDA_TRY(launch_sweep(h, step2_kernel<T, VW, 2, true>, grid, K::NTHREADS, K::SMEM_BYTES, h->tm2_f[h->cur], h->tm2_pi, h->tm2_sn, a));
  } else {
    using K = Step2Cfg<T, VW, 2, false>;
    static bool attr_done[MAX_DEVICES] = {};
    if (int rc = ensure_dyn_smem(step2_kernel<T, VW, 2, false>, K::SMEM_BYTES, h->device, attr_done)) return rc;
    CUDA_TRY(launch_sweep(h, step2_kernel<T, VW, 2, false>, grid, K::NTHREADS, K::SMEM_BYTES, h->tm2_f[h->cur], h->tm2_pi, h->tm2_cs, a));
  }
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  h->cur ^= 1;
  return LPC_OK;   // the sweeps store every ghost image themselves: the shell stays valid
}

int launch_step2(lpc_lattice* h) { return h->cfg.precision ? launch_step2_t<float>(h) : launch_step2_t<double>(h); }

template <typename T>
int set_g_from(lpc_lattice* h, const void* g) {
  T* f = wsp<T>(h, h->cur ? h->off.f1 : h->off.f0);
  int rc = for_chunks_in(h, g, 16, [&](const void* d, long long i0, long long n) {
    set_h_kernel<T><<<aux_grid(n), 256, 0, h->stream>>>(static_cast<const double*>(d), i0, n, h->L, wsp<T>(h, h->off.pi), f);
    CUDA_TRY(cudaGetLastError());
    h->launches++;
    return LPC_OK;
  });
  if (rc) return rc;
  reduce_g_kernel<T><<<aux_grid(h->N), 256, 0, h->stream>>>(h->L, wsp<T>(h, h->off.pi), f, wsp<double>(h, h->off.partials),
                                                             wsp<Ctl>(h, h->off.ctl), wsp<double2>(h, h->off.fid));
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  return LPC_OK;
}

// Pass 1 of the precompute: e_i = exp(-dF_i) on open sites into the dense scratch (which aliases the back
// buffer) and their fixed-order sum into ctl->zsum.  dF and blocked travel through the staging buffer together.
int boltzmann_pass(lpc_lattice* h, const double* dF, const uint8_t* blocked, Ctl* hc) {
  Ctl* ctl = wsp<Ctl>(h, h->off.ctl);
  double* e = wsp<double>(h, h->off.f1);
  const bool dev_in = is_device_ptr(dF) && is_device_ptr(blocked);
  if (dev_in) {
    boltzmann_factor_kernel<<<aux_grid(h->N), 256, 0, h->stream>>>(dF, blocked, 0, h->N, e, ctl);
    CUDA_TRY(cudaGetLastError());
    h->launches++;
  } else {
    // as for_chunks_in: two halves of the staging region, ordered by the stream alone
    const long long chunk = stage_chunk_sites(h->N);
    const size_t half_bytes = (size_t)chunk * 16;
    int half = 0;
    for (long long i0 = 0; i0 < h->N; i0 += chunk) {
      const long long n = std::min(chunk, h->N - i0);
      unsigned char* stg = h->ws + h->off.staging + (size_t)half * half_bytes;
      CUDA_TRY(cudaMemcpyAsync(stg, dF + i0, (size_t)n * 8, cudaMemcpyDefault, h->stream));
      CUDA_TRY(cudaMemcpyAsync(stg + (size_t)chunk * 8, blocked + i0, (size_t)n, cudaMemcpyDefault, h->stream));
      boltzmann_factor_kernel<<<aux_grid(n), 256, 0, h->stream>>>(reinterpret_cast<const double*>(stg), stg + (size_t)chunk * 8, i0, n, e,
                                                                   ctl);
      CUDA_TRY(cudaGetLastError());
      h->launches++;
      half ^= 1;
    }
  }
  sum_kernel<<<aux_grid(h->N), 256, 0, h->stream>>>(e, h->N, wsp<double>(h, h->off.partials), ctl);
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  CUDA_TRY(cudaMemcpyAsync(hc, ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (hc->bad != 0) return fail(LPC_EINVAL, "exp(-dF) under- or overflows on %llu open sites: the spread of dF is too wide", hc->bad);
  return LPC_OK;
}

// Initial state: h = 1 (g(0) = pi), r = 1, q^d(1), and the sums G[0], Z_d[1]; uses the link weights if they are set.
template <typename T>
int init_state_t(lpc_lattice* h) {
  const Layout& L = h->L;
  Ctl* ctl = wsp<Ctl>(h, h->off.ctl);
  h->cur = 0;
  T* f = wsp<T>(h, h->off.f0);
  auto init = [&](auto kern) {
    kern<<<aux_grid(h->N), 256, 0, h->stream>>>(L, wsp<T>(h, h->off.pi), mlink_of<T>(h), (T)(h->cfg.alpha / 6.0), f, h->cfg.a,
                                                 wsp<double>(h, h->off.partials), ctl, wsp<double2>(h, h->off.fid),
                                                 wsp<double>(h, h->off.vacf), h->cfg.max_steps + 2,
                                                 h->cfg.a * h->cfg.a * h->cfg.alpha / 6.0);
  };
  if (h->nrho == 0 && h->nmom == 0) init(init_state_kernel<T, 0, 0>);
  else if (h->nrho == 1 && h->nmom == 0) init(init_state_kernel<T, 1, 0>);
  else if (h->nrho == 0 && h->nmom == 3) init(init_state_kernel<T, 0, 3>);
  else init(init_state_kernel<T, 1, 3>);
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  return LPC_OK;
}

template <typename T>
int set_site_params_t(lpc_lattice* h, const double* dF, const uint8_t* blocked, const double* omega, const void* g0) {
  const Layout& L = h->L;
  Ctl* ctl = wsp<Ctl>(h, h->off.ctl);
  CUDA_TRY(cudaMemsetAsync(h->ws, 0, h->off.staging, h->stream));  // ghosts, series, control block, state: all zero
  double* e = wsp<double>(h, h->off.f1);                            // dense scratch for exp(-dF), aliases the back buffer
  Ctl hc;
  int rc = boltzmann_pass(h, dF, blocked, &hc);
  if (rc) return rc;
  if (h->z_override > 0.0) {
    // slab mode: Eq. 2 normalises over the whole lattice, the caller supplies that sum
    hc.zsum = h->z_override;
    CUDA_TRY(cudaMemcpyAsync(&ctl->zsum, &h->z_override, sizeof(double), cudaMemcpyHostToDevice, h->stream));
  }
  if (!(hc.zsum > 0.0) || !std::isfinite(hc.zsum)) return fail(LPC_EINVAL, "every site is blocked (sum of Boltzmann factors = %g)", hc.zsum);

  // pass 2: pi, kappa, phase factors
  rc = for_chunks_in(h, omega, 8, [&](const void* d, long long i0, long long n) {
    site_params_kernel<T><<<aux_grid(n), 256, 0, h->stream>>>(e, static_cast<const double*>(d), i0, n, L, h->cfg.dt, ctl,
                                                               wsp<T>(h, h->off.pi), wsp<T>(h, h->off.cs));
    CUDA_TRY(cudaGetLastError());
    h->launches++;
    return LPC_OK;
  });
  if (rc) return rc;
  CUDA_TRY(cudaMemcpyAsync(&hc, ctl, sizeof(Ctl), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (hc.bad != 0)
    return fail(LPC_EINVAL, "the equilibrium density underflows on %llu open sites: the spread of dF is too wide for %s", hc.bad,
                h->cfg.precision ? "fp32" : "fp64");
  h->phase_small = (hc.wide_phase == 0);
  {
    // ghosts of pi (wrapped value, or 0 beyond a wall) and of cos, sin (the two-step sweep rotates ghost sites too)
    const long long cells = ghost_cells(L);
    fill_ghosts_kernel<T><<<aux_grid(cells), 256, 0, h->stream>>>(wsp<T>(h, h->off.pi), 1, L, xghost_mode(h), h->cfg.bc[1] == 0,
                                                                   h->cfg.bc[2] == 0);
    CUDA_TRY(cudaGetLastError());
    fill_ghosts_kernel<T><<<aux_grid(2 * cells), 256, 0, h->stream>>>(wsp<T>(h, h->off.cs), 2, L, xghost_mode(h), h->cfg.bc[1] == 0,
                                                                       h->cfg.bc[2] == 0);
    CUDA_TRY(cudaGetLastError());
    h->launches += 2;
  }
  // the scratch aliased the back buffer: clear it again so that its ghosts and carbon sites are 0
  CUDA_TRY(cudaMemsetAsync(h->ws + h->off.f1, 0, (size_t)h->C * L.np * h->sT, h->stream));

  // initial state
  rc = init_state_t<T>(h);
  if (rc) return rc;
  if (g0) {
    rc = set_g_from<T>(h, g0);
    if (rc) return rc;
  }
  rc = fill_state_ghosts<T>(h);
  if (rc) return rc;
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  h->steps = 0;
  h->have_params = true;
  return LPC_OK;
}

// Per-link mobility factors: stored link weights m_{i,+d} = alpha_{i,i+e_d} min(pi_i, pi_{i+e_d}), then the initial state again
// (q^d(1) and Z_d[1] depend on the hop probabilities).
template <typename T>
int set_link_mobility_t(lpc_lattice* h, const double* alpha_link) {
  const Layout& L = h->L;
  Ctl* ctl = wsp<Ctl>(h, h->off.ctl);
  h->have_links = false;
  int rc;
  if (alpha_link) {
    T* m = wsp<T>(h, h->off.mlink);
    CUDA_TRY(cudaMemsetAsync(m, 0, (size_t)3 * L.np * sizeof(T), h->stream));
    CUDA_TRY(cudaMemsetAsync(&ctl->bad, 0, sizeof(ctl->bad), h->stream));
    const long long stride[3] = {L.sx, L.sy, 1};
    for (int d = 0; d < 3; ++d) {
      rc = for_chunks_in(h, alpha_link + (size_t)d * h->N, 8, [&](const void* src, long long i0, long long n) {
        link_weights_kernel<T><<<aux_grid(n), 256, 0, h->stream>>>(static_cast<const double*>(src), i0, n, L, stride[d],
                                                                    wsp<T>(h, h->off.pi), m + (long long)d * L.np, ctl);
        CUDA_TRY(cudaGetLastError());
        h->launches++;
        return LPC_OK;
      });
      if (rc) return rc;
    }
    const long long cells = ghost_cells(L) * 3;
    fill_ghosts_kernel<T><<<aux_grid(cells), 256, 0, h->stream>>>(m, 3, L, h->cfg.bc[0] == 0, h->cfg.bc[1] == 0, h->cfg.bc[2] == 0);
    CUDA_TRY(cudaGetLastError());
    h->launches++;
    unsigned long long bad = 0;
    CUDA_TRY(cudaMemcpyAsync(&bad, &ctl->bad, sizeof(bad), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    if (bad) return fail(LPC_EINVAL, "%llu link factors lie outside [0, 1]", bad);
    h->have_links = true;
  }
  CUDA_TRY(cudaMemsetAsync(h->ws + h->off.f0, 0, (size_t)h->C * L.np * h->sT, h->stream));
  CUDA_TRY(cudaMemsetAsync(h->ws + h->off.f1, 0, (size_t)h->C * L.np * h->sT, h->stream));
  rc = init_state_t<T>(h);
  if (rc) return rc;
  rc = fill_state_ghosts<T>(h);
  if (rc) return rc;
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

template <typename T>
int read_field_t(lpc_lattice* h, int which, void* out) {
  const Layout& L = h->L;
  const T* f = wsp<T>(h, h->cur ? h->off.f1 : h->off.f0);
  int mode;
  const T* ch;
  size_t bps = 8;
  if (which == LPC_FIELD_G) { mode = 0; ch = f; bps = 16; }
  else if (which == LPC_FIELD_PI) { mode = 1; ch = f; }
  else if (which >= LPC_FIELD_PX && which <= LPC_FIELD_PZ) {
    if (h->nmom != 3) return fail(LPC_ESTATE, "moment fields are not propagated (n_moments = 0)");
    mode = 2; ch = f + (long long)(2 + h->nrho + (which - LPC_FIELD_PX)) * L.np;
  } else if (which == LPC_FIELD_RHO) {
    if (h->nrho != 1) return fail(LPC_ESTATE, "the density field is not propagated (n_density = 0)");
    mode = 2; ch = f + 2 * L.np;
  } else return fail(LPC_EINVAL, "unknown field %d", which);
  const T* pi = wsp<T>(h, h->off.pi);
  if (is_device_ptr(out)) {
    gather_field_kernel<T><<<aux_grid(h->N), 256, 0, h->stream>>>(mode, 0, h->N, L, pi, ch, static_cast<double*>(out));
    CUDA_TRY(cudaGetLastError());
    h->launches++;
  } else {
    const long long chunk = stage_chunk_sites(h->N);
    int half = 0;
    for (long long i0 = 0; i0 < h->N; i0 += chunk) {
      const long long n = std::min(chunk, h->N - i0);
      double* stg = wsp<double>(h, h->off.staging) + (size_t)half * chunk * 2;
      gather_field_kernel<T><<<aux_grid(n), 256, 0, h->stream>>>(mode, i0, n, L, pi, ch, stg);
      CUDA_TRY(cudaGetLastError());
      h->launches++;
      CUDA_TRY(cudaMemcpyAsync(static_cast<unsigned char*>(out) + (size_t)i0 * bps, stg, (size_t)n * bps, cudaMemcpyDeviceToHost, h->stream));
      half ^= 1;
    }
  }
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

template <typename T>
int set_state_t(lpc_lattice* h, int which, const void* in) {
  int rc;
  if (which == LPC_FIELD_G) {
    rc = set_g_from<T>(h, in);
    if (rc) return rc;
    h->steps = 0;
    if (h->have_regions) {
      h->region_first = 0;
      rc = region_reduce_t<T>(h, 0);
      if (rc) return rc;
    }
  } else if (which == LPC_FIELD_RHO) {
    if (h->nrho != 1) return fail(LPC_ESTATE, "the density field is not propagated (n_density = 0)");
    T* ch = wsp<T>(h, h->cur ? h->off.f1 : h->off.f0) + 2 * h->L.np;
    rc = for_chunks_in(h, in, 8, [&](const void* d, long long i0, long long n) {
      set_real_kernel<T><<<aux_grid(n), 256, 0, h->stream>>>(static_cast<const double*>(d), i0, n, h->L, wsp<T>(h, h->off.pi), ch);
      CUDA_TRY(cudaGetLastError());
      h->launches++;
      return LPC_OK;
    });
    if (rc) return rc;
  } else {
    return fail(LPC_EINVAL, "field %d cannot be set", which);
  }
  rc = fill_state_ghosts<T>(h);
  if (rc) return rc;
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

template <typename T>
int equilibrate_t(lpc_lattice* h, double threshold, int64_t max_iters, int64_t check_every, int64_t* iters_done, double* last_delta) {
  const Layout& L = h->L;
  Ctl* ctl = wsp<Ctl>(h, h->off.ctl);
  T* ch[2] = {wsp<T>(h, h->off.f0) + 2 * L.np, wsp<T>(h, h->off.f1) + 2 * L.np};  // density channel of F0 / F1
  int src = h->cur;  // the current state buffer holds rho(t)
  CUDA_TRY(cudaMemsetAsync(&ctl->scratch[4], 0, 2 * sizeof(double), h->stream));
  EquilArgs<T> a;
  a.L = L;
  a.pi = wsp<T>(h, h->off.pi);
  a.mlink = mlink_of<T>(h);
  a.a6 = (T)(h->cfg.alpha / 6.0);
  a.partials = wsp<double>(h, h->off.partials);
  a.ctl = ctl;
  for (int d = 0; d < 3; ++d) a.per[d] = h->cfg.bc[d] == 0;
  const long long npairs = (long long)((L.nz + 1) / 2) * L.ny * L.nx;
  const int grid = (int)std::max<long long>(1, std::min<long long>((npairs + 255) / 256, DIRECT_MAX_BLOCKS));
  // The same sweep on the TMA march (the density channel alone: NH = 0, NRHO = 1), unless the direct kernel is asked for
  const bool use_tma = h->tma_ok && h->kernel != LPC_KERNEL_DIRECT;
  StepArgs<T> sa;
  sa.L = L; sa.fin = nullptr; sa.pi = a.pi; sa.cs = wsp<T>(h, h->off.cs); sa.mlink = a.mlink; sa.a6 = a.a6;
  sa.partials = a.partials; sa.ctl = ctl; sa.fid = nullptr; sa.vacf = nullptr; sa.vacf_stride = 0; sa.zscale = 0.0;
  for (int d = 0; d < 3; ++d) sa.per[d] = a.per[d];
  sa.peer[0] = sa.peer[1] = nullptr; sa.peer_stride[0] = sa.peer_stride[1] = 0;
  sa.label = nullptr; sa.rpartials = nullptr; sa.fidr = nullptr; sa.fidr_stride = 0; sa.region_sample = 0; sa.n_regions = 0;
  sa.vacfr = nullptr; sa.wr = nullptr; sa.vacfr_stride = 0;
  sa.c0 = 2; sa.xc = h->xc; sa.tiles_z = h->tiles_z; sa.tiles_y = h->tiles_y; sa.chunks_x = h->chunks_x;
  constexpr int VW = 16 / (int)sizeof(T), TY = sizeof(T) == 8 ? LPC_TY64 : 4 * VW;
  using KP = TmaCfg<T, 0, 1, 0, TY, 64, 4, 0, VW>;
  using KL = TmaCfg<T, 0, 1, 0, TY, 64, 4, 1, VW>;
  if (use_tma) {
    static bool attr_done[MAX_DEVICES] = {}, attr_done_l[MAX_DEVICES] = {};
    if (int rc = ensure_dyn_smem(step_tma_kernel<T, 0, 1, 0, TY, 64, 4, VW>, KP::SMEM_BYTES, h->device, attr_done)) return rc;
    if (int rc = ensure_dyn_smem(step_tma_links_kernel<T, 0, 1, 0, TY, 64, 4, VW>, KL::SMEM_BYTES, h->device, attr_done_l)) return rc;
  }
  h->ghosts_full = false;
  const unsigned tgrid = (unsigned)(h->tiles_z * h->tiles_y * h->chunks_x);
  int64_t done = 0;
  double delta = 0.0;
  while (done < max_iters) {
    const int64_t batch = std::min<int64_t>(check_every, max_iters - done);
    for (int64_t k = 0; k < batch; ++k) {
      if (use_tma) {
        sa.fout = ch[src ^ 1];
        if (h->have_links)
          CUDA_TRY(launch_sweep(h, step_tma_links_kernel<T, 0, 1, 0, TY, 64, 4, VW>, tgrid, KL::NTHREADS, KL::SMEM_BYTES, h->tm_r[src], h->tm_cs, h->tm_l, sa));
        else
          CUDA_TRY(launch_sweep(h, step_tma_kernel<T, 0, 1, 0, TY, 64, 4, VW>, tgrid, KP::NTHREADS, KP::SMEM_BYTES, h->tm_r[src], h->tm_pi, h->tm_cs, sa));
      } else {
        a.rin = ch[src];
        a.rout = ch[src ^ 1];
        equil_kernel<T><<<grid, 256, 0, h->stream>>>(a);
      }
      CUDA_TRY(cudaGetLastError());
      h->launches++;
      src ^= 1;
    }
    done += batch;
    CUDA_TRY(cudaMemcpyAsync(&delta, &ctl->scratch[4], sizeof(double), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    if (delta < threshold) break;
  }
  // the other channels live in buffer `cur`: bring the density back there if it ended in the other one
  if (src != h->cur) CUDA_TRY(cudaMemcpyAsync(ch[h->cur], ch[src], (size_t)L.np * sizeof(T), cudaMemcpyDeviceToDevice, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (iters_done) *iters_done = done;
  if (last_delta) *last_delta = delta;
  return LPC_OK;
}

template <typename T>
int seed_from_density_t(lpc_lattice* h) {
  const Layout& L = h->L;
  T* f = wsp<T>(h, h->cur ? h->off.f1 : h->off.f0);
  seed_h_from_r_kernel<T><<<aux_grid(L.np), 256, 0, h->stream>>>(L.np, f + 2 * L.np, f, f + L.np);
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  reduce_g_kernel<T><<<aux_grid(h->N), 256, 0, h->stream>>>(L, wsp<T>(h, h->off.pi), f, wsp<double>(h, h->off.partials),
                                                             wsp<Ctl>(h, h->off.ctl), wsp<double2>(h, h->off.fid));
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  h->steps = 0;
  if (h->have_regions) {
    h->region_first = 0;
    int rc = region_reduce_t<T>(h, 0);
    if (rc) return rc;
  }
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

}  // namespace

// ================================================================================================
extern "C" {

const char* lpc_last_error(void) { return g_err; }

int lpc_workspace_bytes(const lpc_config* cfg, size_t* bytes) {
  int rc = check_cfg(cfg);
  if (rc) return rc;
  if (!bytes) return fail(LPC_EINVAL, "bytes is NULL");
  *bytes = make_offsets(cfg, make_layout(cfg)).total;
  return LPC_OK;
}

int lpc_create_lattice(const lpc_config* cfg, void* workspace_dev, size_t bytes, lpc_lattice** out) {
  int rc = check_cfg(cfg);
  if (rc) return rc;
  if (!out) return fail(LPC_EINVAL, "out is NULL");
  *out = nullptr;
  if (!workspace_dev) return fail(LPC_EINVAL, "workspace is NULL");
  int dev = 0, major = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&major, cudaDevAttrComputeCapabilityMajor, dev));
  if (major != 10) return fail(LPC_ECUDA, "liblpc is built for sm_100a only; device %d has compute capability major %d", dev, major);
  lpc_lattice* h = new (std::nothrow) lpc_lattice();
  if (!h) return fail(LPC_ENOMEM, "host allocation failed");
  h->cfg = *cfg;
  h->L = make_layout(cfg);
  h->off = make_offsets(cfg, h->L);
  if (bytes < h->off.total) {
    delete h;
    return fail(LPC_ENOMEM, "workspace of %zu bytes is smaller than the %zu needed", bytes, make_offsets(cfg, make_layout(cfg)).total);
  }
  if (reinterpret_cast<uintptr_t>(workspace_dev) % ALIGN != 0) {
    delete h;
    return fail(LPC_ENOMEM, "workspace must be %zu-byte aligned", ALIGN);
  }
  if (!is_device_ptr(workspace_dev)) {
    delete h;
    return fail(LPC_EINVAL, "workspace is not device memory");
  }
  h->nrho = cfg->n_density;
  h->nmom = cfg->n_moments;
  h->C = 2 + h->nrho + h->nmom;
  h->sT = cfg->precision ? 4 : 8;
  h->N = (long long)cfg->nx * cfg->ny * cfg->nz;
  h->ws = static_cast<unsigned char*>(workspace_dev);
  h->stream = static_cast<cudaStream_t>(cfg->stream);
  h->have_params = false;
  h->have_regions = false;
  h->region_moments = false;
  h->have_links = false;
  h->regions_fused = false;
  h->halo = cfg->bc[0] == LPC_BC_HALO;
  h->halo_ready = false;
  h->z_override = 0.0;
  for (int s = 0; s < 2; ++s) h->peer[s][0] = h->peer[s][1] = nullptr, h->peer_stride[s] = 0;
  h->region_first = 0;
  h->cur = 0;
  h->steps = 0;
  h->launches = 0;
  h->kernel = LPC_KERNEL_AUTO;
  h->device = dev;
  h->time_block = 0;
  h->ghosts_full = false;
  h->opt_xc = h->opt_persist_mb = h->opt_region_fusion = h->opt_full_phase = h->opt_serial_launch = 0;
  h->phase_small = false;
  tma_geometry(h->C, cfg->precision == 1, cfg->nx, cfg->ny, cfg->nz, 0, &h->ty, &h->tz, &h->nstage, &h->xc, &h->tiles_z, &h->tiles_y, &h->chunks_x);
  h->tma_ok = (size_t)h->tiles_z * h->tiles_y * h->chunks_x <= h->off.partial_slots;
  {
    int ty, tz, ns, tzs, tys;
    tma_geometry(h->C, cfg->precision == 1, cfg->nx, cfg->ny, cfg->nz, 0, &ty, &tz, &ns, &h->xc_reg, &tzs, &tys, &h->chunks_x_reg, 64);
  }
  // two steps per sweep: the magnetisation channels alone, no slab, and every periodic axis long enough for two ghost layers
  h->ty2 = 8; h->tz2 = 32 * (16 / h->sT);
  h->tiles_z2 = (cfg->nz + h->tz2 - 1) / h->tz2;
  h->tiles_y2 = (cfg->ny + h->ty2 - 1) / h->ty2;
  step2_geometry(cfg->nx, (long long)h->tiles_z2 * h->tiles_y2, 0, &h->xc2, &h->chunks_x2);
  h->step2_ok = h->tma_ok && h->nrho == 0 && !(h->halo && cfg->nx < 2) &&
                (size_t)h->tiles_z2 * h->tiles_y2 * h->chunks_x2 <= h->off.partial_slots;
  for (int d = 0; d < 3; ++d) {
    const int n = d == 0 ? cfg->nx : d == 1 ? cfg->ny : cfg->nz;
    if (cfg->bc[d] == 0 && n < 4) h->step2_ok = false;
  }
  if (h->tma_ok) {
    const Layout& L = h->L;
    const bool f32 = cfg->precision == 1;
    const cuuint64_t d4[4] = {(cuuint64_t)L.nzp, (cuuint64_t)L.nyp, (cuuint64_t)L.nxp, (cuuint64_t)h->C};
    const cuuint32_t b4[4] = {(cuuint32_t)(h->tz + 2 * (16 / h->sT)), (cuuint32_t)(h->ty + 2), 1, (cuuint32_t)h->C};
    const cuuint64_t dk[4] = {(cuuint64_t)L.nzp, (cuuint64_t)L.nyp, (cuuint64_t)L.nxp, 2};
    const cuuint32_t bk[4] = {(cuuint32_t)h->tz, (cuuint32_t)h->ty, 1, 2};
    // the channel dimension of the box: the magnetisation (+ density) channels, and the 3 moment channels
    const cuuint32_t bf[4] = {b4[0], b4[1], 1, (cuuint32_t)(2 + h->nrho)};
    const cuuint32_t bm[4] = {b4[0], b4[1], 1, 3};
    rc = encode_map(&h->tm_f[0], f32, h->ws + h->off.f0, 4, d4, bf);
    if (!rc) rc = encode_map(&h->tm_f[1], f32, h->ws + h->off.f1, 4, d4, bf);
    if (!rc && h->nmom == 3) rc = encode_map(&h->tm_m[0], f32, h->ws + h->off.f0, 4, d4, bm);
    if (!rc && h->nmom == 3) rc = encode_map(&h->tm_m[1], f32, h->ws + h->off.f1, 4, d4, bm);
    const cuuint32_t br[4] = {b4[0], b4[1], 1, 1};
    if (!rc && h->nrho == 1) rc = encode_map(&h->tm_r[0], f32, h->ws + h->off.f0, 4, d4, br);
    if (!rc && h->nrho == 1) rc = encode_map(&h->tm_r[1], f32, h->ws + h->off.f1, 4, d4, br);
    if (!rc) rc = encode_map(&h->tm_pi, f32, h->ws + h->off.pi, 3, d4, b4);
    if (!rc) rc = encode_map(&h->tm_cs, f32, h->ws + h->off.cs, 4, dk, bk);
    const cuuint32_t bs[4] = {bk[0], bk[1], 1, 1};   // the sine channel alone
    if (!rc) rc = encode_map(&h->tm_sn, f32, h->ws + h->off.cs, 4, dk, bs);
    if (!rc && h->step2_ok) {
      // the two-step sweep: h and pi with two halo rows / one 16-byte halo group, cos and sin with one halo row
      const cuuint32_t zw = (cuuint32_t)(h->tz2 + 2 * (16 / h->sT));
      const cuuint32_t b2f[4] = {zw, (cuuint32_t)(h->ty2 + 4), 1, 2};
      const cuuint32_t b2k[4] = {zw, (cuuint32_t)(h->ty2 + 2), 1, 2};
      rc = encode_map(&h->tm2_f[0], f32, h->ws + h->off.f0, 4, d4, b2f);
      if (!rc) rc = encode_map(&h->tm2_f[1], f32, h->ws + h->off.f1, 4, d4, b2f);
      const cuuint32_t b2m[4] = {zw, (cuuint32_t)(h->ty2 + 4), 1, 3};
      if (!rc && h->nmom == 3) rc = encode_map(&h->tm2_m[0], f32, h->ws + h->off.f0, 4, d4, b2m);
      if (!rc && h->nmom == 3) rc = encode_map(&h->tm2_m[1], f32, h->ws + h->off.f1, 4, d4, b2m);
      if (!rc) rc = encode_map(&h->tm2_pi, f32, h->ws + h->off.pi, 3, d4, b2f);
      if (!rc) rc = encode_map(&h->tm2_cs, f32, h->ws + h->off.cs, 4, dk, b2k);
      const cuuint32_t b2s[4] = {zw, (cuuint32_t)(h->ty2 + 2), 1, 1};
      if (!rc) rc = encode_map(&h->tm2_sn, f32, h->ws + h->off.cs, 4, dk, b2s);
    }
    if (!rc && cfg->link_mobility) {
      // pi centres and m_x: the tile itself; m_y: one more row below; m_z: 16 bytes of columns below
      const size_t chan = (size_t)L.np * h->sT;
      const cuuint32_t bc[3] = {(cuuint32_t)h->tz, (cuuint32_t)h->ty, 1};
      const cuuint32_t by[3] = {(cuuint32_t)h->tz, (cuuint32_t)(h->ty + 1), 1};
      const cuuint32_t bz[3] = {(cuuint32_t)(h->tz + 16 / h->sT), (cuuint32_t)h->ty, 1};
      rc = encode_map(&h->tm_l.pic, f32, h->ws + h->off.pi, 3, d4, bc);
      if (!rc) rc = encode_map(&h->tm_l.mx, f32, h->ws + h->off.mlink, 3, d4, bc);
      if (!rc) rc = encode_map(&h->tm_l.my, f32, h->ws + h->off.mlink + chan, 3, d4, by);
      if (!rc) rc = encode_map(&h->tm_l.mz, f32, h->ws + h->off.mlink + 2 * chan, 3, d4, bz);
    }
    if (rc) {
      delete h;
      return rc;
    }
  }
  *out = h;
  return LPC_OK;
}

int lpc_set_site_params(lpc_lattice* h, const double* dF, const uint8_t* blocked, const double* omega, const void* g0) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!dF || !blocked || !omega) return fail(LPC_EINVAL, "dF, blocked and omega must not be NULL");
  h->have_params = false;
  h->have_regions = false;
  h->region_moments = false;
  h->have_links = false;
  h->halo_ready = false;
  return h->cfg.precision ? set_site_params_t<float>(h, dF, blocked, omega, g0) : set_site_params_t<double>(h, dF, blocked, omega, g0);
}

int lpc_set_link_mobility(lpc_lattice* h, const double* alpha_link) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (!h->cfg.link_mobility) return fail(LPC_ESTATE, "the lattice was created without link_mobility = 1");
  if (h->steps != 0) return fail(LPC_ESTATE, "link factors must be set before the first step");
  h->have_regions = false;
  h->region_moments = false;
  return h->cfg.precision ? set_link_mobility_t<float>(h, alpha_link) : set_link_mobility_t<double>(h, alpha_link);
}

int lpc_partition_sum(lpc_lattice* h, const double* dF, const uint8_t* blocked, double* out) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!dF || !blocked || !out) return fail(LPC_EINVAL, "dF, blocked and out must not be NULL");
  // the pass uses the back buffer as scratch: whatever the lattice held is gone
  h->have_params = false;
  h->halo_ready = false;
  CUDA_TRY(cudaMemsetAsync(h->ws, 0, h->off.staging, h->stream));
  Ctl hc;
  int rc = boltzmann_pass(h, dF, blocked, &hc);
  if (rc) return rc;
  *out = hc.zsum;
  return LPC_OK;
}

int lpc_set_partition_sum(lpc_lattice* h, double Z) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!std::isfinite(Z)) return fail(LPC_EINVAL, "Z is not finite");
  h->z_override = Z > 0.0 ? Z : 0.0;
  return LPC_OK;
}

int lpc_halo_view(lpc_lattice* h, int32_t set, int32_t side, int32_t role, void** plane, size_t* plane_bytes, size_t* stride_bytes,
                  int32_t* n_channels) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (set < LPC_HALO_PARAMS || set > LPC_HALO_PHASE2 || (side != 0 && side != 1) || (role != LPC_HALO_SEND && role != LPC_HALO_RECV))
    return fail(LPC_EINVAL, "bad selector (set %d, side %d, role %d)", set, side, role);
  if (!plane || !plane_bytes || !stride_bytes || !n_channels) return fail(LPC_EINVAL, "output pointers must not be NULL");
  const Layout& L = h->L;
  if (set >= LPC_HALO_STATE2) {
    // two planes per face, one contiguous run: owned planes gh, gh+1 / gh+nx-2, gh+nx-1; ghost planes 0, 1 / gh+nx, gh+nx+1
    if (L.nx < 2) return fail(LPC_ESTATE, "a two-plane halo needs at least two owned planes");
    const long long xp2 = side == 0 ? (role == LPC_HALO_SEND ? L.gh : L.gh - 2) : (role == LPC_HALO_SEND ? L.gh + L.nx - 2 : L.gh + L.nx);
    const size_t base2 = set == LPC_HALO_PARAMS2 ? h->off.pi : set == LPC_HALO_PHASE2 ? h->off.cs : (h->cur ? h->off.f1 : h->off.f0);
    *plane = h->ws + base2 + (size_t)xp2 * L.sx * h->sT;
    *plane_bytes = 2 * (size_t)L.sx * h->sT;
    *stride_bytes = (size_t)L.np * h->sT;
    *n_channels = set == LPC_HALO_PARAMS2 ? 1 : set == LPC_HALO_PHASE2 ? 2 : h->C;
    return LPC_OK;
  }
  // padded x index: ghost planes 0 .. gh-1, owned gh .. gh+nx-1, ghost planes gh+nx ..; the exchange moves the innermost ghost plane
  const long long xp = side == 0 ? (role == LPC_HALO_SEND ? L.gh : L.gh - 1) : (role == LPC_HALO_SEND ? L.gh + L.nx - 1 : L.gh + L.nx);
  const size_t base = set == LPC_HALO_PARAMS ? h->off.pi
                    : set == LPC_HALO_STATE0 ? h->off.f0
                    : set == LPC_HALO_STATE1 ? h->off.f1
                                             : (h->cur ? h->off.f1 : h->off.f0);
  *plane = h->ws + base + (size_t)xp * L.sx * h->sT;
  *plane_bytes = (size_t)L.sx * h->sT;
  *stride_bytes = (size_t)L.np * h->sT;
  *n_channels = set == LPC_HALO_PARAMS ? 1 : h->C;
  return LPC_OK;
}

int lpc_set_halo_peers(lpc_lattice* h, void* lo0, void* lo1, size_t lo_stride, void* hi0, void* hi1, size_t hi_stride) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->halo) return fail(LPC_ESTATE, "the lattice was not created with bc[0] = LPC_BC_HALO");
  if ((lo0 == nullptr) != (lo1 == nullptr) || (hi0 == nullptr) != (hi1 == nullptr))
    return fail(LPC_EINVAL, "give both buffers of a neighbour or neither");
  if ((lo0 && lo_stride % h->sT) || (hi0 && hi_stride % h->sT)) return fail(LPC_EINVAL, "channel stride is not a multiple of the element size");
  if ((lo0 || hi0) && !h->tma_ok) return fail(LPC_ESTATE, "direct halo stores need the TMA kernel, which this lattice cannot run");
  h->peer[0][0] = static_cast<unsigned char*>(lo0); h->peer[0][1] = static_cast<unsigned char*>(lo1); h->peer_stride[0] = lo_stride;
  h->peer[1][0] = static_cast<unsigned char*>(hi0); h->peer[1][1] = static_cast<unsigned char*>(hi1); h->peer_stride[1] = hi_stride;
  return LPC_OK;
}

int lpc_ipc_export(lpc_lattice* h, void* handle_out, size_t* offset_out) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!handle_out || !offset_out) return fail(LPC_EINVAL, "output pointers must not be NULL");
  static_assert(sizeof(cudaIpcMemHandle_t) == LPC_IPC_HANDLE_BYTES, "LPC_IPC_HANDLE_BYTES is the size of a cudaIpcMemHandle_t");
  // the handle names the whole allocation the workspace lies in: find its base
  typedef CUresult (*RangeFn)(CUdeviceptr*, size_t*, CUdeviceptr);
  static RangeFn range_fn = nullptr;
  if (!range_fn) {
    void* p = nullptr;
    cudaDriverEntryPointQueryResult q;
    CUDA_TRY(cudaGetDriverEntryPoint("cuMemGetAddressRange", &p, cudaEnableDefault, &q));
    if (q != cudaDriverEntryPointSuccess || !p) return fail(LPC_ECUDA, "cuMemGetAddressRange not available in this driver");
    range_fn = reinterpret_cast<RangeFn>(p);
  }
  CUdeviceptr base = 0;
  size_t size = 0;
  const CUresult r = range_fn(&base, &size, reinterpret_cast<CUdeviceptr>(h->ws));
  if (r != CUDA_SUCCESS) return fail(LPC_ECUDA, "cuMemGetAddressRange failed with CUresult %d", (int)r);
  cudaIpcMemHandle_t hd;
  CUDA_TRY(cudaIpcGetMemHandle(&hd, reinterpret_cast<void*>(base)));
  memcpy(handle_out, &hd, sizeof(hd));
  *offset_out = (size_t)(reinterpret_cast<CUdeviceptr>(h->ws) - base);
  return LPC_OK;
}

int lpc_ipc_open(const void* handle, void** base_out) {
  if (!handle || !base_out) return fail(LPC_EINVAL, "handle and base_out must not be NULL");
  cudaIpcMemHandle_t hd;
  memcpy(&hd, handle, sizeof(hd));
  void* p = nullptr;
  CUDA_TRY(cudaIpcOpenMemHandle(&p, hd, cudaIpcMemLazyEnablePeerAccess));
  *base_out = p;
  return LPC_OK;
}

int lpc_ipc_close(void* base) {
  if (!base) return fail(LPC_EINVAL, "base is NULL");
  CUDA_TRY(cudaIpcCloseMemHandle(base));
  return LPC_OK;
}

int lpc_slab_finish(lpc_lattice* h) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->halo) return fail(LPC_ESTATE, "the lattice was not created with bc[0] = LPC_BC_HALO");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  h->have_regions = false;
  h->region_moments = false;
  CUDA_TRY(cudaMemsetAsync(h->ws + h->off.f0, 0, (size_t)h->C * h->L.np * h->sT, h->stream));
  CUDA_TRY(cudaMemsetAsync(h->ws + h->off.f1, 0, (size_t)h->C * h->L.np * h->sT, h->stream));
  int rc = h->cfg.precision ? init_state_t<float>(h) : init_state_t<double>(h);
  if (rc) return rc;
  rc = h->cfg.precision ? fill_state_ghosts<float>(h) : fill_state_ghosts<double>(h);
  if (rc) return rc;
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  h->steps = 0;
  h->halo_ready = true;
  return LPC_OK;
}

int lpc_step_n(lpc_lattice* h, int64_t n) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (n < 0) return fail(LPC_EINVAL, "n must be >= 0");
  if (h->steps + n > h->cfg.max_steps) return fail(LPC_EINVAL, "steps_done + n = %lld exceeds max_steps = %lld", (long long)(h->steps + n), (long long)h->cfg.max_steps);
  if (h->halo && !h->halo_ready) return fail(LPC_ESTATE, "slab mode: lpc_slab_finish has not been called");
  if (h->halo && n > 1 && !(n == 2 && step2_usable(h)))
    return fail(LPC_ESTATE, "slab mode: the x ghost planes must be exchanged after every sweep (n <= 1, or n = 2 on a lattice with lpc_time_block_steps = 2 and two-plane exchanges)");
  // (never on a slab: the persistent kernel would take both steps of a two-step call without the ghost planes of the second)
  const bool persist = !h->have_regions && !h->halo && n >= 2 &&
                       (h->kernel == LPC_KERNEL_PERSIST || (h->kernel == LPC_KERNEL_AUTO && persist_by_default(h)));
  if (persist) return h->cfg.precision ? launch_persist<float>(h, n) : launch_persist<double>(h, n);
  // two steps per sweep while at least two are left (lpc_step2.cuh); an odd last step takes the one-step sweep
  if (step2_usable(h)) {
    while (n >= 2) {
      int rc = launch_step2(h);
      if (rc) return rc;
      h->steps += 2;
      n -= 2;
    }
  }
  for (int64_t k = 0; k < n; ++k) {
    if (h->region_moments && !will_fuse_regions(h)) {   // else the moment sweep books the regional VACF itself
      int rc = region_moment<false>(h);
      if (rc) return rc;
    }
    int rc = h->cfg.precision ? launch_step<float>(h) : launch_step<double>(h);
    if (rc) return rc;
    h->steps++;
    if (h->have_regions && !h->regions_fused) {
      rc = region_reduce(h, h->steps);
      if (rc) return rc;
    }
  }
  // a slab that may take two steps per sweep hands whole planes to its neighbours, y and z ghosts included: after a
  // one-step sweep bring the full shell of the owned planes up to date before the caller's exchange
  if (h->halo && n > 0 && step2_usable(h) && !h->ghosts_full) {
    int rc = h->cfg.precision ? fill_state_ghosts<float>(h) : fill_state_ghosts<double>(h);
    if (rc) return rc;
  }
  return LPC_OK;
}

int lpc_read_fid(lpc_lattice* h, int64_t first, int64_t count, double* out) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (first < 0 || count < 0 || first + count > h->steps + 1) return fail(LPC_EINVAL, "range [%lld, %lld) is outside the %lld samples of the series", (long long)first, (long long)(first + count), (long long)(h->steps + 1));
  if (count > 0 && !out) return fail(LPC_EINVAL, "out is NULL");
  if (count > 0)
    CUDA_TRY(cudaMemcpyAsync(out, wsp<double2>(h, h->off.fid) + first, (size_t)count * sizeof(double2), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

int lpc_moments(lpc_lattice* h, int64_t count, double* vacf_host, double D[3]) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (h->nmom != 3) return fail(LPC_ESTATE, "moment fields are not propagated (n_moments = 0)");
  if (count < 1 || count > h->steps + 1) return fail(LPC_EINVAL, "count must lie in [1, steps_done + 1]");
  if (!D) return fail(LPC_EINVAL, "D is NULL");
  const long long stride = h->cfg.max_steps + 2;
  double* vacf = wsp<double>(h, h->off.vacf);
  Ctl* ctl = wsp<Ctl>(h, h->off.ctl);
  diffusion_kernel<<<3, 256, 0, h->stream>>>(vacf, stride, count, h->cfg.dt, ctl);
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  CUDA_TRY(cudaMemcpyAsync(D, ctl->scratch, 3 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  if (vacf_host)
    for (int d = 0; d < 3; ++d)
      CUDA_TRY(cudaMemcpyAsync(vacf_host + (size_t)d * count, vacf + d * stride + 1, (size_t)count * sizeof(double), cudaMemcpyDeviceToHost,
                               h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

int lpc_read_field(lpc_lattice* h, int32_t which, void* out) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (!out) return fail(LPC_EINVAL, "out is NULL");
  return h->cfg.precision ? read_field_t<float>(h, which, out) : read_field_t<double>(h, which, out);
}

int lpc_set_state(lpc_lattice* h, int32_t which, const void* in) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (!in) return fail(LPC_EINVAL, "in is NULL");
  return h->cfg.precision ? set_state_t<float>(h, which, in) : set_state_t<double>(h, which, in);
}

int lpc_equilibrate(lpc_lattice* h, double threshold, int64_t max_iters, int64_t check_every, int64_t* iters_done, double* last_delta) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (h->nrho != 1) return fail(LPC_ESTATE, "the density field is not propagated (n_density = 0)");
  if (h->halo && !h->halo_ready) return fail(LPC_ESTATE, "slab mode: lpc_slab_finish has not been called");
  if (h->halo && max_iters > 1)
    return fail(LPC_ESTATE, "slab mode: the x ghost planes must be exchanged after every sweep (max_iters <= 1)");
  if (max_iters < 0) return fail(LPC_EINVAL, "max_iters must be >= 0");
  if (check_every < 1) return fail(LPC_EINVAL, "check_every must be >= 1");
  if (!(threshold == threshold)) return fail(LPC_EINVAL, "threshold is NaN");
  return h->cfg.precision ? equilibrate_t<float>(h, threshold, max_iters, check_every, iters_done, last_delta)
                          : equilibrate_t<double>(h, threshold, max_iters, check_every, iters_done, last_delta);
}

int lpc_seed_from_density(lpc_lattice* h) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (h->nrho != 1) return fail(LPC_ESTATE, "the density field is not propagated (n_density = 0)");
  return h->cfg.precision ? seed_from_density_t<float>(h) : seed_from_density_t<double>(h);
}

int lpc_set_regions(lpc_lattice* h, const uint8_t* region) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (h->cfg.n_regions < 1) return fail(LPC_ESTATE, "the lattice was created with n_regions = 0");
  if (!region) return fail(LPC_EINVAL, "region is NULL");
  CUDA_TRY(cudaMemcpyAsync(h->ws + h->off.regions, region, (size_t)h->N, cudaMemcpyDefault, h->stream));
  h->have_regions = true;
  h->region_first = h->steps;
  int rc = region_reduce(h, h->steps);
  if (rc) return rc;
  // the regional VACF needs the whole series: it is recorded when the labels arrive before the first step
  h->region_moments = (h->nmom == 3 && h->steps == 0);
  if (h->region_moments) {
    rc = region_moment<true>(h);
    if (rc) return rc;
  }
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

int lpc_read_fid_region(lpc_lattice* h, int32_t region, int64_t first, int64_t count, double* out) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (!h->have_regions) return fail(LPC_ESTATE, "lpc_set_regions has not been called");
  if (region < 0 || region >= h->cfg.n_regions) return fail(LPC_EINVAL, "region %d is outside [0, %d)", region, h->cfg.n_regions);
  if (first < h->region_first || count < 0 || first + count > h->steps + 1)
    return fail(LPC_EINVAL, "range [%lld, %lld) is outside the recorded samples [%lld, %lld]", (long long)first, (long long)(first + count),
                h->region_first, (long long)h->steps);
  if (count > 0 && !out) return fail(LPC_EINVAL, "out is NULL");
  if (count > 0)
    CUDA_TRY(cudaMemcpyAsync(out, wsp<double2>(h, h->off.fidr) + (size_t)region * (h->cfg.max_steps + 1) + first,
                             (size_t)count * sizeof(double2), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

int lpc_spectrum(lpc_lattice* h, int32_t region, int64_t count, double f0, double df, int64_t n_freq, double lb, double* out) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (count < 1 || count > h->steps + 1) return fail(LPC_EINVAL, "count must lie in [1, steps_done + 1]");
  if (n_freq < 0) return fail(LPC_EINVAL, "n_freq must be >= 0");
  if (!(lb >= 0.0) || !std::isfinite(f0) || !std::isfinite(df)) return fail(LPC_EINVAL, "lb must be >= 0 and the frequency grid finite");
  if (n_freq > 0 && !out) return fail(LPC_EINVAL, "out is NULL");
  const double2* series;
  if (region == -1) {
    series = wsp<double2>(h, h->off.fid);
  } else {
    if (!h->have_regions) return fail(LPC_ESTATE, "lpc_set_regions has not been called");
    if (region < 0 || region >= h->cfg.n_regions) return fail(LPC_EINVAL, "region %d is outside [-1, %d)", region, h->cfg.n_regions);
    if (h->region_first != 0) return fail(LPC_ESTATE, "the regional series starts at step %lld, not 0", h->region_first);
    series = wsp<double2>(h, h->off.fidr) + (size_t)region * (h->cfg.max_steps + 1);
  }
  double2* spec = wsp<double2>(h, h->off.spec);
  for (int64_t k0 = 0; k0 < n_freq; k0 += SPEC_BATCH) {
    const int64_t nb = std::min<int64_t>(SPEC_BATCH, n_freq - k0);
    spectrum_kernel<<<(unsigned)nb, 256, 0, h->stream>>>(series, count, h->cfg.dt, f0, df, k0, lb, spec);
    CUDA_TRY(cudaGetLastError());
    h->launches++;
    CUDA_TRY(cudaMemcpyAsync(out + 2 * k0, spec, (size_t)nb * sizeof(double2), cudaMemcpyDeviceToHost, h->stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
  }
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

int lpc_moments_region(lpc_lattice* h, int32_t region, int64_t count, double* vacf_host, double D[3]) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  if (h->nmom != 3) return fail(LPC_ESTATE, "moment fields are not propagated (n_moments = 0)");
  if (!h->have_regions || !h->region_moments) return fail(LPC_ESTATE, "region labels must be set before the first step to record the regional VACF");
  if (region < 0 || region >= h->cfg.n_regions) return fail(LPC_EINVAL, "region %d is outside [0, %d)", region, h->cfg.n_regions);
  if (count < 1 || count > h->steps + 1) return fail(LPC_EINVAL, "count must lie in [1, steps_done + 1]");
  if (!D) return fail(LPC_EINVAL, "D is NULL");
  const long long stride = h->cfg.max_steps + 2;
  double* vacf = wsp<double>(h, h->off.vacfr) + (size_t)region * 3 * stride;
  Ctl* ctl = wsp<Ctl>(h, h->off.ctl);
  diffusion_kernel<<<3, 256, 0, h->stream>>>(vacf, stride, count, h->cfg.dt, ctl);
  CUDA_TRY(cudaGetLastError());
  h->launches++;
  CUDA_TRY(cudaMemcpyAsync(D, ctl->scratch, 3 * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  if (vacf_host)
    for (int d = 0; d < 3; ++d)
      CUDA_TRY(cudaMemcpyAsync(vacf_host + (size_t)d * count, vacf + d * stride + 1, (size_t)count * sizeof(double), cudaMemcpyDeviceToHost,
                               h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return LPC_OK;
}

int lpc_set_kernel(lpc_lattice* h, int32_t which) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (which < LPC_KERNEL_AUTO || which > LPC_KERNEL_PERSIST) return fail(LPC_EINVAL, "unknown kernel selector %d", which);
  if (which == LPC_KERNEL_TMA && !h->tma_ok) return fail(LPC_EINVAL, "the TMA kernel is not available for this lattice");
  h->kernel = which;
  return LPC_OK;
}

int lpc_set_option(lpc_lattice* h, int32_t key, int64_t value) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (value < 0) return fail(LPC_EINVAL, "option values are >= 0");
  switch (key) {
    case LPC_OPT_TIME_BLOCK:
      if (value > 2) return fail(LPC_EINVAL, "LPC_OPT_TIME_BLOCK takes 0 (auto), 1 (one step per sweep) or 2 (two steps per sweep)");
      if (value == 2 && !h->step2_ok) return fail(LPC_EINVAL, "this lattice cannot run the two-step sweep (channels, slab mode or a periodic axis shorter than 4)");
      h->time_block = (int)value;
      return LPC_OK;
    case LPC_OPT_X_CHUNK: {
      if (value > h->cfg.nx) value = h->cfg.nx;
      h->opt_xc = (int)value;
      tma_geometry(h->C, h->cfg.precision == 1, h->cfg.nx, h->cfg.ny, h->cfg.nz, h->opt_xc, &h->ty, &h->tz, &h->nstage, &h->xc, &h->tiles_z, &h->tiles_y, &h->chunks_x);
      return LPC_OK;
    }
    case LPC_OPT_X_CHUNK2:
      if (value > h->cfg.nx) value = h->cfg.nx;
      step2_geometry(h->cfg.nx, (long long)h->tiles_z2 * h->tiles_y2, (int)value, &h->xc2, &h->chunks_x2);
      if ((size_t)h->tiles_z2 * h->tiles_y2 * h->chunks_x2 > h->off.partial_slots) {   // too many CTAs for the partial sums: back to the default
        step2_geometry(h->cfg.nx, (long long)h->tiles_z2 * h->tiles_y2, 0, &h->xc2, &h->chunks_x2);
        return fail(LPC_EINVAL, "LPC_OPT_X_CHUNK2 = %lld gives more CTAs than the workspace has partial-sum slots", (long long)value);
      }
      return LPC_OK;
    case LPC_OPT_PERSIST_MAX_MB:
      if (value > (1 << 20)) return fail(LPC_EINVAL, "LPC_OPT_PERSIST_MAX_MB is in MiB");
      h->opt_persist_mb = (int)value;
      return LPC_OK;
    case LPC_OPT_FULL_PHASE:
      if (value > 1) return fail(LPC_EINVAL, "LPC_OPT_FULL_PHASE takes 0 (sin alone where every phase angle is small) or 1 (always cos and sin)");
      h->opt_full_phase = (int)value;
      return LPC_OK;
    case LPC_OPT_SERIAL_LAUNCH:
      if (value > 1) return fail(LPC_EINVAL, "LPC_OPT_SERIAL_LAUNCH takes 0 (a sweep may start behind the one before it) or 1 (plain launches)");
      h->opt_serial_launch = (int)value;
      return LPC_OK;
    case LPC_OPT_REGION_FUSION:
      if (value > 1) return fail(LPC_EINVAL, "LPC_OPT_REGION_FUSION takes 0 (inside the sweep when possible) or 1 (separate pass)");
      h->opt_region_fusion = (int)value;
      return LPC_OK;
    default:
      return fail(LPC_EINVAL, "unknown option %d", key);
  }
}

int32_t lpc_time_block_steps(const lpc_lattice* h) { return (h && step2_usable(h)) ? 2 : 1; }
int32_t lpc_reads_sin_alone(const lpc_lattice* h) { return (h && h->have_params && sin_only(h)) ? 1 : 0; }
int64_t lpc_steps_done(const lpc_lattice* h) { return h ? h->steps : 0; }

int lpc_sync_steps(lpc_lattice* h, int64_t* steps_done) {
  if (!h) return fail(LPC_EINVAL, "lattice is NULL");
  if (!h->have_params) return fail(LPC_ESTATE, "lpc_set_site_params has not been called");
  long long s = 0;
  CUDA_TRY(cudaMemcpyAsync(&s, &wsp<Ctl>(h, h->off.ctl)->step, sizeof(s), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  if (s < 0 || s > h->cfg.max_steps)
    return fail(LPC_ESTATE, "the device has taken %lld steps but the series hold max_steps = %lld: graph replays overflowed them", s,
                (long long)h->cfg.max_steps);
  h->steps = s;
  if (steps_done) *steps_done = s;
  return LPC_OK;
}
int64_t lpc_launch_count(const lpc_lattice* h) { return h ? h->launches : 0; }

double lpc_bytes_per_site_step(const lpc_lattice* h) {
  if (!h) return 0.0;
  // read C state channels + pi + cos + sin, write C state channels; with region labels one more pass
  // reads h (2 channels), pi and the label
  // with per-link mobility factors the sweep also reads three stored link weights per site
  // region labels: one byte per site inside the sweep, or one more pass over h (2 channels), pi and the label
  const double regions = !h->have_regions ? 0.0 : regions_fusable(h) ? 1.0 : 3.0 * h->sT + 1.0;
  // lattices whose phase angles are all small: the plain magnetisation sweeps read sin alone
  const bool sn = sin_only(h) && h->tma_ok && h->kernel != LPC_KERNEL_DIRECT && h->kernel != LPC_KERNEL_PERSIST &&
                  !(h->kernel == LPC_KERNEL_AUTO && persist_by_default(h) && !h->have_regions) && h->nrho == 0 && !h->have_links;
  // moment fields on the TMA path: the step is two sweeps (moment channels, then magnetisation) and each stages pi
  const bool tma = h->tma_ok && h->kernel != LPC_KERNEL_DIRECT && h->kernel != LPC_KERNEL_PERSIST &&
                   !(h->kernel == LPC_KERNEL_AUTO && persist_by_default(h) && !h->have_regions);
  const double pi_again = (h->nmom == 3 && tma) ? 1.0 : 0.0;
  return (double)h->sT * (2.0 * h->C + (sn ? 2.0 : 3.0) + pi_again + (h->have_links ? 3.0 : 0.0)) + regions;
}

void lpc_destroy(lpc_lattice* h) { delete h; }

}  // extern "C"

// ================================================================================================
// lpc_fid_sample_noalloc: Eq. 12 of a dense complex array with NO memory of the caller's or of an
// allocator: the block partials and the ticket counter of the reduction -- what reduce_g_kernel keeps in the workspace --
// live in a file-scope device array.  Everything that touches the array is in this file: in host code its name is a
// host-side stand-in, not a device address, so the entry point asks cudaGetSymbolAddress once per device (with that
// device current) and hands the kernel the pointer it got.
// ================================================================================================
namespace {

constexpr int NA_CHUNK = 1 << 15;       // sites per block partial
constexpr int NA_MAX_BLOCKS = 8192;     // partials the array holds: LPC_NOALLOC_MAX_SITES = NA_CHUNK * NA_MAX_BLOCKS
constexpr int NA_HEADER = 256;          // the ticket counter, on a 256-byte line of its own
static_assert((long long)NA_CHUNK * NA_MAX_BLOCKS == LPC_NOALLOC_MAX_SITES, "lpc.h states the limit");
static_assert(NA_HEADER + NA_MAX_BLOCKS * (int)sizeof(double2) == LPC_NOALLOC_SCRATCH_BYTES, "lpc.h states the size");

static __device__ __align__(256) unsigned char g_noalloc_scratch[LPC_NOALLOC_SCRATCH_BYTES];

// Block b adds the sites [b NA_CHUNK, (b+1) NA_CHUNK) (thread-strided, then warp shuffles, then the warps in order) and
// stores one partial; the block that takes the last ticket adds all partials in block order and writes out[0..1].
// Deterministic: the order depends on n alone.  `scratch` is the device address of g_noalloc_scratch.
__global__ void __launch_bounds__(256) fid_sample_noalloc_kernel(const double2* __restrict__ g, long long n, unsigned char* scratch,
                                                                  double* __restrict__ out) {
  unsigned int* ticket = reinterpret_cast<unsigned int*>(scratch);
  double2* partial = reinterpret_cast<double2*>(scratch + NA_HEADER);
  __shared__ double red[2 * 8];
  __shared__ unsigned int s_last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const long long i0 = (long long)blockIdx.x * NA_CHUNK;
  const long long i1 = (i0 + NA_CHUNK < n) ? i0 + NA_CHUNK : n;
  double re = 0.0, im = 0.0;
  for (long long i = i0 + threadIdx.x; i < i1; i += blockDim.x) {
    const double2 v = g[i];
    re += v.x;
    im += v.y;
  }
  re = warp_sum(re);
  im = warp_sum(im);
  if (lane == 0) {
    red[2 * warp] = re;
    red[2 * warp + 1] = im;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double sr = 0.0, si = 0.0;
    for (int w = 0; w < 8; ++w) {
      sr += red[2 * w];
      si += red[2 * w + 1];
    }
    partial[blockIdx.x] = make_double2(sr, si);
    __threadfence();
    s_last = (atomicAdd(ticket, 1u) == gridDim.x - 1) ? 1u : 0u;
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  re = im = 0.0;
  for (unsigned int b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
    const double2 v = __ldcg(&partial[b]);
    re += v.x;
    im += v.y;
  }
  re = warp_sum(re);
  im = warp_sum(im);
  __syncthreads();   // red is reused
  if (lane == 0) {
    red[2 * warp] = re;
    red[2 * warp + 1] = im;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double sr = 0.0, si = 0.0;
    for (int w = 0; w < 8; ++w) {
      sr += red[2 * w];
      si += red[2 * w + 1];
    }
    out[0] = sr;
    out[1] = si;
    *ticket = 0u;   // (the next call clears it as well: it does not rely on this)
  }
}

}  // namespace

extern "C" int lpc_fid_sample_noalloc(const double* g, int64_t n_sites, double* out, void* stream) {
  if (!g || !out) return fail(LPC_EINVAL, "g and out must not be NULL");
  if (n_sites < 0) return fail(LPC_EINVAL, "n_sites must be >= 0");
  if (n_sites > LPC_NOALLOC_MAX_SITES)
    return fail(LPC_EINVAL, "n_sites = %lld exceeds LPC_NOALLOC_MAX_SITES = %lld, what the library's static scratch array (%d bytes) covers",
                (long long)n_sites, (long long)LPC_NOALLOC_MAX_SITES, (int)LPC_NOALLOC_SCRATCH_BYTES);
  if ((n_sites > 0 && !is_device_ptr(g)) || !is_device_ptr(out)) return fail(LPC_EINVAL, "g and out must be device pointers");
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= MAX_DEVICES) return fail(LPC_ECUDA, "device ordinal %d is beyond the %d this library keeps track of", dev, MAX_DEVICES);
  // the device address of the array on THIS device: asked for once per device, with that device current
  static unsigned char* scratch_of[MAX_DEVICES] = {};
  unsigned char* scratch = scratch_of[dev];
  if (!scratch) {
    CUDA_TRY(cudaGetSymbolAddress(reinterpret_cast<void**>(&scratch), g_noalloc_scratch));
    if (!scratch) return fail(LPC_ECUDA, "cudaGetSymbolAddress gave no address for the scratch array on device %d", dev);
    scratch_of[dev] = scratch;
  }
  cudaStream_t st = static_cast<cudaStream_t>(stream);
  // the ticket must start at zero whatever an earlier (perhaps failed) call left; the partials are overwritten before they are read
  CUDA_TRY(cudaMemsetAsync(scratch, 0, NA_HEADER, st));
  const unsigned grid = (unsigned)std::max<long long>(1, (n_sites + NA_CHUNK - 1) / NA_CHUNK);
  fid_sample_noalloc_kernel<<<grid, 256, 0, st>>>(reinterpret_cast<const double2*>(g), (long long)n_sites, scratch, out);
  CUDA_TRY(cudaGetLastError());
  return LPC_OK;
}
