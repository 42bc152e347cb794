// lpc_step.cuh -- the fused propagate + phase-rotate + reduce sweep.
//
// Two kernels compute the same thing with the same per-site arithmetic (SiteUpdate):
//   step_direct_kernel : one thread per z-pair of sites, neighbours read straight from global
//                        memory (L1/L2 serve the reuse).  Works for every size; the fallback.
//   step_tma_kernel    : a CTA owns a (TY x TZ) tile of the y-z plane and marches along x.  One
//                        x-plane per stage is streamed into shared memory with cp.async.bulk.tensor
//                        (TMA, halo included) behind a full/empty mbarrier ring; thread 0 issues the
//                        loads between planes (no producer warp: 16 warps per SM leave 128 registers
//                        per thread).  The threads keep the x-1 / x / x+1 centre values in registers
//                        and read the in-plane neighbours from shared memory.
// Both end with one block partial per CTA and a fixed-order final sum by the last CTA.
#pragma once

#include "lpc_internal.cuh"

namespace lpc {

// Store a pair of outputs (sites z, z+1) and their periodic ghost copies.
template <typename T>
__device__ __forceinline__ void store_pair(T* __restrict__ base, long long i, T oa, T ob, bool vb) {
  using V2 = typename Vec2<T>::type;
  if (vb) {
    V2 v; v.x = oa; v.y = ob;
    *reinterpret_cast<V2*>(base + i) = v;
  } else {
    base[i] = oa;
  }
}

template <typename T>
__device__ __forceinline__ void store_with_ghosts(T* __restrict__ base, const Layout& L, const int* per, long long i, int x, int y,
                                                  int z, T oa, T ob, bool vb) {
  store_pair(base, i, oa, ob, vb);
  if (per[2]) {
    if (z == 0) base[i + L.nz] = oa;                      // ghost column z = nz
    if (z == L.nz - 1) base[i - L.nz] = oa;               // ghost column z = -1
    if (vb && z + 1 == L.nz - 1) base[i + 1 - L.nz] = ob;
  }
  if (per[1]) {
    if (y == 0) store_pair(base, i + (long long)L.ny * L.sy, oa, ob, vb);
    if (y == L.ny - 1) store_pair(base, i - (long long)L.ny * L.sy, oa, ob, vb);
  }
  if (per[0]) {
    if (x == 0) store_pair(base, i + (long long)L.nx * L.sx, oa, ob, vb);
    if (x == L.nx - 1) store_pair(base, i - (long long)L.nx * L.sx, oa, ob, vb);
  }
}

// One channel of a pair that lies on a periodic face (rare; kept out of line, with scalar arguments
// only, so that the march of the TMA kernel stays small and the kernel parameters stay in the
// constant bank).  i is the padded index of (x, y, z); permask bit d = axis d is periodic.
template <typename T>
__device__ __noinline__ void store_face_pair(T* __restrict__ base, long long i, int nx, int ny, int nz, long long sy, long long sx,
                                             int permask, int x, int y, int z, T oa, T ob, bool vb) {
  store_pair(base, i, oa, ob, vb);
  if (permask & 4) {
    if (z == 0) base[i + nz] = oa;
    if (z == nz - 1) base[i - nz] = oa;
    if (vb && z + 1 == nz - 1) base[i + 1 - nz] = ob;
  }
  if (permask & 2) {
    if (y == 0) store_pair(base, i + (long long)ny * sy, oa, ob, vb);
    if (y == ny - 1) store_pair(base, i - (long long)ny * sy, oa, ob, vb);
  }
  if (permask & 1) {
    if (x == 0) store_pair(base, i + (long long)nx * sx, oa, ob, vb);
    if (x == nx - 1) store_pair(base, i - (long long)nx * sx, oa, ob, vb);
  }
}

// ---------------------------------------------------------------------------------------------
// Direct kernel.
// ---------------------------------------------------------------------------------------------
// One sweep over all site pairs, grid-stride.  COHERENT reads the state with ld.global.cg (L2 only): the
// persistent kernel needs that, because another CTA wrote those values one grid barrier ago and L1 is not
// coherent.  The parameters (pi, cos, sin) are read-only and always go through L1.
template <typename T, bool COHERENT>
__device__ __forceinline__ T ld_state(const T* p) {
  return COHERENT ? __ldcg(p) : *p;
}

template <typename T, int NRHO, int NMOM, bool COHERENT>
__device__ __forceinline__ void direct_sweep(const StepArgs<T>& a, const T* __restrict__ fin, T* __restrict__ fout,
                                             double (&acc)[2 + NMOM]) {
  constexpr int C = 2 + NRHO + NMOM;
  const Layout& L = a.L;
  const long long zpairs = (L.nz + 1) / 2;
  const long long npairs = zpairs * L.ny * L.nx;
  const T* __restrict__ pi = a.pi;
  const T* __restrict__ csv = a.cs;
  const T* __restrict__ snv = a.cs + L.np;

  for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < npairs; p += (long long)gridDim.x * blockDim.x) {
    const int z = 2 * (int)(p % zpairs);
    const long long r = p / zpairs;
    const int y = (int)(r % L.ny);
    const int x = (int)(r / L.ny);
    const long long i = L.idx(x, y, z);
    const bool vb = (z + 1 < L.nz);
    T out[2][C];
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      if (s == 1 && !vb) break;
      const long long j = i + s;
      SiteUpdate<T, NRHO, NMOM> u;
      if (a.mlink)
        u.weights_links(pi[j], a.mlink + j, L.np, L.sx, L.sy, a.a6, csv[j], snv[j]);
      else
        u.weights(pi[j], pi[j - L.sx], pi[j + L.sx], pi[j - L.sy], pi[j + L.sy], pi[j - 1], pi[j + 1], a.a6, csv[j], snv[j]);
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const T* __restrict__ f = fin + (long long)c * L.np;
        const T fc = ld_state<T, COHERENT>(f + j);
        if (NMOM == 3 && c >= 2 + NRHO) {
          const int d = c - 2 - NRHO;
          const T dm = (d == 0) ? (u.mxp - u.mxm) : (d == 1) ? (u.myp - u.mym) : (u.mzp - u.mzm);
          acc[2 + d] += (double)fc * (double)dm;  // P^d_i u^d_i / (a alpha/6), before propagation
        }
        out[s][c] = u.gather(fc, ld_state<T, COHERENT>(f + j - L.sx), ld_state<T, COHERENT>(f + j + L.sx),
                             ld_state<T, COHERENT>(f + j - L.sy), ld_state<T, COHERENT>(f + j + L.sy),
                             ld_state<T, COHERENT>(f + j - 1), ld_state<T, COHERENT>(f + j + 1));
      }
      const T hr = out[s][0], hi = out[s][1];
      out[s][0] = u.cs * hr - u.sn * hi;
      out[s][1] = u.cs * hi + u.sn * hr;
      acc[0] += (double)u.pc * (double)out[s][0];
      acc[1] += (double)u.pc * (double)out[s][1];
    }
#pragma unroll
    for (int c = 0; c < C; ++c)
      store_with_ghosts(fout + (long long)c * L.np, L, a.per, i, x, y, z, out[0][c], vb ? out[1][c] : (T)0, vb);
  }
}

template <typename T, int NRHO, int NMOM>
__global__ void __launch_bounds__(256) step_direct_kernel(StepArgs<T> a) {
  constexpr int NRED = 2 + NMOM;
  double acc[NRED];
#pragma unroll
  for (int r = 0; r < NRED; ++r) acc[r] = 0.0;
  direct_sweep<T, NRHO, NMOM, false>(a, a.fin, a.fout, acc);
  __shared__ double red[8 * NRED + 1];
  block_reduce_finalize<NRED, FIN_STEP, NMOM>(acc, red, a.partials, a.ctl, a.fid, a.vacf, a.vacf_stride, a.zscale, gridDim.x,
                                              blockIdx.x);
}

// ---------------------------------------------------------------------------------------------
// Persistent kernel for lattices whose state and parameters stay in L2: all n steps of lpc_step_n in
// ONE cooperative launch, a grid barrier between steps instead of a kernel boundary (a launch costs
// more than a 32^3 .. 64^3 sweep).  Same per-site arithmetic as the other kernels.  Per step: sweep ->
// block partial into partials[step parity] -> grid barrier -> block 0 sums the partials in block order
// and writes G[step+1] (Z_d[step+2]) while the others start the next sweep; block 0 joins the next
// barrier only after that, so a partial slot is never overwritten while it is still being read.
// ---------------------------------------------------------------------------------------------
__device__ __forceinline__ void grid_barrier(unsigned long long* bar, unsigned long long target) {
  __syncthreads();
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(bar, 1ull);
    unsigned long long v;
    do {
      asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(bar) : "memory");
    } while (v < target);
  }
  __syncthreads();
}

template <typename T, int NRHO, int NMOM>
__global__ void __launch_bounds__(256) step_persist_kernel(StepArgs<T> a, T* buf_a, T* buf_b, int nsteps, unsigned long long* bar) {
  constexpr int NRED = 2 + NMOM;
  __shared__ double red[8 * NRED];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  const size_t slot = (size_t)gridDim.x * NRED;   // partials of one step parity
  T* fin = buf_a;
  T* fout = buf_b;
  for (int s = 0; s < nsteps; ++s) {
    double acc[NRED];
#pragma unroll
    for (int r = 0; r < NRED; ++r) acc[r] = 0.0;
    direct_sweep<T, NRHO, NMOM, true>(a, fin, fout, acc);
    double* part = a.partials + (size_t)(s & 1) * slot;
#pragma unroll
    for (int r = 0; r < NRED; ++r) {
      const double v = warp_sum(acc[r]);
      if (lane == 0) red[warp * NRED + r] = v;
    }
    __syncthreads();
    if (threadIdx.x < NRED) {
      double v = 0.0;
      for (int w = 0; w < 8; ++w) v += red[w * NRED + threadIdx.x];
      part[(size_t)blockIdx.x * NRED + threadIdx.x] = v;
    }
    grid_barrier(bar, (unsigned long long)(s + 1) * gridDim.x);
    if (blockIdx.x == 0) {
      // fixed-order sum of the block partials: thread r < NRED takes column r
      double tot[NRED];
#pragma unroll
      for (int r = 0; r < NRED; ++r) tot[r] = 0.0;
      for (unsigned int b = threadIdx.x; b < gridDim.x; b += blockDim.x) {
#pragma unroll
        for (int r = 0; r < NRED; ++r) tot[r] += __ldcg(&part[(size_t)b * NRED + r]);
      }
#pragma unroll
      for (int r = 0; r < NRED; ++r) {
        const double v = warp_sum(tot[r]);
        if (lane == 0) red[warp * NRED + r] = v;
      }
      __syncthreads();
      if (threadIdx.x == 0) {
        double out[NRED];
        for (int r = 0; r < NRED; ++r) {
          double v = 0.0;
          for (int w = 0; w < 8; ++w) v += red[w * NRED + r];
          out[r] = v;
        }
        const long long st = a.ctl->step;
        a.fid[st + 1] = make_double2(out[0], out[1]);
        if (NMOM == 3)
          for (int d = 0; d < 3; ++d) a.vacf[d * a.vacf_stride + st + 2] = a.zscale * out[2 + d];
        a.ctl->step = st + 1;
      }
      __syncthreads();
    }
    T* t = fin;
    fin = fout;
    fout = t;
  }
}

// ---------------------------------------------------------------------------------------------
// TMA kernel.
// ---------------------------------------------------------------------------------------------
// NH = 2: the sweep carries the magnetisation (h_re, h_im, phase multiply, G); NH = 0: real channels only.
// LK = 1: per-link mobility factors.  The symmetric link weights m_{i,+d} are stored (3 channels) and
// staged per plane instead of being rebuilt from pi: m_x without halo (the -x link is the +x link of the plane
// below, carried in registers), m_y with one halo row below, m_z with one halo column (HZ wide) below; pi is then
// needed at the centres only.
struct TmaLinkMaps {
  CUtensorMap pic, mx, my, mz;   // pi centres, the three link channels
};

// VW: sites per thread along z (one 16-byte vector: 2 in fp64, 4 in the fp32 march of lpc_step_vec.cuh).
template <typename T, int NH, int NRHO, int NMOM, int TY, int TZ, int NSTAGE, int LK = 0, int VW = 2>
struct TmaCfg {
  static constexpr int C = NH + NRHO + NMOM;
  static constexpr int NRED = 2 + NMOM;
  static constexpr int HZ = 16 / (int)sizeof(T);  // z halo of 16 bytes on each side keeps the centre pairs 16-byte aligned
  static constexpr int TZW = TZ + 2 * HZ;
  static constexpr int TYH = TY + 2;
  static constexpr int NCONS = TY * TZ / VW;  // consumer threads, one per z-pair (z-quad with VW = 4)
  static constexpr int NCW = NCONS / 32;
  static constexpr int NTHREADS = NCONS;      // no producer warp: thread 0 issues the TMA loads between planes
  static constexpr int F_RAW = C * TYH * TZW * (int)sizeof(T);
  static constexpr int TZM = TZ + HZ;         // row length of the staged m_z box
  static constexpr int PI_RAW = (LK ? TY * TZ : TYH * TZW) * (int)sizeof(T);
  static constexpr int MX_RAW = LK ? TY * TZ * (int)sizeof(T) : 0;
  static constexpr int MY_RAW = LK ? (TY + 1) * TZ * (int)sizeof(T) : 0;
  static constexpr int MZ_RAW = LK ? TY * TZM * (int)sizeof(T) : 0;
  static constexpr int MX_BYTES = (MX_RAW + 127) / 128 * 128;
  static constexpr int MY_BYTES = (MY_RAW + 127) / 128 * 128;
  static constexpr int MZ_BYTES = (MZ_RAW + 127) / 128 * 128;
  static constexpr int KCS_RAW = NH * TY * TZ * (int)sizeof(T);  // cos, sin (no halo); none without the magnetisation
  static constexpr int F_BYTES = (F_RAW + 127) / 128 * 128;
  static constexpr int PI_BYTES = (PI_RAW + 127) / 128 * 128;
  static constexpr int KCS_BYTES = (KCS_RAW + 127) / 128 * 128;
  static constexpr int MX_OFF = F_BYTES + PI_BYTES + KCS_BYTES;
  static constexpr int MY_OFF = MX_OFF + MX_BYTES;
  static constexpr int MZ_OFF = MY_OFF + MY_BYTES;
  static constexpr int STAGE_BYTES = MZ_OFF + MZ_BYTES;
  static constexpr int TX_BYTES = F_RAW + PI_RAW + MX_RAW + MY_RAW + MZ_RAW;   // per stage, without cos/sin
  static constexpr int BAR_OFF = NSTAGE * STAGE_BYTES;
  static constexpr int RED_OFF = BAR_OFF + 2 * NSTAGE * 8;
  static constexpr int SMEM_BYTES = RED_OFF + ((NTHREADS / 32) * NRED + 1) * 8 + 128;  // +128: manual alignment slack
  // Resident CTAs per SM the registers are budgeted for: two 8-warp CTAs (TY = 8, up to 3 channels) or
  // one.  16 warps per SM are 4 per scheduler, i.e. up to 128 registers per thread.
  static constexpr int LB_CTAS = (NCONS == 256 && C <= 3) ? 2 : 1;
  static constexpr int LB_THREADS = NTHREADS;
  static_assert(NCONS % 32 == 0, "consumer threads must fill whole warps");
  static_assert(TZ % VW == 0, "TZ must be a multiple of the vector width");
};

template <typename T, int NH, int NRHO, int NMOM, int TY, int TZ, int NSTAGE, int LK, typename LM>
__device__ __forceinline__ void step_tma_body(const CUtensorMap& tm_f, const CUtensorMap& tm_pi, const CUtensorMap& tm_cs, const LM& lm,
                                              const StepArgs<T>& a) {
  using K = TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, LK>;
  using V2 = typename Vec2<T>::type;
  constexpr int C = K::C, NRED = K::NRED, TZW = K::TZW, TYH = K::TYH, HZ = K::HZ;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  // round the base up to 128 bytes by offset arithmetic so that the pointer stays in the shared window
  unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + K::BAR_OFF);
  uint64_t* empty = full + NSTAGE;
  double* red = reinterpret_cast<double*>(smem + K::RED_OFF);

  const Layout& L = a.L;
  const int bz = blockIdx.x % a.tiles_z;
  const int by = (blockIdx.x / a.tiles_z) % a.tiles_y;
  const int bx = blockIdx.x / (a.tiles_z * a.tiles_y);
  const int z0 = bz * TZ, y0 = by * TY, x0 = bx * a.xc;
  const int nplanes = min(a.xc, L.nx - x0);
  const int nloads = nplanes + 2;
  const int lane = threadIdx.x & 31;

  if (threadIdx.x == 0) {
    for (int s = 0; s < NSTAGE; ++s) {
      mbar_init(&full[s], 1);
      mbar_init(&empty[s], K::NCW);
    }
    mbar_fence_init();
  }
  __syncthreads();

  double acc[NRED];
#pragma unroll
  for (int r = 0; r < NRED; ++r) acc[r] = 0.0;

  // ----- TMA issue (thread 0): load j brings plane x0-1+j into stage j % NSTAGE -----
  int jl = 0;  // next load to issue (thread 0 only)
  auto issue_load = [&]() {
    const int s = jl % NSTAGE;
    if (jl >= NSTAGE) mbar_wait(&empty[s], ((jl / NSTAGE) - 1) & 1);   // every warp is done with the plane it held
    unsigned char* st = smem + s * K::STAGE_BYTES;
    const bool need_kcs = (NH == 2) && (jl >= 1 && jl <= nplanes);
    mbar_expect_tx(&full[s], K::TX_BYTES + (need_kcs ? K::KCS_RAW : 0));
    // plane x0-1+j lives at padded x coordinate x0+j; box starts HZ columns / 1 row before the tile
    tma_load_4d(st, &tm_f, &full[s], L.padz + z0 - HZ, y0, x0 + jl, a.c0);
    if constexpr (LK) {
      tma_load_3d(st + K::F_BYTES, &lm.pic, &full[s], L.padz + z0, y0 + 1, x0 + jl);
      tma_load_3d(st + K::MX_OFF, &lm.mx, &full[s], L.padz + z0, y0 + 1, x0 + jl);
      tma_load_3d(st + K::MY_OFF, &lm.my, &full[s], L.padz + z0, y0, x0 + jl);           // rows y0-1 .. y0+TY-1
      tma_load_3d(st + K::MZ_OFF, &lm.mz, &full[s], L.padz + z0 - HZ, y0 + 1, x0 + jl);  // columns z0-HZ .. z0+TZ-1
    } else {
      tma_load_3d(st + K::F_BYTES, &tm_pi, &full[s], L.padz + z0 - HZ, y0, x0 + jl);
    }
    if (need_kcs) tma_load_4d(st + K::F_BYTES + K::PI_BYTES, &tm_cs, &full[s], L.padz + z0, y0 + 1, x0 + jl, 0);
    ++jl;
  };
  if (threadIdx.x == 0) {
    tma_prefetch_desc(&tm_f);
    if constexpr (LK) {
      tma_prefetch_desc(&lm.pic);
      tma_prefetch_desc(&lm.mx);
      tma_prefetch_desc(&lm.my);
      tma_prefetch_desc(&lm.mz);
    } else {
      tma_prefetch_desc(&tm_pi);
    }
    tma_prefetch_desc(&tm_cs);
    for (int j = 0; j < NSTAGE && j < nloads; ++j) issue_load();
  }
  {
    // ===== consumer warps =====
    const int ty = threadIdx.x / (TZ / 2);   // row inside the tile
    const int tp = threadIdx.x % (TZ / 2);   // pair inside the row
    const int y = y0 + ty, z = z0 + 2 * tp;
    const bool va = (y < L.ny) && (z < L.nz);
    const bool vb = (y < L.ny) && (z + 1 < L.nz);
    const int ec = (ty + 1) * TZW + 2 * tp + HZ;  // element offset of the centre pair in a halo'd tile
    const int ek = ty * TZ + 2 * tp;              // element offset of the pair in a tile without halo
    // sites on a periodic face also write their ghost copies: rare, so it is a separate path
    const bool edge_yz = (a.per[1] && (y == 0 || y == L.ny - 1)) || (a.per[2] && (z == 0 || z + 2 >= L.nz - 1));
    const int permask = (a.per[0] ? 1 : 0) | (a.per[1] ? 2 : 0) | (a.per[2] ? 4 : 0);
    T* outp = a.fout + L.idx(x0, y, z);

    // One x-plane as a consumer thread holds it: the centre pair of every channel and of pi, kappa of
    // the pair, and mlo = min(pi, pi of the plane below) -- the symmetric link weight m_ij of the -x
    // link (which is the +x link of the plane below).  With stored link weights (LK) mlo holds the plane's
    // own +x link weight instead, which is the -x link of the plane above.
    struct Plane {
      V2 f[C];
      V2 pi, kap, mlo;
    };
    Plane P0, P1, P2;
    int sj = 0;            // stage of the next plane to take from the ring
    uint32_t phj = 0;      // and its phase bit
    auto take = [&](Plane& n, const Plane* below) {
      mbar_wait(&full[sj], phj);
      const T* sf = reinterpret_cast<const T*>(smem + sj * K::STAGE_BYTES);
      const T* sp = reinterpret_cast<const T*>(smem + sj * K::STAGE_BYTES + K::F_BYTES);
#pragma unroll
      for (int c = 0; c < C; ++c) n.f[c] = *reinterpret_cast<const V2*>(sf + c * TYH * TZW + ec);
      n.pi = *reinterpret_cast<const V2*>(sp + (LK ? ek : ec));
      n.kap.x = kappa_of(n.pi.x, a.a6);
      n.kap.y = kappa_of(n.pi.y, a.a6);
      if constexpr (LK) {
        n.mlo = *reinterpret_cast<const V2*>(reinterpret_cast<const T*>(smem + sj * K::STAGE_BYTES + K::MX_OFF) + ek);
      } else if (below) {
        n.mlo.x = tmin(n.pi.x, below->pi.x);
        n.mlo.y = tmin(n.pi.y, below->pi.y);
      }
      if (++sj == NSTAGE) {
        sj = 0;
        phj ^= 1u;
      }
    };

    // one plane of the march: prv / ctr / nxt are the planes x-1 / x / x+1, sc the stage that holds x
    auto plane = [&](int x, int sc, const Plane& prv, const Plane& ctr, Plane& nxt) {
      // refill the stage that held plane x-1 (released when the previous plane was finished)
      if (threadIdx.x == 0 && jl < nloads) issue_load();
      take(nxt, &ctr);
      const T* sf = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES);
      const T* sp = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::F_BYTES);
      const T* sk = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::F_BYTES + K::PI_BYTES);
      V2 csv, snv;
      if (NH == 2) {
        csv = *reinterpret_cast<const V2*>(sk + ek);
        snv = *reinterpret_cast<const V2*>(sk + TY * TZ + ek);
      }
      SiteUpdate<T, NRHO, NMOM> ua, ub;
      ua.pc = ctr.pi.x; ub.pc = ctr.pi.y;
      ua.kap = ctr.kap.x; ub.kap = ctr.kap.y;
      if constexpr (LK) {
        const T* smy = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::MY_OFF) + ek;          // row y-1 of the box
        const T* smz = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::MZ_OFF) + ty * K::TZM + HZ + 2 * tp;
        const V2 mym = *reinterpret_cast<const V2*>(smy);
        const V2 myp = *reinterpret_cast<const V2*>(smy + TZ);
        const V2 mzp = *reinterpret_cast<const V2*>(smz);
        ua.mxm = prv.mlo.x; ub.mxm = prv.mlo.y;
        ua.mxp = ctr.mlo.x; ub.mxp = ctr.mlo.y;
        ua.mym = mym.x; ub.mym = mym.y;
        ua.myp = myp.x; ub.myp = myp.y;
        ua.mzm = smz[-1];
        ua.mzp = mzp.x;
        ub.mzm = mzp.x;
        ub.mzp = mzp.y;
      } else {
        const V2 pym = *reinterpret_cast<const V2*>(sp + ec - TZW);
        const V2 pyp = *reinterpret_cast<const V2*>(sp + ec + TZW);
        const T pzm = sp[ec - 1], pzp = sp[ec + 2];
        ua.mxm = ctr.mlo.x; ub.mxm = ctr.mlo.y;
        ua.mxp = nxt.mlo.x; ub.mxp = nxt.mlo.y;
        ua.mym = tmin(ctr.pi.x, pym.x); ub.mym = tmin(ctr.pi.y, pym.y);
        ua.myp = tmin(ctr.pi.x, pyp.x); ub.myp = tmin(ctr.pi.y, pyp.y);
        ua.mzm = tmin(ctr.pi.x, pzm);
        ua.mzp = tmin(ctr.pi.x, ctr.pi.y);
        ub.mzm = ua.mzp;
        ub.mzp = tmin(ctr.pi.y, pzp);
      }

      T oa[C], ob[C];
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const T* fcn = sf + c * TYH * TZW;
        const V2 fym = *reinterpret_cast<const V2*>(fcn + ec - TZW);
        const V2 fyp = *reinterpret_cast<const V2*>(fcn + ec + TZW);
        const T fzm = fcn[ec - 1], fzp = fcn[ec + 2];
        if (NMOM == 3 && c >= NH + NRHO) {
          const int d = c - NH - NRHO;
          const T dma = (d == 0) ? (ua.mxp - ua.mxm) : (d == 1) ? (ua.myp - ua.mym) : (ua.mzp - ua.mzm);
          const T dmb = (d == 0) ? (ub.mxp - ub.mxm) : (d == 1) ? (ub.myp - ub.mym) : (ub.mzp - ub.mzm);
          double t = 0.0;
          if (va) t += (double)ctr.f[c].x * (double)dma;
          if (vb) t += (double)ctr.f[c].y * (double)dmb;
          acc[2 + d] += t;
        }
        oa[c] = ua.gather(ctr.f[c].x, prv.f[c].x, nxt.f[c].x, fym.x, fyp.x, fzm, ctr.f[c].y);
        ob[c] = ub.gather(ctr.f[c].y, prv.f[c].y, nxt.f[c].y, fym.y, fyp.y, ctr.f[c].x, fzp);
      }
      // every shared-memory read of stage sc is done: hand it back to the producer
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[sc]);

      if (NH == 2) {
        const T ar = oa[0], ai = oa[1], br = ob[0], bi = ob[1];
        oa[0] = csv.x * ar - snv.x * ai;
        oa[1] = csv.x * ai + snv.x * ar;
        ob[0] = csv.y * br - snv.y * bi;
        ob[1] = csv.y * bi + snv.y * br;
      }
      if (va) {
        if (NH == 2) {
          acc[0] += (double)ctr.pi.x * (double)oa[0];
          acc[1] += (double)ctr.pi.x * (double)oa[1];
          if (vb) {
            acc[0] += (double)ctr.pi.y * (double)ob[0];
            acc[1] += (double)ctr.pi.y * (double)ob[1];
          }
        }
        if (edge_yz || (a.per[0] && (x == 0 || x == L.nx - 1))) {
          const long long i = L.idx(x, y, z);
#pragma unroll
          for (int c = 0; c < C; ++c)
            store_face_pair<T>(a.fout + (long long)c * L.np, i, L.nx, L.ny, L.nz, L.sy, L.sx, permask, x, y, z, oa[c], ob[c], vb);
        } else {
#pragma unroll
          for (int c = 0; c < C; ++c) store_pair(outp + (long long)c * L.np, 0, oa[c], ob[c], vb);
        }
      }
      outp += L.sx;
    };

    take(P0, nullptr);
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[0]);   // the plane below the chunk is only needed for its centres
    take(P1, &P0);

    // the march, unrolled by three so that the planes keep their registers while their roles rotate
    int sc = 1 % NSTAGE;
    auto next_stage = [&]() { if (++sc == NSTAGE) sc = 0; };
    int p = 0;
    for (; p + 3 <= nplanes; p += 3) {
      plane(x0 + p, sc, P0, P1, P2); next_stage();
      plane(x0 + p + 1, sc, P1, P2, P0); next_stage();
      plane(x0 + p + 2, sc, P2, P0, P1); next_stage();
    }
    if (p < nplanes) { plane(x0 + p, sc, P0, P1, P2); next_stage(); ++p; }
    if (p < nplanes) { plane(x0 + p, sc, P1, P2, P0); next_stage(); ++p; }
  }
  block_reduce_finalize<NRED, (NH == 2) ? FIN_STEP : FIN_MOM, NMOM>(acc, red, a.partials, a.ctl, a.fid, a.vacf, a.vacf_stride, a.zscale, gridDim.x,
                                              blockIdx.x);
}

struct NoLinkMaps {};

template <typename T, int NH, int NRHO, int NMOM, int TY, int TZ, int NSTAGE>
__global__ void __launch_bounds__(TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE>::LB_THREADS, TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE>::LB_CTAS)
    step_tma_kernel(const __grid_constant__ CUtensorMap tm_f, const __grid_constant__ CUtensorMap tm_pi,
                    const __grid_constant__ CUtensorMap tm_cs, StepArgs<T> a) {
  step_tma_body<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, 0>(tm_f, tm_pi, tm_cs, NoLinkMaps(), a);
}

// the same sweep with stored link weights (per-link mobility factors)
template <typename T, int NH, int NRHO, int NMOM, int TY, int TZ, int NSTAGE>
__global__ void __launch_bounds__(TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, 1>::LB_THREADS, TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, 1>::LB_CTAS)
    step_tma_links_kernel(const __grid_constant__ CUtensorMap tm_f, const __grid_constant__ CUtensorMap tm_cs,
                          const __grid_constant__ TmaLinkMaps lm, StepArgs<T> a) {
  step_tma_body<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, 1>(tm_f, tm_f, tm_cs, lm, a);
}

}  // namespace lpc

#include "lpc_step_vec.cuh"
