// lpc_step.cuh -- the fused propagate + phase-rotate + reduce sweep.
//
// Two kernels compute the same thing with the same per-site arithmetic (SiteUpdate):
//   step_direct_kernel : one thread per z-pair of sites, neighbours read straight from global
//                        memory (L1/L2 serve the reuse).  Works for every size; the fallback.
//   step_tma_kernel    : (lpc_step_vec.cuh) a CTA owns a (TY x TZ) tile of the y-z plane and marches along x.  One
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
      phase_rotate(u.cs, u.sn, hr, hi, out[s][0], out[s][1]);
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
// FEAT bit 0: the region-resolved FID (magnetisation sweep) or VACF (moment sweep) is accumulated in the same sweep;
// bit 1: slab mode with direct halo stores (no shared memory of its own).
// bit 2: the sweep stages sin alone and rebuilds cos (cos_from_sin): 8 bytes per site less (fp64).
template <typename T, int NH, int NRHO, int NMOM, int TY, int TZ, int NSTAGE, int LK = 0, int VW = 2, int FEAT = 0>
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
  static constexpr int KCS_RAW = ((FEAT & 4) ? 1 : NH) * TY * TZ * (int)sizeof(T);  // cos, sin (no halo), or sin alone (FEAT bit 2); none without the magnetisation
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
  static constexpr int RSLOT_OFF = (RED_OFF + ((NTHREADS / 32) * NRED + 1) * 8 + 15) / 16 * 16;
  static constexpr int RSLOT_BYTES = (FEAT & 1) ? NTHREADS * 8 : 0;   // scratch of the regional column sums (<= NTHREADS doubles)
  static constexpr int SMEM_BYTES = RSLOT_OFF + RSLOT_BYTES + 128;  // +128: manual alignment slack
  // Resident CTAs per SM the registers are budgeted for: two 8-warp CTAs (TY = 8, up to 3 channels) or
  // one.  16 warps per SM are 4 per scheduler, i.e. up to 128 registers per thread.
  static constexpr int LB_CTAS = (NCONS == 256 && C <= 3) ? 2 : 1;
  static constexpr int LB_THREADS = NTHREADS;
  static_assert(NCONS % 32 == 0, "consumer threads must fill whole warps");
  static_assert(TZ % VW == 0, "TZ must be a multiple of the vector width");
};

struct NoLinkMaps {};

}  // namespace lpc

#include "lpc_step_vec.cuh"
