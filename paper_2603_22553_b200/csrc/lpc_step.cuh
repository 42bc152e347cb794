// lpc_step.cuh -- the fused propagate + phase-rotate + reduce sweep.
//
// Two kernels compute the same thing with the same per-site arithmetic (SiteUpdate):
//   step_direct_kernel : one thread per z-pair of sites, neighbours read straight from global
//                        memory (L1/L2 serve the reuse).  Works for every size; the fallback.
//   step_tma_kernel    : a CTA owns a (TY x TZ) tile of the y-z plane and marches along x.  A
//                        producer warp streams one x-plane per stage into shared memory with
//                        cp.async.bulk.tensor (TMA, halo included) behind a full/empty mbarrier
//                        ring; consumer warps keep the x-1 / x / x+1 centre values in registers
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
template <typename T, int NRHO, int NMOM>
__global__ void __launch_bounds__(256) step_direct_kernel(StepArgs<T> a) {
  constexpr int C = 2 + NRHO + NMOM;
  constexpr int NRED = 2 + NMOM;
  const Layout& L = a.L;
  const long long zpairs = (L.nz + 1) / 2;
  const long long npairs = zpairs * L.ny * L.nx;
  double acc[NRED];
#pragma unroll
  for (int r = 0; r < NRED; ++r) acc[r] = 0.0;

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
      u.weights(pi[j], pi[j - L.sx], pi[j + L.sx], pi[j - L.sy], pi[j + L.sy], pi[j - 1], pi[j + 1], a.a6, csv[j], snv[j]);
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const T* __restrict__ f = a.fin + (long long)c * L.np;
        const T fc = f[j];
        if (NMOM == 3 && c >= 2 + NRHO) {
          const int d = c - 2 - NRHO;
          const T dm = (d == 0) ? (u.mxp - u.mxm) : (d == 1) ? (u.myp - u.mym) : (u.mzp - u.mzm);
          acc[2 + d] += (double)fc * (double)dm;  // P^d_i u^d_i / (a alpha/6), before propagation
        }
        out[s][c] = u.gather(fc, f[j - L.sx], f[j + L.sx], f[j - L.sy], f[j + L.sy], f[j - 1], f[j + 1]);
      }
      const T hr = out[s][0], hi = out[s][1];
      out[s][0] = u.cs * hr - u.sn * hi;
      out[s][1] = u.cs * hi + u.sn * hr;
      acc[0] += (double)u.pc * (double)out[s][0];
      acc[1] += (double)u.pc * (double)out[s][1];
    }
#pragma unroll
    for (int c = 0; c < C; ++c)
      store_with_ghosts(a.fout + (long long)c * L.np, L, a.per, i, x, y, z, out[0][c], vb ? out[1][c] : (T)0, vb);
  }
  __shared__ double red[8 * NRED + 1];
  block_reduce_finalize<NRED, FIN_STEP, NMOM>(acc, red, a.partials, a.ctl, a.fid, a.vacf, a.vacf_stride, a.zscale, gridDim.x,
                                              blockIdx.x);
}

// ---------------------------------------------------------------------------------------------
// TMA kernel.
// ---------------------------------------------------------------------------------------------
template <typename T, int NRHO, int NMOM, int TY, int TZ, int NSTAGE>
struct TmaCfg {
  static constexpr int C = 2 + NRHO + NMOM;
  static constexpr int NRED = 2 + NMOM;
  static constexpr int HZ = 16 / (int)sizeof(T);  // z halo of 16 bytes on each side keeps the centre pairs 16-byte aligned
  static constexpr int TZW = TZ + 2 * HZ;
  static constexpr int TYH = TY + 2;
  static constexpr int NCONS = TY * TZ / 2;  // consumer threads, one per z-pair
  static constexpr int NCW = NCONS / 32;
  static constexpr int NTHREADS = NCONS + 32;
  static constexpr int F_RAW = C * TYH * TZW * (int)sizeof(T);
  static constexpr int PI_RAW = TYH * TZW * (int)sizeof(T);
  static constexpr int KCS_RAW = 2 * TY * TZ * (int)sizeof(T);  // cos, sin (no halo)
  static constexpr int F_BYTES = (F_RAW + 127) / 128 * 128;
  static constexpr int PI_BYTES = (PI_RAW + 127) / 128 * 128;
  static constexpr int KCS_BYTES = (KCS_RAW + 127) / 128 * 128;
  static constexpr int STAGE_BYTES = F_BYTES + PI_BYTES + KCS_BYTES;
  static constexpr int BAR_OFF = NSTAGE * STAGE_BYTES;
  static constexpr int RED_OFF = BAR_OFF + 2 * NSTAGE * 8;
  static constexpr int SMEM_BYTES = RED_OFF + ((NTHREADS / 32) * NRED + 1) * 8 + 128;  // +128: manual alignment slack
  static_assert(NCONS % 32 == 0, "consumer threads must fill whole warps");
  static_assert(TZ % 2 == 0, "TZ must be even");
};

template <typename T, int NRHO, int NMOM, int TY, int TZ, int NSTAGE>
__global__ void __launch_bounds__(TY* TZ / 2 + 64, (2 + NRHO + NMOM <= 3) ? 2 : 1)
    step_tma_kernel(const __grid_constant__ CUtensorMap tm_f, const __grid_constant__ CUtensorMap tm_pi,
                    const __grid_constant__ CUtensorMap tm_cs, StepArgs<T> a) {
  using K = TmaCfg<T, NRHO, NMOM, TY, TZ, NSTAGE>;
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
  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;

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

  if (warp == K::NCW) {
    // ===== producer warp: one elected lane issues the TMA loads =====
    if (lane == 0) {
      tma_prefetch_desc(&tm_f);
      tma_prefetch_desc(&tm_pi);
      tma_prefetch_desc(&tm_cs);
      for (int j = 0; j < nloads; ++j) {
        const int s = j % NSTAGE;
        if (j >= NSTAGE) mbar_wait(&empty[s], ((j / NSTAGE) - 1) & 1);
        unsigned char* st = smem + s * K::STAGE_BYTES;
        const bool need_kcs = (j >= 1 && j <= nplanes);
        mbar_expect_tx(&full[s], K::F_RAW + K::PI_RAW + (need_kcs ? K::KCS_RAW : 0));
        // plane x0-1+j lives at padded x coordinate x0+j; box starts HZ columns / 1 row before the tile
        tma_load_4d(st, &tm_f, &full[s], L.padz + z0 - HZ, y0, x0 + j, 0);
        tma_load_3d(st + K::F_BYTES, &tm_pi, &full[s], L.padz + z0 - HZ, y0, x0 + j);
        if (need_kcs) tma_load_4d(st + K::F_BYTES + K::PI_BYTES, &tm_cs, &full[s], L.padz + z0, y0 + 1, x0 + j, 0);
      }
    }
  } else {
    // ===== consumer warps =====
    const int ty = threadIdx.x / (TZ / 2);   // row inside the tile
    const int tp = threadIdx.x % (TZ / 2);   // pair inside the row
    const int y = y0 + ty, z = z0 + 2 * tp;
    const bool va = (y < L.ny) && (z < L.nz);
    const bool vb = (y < L.ny) && (z + 1 < L.nz);
    const int ec = (ty + 1) * TZW + 2 * tp + HZ;  // element offset of the centre pair in a halo'd tile

    V2 prev[C], ctr[C], nxt[C], ppi, cpi, npi;
    auto load_centres = [&](int s, V2(&f)[C], V2& p) {
      const T* sf = reinterpret_cast<const T*>(smem + s * K::STAGE_BYTES);
      const T* sp = reinterpret_cast<const T*>(smem + s * K::STAGE_BYTES + K::F_BYTES);
#pragma unroll
      for (int c = 0; c < C; ++c) f[c] = *reinterpret_cast<const V2*>(sf + c * TYH * TZW + ec);
      p = *reinterpret_cast<const V2*>(sp + ec);
    };

    mbar_wait(&full[0], 0);
    load_centres(0, prev, ppi);
    __syncwarp();
    if (lane == 0) mbar_arrive(&empty[0]);
    mbar_wait(&full[1 % NSTAGE], (1 / NSTAGE) & 1);
    load_centres(1 % NSTAGE, ctr, cpi);

    for (int p = 0; p < nplanes; ++p) {
      const int x = x0 + p;
      const int jn = p + 2, sn_ = jn % NSTAGE;
      mbar_wait(&full[sn_], (jn / NSTAGE) & 1);
      load_centres(sn_, nxt, npi);

      const int sc = (p + 1) % NSTAGE;
      const T* sf = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES);
      const T* sp = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::F_BYTES);
      const T* sk = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::F_BYTES + K::PI_BYTES);
      const int ek = ty * TZ + 2 * tp;
      const V2 csv = *reinterpret_cast<const V2*>(sk + ek);
      const V2 snv = *reinterpret_cast<const V2*>(sk + TY * TZ + ek);
      const V2 pym = *reinterpret_cast<const V2*>(sp + ec - TZW);
      const V2 pyp = *reinterpret_cast<const V2*>(sp + ec + TZW);
      const T pzm = sp[ec - 1], pzp = sp[ec + 2];

      SiteUpdate<T, NRHO, NMOM> ua, ub;
      ua.weights(cpi.x, ppi.x, npi.x, pym.x, pyp.x, pzm, cpi.y, a.a6, csv.x, snv.x);
      ub.weights(cpi.y, ppi.y, npi.y, pym.y, pyp.y, cpi.x, pzp, a.a6, csv.y, snv.y);

      T oa[C], ob[C];
#pragma unroll
      for (int c = 0; c < C; ++c) {
        const T* fcn = sf + c * TYH * TZW;
        const V2 fym = *reinterpret_cast<const V2*>(fcn + ec - TZW);
        const V2 fyp = *reinterpret_cast<const V2*>(fcn + ec + TZW);
        const T fzm = fcn[ec - 1], fzp = fcn[ec + 2];
        if (NMOM == 3 && c >= 2 + NRHO) {
          const int d = c - 2 - NRHO;
          const T dma = (d == 0) ? (ua.mxp - ua.mxm) : (d == 1) ? (ua.myp - ua.mym) : (ua.mzp - ua.mzm);
          const T dmb = (d == 0) ? (ub.mxp - ub.mxm) : (d == 1) ? (ub.myp - ub.mym) : (ub.mzp - ub.mzm);
          double t = 0.0;
          if (va) t += (double)ctr[c].x * (double)dma;
          if (vb) t += (double)ctr[c].y * (double)dmb;
          acc[2 + d] += t;
        }
        oa[c] = ua.gather(ctr[c].x, prev[c].x, nxt[c].x, fym.x, fyp.x, fzm, ctr[c].y);
        ob[c] = ub.gather(ctr[c].y, prev[c].y, nxt[c].y, fym.y, fyp.y, ctr[c].x, fzp);
      }
      // every shared-memory read of stage sc is done: hand it back to the producer
      __syncwarp();
      if (lane == 0) mbar_arrive(&empty[sc]);

      {
        const T ar = oa[0], ai = oa[1], br = ob[0], bi = ob[1];
        oa[0] = ua.cs * ar - ua.sn * ai;
        oa[1] = ua.cs * ai + ua.sn * ar;
        ob[0] = ub.cs * br - ub.sn * bi;
        ob[1] = ub.cs * bi + ub.sn * br;
      }
      if (va) {
        acc[0] += (double)cpi.x * (double)oa[0];
        acc[1] += (double)cpi.x * (double)oa[1];
        if (vb) {
          acc[0] += (double)cpi.y * (double)ob[0];
          acc[1] += (double)cpi.y * (double)ob[1];
        }
        const long long i = L.idx(x, y, z);
#pragma unroll
        for (int c = 0; c < C; ++c) store_with_ghosts(a.fout + (long long)c * L.np, L, a.per, i, x, y, z, oa[c], ob[c], vb);
      }
#pragma unroll
      for (int c = 0; c < C; ++c) {
        prev[c] = ctr[c];
        ctr[c] = nxt[c];
      }
      ppi = cpi;
      cpi = npi;
    }
  }
  block_reduce_finalize<NRED, FIN_STEP, NMOM>(acc, red, a.partials, a.ctl, a.fid, a.vacf, a.vacf_stride, a.zscale, gridDim.x,
                                              blockIdx.x);
}

}  // namespace lpc
