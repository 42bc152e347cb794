// lpc_regions.cuh -- region-resolved FID and the spectrum.
//
// The paper splits the system into "blocks" (electrodes, bulk) and plots the NMR signal of
// "different parts" of it (Fig. 9, :275-281).  A region is a per-site label 0..n_regions-1 (any other
// value = in no region); the regional FID is Eq. 12 (:137) restricted to the region,
//     G_r[n] = sum_{i in r} g_i(n),
// and the spectrum is Eq. 9 (:115) of a FID series on a caller-chosen frequency grid.
#pragma once

#include "lpc_internal.cuh"
#include "lpc_precompute.cuh"

namespace lpc {


// Region accumulators of one thread.  Regions are blobs, so consecutive sites of a thread mostly carry the same
// label: the running sums of the current region stay in registers (cur) and move to the per-region array only
// when the label changes (that array is indexed at run time and lives in local memory; it is touched rarely).
// Thread-private throughout, so the result does not depend on timing.
template <int NV>
struct RegionAcc {
  double acc[MAX_REGIONS][NV];
  double cur[NV];
  int rcur;
  __device__ __forceinline__ void init() {
#pragma unroll
    for (int r = 0; r < MAX_REGIONS; ++r)
#pragma unroll
      for (int v = 0; v < NV; ++v) acc[r][v] = 0.0;
#pragma unroll
    for (int v = 0; v < NV; ++v) cur[v] = 0.0;
    rcur = 255;
  }
  __device__ __forceinline__ void flush(int next) {
    if (rcur < MAX_REGIONS) {
#pragma unroll
      for (int v = 0; v < NV; ++v) acc[rcur][v] += cur[v];
    }
#pragma unroll
    for (int v = 0; v < NV; ++v) cur[v] = 0.0;
    rcur = next;
  }
  __device__ __forceinline__ void add(int lab, const double (&v)[NV]) {
    if (lab != rcur) flush(lab);
#pragma unroll
    for (int k = 0; k < NV; ++k) cur[k] += v[k];
  }
};

// Rows (x, y) are dealt to warps, the lanes of a warp stride along z: coalesced, and the index arithmetic is paid
// once per row.  body(i_dense, j_padded) is called for every site.
template <typename F>
__device__ __forceinline__ void for_sites_by_rows(const Layout& L, F body) {
  const long long rows = (long long)L.nx * L.ny;
  const int lane = threadIdx.x & 31;
  const long long warps = (long long)gridDim.x * (blockDim.x >> 5);
  for (long long r = (long long)blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5); r < rows; r += warps) {
    const int x = (int)(r / L.ny), y = (int)(r % L.ny);
    const long long i0 = r * L.nz, j0 = L.idx(x, y, 0);
    for (int z = lane; z < L.nz; z += 32) body(i0 + z, j0 + z);
  }
}

// G_r[sample] for all regions: one pass over the current state (16 B) + pi (8 B) + label (1 B) per site.
// Per-thread region accumulators (RegionAcc), reduced per warp and block,
// and the last block sums the block partials in a fixed order.
template <typename T>
__global__ void __launch_bounds__(256)
    region_reduce_kernel(Layout L, const T* __restrict__ pi, const T* __restrict__ f, const uint8_t* __restrict__ label, int n_regions,
                         double* partials, Ctl* ctl, double2* fidr, long long stride, long long sample) {
  RegionAcc<2> ra;
  ra.init();
  for_sites_by_rows(L, [&](long long i, long long j) {
    const double p = (double)pi[j];
    const double g[2] = {p * (double)f[j], p * (double)f[L.np + j]};
    ra.add(label[i], g);
  });
  ra.flush(255);
  __shared__ double red[8][2 * MAX_REGIONS];
  __shared__ unsigned int s_last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int r = 0; r < MAX_REGIONS; ++r) {
    const double vr = warp_sum(ra.acc[r][0]), vi = warp_sum(ra.acc[r][1]);
    if (lane == 0) {
      red[warp][2 * r] = vr;
      red[warp][2 * r + 1] = vi;
    }
  }
  __syncthreads();
  if (threadIdx.x < 2 * MAX_REGIONS) {
    double v = 0.0;
    for (int w = 0; w < 8; ++w) v += red[w][threadIdx.x];
    partials[(size_t)blockIdx.x * 2 * MAX_REGIONS + threadIdx.x] = v;
    __threadfence();
  }
  __syncthreads();
  if (threadIdx.x == 0) s_last = (atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1);
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  // 16 threads, one per (region, re/im), each sums its column of the partials in block order
  if (threadIdx.x < 2 * MAX_REGIONS) {
    double v = 0.0;
    for (unsigned int b = 0; b < gridDim.x; ++b) v += __ldcg(&partials[(size_t)b * 2 * MAX_REGIONS + threadIdx.x]);
    const int r = threadIdx.x >> 1;
    if (r < n_regions) reinterpret_cast<double*>(fidr + r * stride + sample)[threadIdx.x & 1] = v;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    ctl->ticket = 0;
    __threadfence();
  }
}

// Regional VACF (the regional diffusion coefficients of Table 1):
// the sum of Eq. 4 (:79) restricted to the particles that sit in region r when the later displacement
// starts, normalised by the region's equilibrium population w_r = sum_{i in r} pi_i (Q27):
//   INIT: w_r, and Z^r_d[1]   = (a^2 alpha/6) sum_{i in r} (m_{i,+d} + m_{i,-d}) / w_r
//   STEP: Z^r_d[k+1] = (a alpha/6) sum_{i in r} q^d_i(k) (m_{i,+d} - m_{i,-d}) / w_r     (q = P/pi before the sweep)
// One pass over pi (with neighbours), the three moment channels and the labels; per-thread region accumulators
// (RegionAcc), block partials, fixed-order sum by the last block.
template <typename T, bool INIT>
__global__ void __launch_bounds__(256)
    region_moment_kernel(Layout L, const T* __restrict__ pi, const T* __restrict__ mlink, const T* __restrict__ q,
                         const uint8_t* __restrict__ label, int n_regions,
                         double* partials, Ctl* ctl, double* wr, double* vacfr, long long stride, long long index, double scale) {
  constexpr int NV = INIT ? 4 : 3;   // INIT also sums pi
  RegionAcc<NV> ra;
  ra.init();
  const long long st[3] = {L.sx, L.sy, 1};
  for_sites_by_rows(L, [&](long long i, long long j) {
    const T p = pi[j];
    double v[NV];
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      const T* ml = mlink + (long long)d * L.np + j;
      const T mm = mlink ? ml[-st[d]] : tmin(p, pi[j - st[d]]), mp = mlink ? ml[0] : tmin(p, pi[j + st[d]]);
      v[d] = INIT ? (double)mp + (double)mm : (double)q[(long long)d * L.np + j] * (double)(mp - mm);
    }
    if (INIT) v[NV - 1] = (double)p;
    ra.add(label[i], v);
  });
  ra.flush(255);
  constexpr int NC = MAX_REGIONS * NV;
  __shared__ double red[8][NC];
  __shared__ unsigned int s_last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
#pragma unroll
  for (int r = 0; r < MAX_REGIONS; ++r)
#pragma unroll
    for (int k = 0; k < NV; ++k) {
      const double t = warp_sum(ra.acc[r][k]);
      if (lane == 0) red[warp][r * NV + k] = t;
    }
  __syncthreads();
  if (threadIdx.x < NC) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += red[w][threadIdx.x];
    partials[(size_t)blockIdx.x * NC + threadIdx.x] = t;
    __threadfence();
  }
  __syncthreads();
  if (threadIdx.x == 0) s_last = (atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1);
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  double* tot = &red[0][0];
  if (threadIdx.x < NC) {
    double t = 0.0;
    for (unsigned int b = 0; b < gridDim.x; ++b) t += __ldcg(&partials[(size_t)b * NC + threadIdx.x]);
    tot[threadIdx.x] = t;
  }
  __syncthreads();
  if (threadIdx.x < n_regions) {
    const int r = threadIdx.x;
    if (INIT) wr[r] = tot[r * NV + 3];
    const double w = INIT ? tot[r * NV + 3] : wr[r];
    for (int d = 0; d < 3; ++d) vacfr[((long long)r * 3 + d) * stride + index] = (w > 0.0) ? scale * tot[r * NV + d] / w : 0.0;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    ctl->ticket = 0;
    __threadfence();
  }
}

// F(f_k) = dt * sum_{n=0}^{M-1} G[n] exp(-pi lb n dt) exp(-2 pi i f_k n dt),  f_k = f0 + k df
// (Eq. 9, as a plain discrete sum over the samples; lb = Lorentzian line broadening in Hz,
// 0 = none).  One block per frequency, fixed summation order.
__global__ void __launch_bounds__(256)
    spectrum_kernel(const double2* __restrict__ series, long long M, double dt, double f0, double df, long long k0, double lb,
                    double2* __restrict__ out) {
  const double f = f0 + (double)(k0 + blockIdx.x) * df;
  double sr = 0.0, si = 0.0;
  for (long long n = threadIdx.x; n < M; n += blockDim.x) {
    const double t = (double)n * dt;
    double s, c;
    sincospi(2.0 * f * t, &s, &c);        // e^{-2 pi i f t} = c - i s
    const double w = exp(-M_PI * lb * t);
    const double2 g = series[n];
    sr += w * (g.x * c + g.y * s);
    si += w * (g.y * c - g.x * s);
  }
  __shared__ double red[8][2];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  sr = warp_sum(sr);
  si = warp_sum(si);
  if (lane == 0) {
    red[warp][0] = sr;
    red[warp][1] = si;
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    double a = 0.0, b = 0.0;
    for (int w = 0; w < 8; ++w) {
      a += red[w][0];
      b += red[w][1];
    }
    out[blockIdx.x] = make_double2(dt * a, dt * b);
  }
}

}  // namespace lpc
