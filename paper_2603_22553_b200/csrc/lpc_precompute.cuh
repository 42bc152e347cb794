// lpc_precompute.cuh -- site-parameter precompute and state set-up kernels,
// plus the read-out kernels.  All of them run once per lpc_set_site_params / read call; they are
// plain grid-stride kernels over dense site indices i = (x*ny + y)*nz + z.
#pragma once

#include "lpc_internal.cuh"

namespace lpc {

__device__ __forceinline__ long long dense_to_padded(const Layout& L, long long i) {
  const int z = (int)(i % L.nz);
  const long long r = i / L.nz;
  const int y = (int)(r % L.ny);
  const int x = (int)(r / L.ny);
  return L.idx(x, y, z);
}

// e_i = blocked ? 0 : exp(-dF_i)   (Eq. 2 numerator).  dF/blocked point at site i0.
__global__ void boltzmann_factor_kernel(const double* __restrict__ dF, const uint8_t* __restrict__ blocked, long long i0,
                                        long long n, double* __restrict__ e, Ctl* ctl) {
  unsigned long long bad = 0;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
    double v = 0.0;
    if (!blocked[k]) {
      v = exp(-dF[k]);
      if (!(v > 0.0) || isinf(v)) bad++;
    }
    e[i0 + k] = v;
  }
  if (bad) atomicAdd(&ctl->bad, bad);
}

// Fixed-order sum of a dense double array into ctl->zsum.
__global__ void __launch_bounds__(256) sum_kernel(const double* __restrict__ e, long long n, double* partials, Ctl* ctl) {
  double acc = 0.0;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) acc += e[k];
  __shared__ double red[8];
  __shared__ unsigned int s_last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double v = warp_sum(acc);
  if (lane == 0) red[warp] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += red[w];
    partials[blockIdx.x] = t;
    __threadfence();
    s_last = (atomicAdd(&ctl->ticket, 1u) == gridDim.x - 1);
  }
  __syncthreads();
  if (!s_last) return;
  __threadfence();
  double tot = 0.0;
  for (unsigned int b = threadIdx.x; b < gridDim.x; b += blockDim.x) tot += __ldcg(&partials[b]);
  __syncthreads();
  v = warp_sum(tot);
  if (lane == 0) red[warp] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += red[w];
    ctl->zsum = t;
    ctl->ticket = 0;
  }
}

// pi_i = e_i / Z and the phase factors cos, sin of omega_i dt of Eq. 13.
// omega points at site i0.
template <typename T>
__global__ void site_params_kernel(const double* __restrict__ e, const double* __restrict__ omega, long long i0, long long n,
                                   Layout L, double dt, Ctl* ctl, T* __restrict__ pi, T* __restrict__ cs) {
  const double Z = ctl->zsum;
  unsigned long long bad = 0;
  bool wide = false;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
    const long long i = i0 + k;
    const long long j = dense_to_padded(L, i);
    const double p = e[i] / Z;
    double c = 1.0, s = 0.0;
    if (p > 0.0) sincos(omega[k] * dt, &s, &c);
    // small phase angles (every BASELINE config: |omega dt| <= 0.13): the stored cosine is the one a sweep rebuilds from
    // the stored sine (cos_from_sin), so sweeps that read sin alone agree bit for bit with those that read both
    T sT = (T)s, cT = (T)c;
    if (c >= COMPACT_PHASE_MIN_COS) cT = cos_from_sin(sT);
    else wide = true;
    // kappa_of() needs pi to be a normal number of T on every open site
    if (e[i] > 0.0 && !((T)p >= (sizeof(T) == 8 ? (T)2.2250738585072014e-308 : (T)1.17549435e-38f))) bad++;
    pi[j] = (T)p;
    cs[j] = cT;
    cs[L.np + j] = sT;
  }
  if (bad) atomicAdd(&ctl->bad, bad);
  if (wide) ctl->wide_phase = 1u;
}

// Ghost layers of nch channel planes, all of them: L.gh planes / rows in x and y, GHZ columns in z, edges and corners
// included.  A ghost cell takes the interior value it wraps to when every axis on which it lies outside is periodic (1),
// and 0 as soon as one of them is reflective (0): nothing crosses a wall.  perx = 2 (slab mode): cells outside in x
// belong to the caller and are left alone.  The shell is enumerated as x slabs (all of y, z), then y slabs (interior x,
// all of z), then z columns (interior x and y).
template <typename T>
__global__ void fill_ghosts_kernel(T* __restrict__ f, int nch, Layout L, int perx, int pery, int perz) {
  const int gh = L.gh;
  const long long wy = L.ny + 2 * gh, wz = L.nz + 2 * GHZ;
  const long long ca = 2ll * gh * wy * wz, cb = (long long)L.nx * 2 * gh * wz, cc = (long long)L.nx * L.ny * 2 * GHZ;
  const long long per_ch = ca + cb + cc;
  for (long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x; t < per_ch * nch; t += (long long)gridDim.x * blockDim.x) {
    const int c = (int)(t / per_ch);
    long long r = t % per_ch;
    int x, y, z;
    if (r < ca) {
      z = (int)(r % wz) - GHZ; r /= wz;
      y = (int)(r % wy) - gh; r /= wy;
      x = (int)r; x = x < gh ? x - gh : L.nx + (x - gh);
    } else if (r < ca + cb) {
      r -= ca;
      z = (int)(r % wz) - GHZ; r /= wz;
      y = (int)(r % (2 * gh)); r /= 2 * gh;
      y = y < gh ? y - gh : L.ny + (y - gh);
      x = (int)r;
    } else {
      r -= ca + cb;
      z = (int)(r % (2 * GHZ)); r /= 2 * GHZ;
      z = z < GHZ ? z - GHZ : L.nz + (z - GHZ);
      y = (int)(r % L.ny);
      x = (int)(r / L.ny);
    }
    const bool ox = x < 0 || x >= L.nx, oy = y < 0 || y >= L.ny, oz = z < 0 || z >= L.nz;
    if (ox && perx == 2) continue;
    const bool wall = (ox && !perx) || (oy && !pery) || (oz && !perz);
    T* g = f + (long long)c * L.np;
    T v = (T)0;
    if (!wall) {
      const int sx = ((x % L.nx) + L.nx) % L.nx, sy = ((y % L.ny) + L.ny) % L.ny, sz = ((z % L.nz) + L.nz) % L.nz;
      v = g[L.idx(sx, sy, sz)];
    }
    g[L.idx(x, y, z)] = v;
  }
}

// Stored link weights for per-link mobility factors: m_{i,+d} = alpha_{i,i+e_d} min(pi_i, pi_{i+e_d})
// for the interior sites of channel d; `link` points at site i0 of the dense factor array of that axis.  The
// ghosts of pi are in place (wrapped value or 0), so a link through a reflective wall gets weight 0.
template <typename T>
__global__ void link_weights_kernel(const double* __restrict__ link, long long i0, long long n, Layout L, long long stride,
                                    const T* __restrict__ pi, T* __restrict__ m, Ctl* ctl) {
  unsigned long long bad = 0;
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
    const long long j = dense_to_padded(L, i0 + k);
    const double a = link[k];
    if (!(a >= 0.0 && a <= 1.0)) bad++;
    m[j] = (T)a * tmin(pi[j], pi[j + stride]);
  }
  if (bad) atomicAdd(&ctl->bad, bad);
}

// Initial state in density-normalised form:
//   h = 1 on open sites (g(0) = pi, real), r = 1 (rho(0) = pi),
//   q^d(1) = P^d(1)/pi = a kappa_i [m_{i,-d} - m_{i,+d}]                       (O7; Eq. 4, 5)
// and the sums G[0] = sum pi h, Z_d[1] = a^2 (alpha/6) sum_i [m_{i,+d} + m_{i,-d}].
template <typename T, int NRHO, int NMOM>
__global__ void __launch_bounds__(256)
    init_state_kernel(Layout L, const T* __restrict__ pi, const T* __restrict__ mlink, T a6, T* __restrict__ f, double a_len,
                      double* partials, Ctl* ctl, double2* fid, double* vacf, long long vacf_stride, double zscale) {
  constexpr int NRED = 2 + NMOM;
  double acc[NRED];
#pragma unroll
  for (int r = 0; r < NRED; ++r) acc[r] = 0.0;
  const long long n = (long long)L.nx * L.ny * L.nz;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const long long j = dense_to_padded(L, i);
    const T p = pi[j];
    const T one = (p > (T)0) ? (T)1 : (T)0;
    f[j] = one;
    f[L.np + j] = (T)0;
    acc[0] += (double)p * (double)one;
    if (NRHO) f[2 * L.np + j] = one;
    if (NMOM == 3) {
      const long long st[3] = {L.sx, L.sy, 1};
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const T* ml = mlink + (long long)d * L.np + j;
        const T mm = mlink ? ml[-st[d]] : tmin(p, pi[j - st[d]]), mp = mlink ? ml[0] : tmin(p, pi[j + st[d]]);
        f[(long long)(2 + NRHO + d) * L.np + j] = (T)a_len * kappa_of(p, a6) * (mm - mp);
        acc[2 + d] += (double)mp + (double)mm;
      }
    }
  }
  __shared__ double red[8 * NRED + 1];
  block_reduce_finalize<NRED, FIN_INIT, NMOM>(acc, red, partials, ctl, fid, vacf, vacf_stride, zscale, gridDim.x, blockIdx.x);
}

// h = g / pi from a dense interleaved complex array (points at site i0); carbon sites -> 0.
template <typename T>
__global__ void set_h_kernel(const double* __restrict__ g_re_im, long long i0, long long n, Layout L, const T* __restrict__ pi,
                             T* __restrict__ f) {
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
    const long long j = dense_to_padded(L, i0 + k);
    const double p = (double)pi[j];
    f[j] = (T)(p > 0.0 ? g_re_im[2 * k] / p : 0.0);
    f[L.np + j] = (T)(p > 0.0 ? g_re_im[2 * k + 1] / p : 0.0);
  }
}

// one real channel phi = v / pi from a dense array
template <typename T>
__global__ void set_real_kernel(const double* __restrict__ v, long long i0, long long n, Layout L, const T* __restrict__ pi,
                                T* __restrict__ fch) {
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
    const long long j = dense_to_padded(L, i0 + k);
    const double p = (double)pi[j];
    fch[j] = (T)(p > 0.0 ? v[k] / p : 0.0);
  }
}

// G[0] = sum_i pi_i h_i for a state that was set from outside.
template <typename T>
__global__ void __launch_bounds__(256)
    reduce_g_kernel(Layout L, const T* __restrict__ pi, const T* __restrict__ f, double* partials, Ctl* ctl, double2* fid) {
  double acc[2] = {0.0, 0.0};
  const long long n = (long long)L.nx * L.ny * L.nz;
  for (long long i = (long long)blockIdx.x * blockDim.x + threadIdx.x; i < n; i += (long long)gridDim.x * blockDim.x) {
    const long long j = dense_to_padded(L, i);
    acc[0] += (double)pi[j] * (double)f[j];
    acc[1] += (double)pi[j] * (double)f[L.np + j];
  }
  __shared__ double red[8 * 2 + 1];
  block_reduce_finalize<2, FIN_INIT, 0>(acc, red, partials, ctl, fid, nullptr, 0, 0.0, gridDim.x, blockIdx.x);
}

// Dense read-out of sites [i0, i0+n): mode 0 complex g = pi h (2 doubles per site), mode 1 pi,
// mode 2 real channel times pi.
template <typename T>
__global__ void gather_field_kernel(int mode, long long i0, long long n, Layout L, const T* __restrict__ pi, const T* __restrict__ fch,
                                    double* __restrict__ out) {
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < n; k += (long long)gridDim.x * blockDim.x) {
    const long long j = dense_to_padded(L, i0 + k);
    const double p = (double)pi[j];
    if (mode == 0) {
      out[2 * k] = p * (double)fch[j];
      out[2 * k + 1] = p * (double)fch[L.np + j];
    } else if (mode == 1) {
      out[k] = p;
    } else {
      out[k] = p * (double)fch[j];
    }
  }
}

// D_d = Z_d[1]/(2 dt) + (1/dt) sum_{m=2..count} Z_d[m]   (Eq. 4); block d, fixed order.
__global__ void __launch_bounds__(256) diffusion_kernel(const double* __restrict__ vacf, long long vacf_stride, long long count,
                                                        double dt, Ctl* ctl) {
  const double* z = vacf + blockIdx.x * vacf_stride;
  double acc = 0.0;
  for (long long m = 2 + threadIdx.x; m <= count; m += blockDim.x) acc += z[m];
  __shared__ double red[8];
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  double v = warp_sum(acc);
  if (lane == 0) red[warp] = v;
  __syncthreads();
  if (threadIdx.x == 0) {
    double t = 0.0;
    for (int w = 0; w < 8; ++w) t += red[w];
    ctl->scratch[blockIdx.x] = z[1] / (2.0 * dt) + t / dt;
  }
}

}  // namespace lpc
