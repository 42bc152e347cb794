// lpc_equil.cuh -- the equilibration loop of the paper's workflow (Fig. 3 step 3, PAPER.md:168-172,
// 190-194): iterate the density update rho <- W rho and compare rho(t) with rho(t+1).
//
// One sweep = one launch of equil_kernel: the real-field gather of the step kernel (no phase) on the
// density channel r = rho/pi, fused with the convergence measure
//     delta = max_i |rho_i(t+1) - rho_i(t)| = max_i pi_i |r'_i - r_i|          (reading Q25)
// reduced per warp (shuffle), per block (one partial) and by the last block to finish (fixed data,
// max is order-independent).  The density channel ping-pongs between the two state buffers; the
// other channels are not touched.
#pragma once

#include "lpc_internal.cuh"
#include "lpc_step.cuh"

namespace lpc {

template <typename T>
struct EquilArgs {
  Layout L;
  const T* rin;   // density channel of the buffer that holds rho(t)
  T* rout;        // density channel of the other buffer
  const T* pi;
  const T* mlink;  // nullptr or the stored link weights (per-link mobility)
  T a6;
  double* partials;
  Ctl* ctl;
  int per[3];
};

// ctl->scratch[4] = delta of this sweep, ctl->scratch[5] += 1 (sweeps since the loop started)
template <typename T>
__global__ void __launch_bounds__(256) equil_kernel(EquilArgs<T> a) {
  const Layout& L = a.L;
  const long long zpairs = (L.nz + 1) / 2;
  const long long npairs = zpairs * L.ny * L.nx;
  const T* __restrict__ pi = a.pi;
  const T* __restrict__ f = a.rin;
  double dmax = 0.0;
  for (long long p = (long long)blockIdx.x * blockDim.x + threadIdx.x; p < npairs; p += (long long)gridDim.x * blockDim.x) {
    const int z = 2 * (int)(p % zpairs);
    const long long r = p / zpairs;
    const int y = (int)(r % L.ny);
    const int x = (int)(r / L.ny);
    const long long i = L.idx(x, y, z);
    const bool vb = (z + 1 < L.nz);
    T out[2] = {(T)0, (T)0};
#pragma unroll
    for (int s = 0; s < 2; ++s) {
      if (s == 1 && !vb) break;
      const long long j = i + s;
      SiteUpdate<T, 0, 0> u;
      if (a.mlink)
        u.weights_links(pi[j], a.mlink + j, L.np, L.sx, L.sy, a.a6, (T)1, (T)0);
      else
        u.weights(pi[j], pi[j - L.sx], pi[j + L.sx], pi[j - L.sy], pi[j + L.sy], pi[j - 1], pi[j + 1], a.a6, (T)1, (T)0);
      const T fc = f[j];
      out[s] = u.gather(fc, f[j - L.sx], f[j + L.sx], f[j - L.sy], f[j + L.sy], f[j - 1], f[j + 1]);
      // rho' - rho = pi (r' - r); the product and the difference are taken in fp64
      dmax = fmax(dmax, (double)u.pc * fabs((double)out[s] - (double)fc));
    }
    store_with_ghosts(a.rout, L, a.per, i, x, y, z, out[0], out[1], vb);
  }
  __shared__ double red[8 + 1];
  block_max_finalize(dmax, red, a.partials, a.ctl, gridDim.x, blockIdx.x);
}

// g(0) <- rho: h = r (real) on every site, ghosts included (they already mirror r).
template <typename T>
__global__ void seed_h_from_r_kernel(long long np, const T* __restrict__ r, T* __restrict__ h_re, T* __restrict__ h_im) {
  for (long long k = (long long)blockIdx.x * blockDim.x + threadIdx.x; k < np; k += (long long)gridDim.x * blockDim.x) {
    h_re[k] = r[k];
    h_im[k] = (T)0;
  }
}

}  // namespace lpc
