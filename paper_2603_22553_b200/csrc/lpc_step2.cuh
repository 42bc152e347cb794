// lpc_step2.cuh -- TWO time steps per sweep (temporal blocking of Eq. 13; north star (b) "optional temporal
// blocking of several steps per pass").  The magnetisation channels (h_re, h_im) or the three moment
// channels of the VACF; no density or link channels, no region labels, no direct halo stores.
//
// Eq. 13 is a Jacobi update: g(n+1) depends on g(n) at the site and its six neighbours only.  Two steps therefore depend
// on the sites within two hops, and a CTA that stages a (TY+4) x (TZ+2 VW) window of the y-z plane can advance its
// TY x TZ tile twice without going back to HBM: state and parameters are read once and written once per TWO steps
// (28 B per site-step in fp64 instead of 56, plus the halo rows that L2 does not absorb).
//
// A CTA marches along x like the one-step sweep (lpc_step_vec.cuh).  Input plane j (absolute x0 - 2 + j) comes in by TMA
// into one of six stages: h_re, h_im and pi on the window with two halo rows / one 16-byte halo group, cos and sin on the
// window with one.  Per iteration t every thread does, for ITS group of VW consecutive z sites (one 16-byte vector),
//   first step : plane t+1 on the (TY+2) x (TZ/VW+2) groups of the tile and its ring of neighbours -> shared-memory ring
//                of three planes (the intermediate state g(n+1) never reaches HBM),
//   second step: plane t-1 on the TY x TZ/VW groups of the tile, neighbours from that ring            -> global memory,
// then one __syncthreads.  The two halves of an iteration do not depend on one another (the second step reads what the
// first step wrote one and two iterations earlier), so a thread has two independent instruction streams in flight; the
// x-1 / x / x+1 values of its groups stay in registers for both steps, rotating through three register planes each (the
// loop is unrolled by three).  11 warps, one CTA per SM, about 170 registers per thread.
//
// G[n+1] is accumulated by the first step over the tile's OWN sites only (the ring of neighbours belongs to other
// tiles), G[n+2] by the second step; one block partial of four numbers, fixed-order final sum by the last CTA.
// Per-site arithmetic is SiteUpdate::gather + phase_rotate, the same as in the one-step kernels: after two steps the state
// agrees with theirs bit for bit (tests/test_gpu_parity.py::test_two_step_sweep_*).
//
// Boundaries: the sweep reads ghost cells two deep, including the edges between two axes (a site's second neighbours
// (x+-1, y+-1) ...), so it needs the full ghost shell of the padded layout (fill_ghosts_kernel) on entry and keeps it
// valid itself: sites within two of a periodic face store their ghost images too (store_images, out of line).
#pragma once

#include "lpc_internal.cuh"

namespace lpc {

// NC = 2: the magnetisation (h_re, h_im; phase rotation; G of both steps).  NC = 3: the three moment fields q^d of the
// VACF (Eq. 4; no phase, no cos / sin traffic; Z_d of both steps) -- they propagate independently of the
// magnetisation, so a lattice with moment fields runs one two-step sweep of each kind per two steps.
template <typename T, int VW, int NC = 2, int TZ_ = 64>
struct Step2Cfg {
  static constexpr bool MAG = (NC == 2);
  static constexpr int TZ = TZ_;
  static constexpr int TY = 4 * VW;                 // 8 rows of z-pairs in fp64, 16 rows of z-quads in fp32: 256 own groups
  static constexpr int GZ = TZ / VW;                // own groups per row
  static constexpr int G1 = GZ + 2;                 // groups per row of the first step: one more on each side
  static constexpr int TZW = G1 * VW;               // row pitch of every staged box and of the ring (elements)
  static constexpr int R0 = TY + 4;                 // rows of the h / pi boxes (two halo rows)
  static constexpr int R1 = TY + 2;                 // rows of the first step, of the ring and of the cos / sin box
  static constexpr int N1 = R1 * G1;                // thread slots of the first step (340 / 324)
  static constexpr int N2 = TY * GZ;                // thread slots of the second step (256)
  static constexpr int NTHREADS = (N1 + 31) / 32 * 32;
  static constexpr int NSTAGE = 6;                  // a plane is in use for four iterations; two more are in flight
  static constexpr int F_BYTES = NC * R0 * TZW * (int)sizeof(T);
  static constexpr int PI_BYTES = R0 * TZW * (int)sizeof(T);
  static constexpr int CS_BYTES = MAG ? 2 * R1 * TZW * (int)sizeof(T) : 0;
  static constexpr int STAGE_BYTES = F_BYTES + PI_BYTES + CS_BYTES;
  static constexpr int RING_PLANE = NC * R1 * TZW * (int)sizeof(T);
  static constexpr int RING_OFF = NSTAGE * STAGE_BYTES;
  static constexpr int BAR_OFF = RING_OFF + 3 * RING_PLANE;
  static constexpr int RED_OFF = BAR_OFF + NSTAGE * 8;
  static constexpr int NRED = 2 * (MAG ? 2 : 3);    // G_re, G_im (or Z_x, Z_y, Z_z) of the first and of the second step
  static constexpr int SMEM_BYTES = RED_OFF + ((NTHREADS / 32) * NRED + 2) * 8 + 128;   // +128: manual alignment slack
  static_assert(F_BYTES % 128 == 0 && PI_BYTES % 128 == 0 && CS_BYTES % 128 == 0, "TMA boxes land 128-byte aligned");
  static_assert(RING_PLANE % 16 == 0 && RING_OFF % 128 == 0, "16-byte vector accesses to the ring");
  static_assert(SMEM_BYTES <= 227 * 1024, "one CTA per SM");
};

// A group of a periodic face region and all its ghost images: every combination of the shifts that map the site into the
// ghost shell (two layers in x, y and z; edges and corners included).  Rare, out of line.
template <typename T, int VW>
__device__ __noinline__ void store_images(T* __restrict__ base, long long sx, long long sy, int gh, int padz, int nx, int ny, int nz, int permask, int x,
                                          int y, int z, typename VecN<T, VW>::type v, int nvalid) {
  T o[VW];
  o[0] = v.x; o[1] = v.y;
  if constexpr (VW == 4) { o[2] = v.z; o[3] = v.w; }
  int dx[3], dy[3], ndx = 1, ndy = 1;
  dx[0] = 0; dy[0] = 0;
  if (permask & 1) {
    if (x < GH) dx[ndx++] = nx;
    if (x >= nx - GH) dx[ndx++] = -nx;
  }
  if (permask & 2) {
    if (y < GH) dy[ndy++] = ny;
    if (y >= ny - GH) dy[ndy++] = -ny;
  }
  for (int k = 0; k < VW && k < nvalid; ++k) {
    const int zk = z + k;
    int dz[3], ndz = 1;
    dz[0] = 0;
    if (permask & 4) {
      if (zk < GHZ) dz[ndz++] = nz;
      if (zk >= nz - GHZ) dz[ndz++] = -nz;
    }
    for (int a = 0; a < ndx; ++a)
      for (int b = 0; b < ndy; ++b)
        for (int c = 0; c < ndz; ++c)
          base[(long long)(x + dx[a] + gh) * sx + (long long)(y + dy[b] + gh) * sy + (zk + dz[c] + padz)] = o[k];
  }
}

template <typename T, int VW, int NC>
__global__ void __launch_bounds__(Step2Cfg<T, VW, NC>::NTHREADS, 1)
    step2_kernel(const __grid_constant__ CUtensorMap tm_f, const __grid_constant__ CUtensorMap tm_pi, const __grid_constant__ CUtensorMap tm_cs,
                 StepArgs<T> a) {
  using K = Step2Cfg<T, VW, NC>;
  using V = typename VecN<T, VW>::type;
  constexpr int TZW = K::TZW, R0 = K::R0, R1 = K::R1, NS = K::NSTAGE;
  constexpr bool MAG = K::MAG;
  constexpr int HR = K::NRED / 2;   // reductions per step
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + K::BAR_OFF);
  double* red = reinterpret_cast<double*>(smem + K::RED_OFF);

  const Layout& L = a.L;
  const int bz = blockIdx.x % a.tiles_z;
  const int by = (blockIdx.x / a.tiles_z) % a.tiles_y;
  const int bx = blockIdx.x / (a.tiles_z * a.tiles_y);
  const int z0 = bz * K::TZ, y0 = by * K::TY, x0 = bx * a.xc;
  const int nplanes = min(a.xc, L.nx - x0);   // planes this CTA advances: absolute x0 .. x0 + nplanes - 1 = input planes j = 2 .. nplanes + 1
  const int nin = nplanes + 4;                // input planes j = 0 .. nin - 1, absolute x0 - 2 + j
  const int tid = threadIdx.x;

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    mbar_fence_init();
  }
  __syncthreads();

  // ----- TMA issue (thread 0).  Padded coordinates: plane (x0 - 2 + j) + gh = x0 + j, rows from (y0 - 2) + gh = y0 -----
  auto issue = [&](int j) {
    const int s = j % NS;
    unsigned char* st = smem + s * K::STAGE_BYTES;
    mbar_expect_tx(&full[s], K::STAGE_BYTES);
    const int pz = L.padz + z0 - VW, py = y0 + L.gh - 2, px = x0 + j + L.gh - 2;
    tma_load_4d(st, &tm_f, &full[s], pz, py, px, a.c0);
    tma_load_3d(st + K::F_BYTES, &tm_pi, &full[s], pz, py, px);
    if constexpr (MAG) tma_load_4d(st + K::F_BYTES + K::PI_BYTES, &tm_cs, &full[s], pz, py + 1, px, 0);
  };
  if (tid == 0) {
    tma_prefetch_desc(&tm_f);
    tma_prefetch_desc(&tm_pi);
    if constexpr (MAG) tma_prefetch_desc(&tm_cs);
    for (int j = 0; j < 4 && j < nin; ++j) issue(j);
  }

  // ----- thread slots -----
  // first step: slot s1 = tid over R1 rows of G1 groups; since TZW = G1 * VW the slots are contiguous in shared memory
  const bool act1 = tid < K::N1;
  const int r1 = tid / K::G1, g1 = tid - r1 * K::G1;
  const int e1 = TZW + VW * tid;                      // the group in a box with two halo rows (h, pi)
  const int k1 = VW * tid;                            // ... in a box with one (cos / sin, ring)
  int nv1 = 0;                                        // own sites of the group that exist (they count towards G[n+1])
  if (act1 && r1 >= 1 && r1 <= K::TY && g1 >= 1 && g1 <= K::GZ && y0 - 1 + r1 < L.ny) nv1 = max(0, min(VW, L.nz - (z0 - VW + VW * g1)));
  // second step: slot s2 = tid over TY rows of GZ groups
  const bool act2 = tid < K::N2;
  const int r2 = tid / K::GZ, g2 = tid % K::GZ;
  const int y2 = y0 + r2, z2 = z0 + VW * g2;
  const int e2 = (r2 + 2) * TZW + VW + VW * g2;
  const int k2 = (r2 + 1) * TZW + VW + VW * g2;
  const int nv2 = (act2 && y2 < L.ny) ? max(0, min(VW, L.nz - z2)) : 0;
  const int permask = (a.per[0] ? 1 : 0) | (a.per[1] ? 2 : 0) | (a.per[2] ? 4 : 0);
  const bool edge_yz = (a.per[1] && (y2 < GH || y2 >= L.ny - GH)) || (a.per[2] && (z2 < GHZ || z2 + VW > L.nz - GHZ));
  T* outp = a.fout + L.idx(x0, y2, z2);

  double acc[K::NRED];
#pragma unroll
  for (int r = 0; r < K::NRED; ++r) acc[r] = 0.0;

  // one x-plane as a thread holds it: the group's h and pi, and mlo = the link weight towards the plane below
  struct Plane {
    T f[NC][VW];
    T pi[VW], mlo[VW];
  };
  auto stage_of = [&](int j) -> const unsigned char* { return smem + (j % NS) * K::STAGE_BYTES; };
  auto wait_plane = [&](int j) { mbar_wait(&full[j % NS], (uint32_t)((j / NS) & 1)); };

  // the update of one group whose plane is the centre one: sf = h_re of the centre plane at the group (h_im is fch elements
  // further), sp = pi, sc = cos (sin is kch further); in-plane neighbours at +-TZW (y) and -1 / +VW (z)
  auto update = [&](const Plane& prv, const Plane& ctr, const Plane& nxt, const T* sf, int fch, const T* sp, const T* sc, int kch, T (&o)[NC][VW],
                    double* zacc, int nvz) {
    T pym[VW], pyp[VW], csv[VW], snv[VW];
    ldv<T, VW>(sp - TZW, pym);
    ldv<T, VW>(sp + TZW, pyp);
    const T pzm = sp[-1], pzp = sp[VW];
    if constexpr (MAG) {
      ldv<T, VW>(sc, csv);
      ldv<T, VW>(sc + kch, snv);
    }
    SiteUpdate<T, 0, 0> u[VW];
#pragma unroll
    for (int k = 0; k < VW; ++k) {
      u[k].mxm = ctr.mlo[k]; u[k].mxp = nxt.mlo[k];
      u[k].mym = tmin(ctr.pi[k], pym[k]); u[k].myp = tmin(ctr.pi[k], pyp[k]);
      u[k].mzp = tmin(ctr.pi[k], k == VW - 1 ? pzp : ctr.pi[k == VW - 1 ? k : k + 1]);
    }
    u[0].mzm = tmin(ctr.pi[0], pzm);
#pragma unroll
    for (int k = 1; k < VW; ++k) u[k].mzm = u[k - 1].mzp;
#pragma unroll
    for (int k = 0; k < VW; ++k) {
      u[k].pc = ctr.pi[k];
      u[k].kap = kappa_of(ctr.pi[k], a.a6);
      u[k].sum_weights();
    }
#pragma unroll
    for (int c = 0; c < NC; ++c) {
      const T* fcn = sf + c * fch;
      T fym[VW], fyp[VW];
      ldv<T, VW>(fcn - TZW, fym);
      ldv<T, VW>(fcn + TZW, fyp);
      const T fzm = fcn[-1], fzp = fcn[VW];
      if constexpr (!MAG) {
        // Z_d of this step (Eq. 4): sum over the tile's own sites of q^d_i (m_{i,+d} - m_{i,-d}), from the values BEFORE the update
        if (zacc) {
          double t = 0.0;
#pragma unroll
          for (int k = 0; k < VW; ++k) {
            const T dm = (c == 0) ? (u[k].mxp - u[k].mxm) : (c == 1) ? (u[k].myp - u[k].mym) : (u[k].mzp - u[k].mzm);
            const double qd = (double)ctr.f[c][k] * (double)dm;
            if (k < nvz) t += qd;
          }
          zacc[c] += t;
        }
      }
#pragma unroll
      for (int k = 0; k < VW; ++k)
        o[c][k] = u[k].gather(ctr.f[c][k], prv.f[c][k], nxt.f[c][k], fym[k], fyp[k], k == 0 ? fzm : ctr.f[c][k ? k - 1 : 0],
                              k == VW - 1 ? fzp : ctr.f[c][k == VW - 1 ? k : k + 1]);
    }
    if constexpr (MAG) {
#pragma unroll
      for (int k = 0; k < VW; ++k) {
        const T hr = o[0][k], hi = o[1][k];
        phase_rotate(csv[k], snv[k], hr, hi, o[0][k], o[1][k]);
      }
    }
  };

  // first step: registers of input plane j
  auto take1 = [&](Plane& n, int j, const Plane* below) {
    const T* sf = reinterpret_cast<const T*>(stage_of(j));
    const T* sp = reinterpret_cast<const T*>(stage_of(j) + K::F_BYTES);
#pragma unroll
    for (int c = 0; c < NC; ++c) ldv<T, VW>(sf + c * R0 * TZW + e1, n.f[c]);
    ldv<T, VW>(sp + e1, n.pi);
    if (below) {
#pragma unroll
      for (int k = 0; k < VW; ++k) n.mlo[k] = tmin(n.pi[k], below->pi[k]);
    }
  };
  // second step: registers of intermediate plane j (ring) and pi of input plane j
  auto take2 = [&](Plane& n, int j, const Plane& below) {
    const T* rf = reinterpret_cast<const T*>(smem + K::RING_OFF + (j % 3) * K::RING_PLANE);
    const T* sp = reinterpret_cast<const T*>(stage_of(j) + K::F_BYTES);
#pragma unroll
    for (int c = 0; c < NC; ++c) ldv<T, VW>(rf + c * R1 * TZW + k2, n.f[c]);
    ldv<T, VW>(sp + e2, n.pi);
#pragma unroll
    for (int k = 0; k < VW; ++k) n.mlo[k] = tmin(n.pi[k], below.pi[k]);
  };

  // iteration t: first step of plane t + 1 (needs input planes t, t+1, t+2), second step of plane t - 1 (needs
  // intermediate planes t-2, t-1, t); A* / B* are the register planes in their roles of this iteration
  auto iteration = [&](int t, const Plane& Aprv, const Plane& Actr, Plane& Anxt, const Plane& Bprv, const Plane& Bctr, Plane& Bnxt) {
    if (tid == 0 && t + 4 < nin) issue(t + 4);   // into the stage of plane t - 2, whose last reader passed the barrier of iteration t - 1
    if (act1 && t <= nplanes + 1) {
      const int j = t + 1;
      wait_plane(t + 2);
      take1(Anxt, t + 2, &Actr);
      const unsigned char* st = stage_of(j);
      const T* sf = reinterpret_cast<const T*>(st) + e1;
      const T* sp = reinterpret_cast<const T*>(st + K::F_BYTES) + e1;
      const T* sc = reinterpret_cast<const T*>(st + K::F_BYTES + K::PI_BYTES) + k1;
      T o[NC][VW];
      const bool own_plane = j >= 2 && j <= nplanes + 1;   // a plane of this CTA's own chunk: its own sites count towards the sums
      update(Aprv, Actr, Anxt, sf, R0 * TZW, sp, sc, R1 * TZW, o, (!MAG && own_plane) ? acc : nullptr, nv1);
      T* rf = reinterpret_cast<T*>(smem + K::RING_OFF + (j % 3) * K::RING_PLANE);
#pragma unroll
      for (int c = 0; c < NC; ++c) *reinterpret_cast<V*>(rf + c * R1 * TZW + k1) = packv<T, VW>(o[c]);
      if (MAG && own_plane) {   // G[n+1]
#pragma unroll
        for (int k = 0; k < VW; ++k)
          if (k < nv1) {
            acc[0] += (double)Actr.pi[k] * (double)o[0][k];
            acc[1] += (double)Actr.pi[k] * (double)o[1][k];
          }
      }
    }
    if (act2 && t >= 1) {
      take2(Bnxt, t, Bctr);
      if (t >= 3) {
        const int j = t - 1, x = x0 - 2 + j;
        const unsigned char* st = stage_of(j);
        const T* rf = reinterpret_cast<const T*>(smem + K::RING_OFF + (j % 3) * K::RING_PLANE) + k2;
        const T* sp = reinterpret_cast<const T*>(st + K::F_BYTES) + e2;
        const T* sc = reinterpret_cast<const T*>(st + K::F_BYTES + K::PI_BYTES) + k2;
        T o[NC][VW];
        update(Bprv, Bctr, Bnxt, rf, R1 * TZW, sp, sc, R1 * TZW, o, MAG ? nullptr : acc + HR, nv2);
        if constexpr (MAG) {   // G[n+2]
#pragma unroll
          for (int k = 0; k < VW; ++k)
            if (k < nv2) {
              acc[2] += (double)Bctr.pi[k] * (double)o[0][k];
              acc[3] += (double)Bctr.pi[k] * (double)o[1][k];
            }
        }
        if (nv2 > 0) {
          if (edge_yz || (a.per[0] && (x < GH || x >= L.nx - GH))) {
#pragma unroll
            for (int c = 0; c < NC; ++c)
              store_images<T, VW>(a.fout + (long long)c * L.np, L.sx, L.sy, L.gh, L.padz, L.nx, L.ny, L.nz, permask, x, y2, z2, packv<T, VW>(o[c]), nv2);
          } else {
#pragma unroll
            for (int c = 0; c < NC; ++c) store_vec<T, VW>(outp + (long long)c * L.np, packv<T, VW>(o[c]), nv2);
          }
        }
        outp += L.sx;
      }
    }
    __syncthreads();
  };

  Plane A0, A1, A2, B0, B1, B2;
#pragma unroll
  for (int k = 0; k < VW; ++k) B0.pi[k] = B1.pi[k] = B2.pi[k] = (T)0;
  if (act1) {
    wait_plane(0);
    take1(A0, 0, nullptr);
    wait_plane(1);
    take1(A1, 1, &A0);
  }

  // unrolled by three so that the planes keep their registers while their roles rotate: at iteration t the first step has
  // prv / ctr / nxt = planes t, t+1, t+2 in A[t % 3], A[(t+1) % 3], A[(t+2) % 3]; the second step planes t-2, t-1, t in
  // B[(t+1) % 3], B[(t+2) % 3], B[t % 3]
  const int niter = nplanes + 3;
  int t = 0;
  for (; t + 3 <= niter; t += 3) {
    iteration(t, A0, A1, A2, B1, B2, B0);
    iteration(t + 1, A1, A2, A0, B2, B0, B1);
    iteration(t + 2, A2, A0, A1, B0, B1, B2);
  }
  if (t < niter) { iteration(t, A0, A1, A2, B1, B2, B0); ++t; }
  if (t < niter) { iteration(t, A1, A2, A0, B2, B0, B1); ++t; }

  block_reduce_finalize<K::NRED, MAG ? FIN_STEP2 : FIN_MOM2, MAG ? 0 : 3>(acc, red, a.partials, a.ctl, a.fid, a.vacf, a.vacf_stride, a.zscale, gridDim.x,
                                                                          blockIdx.x);
}

}  // namespace lpc
