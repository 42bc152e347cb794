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
// window with one.  The two steps belong to two groups of warps that run a plane or two apart and meet only through
// mbarriers (no __syncthreads in the march):
//   step-1 warps (TY+2 row warps + one edge warp): iteration t takes the first step of plane t+1 on the (TY+2) x (32+2)
//       groups of the tile and its ring of neighbours and writes it to a shared-memory ring of four planes (the
//       intermediate state g(n+1) never reaches HBM);
//   step-2 warps (TY row warps): iteration t takes the second step of plane t-1 on the TY x 32 groups of the tile, with
//       the neighbours from that ring, and stores it to global memory.
// A warp owns one row of the window and a lane one 16-byte group of VW consecutive z sites, so every shared-memory access
// of a warp is one contiguous 512-byte run; the x-1 / x / x+1 values of a group stay in registers, rotating through three
// register planes (the loops are unrolled by three).  The edge warp takes the two groups left and right of every row.
// Lane 0 of the first step-2 warp issues the TMA loads four planes ahead.  19 warps, one CTA per SM.
//
// Hand-over: adone[t & 3] -- every step-1 warp has finished iteration t (ring plane t+1 is written, stage planes <= t are
// no longer read by step 1); bdone[t & 3] -- every step-2 warp has finished iteration t (ring plane t-1 and stage plane
// t-1 are no longer read).  Step 1 waits for bdone[t-2] before it overwrites ring slot (t+1) & 3, step 2 for adone[t-1]
// before it reads ring plane t, the load of plane t+4 for bdone[t-1].
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
// CPH: the phase factors are staged as sin alone and cos is rebuilt (cos_from_sin; lattices whose phase angles are all small).
template <typename T, int VW, int NC = 2, bool CPH = false, int TY_ = 8>
struct Step2Cfg {
  static constexpr bool MAG = (NC == 2);
  static constexpr int GZ = 32;                     // own groups per row: one per lane of a row warp
  static constexpr int TZ = GZ * VW;                // 64 sites of a row in fp64 (pairs), 128 in fp32 (quads)
  static constexpr int TY = TY_;
  static constexpr int G1 = GZ + 2;                 // groups per row of the first step: one more on each side
  static constexpr int TZW = G1 * VW;               // row pitch of every staged box and of the ring (elements)
  static constexpr int R0 = TY + 4;                 // rows of the h / pi boxes (two halo rows)
  static constexpr int R1 = TY + 2;                 // rows of the first step, of the ring and of the cos / sin box
  static constexpr int NA = R1 + 1;                 // step-1 warps: one per row + the edge warp (groups 0 and G1-1 of every row)
  static constexpr int NB = TY;                     // step-2 warps: one per row
  static constexpr int NTHREADS = 32 * (NA + NB + 1);   // + the warp that issues the loads
  static constexpr int NSTAGE = CPH ? 5 : 4;        // step 1 reads a plane in two iterations; the others are in flight
  static constexpr int NRING = 4;                   // planes of the intermediate state: three in use by step 2, one being written
  static constexpr int ND = 4;                      // hand-over barriers per direction (iterations in flight)
  static constexpr int PF = 0;                      // > 0: every load also sends plane j + PF towards L2 (measured: no gain)
  static constexpr int F_BYTES = NC * R0 * TZW * (int)sizeof(T);
  static constexpr int PI_BYTES = R0 * TZW * (int)sizeof(T);
  static constexpr int NPH = MAG ? (CPH ? 1 : 2) : 0;   // staged phase channels: cos and sin, or sin alone
  static constexpr int CS_RAW = NPH * R1 * TZW * (int)sizeof(T);
  static constexpr int CS_BYTES = (CS_RAW + 127) / 128 * 128;
  static constexpr int STAGE_BYTES = F_BYTES + PI_BYTES + CS_BYTES;
  static constexpr int TX_BYTES = F_BYTES + PI_BYTES + CS_RAW;
  static constexpr int RCH = R1 * TZW;              // elements of one channel of a ring plane
  static constexpr int RING_PLANE = (NC + 1) * RCH * (int)sizeof(T);   // the intermediate state and pi (step 2 reads no stage)
  static constexpr int RING_OFF = NSTAGE * STAGE_BYTES;
  static constexpr int CSB_OFF = RING_OFF + NRING * RING_PLANE;        // step 2's own cos / sin: 16 bytes of each per thread
  static constexpr int CSB_BYTES = 2 * NPH * NB * 32 * 16;   // two slots: the plane in use and the next one
  static constexpr int BAR_OFF = CSB_OFF + CSB_BYTES;
  static constexpr int RED_OFF = BAR_OFF + (NSTAGE + 2 * ND) * 8;
  static constexpr int NRED = 2 * (MAG ? 2 : 3);    // G_re, G_im (or Z_x, Z_y, Z_z) of the first and of the second step
  static constexpr int SMEM_BYTES = RED_OFF + ((NTHREADS / 32) * NRED + 2) * 8 + 128;   // +128: manual alignment slack
  static_assert(2 * R1 <= 32, "the edge warp holds two groups of every row");
  static_assert((NRING & (NRING - 1)) == 0 && (ND & (ND - 1)) == 0, "slots are picked with a mask");
  static_assert(F_BYTES % 128 == 0 && PI_BYTES % 128 == 0 && CS_BYTES % 128 == 0 && (!MAG ? !CPH : true), "TMA boxes land 128-byte aligned");
  static_assert(RING_PLANE % 16 == 0 && RING_OFF % 128 == 0 && CSB_OFF % 16 == 0, "16-byte vector accesses to the ring");
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

template <typename T, int VW, int NC, bool CPH>
__global__ void __launch_bounds__(Step2Cfg<T, VW, NC, CPH>::NTHREADS, 1)
    step2_kernel(const __grid_constant__ CUtensorMap tm_f, const __grid_constant__ CUtensorMap tm_pi, const __grid_constant__ CUtensorMap tm_cs,
                 StepArgs<T> a) {
  using K = Step2Cfg<T, VW, NC, CPH>;
  using V = typename VecN<T, VW>::type;
  constexpr int TZW = K::TZW, R0 = K::R0, R1 = K::R1, NS = K::NSTAGE, RCH = K::RCH;
  constexpr bool MAG = K::MAG;
  constexpr int HR = K::NRED / 2;   // reductions per step
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + K::BAR_OFF);
  uint64_t* adone = full + NS;
  uint64_t* bdone = adone + K::ND;
  double* red = reinterpret_cast<double*>(smem + K::RED_OFF);

  const Layout& L = a.L;
  const int bz = blockIdx.x % a.tiles_z;
  const int by = (blockIdx.x / a.tiles_z) % a.tiles_y;
  const int bx = blockIdx.x / (a.tiles_z * a.tiles_y);
  const int z0 = bz * K::TZ, y0 = by * K::TY, x0 = bx * a.xc;
  const int nplanes = min(a.xc, L.nx - x0);   // planes this CTA advances: absolute x0 .. x0 + nplanes - 1 = input planes j = 2 .. nplanes + 1
  const int nin = nplanes + 4;                // input planes j = 0 .. nin - 1, absolute x0 - 2 + j
  const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;

  if (tid == 0) {
    for (int s = 0; s < NS; ++s) mbar_init(&full[s], 1);
    for (int s = 0; s < K::ND; ++s) {
      mbar_init(&adone[s], K::NA);
      mbar_init(&bdone[s], K::NB);
    }
    mbar_fence_init();
  }
  __syncthreads();
  pdl_launch_dependents();   // as in the one-step sweep (lpc_step_vec.cuh)
  pdl_wait();

  double acc[K::NRED];
#pragma unroll
  for (int r = 0; r < K::NRED; ++r) acc[r] = 0.0;

  // one x-plane as a thread holds it: the group's h and pi, and mlo = the link weight towards the plane below
  struct Plane {
    T f[NC][VW];
    T pi[VW], mlo[VW];
  };

  // the update of one group whose plane is the centre one: sf = h_re of the centre plane at the group (h_im is fch elements
  // further), sp = pi; in-plane neighbours at +-TZW (y) and -1 / +VW (z); phase(csv, snv) fetches cos and sin of the group
  // when the gather is done
  auto update = [&](const Plane& prv, const Plane& ctr, const Plane& nxt, const T* sf, int fch, const T* sp, auto&& phase, T (&o)[NC][VW],
                    double* zacc, int nvz) {
    T pym[VW], pyp[VW];
    ldv<T, VW>(sp - TZW, pym);
    ldv<T, VW>(sp + TZW, pyp);
    const T pzm = sp[-1], pzp = sp[VW];
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
      T csv[VW], snv[VW];
      phase(csv, snv);
#pragma unroll
      for (int k = 0; k < VW; ++k) {
        const T hr = o[0][k], hi = o[1][k];
        phase_rotate(csv[k], snv[k], hr, hi, o[0][k], o[1][k]);
      }
    }
  };

  if (warp == K::NA + K::NB) {
    // =============================== the loads: plane j into stage j % NS ===============================
    if (lane == 0) {
      // padded coordinates: plane (x0 - 2 + j) + gh = x0 + j, rows from (y0 - 2) + gh = y0
      auto issue = [&](int j) {
        const int s = j % NS;
        unsigned char* st = smem + s * K::STAGE_BYTES;
        mbar_expect_tx(&full[s], K::TX_BYTES);
        const int pz = L.padz + z0 - VW, py = y0 + L.gh - 2, px = x0 + j + L.gh - 2;
        tma_load_4d(st, &tm_f, &full[s], pz, py, px, a.c0);
        tma_load_3d(st + K::F_BYTES, &tm_pi, &full[s], pz, py, px);
        if constexpr (MAG) tma_load_4d(st + K::F_BYTES + K::PI_BYTES, &tm_cs, &full[s], pz, py + 1, px, CPH ? 1 : 0);
        if (K::PF > 0 && j + K::PF < nin) {
          tma_prefetch_4d(&tm_f, pz, py, px + K::PF, a.c0);
          tma_prefetch_3d(&tm_pi, pz, py, px + K::PF);
          if constexpr (MAG) tma_prefetch_4d(&tm_cs, pz, py + 1, px + K::PF, CPH ? 1 : 0);
        }
      };
      tma_prefetch_desc(&tm_f);
      tma_prefetch_desc(&tm_pi);
      if constexpr (MAG) tma_prefetch_desc(&tm_cs);
      for (int j = 0; j < NS && j < nin; ++j) issue(j);
      // plane t + NS takes the stage of plane t, which step 1 read last in its iteration t - 1 (plane 0: before iteration 0)
      for (int t = 0; t + NS < nin; ++t) {
        const int w = t > 0 ? t - 1 : 0;
        mbar_wait_parked(&adone[w & (K::ND - 1)], (uint32_t)((w / K::ND) & 1));
        issue(t + NS);
      }
    }
  } else if (warp < K::NA) {
    // =============================== first step: ring plane t + 1 at iteration t ===============================
    const bool roww = warp < R1;                         // a row warp: groups 1 .. 32 of row `warp`; the edge warp: groups 0 and 33 of all rows
    const bool act = roww || lane < 2 * R1;
    const int r1 = roww ? warp : (act ? (lane >> 1) : 0);
    const int g1 = roww ? lane + 1 : ((lane & 1) ? K::GZ + 1 : 0);
    const int e1 = (r1 + 1) * TZW + VW * g1;             // the group in a box with two halo rows (h, pi)
    const int k1 = r1 * TZW + VW * g1;                   // ... in a box with one (cos / sin, ring)
    // own sites of the group that exist (they count towards G[n+1]): rows 1 .. TY of a row warp, inside the lattice
    const bool own_row = roww && r1 >= 1 && r1 <= K::TY && y0 - 1 + r1 < L.ny;
    const int nv1 = own_row ? max(0, min(VW, L.nz - (z0 + VW * (g1 - 1)))) : 0;

    auto take1 = [&](Plane& n, int s, const Plane* below) {
      const T* sf = reinterpret_cast<const T*>(smem + s * K::STAGE_BYTES);
      const T* sp = reinterpret_cast<const T*>(smem + s * K::STAGE_BYTES + K::F_BYTES);
#pragma unroll
      for (int c = 0; c < NC; ++c) ldv<T, VW>(sf + c * R0 * TZW + e1, n.f[c]);
      ldv<T, VW>(sp + e1, n.pi);
      if (below) {
#pragma unroll
        for (int k = 0; k < VW; ++k) n.mlo[k] = tmin(n.pi[k], below->pi[k]);
      }
    };
    int sc = 1 % NS, sn = 2 % NS;   // stages of the centre plane t + 1 and of the plane t + 2 that is taken
    uint32_t pn = (2 / NS) & 1;     // phase of full[sn]
    auto iteration = [&](int t, const Plane& prv, const Plane& ctr, Plane& nxt) {
      if (act) {
        mbar_wait_parked(&full[sn], pn);
        take1(nxt, sn, &ctr);
        const unsigned char* st = smem + sc * K::STAGE_BYTES;
        const T* sf = reinterpret_cast<const T*>(st) + e1;
        const T* sp = reinterpret_cast<const T*>(st + K::F_BYTES) + e1;
        const T* sk = reinterpret_cast<const T*>(st + K::F_BYTES + K::PI_BYTES) + k1;
        T o[NC][VW];
        const bool own_plane = t >= 1 && t <= nplanes;   // plane j = t + 1 of this CTA's own chunk: its own sites count towards the sums
        update(prv, ctr, nxt, sf, R0 * TZW, sp,
               [&](T (&csv)[VW], T (&snv)[VW]) {
                 if constexpr (CPH) {
                   ldv<T, VW>(sk, snv);
#pragma unroll
                   for (int k = 0; k < VW; ++k) csv[k] = cos_from_sin(snv[k]);
                 } else {
                   ldv<T, VW>(sk, csv);
                   ldv<T, VW>(sk + R1 * TZW, snv);
                 }
               },
               o, (!MAG && own_plane) ? acc : nullptr, nv1);
        // ring slot (t + 1) & 3 held plane t - 3, which step 2 read last in its iteration t - 2
        if (t >= 3) mbar_wait_parked(&bdone[(t - 2) & (K::ND - 1)], (uint32_t)(((t - 2) / K::ND) & 1));
        T* rf = reinterpret_cast<T*>(smem + K::RING_OFF + ((t + 1) & (K::NRING - 1)) * K::RING_PLANE) + k1;
#pragma unroll
        for (int c = 0; c < NC; ++c) *reinterpret_cast<V*>(rf + c * RCH) = packv<T, VW>(o[c]);
        *reinterpret_cast<V*>(rf + NC * RCH) = packv<T, VW>(ctr.pi);   // step 2 takes pi from the ring as well
        if (MAG && own_plane) {   // G[n+1]
#pragma unroll
          for (int k = 0; k < VW; ++k)
            if (k < nv1) {
              acc[0] += (double)ctr.pi[k] * (double)o[0][k];
              acc[1] += (double)ctr.pi[k] * (double)o[1][k];
            }
        }
      }
      __syncwarp();
      if (lane == 0) mbar_arrive(&adone[t & (K::ND - 1)]);
      sc = sn;
      if (++sn == NS) {
        sn = 0;
        pn ^= 1u;
      }
    };

    Plane P0, P1, P2;
    if (act) {
      mbar_wait_parked(&full[0], 0);
      take1(P0, 0, nullptr);
      mbar_wait_parked(&full[1 % NS], 0);
      take1(P1, 1 % NS, &P0);
    }
    // unrolled by three so that the planes keep their registers while their roles rotate: at iteration t
    // prv / ctr / nxt = planes t, t+1, t+2 in P[t % 3], P[(t+1) % 3], P[(t+2) % 3]
    const int niter = nplanes + 2;
    int t = 0;
    for (; t + 3 <= niter; t += 3) {
      iteration(t, P0, P1, P2);
      iteration(t + 1, P1, P2, P0);
      iteration(t + 2, P2, P0, P1);
    }
    if (t < niter) { iteration(t, P0, P1, P2); ++t; }
    if (t < niter) { iteration(t, P1, P2, P0); ++t; }
  } else {
    // =============================== second step: output plane t - 1 at iteration t ===============================
    const int r2 = warp - K::NA;
    const int y2 = y0 + r2, z2 = z0 + VW * lane;
    const int k2 = (r2 + 1) * TZW + VW + VW * lane;      // the group in a ring plane
    const int nv2 = (y2 < L.ny) ? max(0, min(VW, L.nz - z2)) : 0;
    const int permask = (a.per[0] ? 1 : 0) | (a.per[1] ? 2 : 0) | (a.per[2] ? 4 : 0);
    const bool edge_yz = (a.per[1] && (y2 < GH || y2 >= L.ny - GH)) || (a.per[2] && (z2 < GHZ || z2 + VW > L.nz - GHZ));
    T* outp = a.fout + L.idx(x0, y2, z2);
    // cos and sin of the thread's own group come straight from global memory into a 16-byte slot of its own (cp.async),
    // one plane ahead: step 2 reads no stage, so the stages turn over at the pace of step 1 alone
    constexpr int CSLOT = K::NPH * K::NB * 32 * VW;      // elements of one slot: cos of every thread, then sin (CPH: sin alone)
    T* csb = reinterpret_cast<T*>(smem + K::CSB_OFF) + (r2 * 32 + lane) * VW;
    const T* csg = a.cs + L.idx(x0, y2, z2);
    // output plane j (absolute x0 - 2 + j) into slot j & 1; one group per call, so that wait<1> leaves only the latest in flight
    auto fetch_cs = [&](int j) {
      if constexpr (MAG) {
        if (nv2 > 0 && j <= nplanes + 1) {
          T* dst = csb + (j & 1) * CSLOT;
          if constexpr (CPH) {
            cp_async16(dst, csg + L.np);
          } else {
            cp_async16(dst, csg);
            cp_async16(dst + K::NB * 32 * VW, csg + L.np);
          }
          csg += L.sx;
        }
        cp_async_commit();
      }
    };

    // registers of intermediate plane j (ring slot j & 3): the state and pi
    auto take2 = [&](Plane& n, int j, const Plane& below) {
      const T* rf = reinterpret_cast<const T*>(smem + K::RING_OFF + (j & (K::NRING - 1)) * K::RING_PLANE) + k2;
#pragma unroll
      for (int c = 0; c < NC; ++c) ldv<T, VW>(rf + c * RCH, n.f[c]);
      ldv<T, VW>(rf + NC * RCH, n.pi);
#pragma unroll
      for (int k = 0; k < VW; ++k) n.mlo[k] = tmin(n.pi[k], below.pi[k]);
    };
    auto iteration = [&](int t, const Plane& prv, const Plane& ctr, Plane& nxt) {
      // ring plane t is complete once every step-1 warp has finished its iteration t - 1
      if (t >= 2) fetch_cs(t);   // cos / sin of the plane that the NEXT iteration rotates
      mbar_wait_parked(&adone[(t - 1) & (K::ND - 1)], (uint32_t)(((t - 1) / K::ND) & 1));
      take2(nxt, t, ctr);
      if (t >= 3) {
        const int j = t - 1, x = x0 - 2 + j;
        const T* rf = reinterpret_cast<const T*>(smem + K::RING_OFF + (j & (K::NRING - 1)) * K::RING_PLANE) + k2;
        T o[NC][VW];
        update(prv, ctr, nxt, rf, RCH, rf + NC * RCH,
               [&](T (&csv)[VW], T (&snv)[VW]) {
                 cp_async_wait<1>();
                 if constexpr (CPH) {
                   ldv<T, VW>(csb + (j & 1) * CSLOT, snv);
#pragma unroll
                   for (int k = 0; k < VW; ++k) csv[k] = cos_from_sin(snv[k]);
                 } else {
                   ldv<T, VW>(csb + (j & 1) * CSLOT, csv);
                   ldv<T, VW>(csb + (j & 1) * CSLOT + K::NB * 32 * VW, snv);
                 }
               },
               o, MAG ? nullptr : acc + HR, nv2);
        if constexpr (MAG) {   // G[n+2]
#pragma unroll
          for (int k = 0; k < VW; ++k)
            if (k < nv2) {
              acc[2] += (double)ctr.pi[k] * (double)o[0][k];
              acc[3] += (double)ctr.pi[k] * (double)o[1][k];
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
      __syncwarp();
      if (lane == 0) mbar_arrive(&bdone[t & (K::ND - 1)]);
    };

    Plane P0, P1, P2;
#pragma unroll
    for (int k = 0; k < VW; ++k) P0.pi[k] = P1.pi[k] = P2.pi[k] = (T)0;
    // step 2 has no iteration 0: arrive for it, so that slot t & 3 of bdone completes its phase (t / 4) & 1 in iteration t
    if (lane == 0) mbar_arrive(&bdone[0]);
    // unrolled by three: at iteration t prv / ctr / nxt = intermediate planes t-2, t-1, t in P[(t+1) % 3], P[(t+2) % 3], P[t % 3]
    const int tend = nplanes + 3;   // iterations 1 .. nplanes + 2
    int t = 1;
    for (; t + 3 <= tend; t += 3) {
      iteration(t, P2, P0, P1);
      iteration(t + 1, P0, P1, P2);
      iteration(t + 2, P1, P2, P0);
    }
    if (t < tend) { iteration(t, P2, P0, P1); ++t; }
    if (t < tend) { iteration(t, P0, P1, P2); ++t; }
  }

  block_reduce_finalize<K::NRED, MAG ? FIN_STEP2 : FIN_MOM2, MAG ? 0 : 3>(acc, red, a.partials, a.ctl, a.fid, a.vacf, a.vacf_stride, a.zscale, gridDim.x,
                                                                          blockIdx.x);
}

}  // namespace lpc
