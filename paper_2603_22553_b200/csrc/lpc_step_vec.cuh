// lpc_step_vec.cuh -- the TMA march (step_tma_kernel, step_tma_links_kernel); included by lpc_step.cuh.
//
// A CTA owns a (TY x TZ) tile of the y-z plane and marches along x.  One x-plane per stage is streamed into shared
// memory with cp.async.bulk.tensor (TMA, halo included) behind a full/empty mbarrier ring; thread 0 issues the loads
// between planes (no producer warp: 16 warps per SM leave 128 registers per thread).  A thread owns ONE 16-BYTE GROUP
// of VW consecutive z sites -- a pair in fp64 (8 x 64 tiles), a quad in fp32 (16 x 64 tiles) -- keeps the x-1 / x / x+1
// values of its group in registers and reads the in-plane neighbours from shared memory, all with 16-byte loads.
// (fp32 first ran with pairs: the same instruction count per site for half the bytes made it issue-bound, 532 M warp
// instructions per 512^3 launch and DRAM at 57% of peak; with quads 410 M and 0.914 -> 0.715 ms.  The fp64 sweep
// measures the same with this body as with the pair-only code it replaced.)
// Per-site arithmetic is SiteUpdate::gather, so the state agrees bit for bit with the direct and persistent kernels.
#pragma once

namespace lpc {

template <typename T, int VW> struct VecN;
template <> struct VecN<double, 2> { using type = double2; };
template <> struct VecN<float, 2> { using type = float2; };
template <> struct VecN<float, 4> { using type = float4; };

template <typename T, int VW>
__device__ __forceinline__ void ldv(const T* p, T (&o)[VW]) {
  const typename VecN<T, VW>::type v = *reinterpret_cast<const typename VecN<T, VW>::type*>(p);
  o[0] = v.x; o[1] = v.y;
  if constexpr (VW == 4) { o[2] = v.z; o[3] = v.w; }
}
template <typename T, int VW>
__device__ __forceinline__ typename VecN<T, VW>::type packv(const T (&o)[VW]) {
  typename VecN<T, VW>::type v;
  v.x = o[0]; v.y = o[1];
  if constexpr (VW == 4) { v.z = o[2]; v.w = o[3]; }
  return v;
}
// the first nvalid of VW consecutive sites
template <typename T, int VW>
__device__ __forceinline__ void store_vec(T* __restrict__ p, typename VecN<T, VW>::type v, int nvalid) {
  if (nvalid == VW) {
    *reinterpret_cast<typename VecN<T, VW>::type*>(p) = v;
  } else {
    T o[VW];
    o[0] = v.x; o[1] = v.y;
    if constexpr (VW == 4) { o[2] = v.z; o[3] = v.w; }
#pragma unroll
    for (int k = 0; k < VW; ++k)
      if (k < nvalid) p[k] = o[k];
  }
}
// one channel of a group that lies on a periodic face: the sites and their ghost copies (rare, out of line)
// store_peer_vec: the same group into the same channel's ghost plane of the x neighbours (slab mode with direct halo
// stores); peer_lo / peer_hi may be nullptr.
template <typename T, int VW>
__device__ __noinline__ void store_peer_vec(T* __restrict__ peer_lo, T* __restrict__ peer_hi, long long po, int nx, int x,
                                            typename VecN<T, VW>::type v, int nvalid) {
  if (peer_lo && x == 0) store_vec<T, VW>(peer_lo + po, v, nvalid);
  if (peer_hi && x == nx - 1) store_vec<T, VW>(peer_hi + po, v, nvalid);
}

template <typename T, int VW>
__device__ __noinline__ void store_face_vec(T* __restrict__ base, long long i, int nx, int ny, int nz, long long sy, long long sx,
                                            int permask, int x, int y, int z, typename VecN<T, VW>::type v, int nvalid) {
  store_vec<T, VW>(base + i, v, nvalid);
  if (permask & 4) {
    T o[VW];
    o[0] = v.x; o[1] = v.y;
    if constexpr (VW == 4) { o[2] = v.z; o[3] = v.w; }
#pragma unroll
    for (int k = 0; k < VW; ++k) {
      if (k < nvalid && z + k == 0) base[i + k + nz] = o[k];        // ghost column z = nz
      if (k < nvalid && z + k == nz - 1) base[i + k - nz] = o[k];   // ghost column z = -1
    }
  }
  if (permask & 2) {
    if (y == 0) store_vec<T, VW>(base + i + (long long)ny * sy, v, nvalid);
    if (y == ny - 1) store_vec<T, VW>(base + i - (long long)ny * sy, v, nvalid);
  }
  if (permask & 1) {
    if (x == 0) store_vec<T, VW>(base + i + (long long)nx * sx, v, nvalid);
    if (x == nx - 1) store_vec<T, VW>(base + i - (long long)nx * sx, v, nvalid);
  }
}

// FEAT bit 0 (REG): region-resolved FID inside the sweep; bit 1 (PEER): slab mode with direct halo stores; bit 2 (CPH): tm_cs
// stages the sine alone (one channel) and the cosine is rebuilt from it (lattices whose phase angles are all small).
template <typename T, int VW, int NH, int NRHO, int NMOM, int TY, int TZ, int NSTAGE, int LK, int FEAT, typename LM>
__device__ __forceinline__ void step_tma_body(const CUtensorMap& tm_f, const CUtensorMap& tm_pi, const CUtensorMap& tm_cs, const LM& lm,
                                                const StepArgs<T>& a) {
  constexpr int REG = FEAT & 1;
  constexpr bool PEER = (FEAT & 2) != 0;
  constexpr bool CPH = (FEAT & 4) != 0;
  static_assert(!CPH || NH == 2, "only a sweep that rotates reads the phase factors");
  using K = TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, LK, VW, FEAT>;
  // REG on the magnetisation sweep: G_r (2 values per site); on the moment sweep: the regional VACF (3 values per site)
  static_assert(!REG || NH == 2 || NMOM == 3, "regional sums ride on the magnetisation or on the moment sweep");
  constexpr int RNV = (NH == 2) ? 2 : 3;
  // NH = 0 without moment fields is the density channel alone: one sweep of the equilibration loop,
  // rho <- W rho with delta = max_i |rho_i(t+1) - rho_i(t)| = max_i pi_i |r'_i - r_i| in acc[0] (a maximum, not a sum)
  constexpr bool EQ = (NH == 0 && NMOM == 0);
  static_assert(!EQ || NRHO == 1, "a sweep needs channels");
  using V = typename VecN<T, VW>::type;
  constexpr int C = K::C, NRED = K::NRED, TZW = K::TZW, TYH = K::TYH, HZ = K::HZ;
  extern __shared__ __align__(128) unsigned char smem_raw[];
  unsigned char* smem = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);
  uint64_t* full = reinterpret_cast<uint64_t*>(smem + K::BAR_OFF);
  uint64_t* empty = full + NSTAGE;
  const uint32_t full_a = smem_u32(full), empty_a = full_a + NSTAGE * 8;   // the consumers' barrier addresses, converted once
  double* red = reinterpret_cast<double*>(smem + K::RED_OFF);
  double* rred = reinterpret_cast<double*>(smem + K::RSLOT_OFF);   // REG: warp partials of the regional columns

  const Layout& L = a.L;
  const int bz = blockIdx.x % a.tiles_z;
  const int by = (blockIdx.x / a.tiles_z) % a.tiles_y;
  int bx = blockIdx.x / (a.tiles_z * a.tiles_y);
  if constexpr (PEER) {
    // direct halo stores: the two x chunks at the ends of the slab go first (block order is launch order), so that their
    // planes are on their way to the neighbours' ghost planes while the interior chunks are still being swept
    const int last = a.chunks_x - 1;
    bx = (bx == 0) ? 0 : (bx == 1) ? last : bx - 1;
  }
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
  // the next sweep of the stream may move in behind this one (its CTAs start as ours leave)
  pdl_launch_dependents();

  double acc[NRED];
#pragma unroll
  for (int r = 0; r < NRED; ++r) acc[r] = 0.0;

  // ----- TMA issue (thread 0): load j brings plane x0-1+j into stage j % NSTAGE (as in step_tma_body) -----
  // what = 1: the parameters of the plane (pi or the link weights, cos / sin), which no sweep writes; 2: its state; 3: both
  int jl = 0;
  auto issue_load = [&](int what = 3) {
    const int s = jl % NSTAGE;
    if (jl >= NSTAGE) mbar_wait(&empty[s], ((jl / NSTAGE) - 1) & 1);
    unsigned char* st = smem + s * K::STAGE_BYTES;
    const bool need_kcs = (NH == 2) && (jl >= 1 && jl <= nplanes);
    if (what & 1) mbar_expect_tx(&full[s], K::TX_BYTES + (need_kcs ? K::KCS_RAW : 0));
    // padded coordinates: plane x0 - 1 + jl, rows from y0 - 1 (boxes with halo) or y0 (boxes without)
    const int px = x0 + jl + L.gh - 1, py = y0 + L.gh - 1;
    if (what & 2) tma_load_4d(st, &tm_f, &full[s], L.padz + z0 - HZ, py, px, a.c0);
    if (what == 2) {
      ++jl;
      return;
    }
    if constexpr (LK) {
      tma_load_3d(st + K::F_BYTES, &lm.pic, &full[s], L.padz + z0, py + 1, px);
      tma_load_3d(st + K::MX_OFF, &lm.mx, &full[s], L.padz + z0, py + 1, px);
      tma_load_3d(st + K::MY_OFF, &lm.my, &full[s], L.padz + z0, py, px);
      tma_load_3d(st + K::MZ_OFF, &lm.mz, &full[s], L.padz + z0 - HZ, py + 1, px);
    } else {
      tma_load_3d(st + K::F_BYTES, &tm_pi, &full[s], L.padz + z0 - HZ, py, px);
    }
    if (need_kcs) tma_load_4d(st + K::F_BYTES + K::PI_BYTES, &tm_cs, &full[s], L.padz + z0, py + 1, px, CPH ? 1 : 0);
    if (what & 2) ++jl;
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
    // the parameters of the first planes do not depend on the sweep before this one: they are on their way while it finishes
    for (jl = 0; jl < NSTAGE && jl < nloads; ++jl) issue_load(1);
    jl = 0;
  }
  // this sweep goes on once the sweep before it has completed: from here on it reads what that one wrote
  pdl_wait();
  if (threadIdx.x == 0) {
    for (int j = 0; j < NSTAGE && j < nloads; ++j) issue_load(2);
  }

  const int ty = threadIdx.x / (TZ / VW);   // row inside the tile
  const int tp = threadIdx.x % (TZ / VW);   // group inside the row
  const int y = y0 + ty, z = z0 + VW * tp;
  const int nvalid = (y < L.ny) ? max(0, min(VW, L.nz - z)) : 0;   // the first nvalid sites of the group exist
  const int ec = (ty + 1) * TZW + VW * tp + HZ;  // element offset of the group in a halo'd tile
  const int ek = ty * TZ + VW * tp;              // and in a tile without halo
  const bool edge_yz = (a.per[1] && (y == 0 || y == L.ny - 1)) || (a.per[2] && (z == 0 || z + VW >= L.nz));
  const int permask = (a.per[0] ? 1 : 0) | (a.per[1] ? 2 : 0) | (a.per[2] ? 4 : 0);
  const bool xface = a.per[0] || PEER;   // the outermost x planes have copies to write
  // planes of this chunk whose groups have copies to write (-1: none), and whether the thread's group takes the plain
  // 16-byte store on all other planes
  const int xlo = (xface && x0 == 0) ? 0 : -1, xhi = (xface && x0 + nplanes == L.nx) ? L.nx - 1 : -1;
  const bool plain = (nvalid == VW) && !edge_yz;
  T* outp = a.fout + L.idx(x0, y, z);
  // REG: the running sum of the region the thread is in; it moves to the thread's slot when the label changes
  const uint8_t* labp = REG ? a.label + ((long long)x0 * L.ny + y) * L.nz + z : nullptr;
  // running sums of the region the thread is in (registers); they move to the thread's own per-region array -- indexed at
  // run time, hence in local memory, touched only when the label changes along the thread's column -- on a change
  // the magnetisation sweep has the registers to request the labels a plane ahead; the moment sweep (at the 128-register
  // cap) reads them at the top of the plane they belong to
  constexpr bool LABEL_AHEAD = (NH == 2);
  int labn[VW];
  if constexpr (REG && LABEL_AHEAD) {
#pragma unroll
    for (int k = 0; k < VW; ++k) labn[k] = (k < nvalid) ? (int)__ldg(labp + k) : 255;
  }
  int rcur = 255;
  double racc[RNV];
  double rall[REG ? MAX_REGIONS * RNV : 1];
  if constexpr (REG) {
    for (int q = 0; q < a.n_regions * RNV; ++q) rall[q] = 0.0;
#pragma unroll
    for (int v = 0; v < RNV; ++v) racc[v] = 0.0;
  }
  const int nrcol = REG ? a.n_regions * RNV : 0;   // regional columns in use: labels beyond n_regions are in no region
  auto rflush = [&](int next) {
    if (rcur < a.n_regions) {
#pragma unroll
      for (int v = 0; v < RNV; ++v) rall[rcur * RNV + v] += racc[v];
    }
#pragma unroll
    for (int v = 0; v < RNV; ++v) racc[v] = 0.0;
    rcur = next;
  };

  // one x-plane as a thread holds it: the group's values of every channel and of pi, and mlo = the link
  // weight towards the plane below (LK: the plane's own +x link weight, i.e. the -x weight of the plane above)
  struct Plane {
    T f[C][VW];
    T pi[VW], mlo[VW];
  };
  Plane P0, P1, P2;
  int sj = 0;
  uint32_t phj = 0;
  auto take = [&](Plane& n, const Plane* below) {
    mbar_wait_a(full_a + sj * 8, phj);
    const T* sf = reinterpret_cast<const T*>(smem + sj * K::STAGE_BYTES);
    const T* sp = reinterpret_cast<const T*>(smem + sj * K::STAGE_BYTES + K::F_BYTES);
#pragma unroll
    for (int c = 0; c < C; ++c) ldv<T, VW>(sf + c * TYH * TZW + ec, n.f[c]);
    ldv<T, VW>(sp + (LK ? ek : ec), n.pi);
    if constexpr (LK) {
      ldv<T, VW>(reinterpret_cast<const T*>(smem + sj * K::STAGE_BYTES + K::MX_OFF) + ek, n.mlo);
    } else if (below) {
#pragma unroll
      for (int k = 0; k < VW; ++k) n.mlo[k] = tmin(n.pi[k], below->pi[k]);
    }
    if (++sj == NSTAGE) {
      sj = 0;
      phj ^= 1u;
    }
  };

  auto plane = [&](int x, int sc, const Plane& prv, const Plane& ctr, Plane& nxt) {
    if (threadIdx.x == 0 && jl < nloads) issue_load();
    int labs[VW];
    if constexpr (REG && LABEL_AHEAD) {
      // the labels of this plane were requested one plane ago; request the next plane's now
#pragma unroll
      for (int k = 0; k < VW; ++k) labs[k] = labn[k];
      labp += (long long)L.ny * L.nz;
      if (x + 1 < x0 + nplanes) {
#pragma unroll
        for (int k = 0; k < VW; ++k) labn[k] = (k < nvalid) ? (int)__ldg(labp + k) : 255;
      }
    } else if constexpr (REG) {
#pragma unroll
      for (int k = 0; k < VW; ++k) labs[k] = (k < nvalid) ? (int)__ldg(labp + k) : 255;
      labp += (long long)L.ny * L.nz;
    }
    take(nxt, &ctr);
    const T* sf = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES);
    const T* sk = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::F_BYTES + K::PI_BYTES);
    T csv[VW], snv[VW];
    if (NH == 2) {
      if constexpr (CPH) {
        ldv<T, VW>(sk + ek, snv);
      } else {
        ldv<T, VW>(sk + ek, csv);
        ldv<T, VW>(sk + TY * TZ + ek, snv);
      }
    }
    SiteUpdate<T, NRHO, NMOM> u[VW];
    if constexpr (LK) {
      const T* smy = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::MY_OFF) + ek;   // row y-1 of the box
      const T* smz = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::MZ_OFF) + ty * K::TZM + HZ + VW * tp;
      T mym[VW], myp[VW], mzp[VW];
      ldv<T, VW>(smy, mym);
      ldv<T, VW>(smy + TZ, myp);
      ldv<T, VW>(smz, mzp);
      const T mz0 = smz[-1];
#pragma unroll
      for (int k = 0; k < VW; ++k) {
        u[k].mxm = prv.mlo[k]; u[k].mxp = ctr.mlo[k];
        u[k].mym = mym[k]; u[k].myp = myp[k];
        u[k].mzm = k == 0 ? mz0 : mzp[k ? k - 1 : 0];
        u[k].mzp = mzp[k];
      }
    } else {
      const T* sp = reinterpret_cast<const T*>(smem + sc * K::STAGE_BYTES + K::F_BYTES);
      T pym[VW], pyp[VW];
      ldv<T, VW>(sp + ec - TZW, pym);
      ldv<T, VW>(sp + ec + TZW, pyp);
      const T pzm = sp[ec - 1], pzp = sp[ec + VW];
#pragma unroll
      for (int k = 0; k < VW; ++k) {
        u[k].mxm = ctr.mlo[k]; u[k].mxp = nxt.mlo[k];
        u[k].mym = tmin(ctr.pi[k], pym[k]); u[k].myp = tmin(ctr.pi[k], pyp[k]);
        u[k].mzp = tmin(ctr.pi[k], k == VW - 1 ? pzp : ctr.pi[k == VW - 1 ? k : k + 1]);
      }
      u[0].mzm = tmin(ctr.pi[0], pzm);
#pragma unroll
      for (int k = 1; k < VW; ++k) u[k].mzm = u[k - 1].mzp;
    }
#pragma unroll
    for (int k = 0; k < VW; ++k) {
      u[k].pc = ctr.pi[k];
      u[k].kap = kappa_of(ctr.pi[k], a.a6);   // once per site and plane, when the plane is the centre one
      u[k].sum_weights();
    }

    T o[C][VW];
#pragma unroll
    for (int c = 0; c < C; ++c) {
      const T* fcn = sf + c * TYH * TZW;
      T fym[VW], fyp[VW];
      ldv<T, VW>(fcn + ec - TZW, fym);
      ldv<T, VW>(fcn + ec + TZW, fyp);
      const T fzm = fcn[ec - 1], fzp = fcn[ec + VW];
      if (NMOM == 3 && c >= NH + NRHO) {
        const int d = c - NH - NRHO;
        double t = 0.0;
#pragma unroll
        for (int k = 0; k < VW; ++k) {
          const T dm = (d == 0) ? (u[k].mxp - u[k].mxm) : (d == 1) ? (u[k].myp - u[k].mym) : (u[k].mzp - u[k].mzm);
          const double qd = (double)ctr.f[c][k] * (double)dm;
          if (k < nvalid) t += qd;
          if constexpr (REG && NMOM == 3) {
            // regional VACF: the same product, booked under the label of the site (labels of a group are visited in
            // d-major order, so a group that straddles two regions flushes more often, never wrongly)
            if (k < nvalid) {
              if (labs[k] != rcur) rflush(labs[k]);
              racc[d] += qd;
            }
          }
        }
        acc[2 + d] += t;
      }
#pragma unroll
      for (int k = 0; k < VW; ++k)
        o[c][k] = u[k].gather(ctr.f[c][k], prv.f[c][k], nxt.f[c][k], fym[k], fyp[k], k == 0 ? fzm : ctr.f[c][k ? k - 1 : 0],
                              k == VW - 1 ? fzp : ctr.f[c][k == VW - 1 ? k : k + 1]);
    }
    // every shared-memory read of stage sc is done: hand it back to the producer
    __syncwarp();
    if (lane == 0) mbar_arrive_a(empty_a + sc * 8);

    if constexpr (EQ) {
#pragma unroll
      for (int k = 0; k < VW; ++k)
        if (k < nvalid) acc[0] = fmax(acc[0], (double)ctr.pi[k] * fabs((double)o[0][k] - (double)ctr.f[0][k]));
    }
    if (NH == 2) {
      T gsum[2] = {(T)0, (T)0};
#pragma unroll
      for (int k = 0; k < VW; ++k) {
        const T hr = o[0][k], hi = o[1][k];
        if constexpr (CPH) csv[k] = cos_from_sin(snv[k]);
        phase_rotate(csv[k], snv[k], hr, hi, o[0][k], o[1][k]);
        if constexpr (!REG && sizeof(T) == 4) {
          // fp32: the four products of the group are added in fp32 (error <= 2.4e-7 of their magnitudes, the tolerance is
          // 1e-5 of sum |g|) and the group sum goes into the fp64 accumulator: 3 instead of 5 instructions per site
          const T w = (nvalid == VW || k < nvalid) ? ctr.pi[k] : (T)0;
          gsum[0] = fma(w, o[0][k], gsum[0]);
          gsum[1] = fma(w, o[1][k], gsum[1]);
        } else if constexpr (!REG) {
          // sites beyond the lattice (ragged tiles) count with weight 0; a full group takes the product as it is
          const double w = (nvalid == VW || k < nvalid) ? (double)ctr.pi[k] : 0.0;
          acc[0] = fma(w, (double)o[0][k], acc[0]);
          acc[1] = fma(w, (double)o[1][k], acc[1]);
        } else if (k < nvalid) {
          acc[0] += (double)ctr.pi[k] * (double)o[0][k];
          acc[1] += (double)ctr.pi[k] * (double)o[1][k];
          if constexpr (REG) {
            if (labs[k] != rcur) rflush(labs[k]);
            racc[0] += (double)ctr.pi[k] * (double)o[0][k];
            racc[1] += (double)ctr.pi[k] * (double)o[1][k];
          }
        }
      }
      if constexpr (!REG && sizeof(T) == 4) {
        acc[0] += (double)gsum[0];
        acc[1] += (double)gsum[1];
      }
    }
    if (plain && x != xlo && x != xhi) {
#pragma unroll
      for (int c = 0; c < C; ++c) *reinterpret_cast<V*>(outp + (long long)c * L.np) = packv<T, VW>(o[c]);
    } else if (nvalid > 0) {
      if (edge_yz || x == xlo || x == xhi) {
        const long long i = L.idx(x, y, z);
#pragma unroll
        for (int c = 0; c < C; ++c) {
          store_face_vec<T, VW>(a.fout + (long long)c * L.np, i, L.nx, L.ny, L.nz, L.sy, L.sx, permask, x, y, z, packv<T, VW>(o[c]), nvalid);
          if constexpr (PEER)   // the neighbours' ghost planes: same offset inside the padded plane
            store_peer_vec<T, VW>(a.peer[0] ? a.peer[0] + c * a.peer_stride[0] : nullptr, a.peer[1] ? a.peer[1] + c * a.peer_stride[1] : nullptr,
                                  i - (long long)(x + L.gh) * L.sx, L.nx, x, packv<T, VW>(o[c]), nvalid);
        }
      } else {
#pragma unroll
        for (int c = 0; c < C; ++c) store_vec<T, VW>(outp + (long long)c * L.np, packv<T, VW>(o[c]), nvalid);
      }
    }
    outp += L.sx;
  };

  take(P0, nullptr);
  __syncwarp();
  if (lane == 0) mbar_arrive_a(empty_a);   // the plane below the chunk is only needed for its centres
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

  constexpr int RNC = MAX_REGIONS * RNV;   // regional columns
  if constexpr (REG) {
    // block partial of every (region, component) column: warp sums, then thread q adds the warps of column q in order
    rflush(255);
    const int warp = threadIdx.x >> 5;
    for (int q = 0; q < nrcol; ++q) {   // only the columns of regions that exist (three regions: 6 of 16)
      const double v = warp_sum(rall[q]);
      if (lane == 0) rred[warp * RNC + q] = v;
    }
    __syncthreads();
    if (threadIdx.x < nrcol) {
      double v = 0.0;
      for (int w = 0; w < K::NTHREADS / 32; ++w) v += rred[w * RNC + threadIdx.x];
      a.rpartials[(size_t)blockIdx.x * RNC + threadIdx.x] = v;
      __threadfence();
    }
  }
  if constexpr (EQ) {
    block_max_finalize(acc[0], red, a.partials, a.ctl, gridDim.x, blockIdx.x);
    return;
  }
  const bool last = block_reduce_finalize<NRED, (NH == 2) ? FIN_STEP : FIN_MOM, NMOM>(acc, red, a.partials, a.ctl, a.fid, a.vacf,
                                                                                      a.vacf_stride, a.zscale, gridDim.x, blockIdx.x);
  if constexpr (REG) {
    if (!last) return;
    // the last CTA adds the block partials: thread t takes column t % RNC over the blocks t / RNC, t / RNC + P, ...
    __threadfence();
    constexpr int P = K::NTHREADS / RNC;
    const int col = threadIdx.x % RNC, part = threadIdx.x / RNC;
    double v = 0.0;
    if (part < P)
      for (unsigned int b = part; b < gridDim.x; b += P) v += __ldcg(&a.rpartials[(size_t)b * RNC + col]);
    __syncthreads();
    if (part < P) rred[part * RNC + col] = v;
    __syncthreads();
    if (threadIdx.x < RNC && threadIdx.x / RNV < a.n_regions) {
      double t = 0.0;
      for (int q = 0; q < P; ++q) t += rred[q * RNC + threadIdx.x];
      const int r = threadIdx.x / RNV, c = threadIdx.x % RNV;
      if (NH == 2) {
        reinterpret_cast<double*>(a.fidr + r * a.fidr_stride + a.region_sample)[c] = t;
      } else {
        // Z^r_d[index] = (a alpha / 6) sum_{i in r} q^d_i (m_{i,+d} - m_{i,-d}) / w_r   (region_moment_kernel, Q27)
        const double w = a.wr[r];
        a.vacfr[((long long)r * 3 + c) * a.vacfr_stride + a.region_sample] = (w > 0.0) ? a.zscale * t / w : 0.0;
      }
    }
  }
}

template <typename T, int NH, int NRHO, int NMOM, int TY, int TZ, int NSTAGE, int VW, int FEAT = 0>
__global__ void __launch_bounds__(TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, 0, VW, FEAT>::LB_THREADS, TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, 0, VW, FEAT>::LB_CTAS)
    step_tma_kernel(const __grid_constant__ CUtensorMap tm_f, const __grid_constant__ CUtensorMap tm_pi,
                    const __grid_constant__ CUtensorMap tm_cs, StepArgs<T> a) {
  step_tma_body<T, VW, NH, NRHO, NMOM, TY, TZ, NSTAGE, 0, FEAT>(tm_f, tm_pi, tm_cs, NoLinkMaps(), a);
}

// the same sweep with stored link weights (per-link mobility factors)
template <typename T, int NH, int NRHO, int NMOM, int TY, int TZ, int NSTAGE, int VW, int FEAT = 0>
__global__ void __launch_bounds__(TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, 1, VW, FEAT>::LB_THREADS, TmaCfg<T, NH, NRHO, NMOM, TY, TZ, NSTAGE, 1, VW, FEAT>::LB_CTAS)
    step_tma_links_kernel(const __grid_constant__ CUtensorMap tm_f, const __grid_constant__ CUtensorMap tm_cs,
                          const __grid_constant__ TmaLinkMaps lm, StepArgs<T> a) {
  step_tma_body<T, VW, NH, NRHO, NMOM, TY, TZ, NSTAGE, 1, FEAT>(tm_f, tm_f, tm_cs, lm, a);
}

}  // namespace lpc
