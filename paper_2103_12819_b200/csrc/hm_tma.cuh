// hm_tma.cuh -- the TMA-fed LLG sweep (one Jacobi iterate r of eqs. 18-21).
//
// Same arithmetic as k_hm_sweep (hm_face_core, kernels.cuh); what differs is how operands reach
// the arithmetic.  A persistent block owns TW x BY columns and marches in z.  One producer thread
// streams the z-planes of every operand into two shared-memory rings with cp.async.bulk.tensor
// (4-D tiles of the workspace tensor, tma.cuh), each plane fetched from HBM/L2 exactly once per
// block and several planes ahead of the arithmetic:
//   H ring  : planes k-1, k, k+1 of H^n [, H^{r-1}], E, Ms with a one-cell rim  (neighbour reads)
//   M ring  : plane k of M^n [, M^{r-1}]                                        (own face only)
// 3*BY compute warps -- warp = (face orientation D, tile row), lane = x -- read their operands
// from shared memory at compile-time offsets (no address arithmetic, no divergence: D is
// warp-uniform), and write M^r, H^r with coalesced 256-byte row stores.  full/empty mbarriers
// pair the producer with the compute warps; there is no block-wide barrier in the march.
// Used when alpha, gamma and mu_r are uniform (all BASELINE configs); k_hm_sweep is the general path.
#pragma once
#include "kernels.cuh"
#include "tma.cuh"

namespace fl {

constexpr int TW = 32;      // tile width: one warp
// TMA needs the first element of a box row on a 16-byte boundary: with 8-byte elements the x
// coordinate of a box must be even.  Tiles start at even x0 (the sweep box starts at an even i), so
// a tile with a left rim starts at x0 - 2.
constexpr int HW = TW + 4;  // row width of the H / Ms tiles: cols x0-2 .. x0+33
constexpr int EW = TW + 2;  // row width of the E tiles:      cols x0   .. x0+33

// a box of cells cut into work items of TW x BY columns x kz planes
struct TileBox {
  int lo[3], hi[3];  // hi exclusive
  int ntx, nty, kz, items;
};

constexpr int up16(int n) { return (n + 15) / 16 * 16; }  // TMA destinations are 128-byte aligned

// shared-memory layout (in doubles) of one stage of each ring
template <int BY, bool FIRST, bool MS_ARR>
struct HmLayout {
  static constexpr int HROWS = BY + 2;  // H tiles: rows y0-1 .. y0+BY,   cols x0-2 .. x0+33
  static constexpr int EROWS = BY + 1;  // E tiles: rows y0   .. y0+BY,   cols x0   .. x0+33
  static constexpr int SROWS = BY + 1;  // Ms tile: rows y0-1 .. y0+BY-1, cols x0-2 .. x0+33
  static constexpr int HSET = up16(3 * HROWS * HW);
  static constexpr int ESET = up16(3 * EROWS * EW);
  static constexpr int SSET = MS_ARR ? up16(SROWS * HW) : 0;
  static constexpr int HN = 0;
  static constexpr int HP = HSET;  // absent when FIRST
  static constexpr int EE = (FIRST ? 1 : 2) * HSET;
  static constexpr int MS = EE + ESET;
  static constexpr int HSTAGE = MS + SSET;
  static constexpr unsigned HBYTES =
      8u * ((FIRST ? 1 : 2) * 3 * HROWS * HW + 3 * EROWS * EW + (MS_ARR ? SROWS * HW : 0));
  static constexpr int MSET = 9 * BY * TW;
  static constexpr int MN = 0;
  static constexpr int MP = MSET;  // absent when FIRST
  static constexpr int MSTAGE = (FIRST ? 1 : 2) * MSET;
  static constexpr unsigned MBYTES = 8u * MSTAGE;
  static constexpr int SH = FIRST ? 5 : 4;  // H ring: 3 planes live + prefetch
  static constexpr int SM = FIRST ? 4 : 3;  // M ring: 1 plane live + prefetch
  static constexpr int NCW = 3 * BY;        // compute warps
  static constexpr int NTHREADS = (NCW + 1) * 32;
  static constexpr size_t SMEM_BYTES =
      128 + 8 * (size_t)(SH * HSTAGE + SM * MSTAGE) + 8 * (2 * SH + 2 * SM) + 8 * NCW;
};

struct HMTArgs {
  HMArgs a;  // scalars, store pointers, residual words (E, Hn, Hp, Mn pointers are not used)
  TileBox tb;
  CUtensorMap mapH, mapE, mapS, mapM;  // box shapes (HW,BY+2,1,3) (EW,BY+1,1,3) (HW,BY+1,1,1) (TW,BY,1,9)
  int aE, aHn, aHp, aMn, aMp, aMs;     // array indices (4th tensor coordinate)
};

// ---- operand fetch from the rings.  hs[0..2] = H-ring stages of planes k-1, k, k+1;
// th = row*HW + lane (H, Ms tiles), te = row*EW + lane (E tiles)

template <class L, int T, int DX, int DY>
__device__ __forceinline__ double ld_h(const double *st, int set, int tb) {
  return st[set + T * L::HROWS * HW + (1 + DY) * HW + (2 + DX) + tb];
}
template <class L, int T, int DX, int DY>
__device__ __forceinline__ double ld_e(const double *st, int tb) {
  return st[L::EE + T * L::EROWS * EW + DY * EW + DX + tb];
}
template <class L, int DX, int DY>
__device__ __forceinline__ double ld_ms(const double *st, int tb) {
  return st[L::MS + (1 + DY) * HW + (2 + DX) + tb];
}

// transverse component T of H at the D-face: four-point average; same
// association as avg4 in kernels.cuh
template <class L, int D, int T>
__device__ __forceinline__ double avg4_s(const double *const *hs, int set, int tb) {
  constexpr int dx = D == 0, dy = D == 1, dz = D == 2;
  constexpr int tx = T == 0, ty = T == 1, tz = T == 2;
  const double v00 = ld_h<L, T, 0, 0>(hs[1], set, tb);
  const double v10 = ld_h<L, T, -dx, -dy>(hs[1 - dz], set, tb);
  const double v01 = ld_h<L, T, tx, ty>(hs[1 + tz], set, tb);
  const double v11 = ld_h<L, T, tx - dx, ty - dy>(hs[1 + tz - dz], set, tb);
  return 0.25 * ((v00 + v10) + (v01 + v11));
}
template <class L, int D>
__device__ __forceinline__ Vec3 h_em_s(const double *const *hs, int set, int tb) {
  Vec3 h;
  if (D == 0) {
    h.x = ld_h<L, 0, 0, 0>(hs[1], set, tb); h.y = avg4_s<L, 0, 1>(hs, set, tb); h.z = avg4_s<L, 0, 2>(hs, set, tb);
  } else if (D == 1) {
    h.x = avg4_s<L, 1, 0>(hs, set, tb); h.y = ld_h<L, 1, 0, 0>(hs[1], set, tb); h.z = avg4_s<L, 1, 2>(hs, set, tb);
  } else {
    h.x = avg4_s<L, 2, 0>(hs, set, tb); h.y = avg4_s<L, 2, 1>(hs, set, tb); h.z = ld_h<L, 2, 0, 0>(hs[1], set, tb);
  }
  return h;
}
// (curl E)_D at the D-face: forward differences; same expression as curl_e in kernels.cuh
template <class L, int D>
__device__ __forceinline__ double curl_e_s(const GridP &g, const double *const *hs, int te) {
  constexpr int d1 = (D + 1) % 3, d2 = (D + 2) % 3;
  const double a0 = ld_e<L, d2, 0, 0>(hs[1], te);
  const double a1 = ld_e<L, d2, d1 == 0, d1 == 1>(hs[1 + (d1 == 2)], te);
  const double b0 = ld_e<L, d1, 0, 0>(hs[1], te);
  const double b1 = ld_e<L, d1, d2 == 0, d2 == 1>(hs[1 + (d2 == 2)], te);
  return (a1 - a0) * g.rd[d1] - (b1 - b0) * g.rd[d2];
}

template <int D, int BY, bool FIRST, bool MS_ARR, bool ANISO>
__device__ __forceinline__ FaceOut hm_face_s(const HMArgs &a, const double *const *hs,
                                             const double *ms, int tb, int te, int tm, bool wall) {
  using L = HmLayout<BY, FIRST, MS_ARR>;
  double Msf = a.Ms_u, rMs = a.rMs_u;
  if (MS_ARR) {
    // face Ms = two-cell mean; Ms_u holds the largest Ms of the map and rMs_u
    // its reciprocal, so that the division only runs on faces with another value
    Msf = 0.5 * (ld_ms<L, 0, 0>(hs[1], tb) + ld_ms<L, -(D == 0), -(D == 1)>(hs[1 - (D == 2)], tb));
    if (Msf != a.Ms_u) rMs = Msf > 0.0 ? 1.0 / Msf : 0.0;
  }
  const Vec3 mn = {ms[L::MN + (3 * D + 0) * BY * TW + tm], ms[L::MN + (3 * D + 1) * BY * TW + tm],
                   ms[L::MN + (3 * D + 2) * BY * TW + tm]};
  Vec3 mp = mn;
  if (!FIRST)
    mp = {ms[L::MP + (3 * D + 0) * BY * TW + tm], ms[L::MP + (3 * D + 1) * BY * TW + tm],
          ms[L::MP + (3 * D + 2) * BY * TW + tm]};
  const Vec3 hn = h_em_s<L, D>(hs, L::HN, tb);
  Vec3 he = hn;
  if (!FIRST) he = h_em_s<L, D>(hs, L::HP, tb);
  const double C = curl_e_s<L, D>(a.g, hs, te);
  return hm_face_core<D, FIRST, ANISO>(a, mn, mp, hn, he, C, Msf, rMs, a.alpha_u, a.gamma_u,
                                       a.ch_uniform, wall);
}

template <int D, int BY, bool FIRST, bool MS_ARR, bool ANISO>
__device__ __forceinline__ double hm_do_face(const HMArgs &a, const double *const *hs,
                                             const double *ms, int tb, int te, int tm, int i, int j, int k,
                                             int c, bool wall, bool edge) {
  const FaceOut o = hm_face_s<D, BY, FIRST, MS_ARR, ANISO>(a, hs, ms, tb, te, tm, wall);
  store_face<D>(a, c, o);
  if (edge) store_face_images<D>(a, i, j, k, c, o);
  return o.res;
}

template <int BY, bool FIRST, bool MS_ARR, bool ANISO>
__global__ void __launch_bounds__((3 * BY + 1) * 32, 1) k_hm_tma(const __grid_constant__ HMTArgs p) {
  using L = HmLayout<BY, FIRST, MS_ARR>;
  const HMArgs &a = p.a;
  // the whole grid takes the same decision: iterate r runs iff iterate r-1 was not converged
  if (!FIRST) {
    if (__longlong_as_double((long long)a.resid[a.r - 1]) < a.tol) return;
  }
  extern __shared__ unsigned char smem_raw[];
  double *const hring =
      reinterpret_cast<double *>((reinterpret_cast<uintptr_t>(smem_raw) + 127) & ~(uintptr_t)127);
  double *const mring = hring + L::SH * L::HSTAGE;
  uint64_t *const fullH = reinterpret_cast<uint64_t *>(mring + L::SM * L::MSTAGE);
  uint64_t *const emptyH = fullH + L::SH;
  uint64_t *const fullM = emptyH + L::SH;
  uint64_t *const emptyM = fullM + L::SM;
  double *const wmax = reinterpret_cast<double *>(emptyM + L::SM);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < L::SH; ++s) { mbar_init(fullH + s, 1); mbar_init(emptyH + s, L::NCW); }
    for (int s = 0; s < L::SM; ++s) { mbar_init(fullM + s, 1); mbar_init(emptyM + s, L::NCW); }
    mbar_fence_init();
  }
  __syncthreads();

  const TileBox &B = p.tb;
  double res = 0.0;
  if (warp == L::NCW) {
    // ===== producer: one thread streams the planes of every operand, in the order the compute
    // warps consume them: H(k0-1), H(k0), then H(k+1), M(k) for k = k0 .. k1-1
    if (lane == 0) {
      tma_prefetch_desc(&p.mapH); tma_prefetch_desc(&p.mapE); tma_prefetch_desc(&p.mapM);
      if (MS_ARR) tma_prefetch_desc(&p.mapS);
      unsigned nH = 0, nM = 0;  // planes issued so far
      for (int it = blockIdx.x; it < B.items; it += gridDim.x) {
        const int tx = it % B.ntx, q = it / B.ntx, ty = q % B.nty, tz = q / B.nty;
        const int x0 = B.lo[0] + tx * TW, y0 = B.lo[1] + ty * BY;
        const int k0 = B.lo[2] + tz * B.kz, k1 = min(k0 + B.kz, B.hi[2]);
        for (int pz = k0 - 1; pz <= k1; ++pz) {
          {
            const unsigned s = nH % L::SH, u = nH / L::SH;
            if (!mbar_wait(emptyH + s, (u & 1) ^ 1, a.pipe_error, 1)) goto done;
            mbar_expect_tx(fullH + s, L::HBYTES);
            double *dst = hring + s * L::HSTAGE;
            // tensor coordinates: x = PADL + i, y = j + 1, z = k + 1 (one ghost layer)
            tma_load_4d(dst + L::HN, &p.mapH, fullH + s, PADL + x0 - 2, y0, pz + 1, p.aHn);
            if (!FIRST) tma_load_4d(dst + L::HP, &p.mapH, fullH + s, PADL + x0 - 2, y0, pz + 1, p.aHp);
            tma_load_4d(dst + L::EE, &p.mapE, fullH + s, PADL + x0, y0 + 1, pz + 1, p.aE);
            if (MS_ARR) tma_load_4d(dst + L::MS, &p.mapS, fullH + s, PADL + x0 - 2, y0, pz + 1, p.aMs);
            ++nH;
          }
          if (pz >= k0 + 1) {
            const unsigned s = nM % L::SM, u = nM / L::SM;
            if (!mbar_wait(emptyM + s, (u & 1) ^ 1, a.pipe_error, 2)) goto done;
            mbar_expect_tx(fullM + s, L::MBYTES);
            double *dst = mring + s * L::MSTAGE;
            tma_load_4d(dst + L::MN, &p.mapM, fullM + s, PADL + x0, y0 + 1, pz, p.aMn);
            if (!FIRST) tma_load_4d(dst + L::MP, &p.mapM, fullM + s, PADL + x0, y0 + 1, pz, p.aMp);
            ++nM;
          }
        }
      }
    }
  } else {
    // ===== compute warps: warp = (D, row), lane = x
    const int D = warp / BY, lj = warp % BY;
    const int tb = lj * HW + lane, te = lj * EW + lane, tm = lj * TW + lane;
    unsigned nH = 0, nM = 0;  // planes consumed so far
    for (int it = blockIdx.x; it < B.items; it += gridDim.x) {
      const int tx = it % B.ntx, q = it / B.ntx, ty = q % B.nty, tz = q / B.nty;
      const int i = B.lo[0] + tx * TW + lane, j = B.lo[1] + ty * BY + lj;
      const int k0 = B.lo[2] + tz * B.kz, k1 = min(k0 + B.kz, B.hi[2]);
      const bool valid = i < B.hi[0] && j < B.hi[1];
      const Column col = make_column(a.g, i, j);
      int c = a.g.org + i + a.g.sy * j + a.g.sz * k0;
      if (!mbar_wait(fullH + nH % L::SH, (nH / L::SH) & 1, a.pipe_error, 3)) goto done;
      if (!mbar_wait(fullH + (nH + 1) % L::SH, ((nH + 1) / L::SH) & 1, a.pipe_error, 4)) goto done;
      for (int k = k0; k < k1; ++k, c += a.g.sz) {
        if (!mbar_wait(fullH + (nH + 2) % L::SH, ((nH + 2) / L::SH) & 1, a.pipe_error, 5)) goto done;
        if (!mbar_wait(fullM + nM % L::SM, (nM / L::SM) & 1, a.pipe_error, 6)) goto done;
        const double *hs[3] = {hring + (nH % L::SH) * L::HSTAGE, hring + ((nH + 1) % L::SH) * L::HSTAGE,
                               hring + ((nH + 2) % L::SH) * L::HSTAGE};
        const double *ms = mring + (nM % L::SM) * L::MSTAGE;
        if (valid) {
          const bool edge = col.edge_ij || edge_k(a.g, k);
          double e;
          if (D == 0)
            e = hm_do_face<0, BY, FIRST, MS_ARR, ANISO>(a, hs, ms, tb, te, tm, i, j, k, c, col.wall[0], edge);
          else if (D == 1)
            e = hm_do_face<1, BY, FIRST, MS_ARR, ANISO>(a, hs, ms, tb, te, tm, i, j, k, c, col.wall[1], edge);
          else
            e = hm_do_face<2, BY, FIRST, MS_ARR, ANISO>(a, hs, ms, tb, te, tm, i, j, k, c, wall_k(a.g, k), edge);
          res = fmax(res, e);
        }
        __syncwarp();
        if (lane == 0) { mbar_arrive(emptyH + nH % L::SH); mbar_arrive(emptyM + nM % L::SM); }
        ++nH; ++nM;
      }
      // planes k1-1 and k1 of this item are not needed again
      if (lane == 0) { mbar_arrive(emptyH + nH % L::SH); mbar_arrive(emptyH + (nH + 1) % L::SH); }
      nH += 2;
    }
    // convergence word: warp shuffles, then (below) ONE atomic per block
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) res = fmax(res, __shfl_xor_sync(0xffffffffu, res, o));
    if (lane == 0) wmax[warp] = res;
  }
done:
  __syncthreads();
  if (threadIdx.x == 0) {
    double m = wmax[0];
    for (int w = 1; w < L::NCW; ++w) m = fmax(m, wmax[w]);
    if (m > 0.0) atomicMax(a.resid + a.r, (unsigned long long)__double_as_longlong(m));
  }
}

}  // namespace fl
