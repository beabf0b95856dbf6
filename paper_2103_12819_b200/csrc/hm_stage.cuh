// hm_stage.cuh -- the staged LLG sweep (one Jacobi iterate r of eqs. 18-21).
//
// Same arithmetic as k_hm_sweep (hm_face_core, kernels.cuh); what differs is how operands reach
// it.  A persistent block owns a tile of SW x BY columns and marches in z; THREAD = CELL (its
// three faces), warp = tile row, lane = x.
//   * Everything a face reads from a NEIGHBOUR (H^n, H^{r-1}, E, Ms) is staged in shared memory by
//     one producer warp with cp.async.bulk.tensor (one 4-D box per array and plane), in a ring of
//     NS stages guarded by full/empty mbarriers; the compute warps read it at compile-time offsets
//     (one LDS per operand, no address arithmetic).
//   * Every array is staged with exactly the one-sided rim its stencil needs (x: cols x0..x0+32 or
//     x0-1..x0+31, y: rows y0..y0+BY or y0-1..y0+BY-1), so a box is (SW+2) x (BY+1) doubles and
//     each component needs only TWO live planes:
//         stage p = { Hx(p), Hy(p), Hz(p+1), Ex(p+1), Ey(p+1), Ez(p), Ms(p) }
//     and plane k is computed from stages k-1 and k (PAPER.md:84, 114 for the four-point averages).
//   * What only the owning thread touches (M^n, M^{r-1} in; M^r, H^r out) goes straight between
//     global memory and registers with coalesced 256-byte rows; the producer warp prefetches the
//     M planes into L2 with cp.async.bulk.prefetch.tensor ahead of the march.
// Used when alpha, gamma and mu_r are uniform (all BASELINE configs); k_hm_sweep is the general path.
#pragma once
#include "kernels.cuh"
#include "tma.cuh"

namespace fl {

constexpr int SW = 32;         // tile width: one warp
constexpr int SROW = SW + 2;   // row width of every staged box (a 16-byte multiple)

constexpr int round16(int n) { return (n + 15) / 16 * 16; }  // TMA destinations: 128-byte aligned

// a box of cells cut into work items of SW x BY columns x kz planes
struct StBox {
  int lo[3], hi[3];  // hi exclusive
  int ntx, nty, kz, items;
};

constexpr int SBY = 16;        // tile rows: one compute warp each

// FIRST: the r = 1 sweep (no H^{r-1} set staged, M^{r-1} = M^n); otherwise an iterate r >= 2
template <bool FIRST, bool MS_ARR>
struct StLayout {
  static constexpr int BY = SBY;
  static constexpr int ROWS = BY + 1;
  static constexpr int SLOT = round16(ROWS * SROW);  // doubles per staged array
  static constexpr int HN = 0;                       // H^n x, y, z
  static constexpr int HP = 3 * SLOT;                // H^{r-1} x, y, z (absent when FIRST)
  static constexpr int EE = (FIRST ? 3 : 6) * SLOT;  // E x, y, z
  static constexpr int MS = EE + 3 * SLOT;
  static constexpr int NSLOT = (FIRST ? 6 : 9) + (MS_ARR ? 1 : 0);
  static constexpr int STAGE = NSLOT * SLOT;
  static constexpr unsigned BYTES = 8u * NSLOT * ROWS * SROW;  // bytes the TMA writes per stage
  // ring depth: two live stages + as many in flight as fit; one block per SM
  static constexpr int BUDGET = 220 * 1024;
  static constexpr int NS_FIT = BUDGET / (8 * STAGE);
  static constexpr int NS = NS_FIT > 8 ? 8 : NS_FIT;
  static constexpr int NCW = BY;  // compute warps
  static constexpr int NTHREADS = (NCW + 1) * 32;
  static constexpr size_t SMEM_BYTES = 128 + 8 * (size_t)(NS * STAGE) + 8 * (2 * NS) + 8 * NCW + 4 * NS;
  static_assert(NS >= 3, "ring too shallow");
};

// registers are granted in steps that allow 512 threads per SM at 128 and 640 at 96
constexpr int ST_MAXREG = (SBY + 1) * 32 <= 512 ? 128 : 96;

struct HMSArgs {
  HMArgs a;  // scalars, M / H pointers, residual words
  StBox tb;
  CUtensorMap mapT;  // box (SROW, BY+1, 1, 1) of the workspace tensor
  CUtensorMap mapM;  // box (SW, BY, 1, 9): L2 prefetch of an M set's plane
  int aE, aHn, aHp, aMn, aMp, aMs;  // array indices (4th tensor coordinate)
  unsigned *work;  // item counter of this launch (zero at launch; k_half_end re-arms it)
  int cond;        // 0: always run; 1: run iff iterate r-1 was not converged
};

__device__ __forceinline__ void tma_prefetch_4d(const CUtensorMap *map, int c0, int c1, int c2, int c3) {
  asm volatile("cp.async.bulk.prefetch.tensor.4d.L2.global.tile [%0, {%1, %2, %3, %4}];" ::"l"(map),
               "r"(c0), "r"(c1), "r"(c2), "r"(c3)
               : "memory");
}

// ---- operand fetch.  A = stage k-1, B = stage k of the ring; t = row*SROW + lane.
// Box origins: Hx (x0, y0-1), Hy (x0-2, y0), Hz (x0-2, y0-1), E (x0, y0), Ms (x0-2, y0-1).
// SET = L::HN or L::HP.  DZ is relative to the computed plane k.
template <class L, int SET, int DX, int DY, int DZ>
__device__ __forceinline__ double s_hx(const double *A, const double *B, int t) {
  static_assert(DX >= 0 && DX <= 1 && DY >= -1 && DY <= 0 && DZ >= -1 && DZ <= 0, "Hx rim");
  return (DZ < 0 ? A : B)[SET + 0 * L::SLOT + (DY + 1) * SROW + DX + t];
}
template <class L, int SET, int DX, int DY, int DZ>
__device__ __forceinline__ double s_hy(const double *A, const double *B, int t) {
  static_assert(DX >= -1 && DX <= 0 && DY >= 0 && DY <= 1 && DZ >= -1 && DZ <= 0, "Hy rim");
  return (DZ < 0 ? A : B)[SET + 1 * L::SLOT + DY * SROW + (DX + 2) + t];
}
template <class L, int SET, int DX, int DY, int DZ>
__device__ __forceinline__ double s_hz(const double *A, const double *B, int t) {
  static_assert(DX >= -1 && DX <= 0 && DY >= -1 && DY <= 0 && DZ >= 0 && DZ <= 1, "Hz rim");
  return (DZ == 0 ? A : B)[SET + 2 * L::SLOT + (DY + 1) * SROW + (DX + 2) + t];
}
template <class L, int DY, int DZ>
__device__ __forceinline__ double s_ex(const double *A, const double *B, int t) {
  static_assert(DY >= 0 && DY <= 1 && DZ >= 0 && DZ <= 1, "Ex rim");
  return (DZ == 0 ? A : B)[L::EE + 0 * L::SLOT + DY * SROW + t];
}
template <class L, int DX, int DZ>
__device__ __forceinline__ double s_ey(const double *A, const double *B, int t) {
  static_assert(DX >= 0 && DX <= 1 && DZ >= 0 && DZ <= 1, "Ey rim");
  return (DZ == 0 ? A : B)[L::EE + 1 * L::SLOT + DX + t];
}
template <class L, int DX, int DY>
__device__ __forceinline__ double s_ez(const double *B, int t) {
  static_assert(DX >= 0 && DX <= 1 && DY >= 0 && DY <= 1, "Ez rim");
  return B[L::EE + 2 * L::SLOT + DY * SROW + DX + t];
}
template <class L, int DX, int DY, int DZ>
__device__ __forceinline__ double s_ms(const double *A, const double *B, int t) {
  static_assert(DX >= -1 && DX <= 0 && DY >= -1 && DY <= 0 && DZ >= -1 && DZ <= 0, "Ms rim");
  return (DZ < 0 ? A : B)[L::MS + (DY + 1) * SROW + (DX + 2) + t];
}

__device__ __forceinline__ double avg4v(double v00, double v10, double v01, double v11) {
  return 0.25 * ((v00 + v10) + (v01 + v11));  // same association as avg4 in kernels.cuh
}

// H_EM at the D-face from the staged H set SET: own normal component + two four-point averages
// (PAPER.md:84, 114); operand order v00 = c, v10 = c - s_D, v01 = c + s_T, v11 = c - s_D + s_T
template <class L, int SET, int D>
__device__ __forceinline__ Vec3 s_hem(const double *A, const double *B, int t) {
  Vec3 h;
  if (D == 0) {
    h.x = s_hx<L, SET, 0, 0, 0>(A, B, t);
    h.y = avg4v(s_hy<L, SET, 0, 0, 0>(A, B, t), s_hy<L, SET, -1, 0, 0>(A, B, t),
                s_hy<L, SET, 0, 1, 0>(A, B, t), s_hy<L, SET, -1, 1, 0>(A, B, t));
    h.z = avg4v(s_hz<L, SET, 0, 0, 0>(A, B, t), s_hz<L, SET, -1, 0, 0>(A, B, t),
                s_hz<L, SET, 0, 0, 1>(A, B, t), s_hz<L, SET, -1, 0, 1>(A, B, t));
  } else if (D == 1) {
    h.x = avg4v(s_hx<L, SET, 0, 0, 0>(A, B, t), s_hx<L, SET, 0, -1, 0>(A, B, t),
                s_hx<L, SET, 1, 0, 0>(A, B, t), s_hx<L, SET, 1, -1, 0>(A, B, t));
    h.y = s_hy<L, SET, 0, 0, 0>(A, B, t);
    h.z = avg4v(s_hz<L, SET, 0, 0, 0>(A, B, t), s_hz<L, SET, 0, -1, 0>(A, B, t),
                s_hz<L, SET, 0, 0, 1>(A, B, t), s_hz<L, SET, 0, -1, 1>(A, B, t));
  } else {
    h.x = avg4v(s_hx<L, SET, 0, 0, 0>(A, B, t), s_hx<L, SET, 0, 0, -1>(A, B, t),
                s_hx<L, SET, 1, 0, 0>(A, B, t), s_hx<L, SET, 1, 0, -1>(A, B, t));
    h.y = avg4v(s_hy<L, SET, 0, 0, 0>(A, B, t), s_hy<L, SET, 0, 0, -1>(A, B, t),
                s_hy<L, SET, 0, 1, 0>(A, B, t), s_hy<L, SET, 0, 1, -1>(A, B, t));
    h.z = s_hz<L, SET, 0, 0, 0>(A, B, t);
  }
  return h;
}

// (curl E)_D at the D-face: forward differences; same expression as curl_e in kernels.cuh
template <class L, int D>
__device__ __forceinline__ double s_curl(const GridP &g, const double *A, const double *B, int t) {
  if (D == 0)
    return (s_ez<L, 0, 1>(B, t) - s_ez<L, 0, 0>(B, t)) * g.rd[1] -
           (s_ey<L, 0, 1>(A, B, t) - s_ey<L, 0, 0>(A, B, t)) * g.rd[2];
  if (D == 1)
    return (s_ex<L, 0, 1>(A, B, t) - s_ex<L, 0, 0>(A, B, t)) * g.rd[2] -
           (s_ez<L, 1, 0>(B, t) - s_ez<L, 0, 0>(B, t)) * g.rd[0];
  return (s_ey<L, 1, 0>(A, B, t) - s_ey<L, 0, 0>(A, B, t)) * g.rd[0] -
         (s_ex<L, 1, 0>(A, B, t) - s_ex<L, 0, 0>(A, B, t)) * g.rd[1];
}

// One Jacobi iterate on the D-face of this thread's cell, neighbour operands from the ring
template <class L, int D, bool FIRST, bool MS_ARR, bool ANISO>
__device__ __forceinline__ FaceOut s_face(const HMArgs &a, const double *A, const double *B, int t,
                                          const Vec3 &mn, const Vec3 &mp, bool wall) {
  double Msf = a.Ms_u, rMs = a.rMs_u;
  if (MS_ARR) {
    // face Ms = two-cell mean; Ms_u holds the largest Ms of the map and rMs_u
    // its reciprocal, so that the division only runs on faces with another value
    Msf = 0.5 * (s_ms<L, 0, 0, 0>(A, B, t) + s_ms<L, -(D == 0), -(D == 1), -(D == 2)>(A, B, t));
    if (Msf != a.Ms_u) rMs = Msf > 0.0 ? 1.0 / Msf : 0.0;
  }
  const Vec3 hn = s_hem<L, L::HN, D>(A, B, t);
  Vec3 he = hn;
  if (!FIRST) he = s_hem<L, L::HP, D>(A, B, t);
  const double C = s_curl<L, D>(a.g, A, B, t);
  return hm_face_core<D, FIRST, ANISO>(a, mn, mp, hn, he, C, Msf, rMs, a.alpha_u, a.cf_u,
                                       a.ch_uniform, wall);
}

template <int D, bool LOAD_MP>
__device__ __forceinline__ void s_load_m(const HMArgs &a, int c, Vec3 &mn, Vec3 &mp) {
  mn = {__ldcs(a.Mn[3 * D + 0] + c), __ldcs(a.Mn[3 * D + 1] + c), __ldcs(a.Mn[3 * D + 2] + c)};
  if (LOAD_MP)
    mp = {__ldcs(a.Mr[3 * D + 0] + c), __ldcs(a.Mr[3 * D + 1] + c), __ldcs(a.Mr[3 * D + 2] + c)};
}

// the TMA loads of stage pz of the tile at (x0, y0): tensor coordinates x = PADL + i, y = j + 1,
// z = k + 1 (one ghost layer)
template <class L, bool FIRST, bool MS_ARR>
__device__ __forceinline__ void s_issue_stage(const HMSArgs &p, double *dst, uint64_t *bar, int x0,
                                              int y0, int pz) {
  const int xa = PADL + x0, xb = PADL + x0 - 2, ya = y0 + 1, yb = y0, z = pz + 1;
#define S_BOX(slot, cx, cy, cz, arr) tma_load_4d(dst + (slot), &p.mapT, bar, cx, cy, cz, arr)
  S_BOX(L::HN + 0 * L::SLOT, xa, yb, z, p.aHn + 0);
  S_BOX(L::HN + 1 * L::SLOT, xb, ya, z, p.aHn + 1);
  S_BOX(L::HN + 2 * L::SLOT, xb, yb, z + 1, p.aHn + 2);
  if (!FIRST) {
    S_BOX(L::HP + 0 * L::SLOT, xa, yb, z, p.aHp + 0);
    S_BOX(L::HP + 1 * L::SLOT, xb, ya, z, p.aHp + 1);
    S_BOX(L::HP + 2 * L::SLOT, xb, yb, z + 1, p.aHp + 2);
  }
  S_BOX(L::EE + 0 * L::SLOT, xa, ya, z + 1, p.aE + 0);
  S_BOX(L::EE + 1 * L::SLOT, xa, ya, z + 1, p.aE + 1);
  S_BOX(L::EE + 2 * L::SLOT, xa, ya, z, p.aE + 2);
  if (MS_ARR) S_BOX(L::MS, xb, yb, z, p.aMs);
#undef S_BOX
}

struct StItem {
  int x0, y0, k0, k1;
};
__device__ __forceinline__ StItem st_decode_by(const StBox &T, int it, int by) {
  const int tx = it % T.ntx, q = it / T.ntx, ty = q % T.nty, tz = q / T.nty;
  StItem w;
  w.x0 = T.lo[0] + tx * SW;
  w.y0 = T.lo[1] + ty * by;
  w.k0 = T.lo[2] + tz * T.kz;
  w.k1 = min(w.k0 + T.kz, T.hi[2]);
  return w;
}
__device__ __forceinline__ StItem st_decode(const StBox &T, int it) {
  const int tx = it % T.ntx, q = it / T.ntx, ty = q % T.nty, tz = q / T.nty;
  StItem w;
  w.x0 = T.lo[0] + tx * SW;
  w.y0 = T.lo[1] + ty * SBY;
  w.k0 = T.lo[2] + tz * T.kz;
  w.k1 = min(w.k0 + T.kz, T.hi[2]);
  return w;
}

// Work items are handed out dynamically (one atomic per item on p.work): SMs do not all stream at
// the same rate, and a static split leaves the fast ones idle at the end.  The producer publishes
// the item of every stage in meta[slot] before arming the stage's barrier; item < 0 ends the march.
template <bool FIRST, bool MS_ARR, bool ANISO>
__global__ void __maxnreg__(ST_MAXREG)
k_hm_stage(const __grid_constant__ HMSArgs p) {
  constexpr bool LOAD_MP = !FIRST;              // M^{r-1} read from memory
  using L = StLayout<FIRST, MS_ARR>;
  const HMArgs &a = p.a;
  // the whole grid takes the same decision (the stopping test is global)
  if (p.cond == 1 && __longlong_as_double((long long)a.resid[a.r - 1]) < a.tol) return;
  // dynamic shared memory starts on a 1 KB boundary of the CTA's window (no static shared memory in
  // this kernel); keeping the pointer a plain offset of the __shared__ array lets the compiler
  // address the ring with LDS instead of generic loads
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double *const ring = reinterpret_cast<double *>(smem_raw);
  uint64_t *const full = reinterpret_cast<uint64_t *>(ring + L::NS * L::STAGE);
  uint64_t *const empty = full + L::NS;
  double *const wmax = reinterpret_cast<double *>(empty + L::NS);
  int *const meta = reinterpret_cast<int *>(wmax + L::NCW);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < L::NS; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, L::NCW); }
    mbar_fence_init();
  }
  if (threadIdx.x < L::NCW) wmax[threadIdx.x] = 0.0;   // a warp that leaves on a pipeline error adds nothing
  __syncthreads();

  const StBox &T = p.tb;
  double res = 0.0;
  if (warp == L::NCW) {
    // ===== producer: one thread streams stage pz = k0-1 .. k1-1 of every item it draws
    if (lane == 0) {
      tma_prefetch_desc(&p.mapT);
      tma_prefetch_desc(&p.mapM);
      unsigned n = 0;  // stages issued so far
      for (;;) {
        const int it = (int)atomicAdd(p.work, 1u);
        const bool end = it >= T.items;
        const StItem w = st_decode(T, end ? 0 : it);
        if (!end) {  // the first M plane of a fresh column, towards L2
          tma_prefetch_4d(&p.mapM, PADL + w.x0, w.y0 + 1, w.k0 + 1, p.aMn);
          if (LOAD_MP) tma_prefetch_4d(&p.mapM, PADL + w.x0, w.y0 + 1, w.k0 + 1, p.aMp);
        }
        for (int pz = w.k0 - 1; pz < (end ? w.k0 : w.k1); ++pz, ++n) {
          const unsigned s = n % L::NS, u = n / L::NS;
          if (!mbar_wait(empty + s, (u & 1) ^ 1, a.pipe_error, 1)) goto done;
          meta[s] = end ? -1 : it;
          if (end) {
            mbar_arrive(full + s);
            break;
          }
          mbar_expect_tx(full + s, L::BYTES);
          s_issue_stage<L, FIRST, MS_ARR>(p, ring + s * L::STAGE, full + s, w.x0, w.y0, pz);
          // towards L2: the M planes the compute warps will load while they work on plane pz - 1
          // (about one plane time ahead: long enough to cover HBM latency, short enough to survive in L2)
          if (pz >= w.k0) {
            tma_prefetch_4d(&p.mapM, PADL + w.x0, w.y0 + 1, pz + 1, p.aMn);
            if (LOAD_MP) tma_prefetch_4d(&p.mapM, PADL + w.x0, w.y0 + 1, pz + 1, p.aMp);
          }
        }
        if (end) break;
      }
    }
  } else {
    // ===== compute warps: warp = tile row, lane = x, thread = cell
    const int t = warp * SROW + lane;
    unsigned n = 0;  // stages released so far
    for (;;) {
      if (!mbar_wait(full + n % L::NS, (n / L::NS) & 1, a.pipe_error, 2)) goto done;
      const int it = *(volatile int *)(meta + n % L::NS);
      if (it < 0) break;
      const StItem w = st_decode(T, it);
      const int i = w.x0 + lane, j = w.y0 + warp;
      const bool valid = i < T.hi[0] && j < T.hi[1];
      const Column col = make_column(a.g, i, j);
      int c = a.g.org + i + a.g.sy * j + a.g.sz * w.k0;
      // own-face operands (M^n, M^{r-1}) rotate through registers one plane ahead: the loads of
      // plane k+1 are issued as soon as the face of plane k has consumed its registers
      Vec3 mn0{}, mp0{}, mn1{}, mp1{}, mn2{}, mp2{};
      if (valid) {
        s_load_m<0, LOAD_MP>(a, c, mn0, mp0);
        s_load_m<1, LOAD_MP>(a, c, mn1, mp1);
        s_load_m<2, LOAD_MP>(a, c, mn2, mp2);
      }
      for (int k = w.k0; k < w.k1; ++k, c += a.g.sz, ++n) {
        const double *A = ring + (n % L::NS) * L::STAGE;
        const double *B = ring + ((n + 1) % L::NS) * L::STAGE;
        if (!mbar_wait(full + (n + 1) % L::NS, ((n + 1) / L::NS) & 1, a.pipe_error, 3)) goto done;
        if (valid) {
          const bool edge = col.edge_ij || edge_k(a.g, k);
          const bool more = k + 1 < w.k1;
          {
            const FaceOut o = s_face<L, 0, FIRST, MS_ARR, ANISO>(a, A, B, t, mn0, LOAD_MP ? mp0 : mn0, col.wall[0]);
            if (more) s_load_m<0, LOAD_MP>(a, c + a.g.sz, mn0, mp0);
            store_face<0>(a, c, o);
            if (edge) store_face_images<0>(a, i, j, k, c, o);
            res = fmax(res, o.res);
          }
          {
            const FaceOut o = s_face<L, 1, FIRST, MS_ARR, ANISO>(a, A, B, t, mn1, LOAD_MP ? mp1 : mn1, col.wall[1]);
            if (more) s_load_m<1, LOAD_MP>(a, c + a.g.sz, mn1, mp1);
            store_face<1>(a, c, o);
            if (edge) store_face_images<1>(a, i, j, k, c, o);
            res = fmax(res, o.res);
          }
          {
            const FaceOut o = s_face<L, 2, FIRST, MS_ARR, ANISO>(a, A, B, t, mn2, LOAD_MP ? mp2 : mn2, wall_k(a.g, k));
            if (more) s_load_m<2, LOAD_MP>(a, c + a.g.sz, mn2, mp2);
            store_face<2>(a, c, o);
            if (edge) store_face_images<2>(a, i, j, k, c, o);
            res = fmax(res, o.res);
          }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(empty + n % L::NS);  // stage k-1 is done with
      }
      if (lane == 0) mbar_arrive(empty + n % L::NS);  // stage k1-1: the next item starts afresh
      ++n;
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
