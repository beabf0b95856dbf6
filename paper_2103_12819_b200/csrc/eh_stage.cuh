// eh_stage.cuh -- the staged Maxwell sweeps: eq. 11 and, FUSED with it on the
// faces no magnetic face reads, the H update that follows it (eq. 21 with M = 0).
//
// Same arithmetic as k_e_update / k_h_update (kernels.cuh: e_edge_val, h_face_val); what differs is
// how operands reach it and how often memory is touched.  A persistent block owns a tile of columns
// and marches in z; THREAD = CELL, warp = tile row, lane = x.  One producer lane stages, per plane,
// a (SW+4) x (rows+2) box of every operand array (H^{n+1/2} x3, E^n x3, eps_r, sigma) in shared
// memory with cp.async.bulk.tensor, in a ring of NS stages under full / empty mbarriers; plane q is
// computed from stages q-1 and q.
//
//   k_eh_stage  E only, tile 32 x 16: the LLG sweep box, whose H lives at integer time.
//   k_eh_fused  E + H, tile 32 x 15 (merged H half-steps, options.merge_h): outside the sweep box
//     the H update that follows the E update -- second half-step of this step and first of the
//     next, both with curl E^{n+1} -- reads nothing but E^{n+1} around the face and
//     its own H.  The block keeps the E^{n+1} plane it just computed in shared memory (with the
//     one-cell rim on the high side) and takes H^{n+1/2} -> H^{n+3/2} in the same pass: per cell
//     and step E 3 + H 3 read, E 3 + H 3 written = 12 words instead of 9 + 9 (27 with two
//     half-steps).  All inputs are sets nobody writes during the pass (every update is out of
//     place), so tiles and planes can be visited in any order.
#pragma once
#include "hm_stage.cuh"

namespace fl {

constexpr int EW = SW + 4;                   // staged row: x0-2 .. x0+33 (16-byte multiples)
constexpr int EROWS = SBY + 2;               // rows y0-1 .. y0+16
constexpr int ESLOT = round16(EROWS * EW);   // doubles per staged array

template <bool EPS_ARR, bool SIG_ARR>
struct EhLayout {   // k_eh_stage: one stage of the ring, the ring, the block
  static constexpr int SLOT = ESLOT;
  static constexpr int HH = 0;                          // H x, y, z
  static constexpr int EE = 3 * ESLOT;                  // E^n x, y, z
  static constexpr int EP = 6 * ESLOT;                  // eps_r
  static constexpr int SG = (6 + (EPS_ARR ? 1 : 0)) * ESLOT;   // sigma
  static constexpr int NARR = 6 + (EPS_ARR ? 1 : 0) + (SIG_ARR ? 1 : 0);
  static constexpr int STAGE = NARR * ESLOT;
  static constexpr unsigned BYTES = 8u * NARR * EROWS * EW;    // bytes the TMA writes per stage
  static constexpr int NS_FIT = 220 * 1024 / (8 * STAGE);
  static constexpr int NS = NS_FIT > 6 ? 6 : NS_FIT;
  static constexpr int NCW = SBY;                       // compute warps
  static constexpr int NTHREADS = (NCW + 1) * 32;
  static constexpr size_t SMEM_BYTES = 128 + 8 * (size_t)(NS * STAGE) + 8 * (2 * NS) + 4 * NS;
  static_assert(NS >= 3, "ring too shallow");
};

struct EHArgs {
  GridP g;
  StBox tb;            // the cells this launch updates, cut into work items
  CUtensorMap map;     // box (EW, EROWS, 1, 1) of the workspace tensor
  int aE, aH, aEps, aSig;   // array indices (4th tensor coordinate) of E^n_x, H_x, eps_r, sigma
  double *Eo[3];       // E^{n+1}: the other E set
  double *Ho[3];       // FUSE: H^{n+3/2}, the other half-time H set
  double eps_u, sigma_u;    // uniform values (eps_u is eps0 * eps_r)
  double rdt;               // 1 / dt
  ECoef k_u;                // e_coef(eps_u, sigma_u, rdt): the coefficients when both maps are uniform
  double chm;          // FUSE: cmul * dt / (2 mu) = dt / mu (uniform mu)
  SourcesP src;
  const DevState *st;
  unsigned *work;      // item counter of this launch (zero at launch; re-armed by k_half_end, or by the
                       // next step's launch when the bookkeeping is folded in, see `book`)
  int *pipe_error;
  // A Maxwell-only step whose E phase is ONE fused launch needs no other kernel: the launch also
  // closes the two H half-steps in the run state (what k_half_end does) and re-arms the item
  // counters of the OTHER step parity (nobody draws from them during this step).
  DevState *book;      // nullptr: k_half_end does the bookkeeping
  unsigned *work_other;  // [8] counters of the other step parity
  int *r_hist;
};

// the TMA loads of stage pz of the tile at (x0, y0): every array with the same box origin
template <class L, bool EPS_ARR, bool SIG_ARR>
__device__ __forceinline__ void eh_issue_stage(const EHArgs &p, double *dst, uint64_t *bar, int x0, int y0, int pz) {
  const int x = PADL + x0 - 2, y = y0, z = pz + 1;   // tensor coordinates: one ghost layer in y, z
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    tma_load_4d(dst + L::HH + d * L::SLOT, &p.map, bar, x, y, z, p.aH + d);
    tma_load_4d(dst + L::EE + d * L::SLOT, &p.map, bar, x, y, z, p.aE + d);
  }
  if (EPS_ARR) tma_load_4d(dst + L::EP, &p.map, bar, x, y, z, p.aEps);
  if (SIG_ARR) tma_load_4d(dst + L::SG, &p.map, bar, x, y, z, p.aSig);
}

// soft sources on the D-edge of cell (i,j,k).  The fused sweep recomputes
// E^{n+1} on the high-side rim of a tile (row y0 + FBY, column x0 + SW, plane k1, the cells at T.hi of
// a ragged tile); at the end of a PERIODIC axis that rim is index n, the image of index 0
// (PAPER.md:185), and carries the current of the source at index 0
template <int D>
__device__ __forceinline__ double eh_source(const EHArgs &a, int i, int j, int k) {
  if (a.g.per[0] && i == a.g.n[0]) i = 0;
  if (a.g.per[1] && j == a.g.n[1]) j = 0;
  if (a.g.per[2] && k == a.g.n[2]) k = 0;
  double J = 0.0;
  for (int s = 0; s < a.src.count; ++s) {
    const SourceP &S = a.src.s[s];
    if (S.kind != 0 || S.comp != D) continue;
    if (i < S.lo[0] || i >= S.hi[0] || j < S.lo[1] || j >= S.hi[1] || k < S.lo[2] || k >= S.hi[2])
      continue;
    double pr = 1.0;
    if (S.profile) {
      const long long bx = S.hi[0] - S.lo[0], by = S.hi[1] - S.lo[1];
      pr = __ldg(S.profile + (i - S.lo[0]) + bx * ((j - S.lo[1]) + by * (long long)(k - S.lo[2])));
    }
    J += a.st->src_amp[s] * pr;
  }
  return J;
}

// E^{n+1} on the D-edge at staged position t (A = stage q-1, B = stage q), grid position (i,j,k):
// the operands of e_edge_val in the order k_e_update fetches them
// `wall`: the edge is tangential to a PEC wall and stays 0: the lower walls, and
// index n of a PEC axis (the upper wall, which the rim of a tile at the end of the grid reaches)
template <class L, int D, bool EPS_ARR, bool SIG_ARR, bool HAS_SRC>
__device__ __forceinline__ double eh_edge(const EHArgs &a, const double *A, const double *B, int t, int i,
                                          int j, int k, bool wall) {
  constexpr int HX = L::HH, HY = L::HH + L::SLOT, HZ = L::HH + 2 * L::SLOT;
  // offsets of the two transverse neighbours: s1 = stride of axis D+1, s2 = stride of axis D+2
  double h2, h2m, h1, h1m, e0, m00 = 0, m10 = 0, m01 = 0, m11 = 0, g00 = 0, g10 = 0, g01 = 0, g11 = 0;
  if (D == 0) {         // s1 = y, s2 = z
    h2 = B[HZ + t]; h2m = B[HZ + t - EW]; h1 = B[HY + t]; h1m = A[HY + t];
    e0 = B[L::EE + t];
    if (EPS_ARR) { m00 = B[L::EP + t]; m10 = B[L::EP + t - EW]; m01 = A[L::EP + t]; m11 = A[L::EP + t - EW]; }
    if (SIG_ARR) { g00 = B[L::SG + t]; g10 = B[L::SG + t - EW]; g01 = A[L::SG + t]; g11 = A[L::SG + t - EW]; }
  } else if (D == 1) {  // s1 = z, s2 = x
    h2 = B[HX + t]; h2m = A[HX + t]; h1 = B[HZ + t]; h1m = B[HZ + t - 1];
    e0 = B[L::EE + L::SLOT + t];
    if (EPS_ARR) { m00 = B[L::EP + t]; m10 = A[L::EP + t]; m01 = B[L::EP + t - 1]; m11 = A[L::EP + t - 1]; }
    if (SIG_ARR) { g00 = B[L::SG + t]; g10 = A[L::SG + t]; g01 = B[L::SG + t - 1]; g11 = A[L::SG + t - 1]; }
  } else {              // s1 = x, s2 = y
    h2 = B[HY + t]; h2m = B[HY + t - 1]; h1 = B[HX + t]; h1m = B[HX + t - EW];
    e0 = B[L::EE + 2 * L::SLOT + t];
    if (EPS_ARR) { m00 = B[L::EP + t]; m10 = B[L::EP + t - 1]; m01 = B[L::EP + t - EW]; m11 = B[L::EP + t - EW - 1]; }
    if (SIG_ARR) { g00 = B[L::SG + t]; g10 = B[L::SG + t - 1]; g01 = B[L::SG + t - EW]; g11 = B[L::SG + t - EW - 1]; }
  }
  double eps = a.eps_u, sig = a.sigma_u;
  if (EPS_ARR) eps = kEps0 * (0.25 * ((m00 + m10) + (m01 + m11)));   // four-cell means
  if (SIG_ARR) sig = 0.25 * ((g00 + g10) + (g01 + g11));
  double J = 0.0;
  if (HAS_SRC) J = eh_source<D>(a, i, j, k);
  ECoef kc = a.k_u;
  if (EPS_ARR || SIG_ARR) kc = e_coef(eps, sig, a.rdt);
  return e_edge_val<D>(a.g, kc, J, e0, h2, h2m, h1, h1m, wall);
}

// index idx lies on a PEC wall of axis d (lower wall at 0, upper wall at n)
__device__ __forceinline__ bool on_wall(const GridP &g, int d, int idx) {
  return (g.wall[d] && idx == 0) || (g.wallhi[d] && idx == g.n[d]);
}

// ------------------------------------------------------------------ E only (the LLG sweep box)
template <bool EPS_ARR, bool SIG_ARR, bool HAS_SRC>
__global__ void __launch_bounds__(EhLayout<EPS_ARR, SIG_ARR>::NTHREADS, 1)
k_eh_stage(const __grid_constant__ EHArgs p) {
  using L = EhLayout<EPS_ARR, SIG_ARR>;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double *const ring = reinterpret_cast<double *>(smem_raw);
  uint64_t *const full = reinterpret_cast<uint64_t *>(ring + L::NS * L::STAGE);
  uint64_t *const empty = full + L::NS;
  int *const meta = reinterpret_cast<int *>(empty + L::NS);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < L::NS; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, L::NCW); }
    mbar_fence_init();
  }
  __syncthreads();

  const StBox &T = p.tb;
  const GridP &g = p.g;
  auto next = [](unsigned &st, unsigned &ph) { if (++st == (unsigned)L::NS) { st = 0; ph ^= 1u; } };
  if (warp == L::NCW) {
    // ===== producer: stages k0-1 .. k1-1 of every item it draws
    if (lane == 0) {
      tma_prefetch_desc(&p.map);
      unsigned s = 0, ph = 1;   // ring position and the parity its empty barrier is waited on
      for (;;) {
        const int it = (int)atomicAdd(p.work, 1u);
        const bool end = it >= T.items;
        const StItem w = st_decode(T, end ? 0 : it);
        // (an L2 tensor prefetch running 3-10 planes ahead of the ring was measured: it costs 3-25 %)
        for (int pz = w.k0 - 1; pz < (end ? w.k0 : w.k1); ++pz) {
          if (!mbar_wait(empty + s, ph, p.pipe_error, 4)) return;
          meta[s] = end ? -1 : it;
          if (end) {
            mbar_arrive(full + s);
            break;
          }
          mbar_expect_tx(full + s, L::BYTES);
          eh_issue_stage<L, EPS_ARR, SIG_ARR>(p, ring + s * L::STAGE, full + s, w.x0, w.y0, pz);
          next(s, ph);
        }
        if (end) break;
      }
    }
    return;
  }
  // ===== compute warps: warp = tile row, lane = x, thread = cell
  const int t0 = (warp + 1) * EW + lane + 2;   // own staged position
  double *const eo0 = p.Eo[0], *const eo1 = p.Eo[1], *const eo2 = p.Eo[2];
  unsigned sa = 0, pa = 0;   // ring position of stage q-1 and its phase (advanced by hand: no division in the march)
  for (;;) {
    if (!mbar_wait(full + sa, pa, p.pipe_error, 5)) return;
    const int it = *(volatile int *)(meta + sa);
    if (it < 0) break;
    const StItem w = st_decode(T, it);
    const int i = w.x0 + lane, j = w.y0 + warp;
    const bool valid = i < T.hi[0] && j < T.hi[1];
    const Column col = make_column(g, i, j);
    const bool wi = on_wall(g, 0, i), wj = on_wall(g, 1, j);   // walls of this thread's edges, per column
    int c = g.org + i + g.sy * j + g.sz * w.k0;
    for (int q = w.k0; q < w.k1; ++q) {
      unsigned sb = sa, pb = pa;
      next(sb, pb);
      const double *A = ring + sa * L::STAGE;
      const double *B = ring + sb * L::STAGE;
      if (!mbar_wait(full + sb, pb, p.pipe_error, 6)) return;
      const bool wk = on_wall(g, 2, q);
      const double ex = eh_edge<L, 0, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, t0, i, j, q, wj || wk);
      const double ey = eh_edge<L, 1, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, t0, i, j, q, wk || wi);
      const double ez = eh_edge<L, 2, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, t0, i, j, q, wi || wj);
      if (valid) {
        eo0[c] = ex;
        eo1[c] = ey;
        eo2[c] = ez;
        if (col.edge_ij || edge_k(g, q)) {
          store_images_inl<exp_of_e<0>()>(eo0, g, i, j, q, c, ex);
          store_images_inl<exp_of_e<1>()>(eo1, g, i, j, q, c, ey);
          store_images_inl<exp_of_e<2>()>(eo2, g, i, j, q, c, ez);
        }
      }
      c += g.sz;
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + sa);  // stage q-1 is done with
      sa = sb; pa = pb;
    }
    if (lane == 0) mbar_arrive(empty + sa);    // the item's last stage: the next item starts afresh
    next(sa, pa);
  }
}

// ------------------------------------------------------------------ E + H fused, warp-specialised
// A first version did the E phase and the H phase of a plane in the SAME 16 + 1 warps, in lockstep
// with one block barrier per plane: 18 warps per SM, each carrying ~375 instructions per plane,
// waited on fixed latencies more than they issued (ncu, profiles/r02_notes.md: issue slots 52 %
// busy, 4.3 TB/s at 256^3).  k_eh_fused gives the two phases to two sets of warps: 15 + 1 E warps
// compute E^{n+1}(q) into one of three rotating planes in shared memory and store it (the 16th
// computes the rim: row y0 + 15 and column x0 + 32); 15 H warps take H(q-1) from E^{n+1}(q-1) and
// E^{n+1}(q).  The sets are coupled by two rings of mbarriers (efull / eempty per plane) instead of
// a block barrier, so the E warps run up to two planes ahead: 32 warps per SM (the most a block
// can have, hence 15 rows), 4.8 TB/s at 256^3.  Same arithmetic, same bits.
// A block has at most 32 warps: 15 tile rows (15 + 1 E warps, 15 H warps, the producer).
constexpr int FBY = 15;
constexpr int FROWS = FBY + 2;                // staged rows y0-1 .. y0+15
constexpr int FSLOT = round16(FROWS * EW);    // doubles per staged array
constexpr int FNSLOT = round16((FBY + 1) * EW);   // E^{n+1} plane: rows y0 .. y0+15, columns x0 .. x0+32

template <bool EPS_ARR, bool SIG_ARR>
struct EfStage {   // one stage of the ring (as EhLayout, 17 rows)
  static constexpr int SLOT = FSLOT;
  static constexpr int HH = 0;
  static constexpr int EE = 3 * FSLOT;
  static constexpr int EP = 6 * FSLOT;
  static constexpr int SG = (6 + (EPS_ARR ? 1 : 0)) * FSLOT;
  static constexpr int NARR = 6 + (EPS_ARR ? 1 : 0) + (SIG_ARR ? 1 : 0);
  static constexpr int STAGE = NARR * FSLOT;
  static constexpr unsigned BYTES = 8u * NARR * FROWS * EW;
};

template <bool EPS_ARR, bool SIG_ARR>
struct EfLayout {
  using S = EfStage<EPS_ARR, SIG_ARR>;          // stage layout and byte counts
  static constexpr int NEB = 3;                 // rotating E^{n+1} planes
  static constexpr int ENEW = NEB * 3 * FNSLOT;
  static constexpr int BUDGET = 220 * 1024 - 8 * ENEW;
  static constexpr int NS_FIT = BUDGET / (8 * S::STAGE);
  static constexpr int NS = NS_FIT > 6 ? 6 : NS_FIT;
  static constexpr int NEW_ = FBY + 1;          // E warps: the tile rows + the rim
  static constexpr int NHW = FBY;               // H warps
  static constexpr int NCW = NEW_ + NHW;        // warps that release a stage
  static constexpr int NTHREADS = (NCW + 1) * 32;
  static constexpr size_t SMEM_BYTES = 128 + 8 * (size_t)(NS * S::STAGE + ENEW) + 8 * (2 * NS + 2 * NEB) + 4 * NS;
  static_assert(NS >= 3, "ring too shallow");
};

template <bool EPS_ARR, bool SIG_ARR, bool HAS_SRC>
__global__ void __launch_bounds__(EfLayout<EPS_ARR, SIG_ARR>::NTHREADS, 1)
k_eh_fused(const __grid_constant__ EHArgs p) {
  using L = EfLayout<EPS_ARR, SIG_ARR>;
  using S = typename L::S;
  extern __shared__ __align__(1024) unsigned char smem_raw[];
  double *const ring = reinterpret_cast<double *>(smem_raw);
  double *const enew = ring + L::NS * S::STAGE;
  uint64_t *const full = reinterpret_cast<uint64_t *>(enew + L::ENEW);
  uint64_t *const empty = full + L::NS;
  uint64_t *const efull = empty + L::NS;     // E^{n+1} plane b is complete (the NEW_ = FBY + 1 E warps arrive)
  uint64_t *const eempty = efull + L::NEB;   // ... is no longer read (the NHW = FBY H warps arrive)
  int *const meta = reinterpret_cast<int *>(eempty + L::NEB);

  const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
  if (threadIdx.x == 0) {
    for (int s = 0; s < L::NS; ++s) { mbar_init(full + s, 1); mbar_init(empty + s, L::NCW); }
    for (int b = 0; b < L::NEB; ++b) { mbar_init(efull + b, L::NEW_); mbar_init(eempty + b, L::NHW); }
    mbar_fence_init();
  }
  __syncthreads();

  if (p.book && blockIdx.x == 0 && threadIdx.x == 0) {   // the step's bookkeeping (k_half_end, twice)
    DevState *st = p.book;
    st->iters_last = 0;
    st->last_R_even = 0;
    p.r_hist[st->halfsteps % 4096] = 0;
    p.r_hist[(st->halfsteps + 1) % 4096] = 0;
    st->halfsteps += 2;
    st->steps++;
    for (int q = 0; q < 8; ++q) p.work_other[q] = 0u;
  }
  const StBox &T = p.tb;
  const GridP &g = p.g;
  auto next = [](unsigned &st, unsigned &ph) { if (++st == (unsigned)L::NS) { st = 0; ph ^= 1u; } };
  auto nextb = [](unsigned &b, unsigned &ph) { if (++b == (unsigned)L::NEB) { b = 0; ph ^= 1u; } };

  if (warp == L::NCW) {
    // ===== producer: stages k0-1 .. k1 of every item it draws
    if (lane == 0) {
      tma_prefetch_desc(&p.map);
      unsigned s = 0, ph = 1;
      for (;;) {
        const int it = (int)atomicAdd(p.work, 1u);
        const bool end = it >= T.items;
        const StItem w = st_decode_by(T, end ? 0 : it, FBY);
        for (int pz = w.k0 - 1; pz < (end ? w.k0 : w.k1 + 1); ++pz) {
          if (!mbar_wait(empty + s, ph, p.pipe_error, 7)) return;
          meta[s] = end ? -1 : it;
          if (end) {
            mbar_arrive(full + s);
            break;
          }
          mbar_expect_tx(full + s, S::BYTES);
          eh_issue_stage<S, EPS_ARR, SIG_ARR>(p, ring + s * S::STAGE, full + s, w.x0, w.y0, pz);
          next(s, ph);
        }
        if (end) break;
      }
    }
    return;
  }

  if (warp < L::NEW_) {
    // ===== E warps.  warp < FBY: tile row, lane = x.  warp == FBY: the rim of the E^{n+1} plane on
    // the high side: row y0 + FBY (E_x, E_z) and column x0 + SW (E_y, E_z)
    const bool rim = warp == FBY;
    const int t0 = (warp + 1) * EW + lane + 2;   // own staged position
    const int u0 = warp * EW + lane;             // own position in the E^{n+1} plane
    double *const eo0 = p.Eo[0], *const eo1 = p.Eo[1], *const eo2 = p.Eo[2];
    unsigned sa = 0, pa = 0;     // ring position of stage q-1
    unsigned eb = 0, ep = 1;     // E^{n+1} plane written next, the parity its eempty barrier is waited on
    for (;;) {
      if (!mbar_wait(full + sa, pa, p.pipe_error, 8)) return;
      const int it = *(volatile int *)(meta + sa);
      if (it < 0) break;
      const StItem w = st_decode_by(T, it, FBY);
      const int i = w.x0 + lane, j = w.y0 + warp;
      const bool valid = !rim && i < T.hi[0] && j < T.hi[1];
      const Column col = make_column(g, i, j);
      const bool wi = on_wall(g, 0, i), wj = on_wall(g, 1, j);
      const bool wj_rim = on_wall(g, 1, w.y0 + FBY), wi_rimrow = on_wall(g, 0, w.x0 + lane);
      const bool wi_rim = on_wall(g, 0, w.x0 + SW), wj_rimcol = on_wall(g, 1, w.y0 + lane);
      int c = g.org + i + g.sy * j + g.sz * w.k0;
      for (int q = w.k0; q <= w.k1; ++q) {
        unsigned sb = sa, pb = pa;
        next(sb, pb);
        const double *A = ring + sa * S::STAGE;
        const double *B = ring + sb * S::STAGE;
        if (!mbar_wait(full + sb, pb, p.pipe_error, 9)) return;
        if (!mbar_wait(eempty + eb, ep, p.pipe_error, 10)) return;   // the H warps are done with this plane
        double *const N = enew + eb * (3 * FNSLOT);
        const bool wk = on_wall(g, 2, q);
        if (!rim) {
          const double ex = eh_edge<S, 0, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, t0, i, j, q, wj || wk);
          const double ey = eh_edge<S, 1, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, t0, i, j, q, wk || wi);
          const double ez = eh_edge<S, 2, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, t0, i, j, q, wi || wj);
          N[u0] = ex; N[FNSLOT + u0] = ey; N[2 * FNSLOT + u0] = ez;
          if (valid && q < w.k1) {
            eo0[c] = ex;
            eo1[c] = ey;
            eo2[c] = ez;
            if (col.edge_ij || edge_k(g, q)) {
              store_images_inl<exp_of_e<0>()>(eo0, g, i, j, q, c, ex);
              store_images_inl<exp_of_e<1>()>(eo1, g, i, j, q, c, ey);
              store_images_inl<exp_of_e<2>()>(eo2, g, i, j, q, c, ez);
            }
          }
        } else {
          {  // row y0 + FBY: E_x, E_z at (x0 + lane, y0 + FBY)
            const int tr = (FBY + 1) * EW + lane + 2, ur = FBY * EW + lane;
            N[ur] = eh_edge<S, 0, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, tr, w.x0 + lane, w.y0 + FBY, q, wj_rim || wk);
            N[2 * FNSLOT + ur] = eh_edge<S, 2, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, tr, w.x0 + lane, w.y0 + FBY, q, wi_rimrow || wj_rim);
          }
          if (lane < FBY) {  // column x0 + SW: E_y, E_z at (x0 + SW, y0 + lane)
            const int tc = (lane + 1) * EW + SW + 2, uc = lane * EW + SW;
            N[FNSLOT + uc] = eh_edge<S, 1, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, tc, w.x0 + SW, w.y0 + lane, q, wk || wi_rim);
            N[2 * FNSLOT + uc] = eh_edge<S, 2, EPS_ARR, SIG_ARR, HAS_SRC>(p, A, B, tc, w.x0 + SW, w.y0 + lane, q, wi_rim || wj_rimcol);
          }
        }
        c += g.sz;
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(efull + eb);   // this warp's part of E^{n+1}(q) is in shared memory
          mbar_arrive(empty + sa);   // stage q-1 is done with (on the E side)
        }
        sa = sb; pa = pb;
        nextb(eb, ep);
      }
      if (lane == 0) mbar_arrive(empty + sa);    // the item's last stage
      next(sa, pa);
    }
    return;
  }

  // ===== H warps: tile row warp - NEW_, lane = x; H(h) for h = k0 .. k1-1 from E^{n+1}(h), E^{n+1}(h+1)
  {
    const int row = warp - L::NEW_;
    const int t0 = (row + 1) * EW + lane + 2;
    const int u0 = row * EW + lane;
    double *const ho0 = p.Ho[0], *const ho1 = p.Ho[1], *const ho2 = p.Ho[2];
    const double chm = p.chm, rdx = g.rd[0], rdy = g.rd[1], rdz = g.rd[2];
    unsigned sh = 0, ph = 0;     // ring position of the stage looked at next
    unsigned hb = 0, hp = 0;     // E^{n+1} plane h and the parity its efull barrier is waited on
    for (;;) {
      if (!mbar_wait(full + sh, ph, p.pipe_error, 11)) return;
      const int it = *(volatile int *)(meta + sh);
      if (it < 0) break;
      const StItem w = st_decode_by(T, it, FBY);
      const int i = w.x0 + lane, j = w.y0 + row;
      const bool valid = i < T.hi[0] && j < T.hi[1];
      const Column col = make_column(g, i, j);
      int c = g.org + i + g.sy * j + g.sz * w.k0;
      __syncwarp();
      if (lane == 0) mbar_arrive(empty + sh);    // stage k0-1 holds nothing an H face reads
      next(sh, ph);
      if (!mbar_wait(efull + hb, hp, p.pipe_error, 12)) return;   // E^{n+1}(k0)
      for (int h = w.k0; h < w.k1; ++h) {
        const double *A = ring + sh * S::STAGE;   // stage h: this face's own H
        if (!mbar_wait(full + sh, ph, p.pipe_error, 13)) return;
        unsigned nb = hb, np = hp;
        nextb(nb, np);
        if (!mbar_wait(efull + nb, np, p.pipe_error, 14)) return;  // E^{n+1}(h+1)
        if (valid) {
          const double *P = enew + hb * (3 * FNSLOT), *Q = enew + nb * (3 * FNSLOT);
          const double ex_h = P[u0], ey_h = P[FNSLOT + u0], ez_h = P[2 * FNSLOT + u0];
          // (curl E^{n+1})_D at the D-face of plane h: forward differences, as curl_e (kernels.cuh)
          const double cx = (P[2 * FNSLOT + u0 + EW] - ez_h) * rdy - (Q[FNSLOT + u0] - ey_h) * rdz;
          const double cy = (Q[u0] - ex_h) * rdz - (P[2 * FNSLOT + u0 + 1] - ez_h) * rdx;
          const double cz = (P[FNSLOT + u0 + 1] - ey_h) * rdx - (P[u0 + EW] - ex_h) * rdy;
          const double hx = h_face_val(A[S::HH + t0], chm, cx, col.wall[0]);
          const double hy = h_face_val(A[S::HH + FSLOT + t0], chm, cy, col.wall[1]);
          const double hz = h_face_val(A[S::HH + 2 * FSLOT + t0], chm, cz, wall_k(g, h));
          ho0[c] = hx;
          ho1[c] = hy;
          ho2[c] = hz;
          if (col.edge_ij || edge_k(g, h)) {
            store_images_inl<exp_of_h<0>()>(ho0, g, i, j, h, c, hx);
            store_images_inl<exp_of_h<1>()>(ho1, g, i, j, h, c, hy);
            store_images_inl<exp_of_h<2>()>(ho2, g, i, j, h, c, hz);
          }
        }
        c += g.sz;
        __syncwarp();
        if (lane == 0) {
          mbar_arrive(eempty + hb);  // E^{n+1}(h) is done with
          mbar_arrive(empty + sh);   // stage h is done with (on the H side)
        }
        next(sh, ph);
        hb = nb; hp = np;
      }
      // E^{n+1}(k1) was read as the plane above the item's last faces; stage k1 holds nothing an H
      // face of this item reads (it was filled: the E warps waited for it before they wrote that plane)
      if (lane == 0) {
        mbar_arrive(eempty + hb);
        mbar_arrive(empty + sh);
      }
      next(sh, ph);
      nextb(hb, hp);
    }
  }
}

}  // namespace fl
