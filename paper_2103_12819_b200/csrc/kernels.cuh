// kernels.cuh -- sm_100a device code of the coupled FDTD-LLG step (fp64 stencils).
//
// Citations are /root/reference/PAPER.md lines of arXiv 2103.12819.  Staggering: include/fdtd_llg.h.
//
// DEVICE LAYOUT.  Every array (fields and cell-centred materials) is stored with one ghost layer:
//   element (i,j,k), -1 <= i <= nx, -1 <= j <= ny, -1 <= k <= nz, lives at
//       org + i + sy*j + sz*k,   sy = row pitch (multiple of 16 doubles), sz = sy*(ny+2),
//   with org chosen so that the interior row start (i = 0) is 128-byte aligned.  Ghosts of a PEC
//   axis are zero for ever (a read beyond a PEC wall is the constant 0: wall-normal H and
//   wall-tangential E vanish there); ghosts of a periodic axis mirror the opposite
//   interior plane and are refreshed IN-KERNEL by the thread that writes the
//   boundary cell.  Hence every stencil neighbour is a constant offset from the centre: no index
//   arithmetic, no predicates in the inner loops.
//   A z side that is an INTERFACE to a neighbouring slab (multi-GPU z-slab decomposition, PAPER.md:195,
//   217) is no wall: its ghost plane holds the neighbour's adjacent plane, and the thread that
//   writes a value of the slab's first / last plane also stores it into the neighbour's ghost plane
//   through peer-mapped memory (store_images_inl), so the halo exchange is part of the update.
//
// THREADING.  A block is TX x TY columns (x fastest, coalesced 256-byte rows) and marches KZ planes
// in z, so the k-1 / k+1 neighbours of consecutive planes are served by L1.  Grids are persistent
// (a multiple of the SM count) and loop over work items; an LLG sweep that finds the previous
// iterate converged exits after one flag read.
//
// Kernels
//   k_h_update   Maxwell (H) half-step on the faces OUTSIDE the LLG sweep box     eq. 21 with M = 0
//   k_hm_sweep   one Jacobi iterate r of the trapezoidal LLG solve + eq. 21 inside the sweep box
//   k_half_end   1 thread: iteration count / statistics from the residual words, re-arm them
//   k_canon      copies H^R into the canonical buffer when R is even
//   k_e_update   eq. 11 with in-kernel edge means of eps_r, sigma and the soft sources
//   k_step_begin source amplitudes g_s((n+1/2) dt) for this step
//   set-up: k_fill_ghosts, k_enforce_walls, k_init_m, k_minmax, k_mag_box
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fl {

constexpr int MAX_SOURCES = 8;
constexpr int PADL = 16;         // doubles left of i = 0 in a row (ghost i = -1 sits at PADL-1)
constexpr int TX = 32, TY = 8;   // thread block = TX x TY columns
constexpr int NTHREADS = TX * TY;
constexpr int KZ_MAX = 16;       // planes marched per work item (fewer on small grids)

constexpr double kPi = 3.14159265358979323846;
constexpr double kMu0 = 4.0e-7 * kPi;
constexpr double kC0 = 299792458.0;
constexpr double kEps0 = 1.0 / (kMu0 * kC0 * kC0);

struct GridP {
  int n[3];    // nx, ny, nz
  int per[3];  // 1 = periodic (the ghost layer mirrors the opposite interior plane)
  int wall[3]; // 1 = PEC wall at index 0
  int wallhi[3]; // 1 = PEC wall at index n (differs from wall[2] on a slab with one interface)
  int ext[2];  // z-low / z-high side is an interface to a neighbouring slab (neither of the above)
  int sy, sz;  // element strides of j and k (the stride of i is 1)
  int org;     // offset of cell (0,0,0)
  // BYTE offsets from an element of this slab's first (dlo) / last (dhi) plane to its image in the
  // lower / upper neighbour's ghost plane (same array, the neighbour's workspace); 0 = not connected
  long long dlo, dhi;
  double rd[3];  // 1/dx, 1/dy, 1/dz
  double dt;
};

// a box of cells cut into work items of TX x TY x kz
struct BoxP {
  int lo[3], hi[3];  // hi exclusive
  int ntx, nty, items;
  int kz;   // planes marched per work item
  int tyr;  // rows of a tile: TY, or a smaller power of two on a box with fewer rows (the block's
            // other thread rows then take further 32-column strips: the tile is TX*TY/tyr wide)
};

// device-resident run state (one per handle)
struct DevState {
  long long steps;
  long long halfsteps;
  long long iters_total;
  long long nonconverged;
  int iters_last;
  int iters_max;
  int last_R_even;  // 1 when the last half-step ended on an even iterate (result in the pong set)
  int init_error;   // set by k_init_m when a magnetic face got a zero averaged M
  int pipe_error;   // set by a TMA-fed kernel whose mbarrier wait timed out (tag of the wait)
  double resid_last;
  double src_amp[MAX_SOURCES];
};

struct SourceP {
  int kind;  // 0 soft E (J of eq. 11), 1 hard E, 2 soft H, 3 hard H (fdtd_llg.h)
  int comp;
  int lo[3], hi[3];
  const double *profile;  // device, box sized, or nullptr
  double amplitude, f0, t0, tp;
};

struct SourcesP {
  int count;
  SourceP s[MAX_SOURCES];
};

template <int D> __device__ __forceinline__ int stride_of(const GridP &g) {
  return D == 0 ? 1 : (D == 1 ? g.sy : g.sz);
}

// this thread's cell
struct Cell {
  int i, j, k;
  int c;      // element offset of (i,j,k)
};

// per-column (i,j) part of the predicates, hoisted out of the z march
struct Column {
  int i, j;
  bool edge_ij;   // periodic first/last plane in x or y
  bool wall[2];   // PEC lower wall in x / y
};
__device__ __forceinline__ Column make_column(const GridP &g, int i, int j) {
  Column q;
  q.i = i; q.j = j;
  q.edge_ij = (g.per[0] && (i == 0 || i == g.n[0] - 1)) || (g.per[1] && (j == 0 || j == g.n[1] - 1));
  q.wall[0] = g.wall[0] && i == 0;
  q.wall[1] = g.wall[1] && j == 0;
  return q;
}
// a value of plane k has images: periodic ghosts, or the ghost plane of a connected neighbour slab
__device__ __forceinline__ bool edge_k(const GridP &g, int k) {
  return ((g.per[2] || g.dlo != 0) && k == 0) || ((g.per[2] || g.dhi != 0) && k == g.n[2] - 1);
}
__device__ __forceinline__ bool wall_k(const GridP &g, int k) { return g.wall[2] && k == 0; }

// What a slab hands to its z neighbours: the curl of E and the four-point averages
// of an x- or y-face reach one plane UP (E_x, E_y, H_z of the upper neighbour's first plane), the curl
// of H and the averages of a z-face one plane DOWN (H_x, H_y of the lower neighbour's last plane).
enum { EXP_NONE = 0, EXP_LO = 1, EXP_HI = 2 };
template <int D> __host__ __device__ constexpr int exp_of_h() { return D == 2 ? EXP_LO : EXP_HI; }
template <int D> __host__ __device__ constexpr int exp_of_e() { return D == 2 ? EXP_NONE : EXP_LO; }

// slow path of a store: the periodic ghost images of an interior value and, for a
// component the neighbouring slab reads (EXP), its image in that slab's ghost plane.  Inlined (no
// call: a call would wait for every load the caller has in flight).  Up to two shifts per axis
// (both when the axis is one cell long).
template <int EXP>
__device__ __forceinline__ void store_images_inl(double *a, const GridP &g, int i, int j, int k,
                                                 int c, double v) {
  const int sx[3] = {0, (g.per[0] && i == 0) ? g.n[0] : 0, (g.per[0] && i == g.n[0] - 1) ? -g.n[0] : 0};
  const int sy[3] = {0, (g.per[1] && j == 0) ? g.n[1] * g.sy : 0,
                     (g.per[1] && j == g.n[1] - 1) ? -g.n[1] * g.sy : 0};
  const int sz[3] = {0, (g.per[2] && k == 0) ? g.n[2] * g.sz : 0,
                     (g.per[2] && k == g.n[2] - 1) ? -g.n[2] * g.sz : 0};
  const bool rlo = (EXP & EXP_LO) && g.dlo != 0 && k == 0;
  const bool rhi = (EXP & EXP_HI) && g.dhi != 0 && k == g.n[2] - 1;
#pragma unroll
  for (int x = 0; x < 3; ++x)
#pragma unroll
    for (int y = 0; y < 3; ++y) {
      if ((x && !sx[x]) || (y && !sy[y])) continue;
      const int cxy = c + sx[x] + sy[y];
#pragma unroll
      for (int z = 0; z < 3; ++z) {
        if (!(x | y | z)) continue;
        if (z && !sz[z]) continue;
        a[cxy + sz[z]] = v;
      }
      // peer stores (NVLink): the neighbour's ghost plane, including its periodic x / y ghosts
      if (EXP & EXP_LO) { if (rlo) *reinterpret_cast<double *>(reinterpret_cast<char *>(a + cxy) + g.dlo) = v; }
      if (EXP & EXP_HI) { if (rhi) *reinterpret_cast<double *>(reinterpret_cast<char *>(a + cxy) + g.dhi) = v; }
    }
}

// (curl E)_D at the D-face: forward differences (standard Yee)
template <int D>
__device__ __forceinline__ double curl_e(const GridP &g, int c, const double *const *E) {
  constexpr int d1 = (D + 1) % 3, d2 = (D + 2) % 3;
  const int s1 = stride_of<d1>(g), s2 = stride_of<d2>(g);
  const double a0 = __ldg(E[d2] + c), a1 = __ldg(E[d2] + c + s1);
  const double b0 = __ldg(E[d1] + c), b1 = __ldg(E[d1] + c + s2);
  return (a1 - a0) * g.rd[d1] - (b1 - b0) * g.rd[d2];
}

// transverse component T of H at the D-face: four-point average
template <int D, int T>
__device__ __forceinline__ double avg4(const GridP &g, int c, const double *__restrict__ Ht) {
  const int sd = stride_of<D>(g), st = stride_of<T>(g);
  const double v00 = __ldg(Ht + c), v10 = __ldg(Ht + c - sd);
  const double v01 = __ldg(Ht + c + st), v11 = __ldg(Ht + c - sd + st);
  return 0.25 * ((v00 + v10) + (v01 + v11));
}

// work-item decode shared by the sweeping kernels
struct Item {
  int i, j, k0, k1;
  bool active;
};
__device__ __forceinline__ Item decode_item(const BoxP &b, int it) {
  const int tx = it % b.ntx, r = it / b.ntx;
  const int ty = r % b.nty, tz = r / b.nty;
  const int strip = (int)threadIdx.y / b.tyr, row = (int)threadIdx.y % b.tyr;
  Item w;
  w.i = b.lo[0] + (tx * (TY / b.tyr) + strip) * TX + (int)threadIdx.x;
  w.j = b.lo[1] + ty * b.tyr + row;
  w.k0 = b.lo[2] + tz * b.kz;
  w.k1 = min(w.k0 + b.kz, b.hi[2]);
  w.active = w.i < b.hi[0] && w.j < b.hi[1];
  return w;
}

// ------------------------------------------------------------------ Maxwell H half-step

struct HArgs {
  GridP g;
  BoxP box;            // the cells this launch updates (a slab of the complement of the LLG box)
  const double *E[3];
  const double *Hn[3];
  double *Hc[3];
  const double *mu_r;  // cell-centred array or nullptr (uniform)
  double ch_uniform;   // dt / (2 mu0 mu_r) when uniform
  double cmul;         // 1: half a step (eq. 21); 2: the two adjacent half-steps of a face that no
                       // magnetic face reads, taken at once with the same curl E
};

// eq. 21 with M = 0 on one face: hn = H on the face, chm = cmul dt / (2 mu), C =
// (curl E)_D there; a PEC wall face stays 0.  Shared by k_h_update and k_eh_stage.
__device__ __forceinline__ double h_face_val(double hn, double chm, double C, bool wall) {
  const double h = hn - chm * C;
  return wall ? 0.0 : h;
}

// eq. 21 with M = 0 and the local mu; a PEC wall face stays 0
template <int D, bool MU_ARR>
__device__ __forceinline__ double h_face(const HArgs &a, int c, bool wall) {
  double ch = a.ch_uniform;
  if (MU_ARR) {
    const double mu = 0.5 * (__ldg(a.mu_r + c) + __ldg(a.mu_r + c - stride_of<D>(a.g)));
    ch = a.g.dt / (2.0 * kMu0 * mu);
  }
  const double C = curl_e<D>(a.g, c, a.E);
  // plain load: Hn aliases Hc when the integer-time H is formed in place (reconstruct_h);
  // cmul = 1, 2: an exact scaling
  return h_face_val(a.Hn[D][c], a.cmul * ch, C, wall);
}

template <bool MU_ARR>
__global__ void __launch_bounds__(NTHREADS) k_h_update(const __grid_constant__ HArgs a) {
  for (int it = blockIdx.x; it < a.box.items; it += gridDim.x) {
    const Item w = decode_item(a.box, it);
    const Column col = make_column(a.g, w.i, w.j);
    if (!w.active) continue;
    int c = a.g.org + w.i + a.g.sy * w.j + a.g.sz * w.k0;
    for (int k = w.k0; k < w.k1; ++k, c += a.g.sz) {
      const double hx = h_face<0, MU_ARR>(a, c, col.wall[0]);
      const double hy = h_face<1, MU_ARR>(a, c, col.wall[1]);
      const double hz = h_face<2, MU_ARR>(a, c, wall_k(a.g, k));
      a.Hc[0][c] = hx;
      a.Hc[1][c] = hy;
      a.Hc[2][c] = hz;
      if (col.edge_ij || edge_k(a.g, k)) {
        store_images_inl<exp_of_h<0>()>(a.Hc[0], a.g, w.i, w.j, k, c, hx);
        store_images_inl<exp_of_h<1>()>(a.Hc[1], a.g, w.i, w.j, k, c, hy);
        store_images_inl<exp_of_h<2>()>(a.Hc[2], a.g, w.i, w.j, k, c, hz);
      }
    }
  }
}

// ------------------------------------------------------------------ LLG sweep

struct HMArgs {
  GridP g;
  BoxP box;             // the LLG sweep box
  const double *E[3];
  const double *Hn[3];  // H^n
  const double *Hp[3];  // H^{r-1}  (== Hn when FIRST)
  double *Hc[3];        // H^r
  const double *Mn[9];  // M^n      [face*3 + comp]
  double *Mr[9];        // M^{r-1} in, M^r out (same thread); FIRST: out only
  const double *Ms, *alpha, *gamma, *mu_r;  // cell-centred arrays or nullptr (uniform)
  double Ms_u, rMs_u, alpha_u, gamma_u, ch_uniform;
  double cf_u;  // mu0 |gamma_u| dt / 4, the coefficient of eqs. 19-20 when gamma is uniform
  double kh;    // dt / (2 mu0), the coefficient of curl E in eq. 21
  double hb[3], hk, u[3];
  double tol;
  int euler;  // 1: first-order scheme: the r = 1 sweep is a forward-Euler step
  unsigned long long *resid;  // [max_iter + 1] bit patterns of the residual of iterate r
  int *pipe_error;            // &DevState::pipe_error
  int r;
};

struct Vec3 { double x, y, z; };
__device__ __forceinline__ Vec3 cross(const Vec3 &a, const Vec3 &b) {
  return {a.y * b.z - a.z * b.y, a.z * b.x - a.x * b.z, a.x * b.y - a.y * b.x};
}
__device__ __forceinline__ double dot(const Vec3 &a, const Vec3 &b) {
  return a.x * b.x + a.y * b.y + a.z * b.z;
}
template <int D> __device__ __forceinline__ double comp(const Vec3 &v) {
  return D == 0 ? v.x : (D == 1 ? v.y : v.z);
}

// H_EM at the D-face from one H set: own normal component + two four-point averages
template <int D>
__device__ __forceinline__ Vec3 h_em(const GridP &g, int c, const double *const *H) {
  Vec3 h;
  if (D == 0) {
    h.x = __ldg(H[0] + c); h.y = avg4<0, 1>(g, c, H[1]); h.z = avg4<0, 2>(g, c, H[2]);
  } else if (D == 1) {
    h.x = avg4<1, 0>(g, c, H[0]); h.y = __ldg(H[1] + c); h.z = avg4<1, 2>(g, c, H[2]);
  } else {
    h.x = avg4<2, 0>(g, c, H[0]); h.y = avg4<2, 1>(g, c, H[1]); h.z = __ldg(H[2] + c);
  }
  return h;
}

// 1/(1+y), y >= 0.  For y < 6e-5 the alternating series through y^3 is exact to 1.3e-17
// relative (y = |a|^2 is ~1e-10 at any physical field strength); otherwise the division.
__device__ __forceinline__ double recip_1p(double y) {
  if (y < 6.0e-5) return fma(y, fma(y, 1.0 - y, -1.0), 1.0);
  return 1.0 / (1.0 + y);
}

// (1+x)^(-1/2) - 1 = Ms/|M^n + Delta| - 1  (PAPER.md:98, 179 applied to the increment).
// |x| < 1e-4: Maclaurin series through x^4 (truncation 63/256 x^5 < 5e-17 relative);
// otherwise -x / (s (1 + s)), s = sqrt(1+x) -- both free of cancellation.
__device__ __forceinline__ double rsqrt_1p_m1(double x) {
  if (fabs(x) < 1.0e-4)
    return x * fma(x, fma(x, fma(x, 35.0 / 128.0, -5.0 / 16.0), 3.0 / 8.0), -0.5);
  const double sq = sqrt(1.0 + x);
  return -x / (sq * (1.0 + sq));
}

// The increment form of eqs. 18-20 + N(M) on one face (reading A24):
//   b = M^n + beta,  tau = a x M^n,  Delta = (18) - M^n,  dM = M^r - M^n.
// mn = M^n, hn = H_eff^n, he = H_eff^{r-1} (FIRST: he == hn).
template <bool FIRST>
__device__ __forceinline__ Vec3 llg_increment(const Vec3 &mn, const Vec3 &hn, const Vec3 &he,
                                              double cf, double aM, double rMs) {
  const Vec3 t0 = cross(mn, hn);
  const Vec3 beta = {-cf * t0.x, -cf * t0.y, -cf * t0.z};                      // (20) - M^n
  const Vec3 av = {-(cf * he.x + aM * mn.x), -(cf * he.y + aM * mn.y), -(cf * he.z + aM * mn.z)};  // (19)
  const Vec3 axb = cross(av, beta);
  const double ab = dot(av, beta);
  const double rden = recip_1p(dot(av, av));
  Vec3 De;  // (18) - M^n
  if (FIRST) {  // tau = -beta
    De = {(2.0 * (beta.x - axb.x) + ab * av.x) * rden, (2.0 * (beta.y - axb.y) + ab * av.y) * rden,
          (2.0 * (beta.z - axb.z) + ab * av.z) * rden};
  } else {
    const Vec3 t1 = cross(mn, he);
    const Vec3 tau = {cf * t1.x, cf * t1.y, cf * t1.z};
    const Vec3 axt = cross(av, tau);
    De = {(beta.x - tau.x + axt.x + ab * av.x - axb.x) * rden,
          (beta.y - tau.y + axt.y + ab * av.y - axb.y) * rden,
          (beta.z - tau.z + axt.z + ab * av.z - axb.z) * rden};
  }
  const double x = (2.0 * dot(mn, De) + dot(De, De)) * (rMs * rMs);
  const double sm1 = rsqrt_1p_m1(x);
  return {De.x + sm1 * (mn.x + De.x), De.y + sm1 * (mn.y + De.y), De.z + sm1 * (mn.z + De.z)};
}

// First-order scheme, Step 1 / Step 3 (eqs. 7 and 12 advance half a step, A22):
//   M' = M + (dt/2) [ mu0 gamma_L (M x H_eff) + (alpha mu0 gamma_L / Ms) M x (M x H_eff) ],
// gamma_L = gamma / (1 + alpha^2) with the electron's negative gamma, then N(M') applied to the
// increment as in llg_increment.  g2 = mu0 |gamma_L| dt / 2.  Returns dM = M' - M.
__device__ __forceinline__ Vec3 llg_euler(const Vec3 &mn, const Vec3 &hn, double g2, double alf,
                                          double rMs) {
  const Vec3 p = cross(mn, hn);
  const Vec3 q = cross(mn, p);
  const double ar = alf * rMs;
  const Vec3 De = {-g2 * (p.x + ar * q.x), -g2 * (p.y + ar * q.y), -g2 * (p.z + ar * q.z)};
  const double x = (2.0 * dot(mn, De) + dot(De, De)) * (rMs * rMs);
  const double sm1 = rsqrt_1p_m1(x);
  return {De.x + sm1 * (mn.x + De.x), De.y + sm1 * (mn.y + De.y), De.z + sm1 * (mn.z + De.z)};
}

// result of one face: M^r, H^r (normal component), residual
struct FaceOut {
  Vec3 m;
  double h;
  double res;
};

// Arithmetic of one Jacobi iterate on a D-face, shared by every sweep kernel (whatever way its
// operands were fetched), BRANCH-FREE: the magnetic / non-magnetic / wall decision is a select at
// the end.  (A non-magnetic face runs the LLG arithmetic on rMs = 0 and discards it.)
//   mn = M^n, mp = M^{r-1}, hn / he = H_EM^n / H_EM^{r-1} (own normal component + the two
//   four-point averages), C = (curl E)_D, Msf / rMs = face Ms and its reciprocal (0 if Msf = 0),
//   alf = face alpha, cf = mu0 |gamma_face| dt / 4, ch = dt / (2 mu) of a non-magnetic face.
// The residual is max_c |M^r_c - M^{r-1}_c| / Ms_f (0 on non-magnetic faces); a non-finite M^r
// (a step far above the Courant limit) gives an infinite residual, so the half-step is never
// reported as converged.
template <int D, bool FIRST, bool ANISO>
__device__ __forceinline__ FaceOut hm_face_core(const HMArgs &a, const Vec3 &mn, const Vec3 &mp_in,
                                                Vec3 hn, Vec3 he, double C, double Msf, double rMs,
                                                double alf, double cf, double ch, bool wall) {
  const Vec3 mp = FIRST ? mn : mp_in;
  const double hn_own = comp<D>(hn), hp_own = comp<D>(he);

  // ---- magnetic face: eqs. 18-21
  const bool magnetic = !wall && Msf > 0.0;
  const Vec3 hb = {a.hb[0], a.hb[1], a.hb[2]};
  const Vec3 u = {a.u[0], a.u[1], a.u[2]};
  // H_eff^n = H_EM^n + H_bias + H_k (M^n.u / Ms) u            (A19)
  hn.x += hb.x; hn.y += hb.y; hn.z += hb.z;
  if (ANISO) {
    const double p = a.hk * (dot(mn, u) * rMs);
    hn.x += p * u.x; hn.y += p * u.y; hn.z += p * u.z;
  }
  // H_eff^{r-1}, lagged; at r = 1 it is H_eff^n
  if (FIRST) {
    he = hn;
  } else {
    he.x += hb.x; he.y += hb.y; he.z += hb.z;
    if (ANISO) {
      const double p = a.hk * (dot(mp, u) * rMs);
      he.x += p * u.x; he.y += p * u.y; he.z += p * u.z;
    }
  }
  Vec3 dM;
  if (FIRST && a.euler)
    dM = llg_euler(mn, hn, 2.0 * cf / (1.0 + alf * alf), alf, rMs);
  else
    dM = llg_increment<FIRST>(mn, hn, he, cf, alf * rMs, rMs);
  const Vec3 mr = {mn.x + dM.x, mn.y + dM.y, mn.z + dM.z};
  // eq. 21, normal component:  H^r = H^n + M^n - M^r - (dt / 2 mu0) curl E
  const double h_mag = hn_own - comp<D>(dM) - a.kh * C;
  // stopping test of PAPER.md:154, per face; reduced by the caller
  const double e = fmax(fmax(fabs(mr.x - mp.x), fabs(mr.y - mp.y)), fabs(mr.z - mp.z)) * rMs;
  const bool finite = fabs(mr.x) + fabs(mr.y) + fabs(mr.z) < INFINITY;   // false for NaN too

  // ---- non-magnetic face inside the sweep box: Maxwell update at r = 1, copy afterwards so that
  // both Jacobi buffers hold it.  PEC wall face: H = 0, M = 0 for ever (A13).
  const double h_non = wall ? 0.0 : (FIRST ? hn_own - ch * C : hp_own);
  FaceOut o;
  o.m = {magnetic ? mr.x : 0.0, magnetic ? mr.y : 0.0, magnetic ? mr.z : 0.0};
  o.h = magnetic ? h_mag : h_non;
  o.res = (magnetic && !(FIRST && a.euler)) ? (finite ? e : INFINITY) : 0.0;  // an explicit sweep has no stopping test
  return o;
}

// One Jacobi iterate on the D-face of the cell at offset c, operands straight from global memory:
// every load is a constant offset from c (always in bounds thanks to the ghost layer) and is
// issued unconditionally, so the compiler batches all of a face's loads ahead of the arithmetic.
// Ms_c / rMs_c: this cell's Ms and its reciprocal, shared by the three faces wherever Ms is
// locally uniform.
template <int D, bool FIRST, bool MS_ARR, bool AG_ARR, bool MU_ARR, bool ANISO>
__device__ __forceinline__ FaceOut hm_face(const HMArgs &a, int c, bool wall, double Ms_c,
                                           double rMs_c) {
  const int cm = c - stride_of<D>(a.g);
  double Ms_m = Ms_c;
  if (MS_ARR) Ms_m = __ldg(a.Ms + cm);
  const Vec3 mn = {__ldcs(a.Mn[3 * D + 0] + c), __ldcs(a.Mn[3 * D + 1] + c),
                   __ldcs(a.Mn[3 * D + 2] + c)};
  Vec3 mp = mn;
  if (!FIRST)
    mp = {__ldcs(a.Mr[3 * D + 0] + c), __ldcs(a.Mr[3 * D + 1] + c), __ldcs(a.Mr[3 * D + 2] + c)};
  const Vec3 hn = h_em<D>(a.g, c, a.Hn);
  Vec3 he = hn;
  if (!FIRST) he = h_em<D>(a.g, c, a.Hp);
  const double C = curl_e<D>(a.g, c, a.E);
  double alf = a.alpha_u, cf = a.cf_u, ch = a.ch_uniform;
  if (AG_ARR) {
    alf = 0.5 * (__ldg(a.alpha + c) + __ldg(a.alpha + cm));
    const double gam = 0.5 * (fabs(__ldg(a.gamma + c)) + fabs(__ldg(a.gamma + cm)));  // |gamma| (eqs. 19-20)
    cf = kMu0 * gam * a.g.dt * 0.25;                                                // mu0 |gamma| dt / 4
  }
  if (MU_ARR) ch = a.g.dt / (2.0 * kMu0 * (0.5 * (__ldg(a.mu_r + c) + __ldg(a.mu_r + cm))));
  const double Msf = 0.5 * (Ms_c + Ms_m);
  double rMs = rMs_c;
  if (MS_ARR && Ms_m != Ms_c) rMs = Msf > 0.0 ? 1.0 / Msf : 0.0;
  return hm_face_core<D, FIRST, ANISO>(a, mn, mp, hn, he, C, Msf, rMs, alf, cf, ch, wall);
}

template <int D>
__device__ __forceinline__ void store_face(const HMArgs &a, int c, const FaceOut &o) {
  __stcs(a.Mr[3 * D + 0] + c, o.m.x);
  __stcs(a.Mr[3 * D + 1] + c, o.m.y);
  __stcs(a.Mr[3 * D + 2] + c, o.m.z);
  a.Hc[D][c] = o.h;
}
// Only H is ever read through a ghost (the four-point averages and curl H); M is read by the
// thread that owns the face, so its ghosts need no refresh.
template <int D>
__device__ __forceinline__ void store_face_images(const HMArgs &a, int i, int j, int k, int c,
                                                  const FaceOut &o) {
  store_images_inl<exp_of_h<D>()>(a.Hc[D], a.g, i, j, k, c, o.h);
}

template <bool FIRST, bool MS_ARR, bool AG_ARR, bool MU_ARR, bool ANISO>
__global__ void __launch_bounds__(NTHREADS) k_hm_sweep(const __grid_constant__ HMArgs a) {
  // the whole grid takes the same decision: iterate r runs iff iterate r-1 was not converged
  if (!FIRST) {
    if (__longlong_as_double((long long)a.resid[a.r - 1]) < a.tol) return;
  }
  double res = 0.0;
  for (int it = blockIdx.x; it < a.box.items; it += gridDim.x) {
    const Item w = decode_item(a.box, it);
    const Column col = make_column(a.g, w.i, w.j);
    if (!w.active) continue;
    int c = a.g.org + w.i + a.g.sy * w.j + a.g.sz * w.k0;
    for (int k = w.k0; k < w.k1; ++k, c += a.g.sz) {
      double Ms_c = a.Ms_u, rMs_c = a.rMs_u;
      if (MS_ARR) {
        Ms_c = __ldg(a.Ms + c);
        rMs_c = Ms_c > 0.0 ? 1.0 / Ms_c : 0.0;
      }
      const bool edge = col.edge_ij || edge_k(a.g, k);
      {
        const FaceOut o = hm_face<0, FIRST, MS_ARR, AG_ARR, MU_ARR, ANISO>(a, c, col.wall[0], Ms_c, rMs_c);
        store_face<0>(a, c, o);
        if (edge) store_face_images<0>(a, w.i, w.j, k, c, o);
        res = fmax(res, o.res);
      }
      {
        const FaceOut o = hm_face<1, FIRST, MS_ARR, AG_ARR, MU_ARR, ANISO>(a, c, col.wall[1], Ms_c, rMs_c);
        store_face<1>(a, c, o);
        if (edge) store_face_images<1>(a, w.i, w.j, k, c, o);
        res = fmax(res, o.res);
      }
      {
        const FaceOut o = hm_face<2, FIRST, MS_ARR, AG_ARR, MU_ARR, ANISO>(a, c, wall_k(a.g, k), Ms_c, rMs_c);
        store_face<2>(a, c, o);
        if (edge) store_face_images<2>(a, w.i, w.j, k, c, o);
        res = fmax(res, o.res);
      }
    }
  }
  // convergence word: warp shuffles, then ONE atomic per block
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) res = fmax(res, __shfl_xor_sync(0xffffffffu, res, o));
  __shared__ double wmax[NTHREADS / 32];
  const int tid = threadIdx.x + TX * threadIdx.y;
  if ((tid & 31) == 0) wmax[tid >> 5] = res;
  __syncthreads();
  if (tid == 0) {
    double m = wmax[0];
#pragma unroll
    for (int w = 1; w < NTHREADS / 32; ++w) m = fmax(m, wmax[w]);
    if (m > 0.0) atomicMax(a.resid + a.r, (unsigned long long)__double_as_longlong(m));
  }
}

// 1 thread: arm the conditional graph node that holds the iterates r >= r_next: they are needed
// only if iterate r_next - 1 ran and missed the tolerance
__global__ void k_set_cond(cudaGraphConditionalHandle h, const unsigned long long *resid, double tol,
                           int r_next) {
  const double res = __longlong_as_double((long long)resid[r_next - 1]);
  cudaGraphSetConditional(h, res < tol ? 0u : 1u);
}

// 1 thread: close an (H,M) half-step of which the iterates 1..r_max were enqueued (fdtd_llg_step:
// all max_iter of them, those after convergence exit on the flag; fdtd_llg_substep: the caller
// stops when an iterate met the tolerance)
__global__ void k_half_end(DevState *st, unsigned long long *resid, unsigned *work, unsigned *work_eh,
                           int *r_hist, int r_max, int max_iter, double tol, int any_magnetic,
                           int last_of_step) {
  for (int q = 0; q < 16; ++q) work_eh[q] = 0u;  // item counters of the staged Maxwell sweeps (both step parities)
  if (any_magnetic) {
    int R = r_max;
    for (int r = 1; r <= r_max; ++r)
      if (__longlong_as_double((long long)resid[r]) < tol) { R = r; break; }
    const double res = __longlong_as_double((long long)resid[R]);
    if (!(res < tol)) st->nonconverged++;
    st->iters_last = R;
    st->iters_total += R;
    if (R > st->iters_max) st->iters_max = R;
    st->resid_last = res;
    st->last_R_even = ((R & 1) == 0);
  } else {
    st->iters_last = 0;
    st->last_R_even = 0;
  }
  // Re-arm the residual words and item counters, magnetic faces or not: a slab WITHOUT magnetic faces
  // still receives the maximum over all slabs in its words (the caller's max-allreduce writes it
  // there, fdtd_llg.h "Z-SLABS") and would otherwise feed that value into every later maximum
  for (int r = 1; r <= max_iter; ++r) { resid[r] = 0ull; work[r] = 0u; }
  work[0] = 0u;
  r_hist[st->halfsteps % 4096] = st->iters_last;
  st->halfsteps++;
  if (last_of_step) st->steps++;
}

struct CanonArgs {
  GridP g;
  BoxP box;
  const double *src[3];
  double *dst[3];
  const DevState *st;
};

__global__ void __launch_bounds__(NTHREADS) k_canon(const __grid_constant__ CanonArgs a) {
  if (!a.st->last_R_even) return;
  for (int it = blockIdx.x; it < a.box.items; it += gridDim.x) {
    const Item w = decode_item(a.box, it);
    if (!w.active) continue;
    const Column col = make_column(a.g, w.i, w.j);
    int c = a.g.org + w.i + a.g.sy * w.j + a.g.sz * w.k0;
    for (int k = w.k0; k < w.k1; ++k, c += a.g.sz) {
      const bool edge = col.edge_ij || edge_k(a.g, k);
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        const double v = __ldg(a.src[d] + c);
        a.dst[d][c] = v;
        if (edge) {
          if (d == 2) store_images_inl<EXP_LO>(a.dst[d], a.g, w.i, w.j, k, c, v);
          else store_images_inl<EXP_HI>(a.dst[d], a.g, w.i, w.j, k, c, v);
        }
      }
    }
  }
}

// ------------------------------------------------------------------ E update (eq. 11)

// Coefficients of eq. 11 on an edge with permittivity eps and conductivity sig (the
// four-cell means): km = sig/2 - eps/dt, rden = 1 / (sig/2 + eps/dt).  The division of eq. 11 is
// taken as a multiplication by this reciprocal (reading A28): with uniform maps the host
// evaluates the very same expressions once, so folding a uniform map changes no bit.
struct ECoef { double km, rden; };
__host__ __device__ __forceinline__ ECoef e_coef(double eps, double sig, double rdt) {
  const double edt = eps * rdt, hs = 0.5 * sig;
  return {hs - edt, 1.0 / (hs + edt)};
}

struct EArgs {
  GridP g;
  BoxP box;  // the cells this launch updates (the whole grid, or one region of it)
  const double *E[3];  // E^n
  double *Eo[3];       // E^{n+1}: the other E set (out of place)
  const double *H[3];
  const double *eps_r, *sigma;  // cell-centred arrays or nullptr (uniform)
  double eps_u, sigma_u;        // uniform values (eps_u is eps0*eps_r)
  double rdt;                   // 1 / dt
  ECoef k_u;                    // e_coef(eps_u, sigma_u, rdt): the coefficients when both maps are uniform
  SourcesP src;
  const DevState *st;
};

// eq. 11 on a D-edge from its operands: k = the edge's coefficients, J = soft source term, e0 = E^n
// on the edge, (curl H)_D by backward differences: h2 - h2m along d1 = D+1, h1 - h1m along
// d2 = D+2.  A wall-tangential edge stays 0.  Shared by k_e_update and k_eh_stage.
template <int D>
__device__ __forceinline__ double e_edge_val(const GridP &g, const ECoef &k, double J, double e0,
                                             double h2, double h2m, double h1, double h1m, bool wall) {
  constexpr int d1 = (D + 1) % 3, d2 = (D + 2) % 3;
  const double curl = (h2 - h2m) * g.rd[d1] - (h1 - h1m) * g.rd[d2];
  const double e1 = (curl - k.km * e0 - J) * k.rden;
  return wall ? 0.0 : e1;
}

// eq. 11 on the D-edge of the cell at offset c, operands by direct loads
template <int D, bool EPS_ARR, bool SIG_ARR>
__device__ __forceinline__ double e_edge(const EArgs &a, int c, bool wall, double J, double e0,
                                         double h2, double h2m, double h1, double h1m) {
  constexpr int d1 = (D + 1) % 3, d2 = (D + 2) % 3;
  const int s1 = stride_of<d1>(a.g), s2 = stride_of<d2>(a.g);
  // four-cell means of eps, sigma at the edge
  double eps = a.eps_u, sig = a.sigma_u;
  if (EPS_ARR)
    eps = kEps0 * (0.25 * ((__ldg(a.eps_r + c) + __ldg(a.eps_r + c - s1)) +
                           (__ldg(a.eps_r + c - s2) + __ldg(a.eps_r + c - s1 - s2))));
  if (SIG_ARR)
    sig = 0.25 * ((__ldg(a.sigma + c) + __ldg(a.sigma + c - s1)) +
                  (__ldg(a.sigma + c - s2) + __ldg(a.sigma + c - s1 - s2)));
  ECoef k = a.k_u;
  if (EPS_ARR || SIG_ARR) k = e_coef(eps, sig, a.rdt);
  return e_edge_val<D>(a.g, k, J, e0, h2, h2m, h1, h1m, wall);
}

// everything the three edges of one cell read
struct EOps {
  double e0, e1, e2;
  double hx, hy, hz;
  double hx_my, hz_my;  // at j-1
  double hy_mx, hz_mx;  // at i-1
  double hx_mz, hy_mz;  // at k-1
};
__device__ __forceinline__ EOps e_load(const EArgs &a, int c) {
  EOps o;
  o.e0 = __ldg(a.E[0] + c); o.e1 = __ldg(a.E[1] + c); o.e2 = __ldg(a.E[2] + c);
  o.hx = __ldg(a.H[0] + c); o.hy = __ldg(a.H[1] + c); o.hz = __ldg(a.H[2] + c);
  o.hx_my = __ldg(a.H[0] + c - a.g.sy); o.hz_my = __ldg(a.H[2] + c - a.g.sy);
  o.hy_mx = __ldg(a.H[1] + c - 1); o.hz_mx = __ldg(a.H[2] + c - 1);
  o.hx_mz = __ldg(a.H[0] + c - a.g.sz); o.hy_mz = __ldg(a.H[1] + c - a.g.sz);
  return o;
}

// soft sources on the D-edge of cell (i,j,k)
template <int D>
__device__ __forceinline__ double source_term(const EArgs &a, int i, int j, int k) {
  double J = 0.0;
  for (int s = 0; s < a.src.count; ++s) {
    const SourceP &S = a.src.s[s];
    if (S.kind != 0 || S.comp != D) continue;
    if (i < S.lo[0] || i >= S.hi[0] || j < S.lo[1] || j >= S.hi[1] || k < S.lo[2] || k >= S.hi[2])
      continue;
    double p = 1.0;
    if (S.profile) {
      const long long bx = S.hi[0] - S.lo[0], by = S.hi[1] - S.lo[1];
      p = __ldg(S.profile + (i - S.lo[0]) + bx * ((j - S.lo[1]) + by * (long long)(k - S.lo[2])));
    }
    J += a.st->src_amp[s] * p;
  }
  return J;
}

template <bool EPS_ARR, bool SIG_ARR, bool HAS_SRC>
__global__ void __launch_bounds__(NTHREADS, 4) k_e_update(const __grid_constant__ EArgs a) {
  for (int it = blockIdx.x; it < a.box.items; it += gridDim.x) {
    const Item w = decode_item(a.box, it);
    if (!w.active) continue;
    const Column col = make_column(a.g, w.i, w.j);
    int c = a.g.org + w.i + a.g.sy * w.j + a.g.sz * w.k0;
    for (int k = w.k0; k < w.k1; ++k, c += a.g.sz) {
      const EOps o = e_load(a, c);
      double Jx = 0.0, Jy = 0.0, Jz = 0.0;
      if (HAS_SRC) {
        Jx = source_term<0>(a, w.i, w.j, k);
        Jy = source_term<1>(a, w.i, w.j, k);
        Jz = source_term<2>(a, w.i, w.j, k);
      }
      const bool wk = wall_k(a.g, k);
      const double ex = e_edge<0, EPS_ARR, SIG_ARR>(a, c, col.wall[1] || wk, Jx, o.e0, o.hz, o.hz_my, o.hy, o.hy_mz);
      const double ey = e_edge<1, EPS_ARR, SIG_ARR>(a, c, wk || col.wall[0], Jy, o.e1, o.hx, o.hx_mz, o.hz, o.hz_mx);
      const double ez = e_edge<2, EPS_ARR, SIG_ARR>(a, c, col.wall[0] || col.wall[1], Jz, o.e2, o.hy, o.hy_mx, o.hx, o.hx_my);
      a.Eo[0][c] = ex;
      a.Eo[1][c] = ey;
      a.Eo[2][c] = ez;
      if (col.edge_ij || edge_k(a.g, k)) {
        store_images_inl<exp_of_e<0>()>(a.Eo[0], a.g, w.i, w.j, k, c, ex);
        store_images_inl<exp_of_e<1>()>(a.Eo[1], a.g, w.i, w.j, k, c, ey);
        store_images_inl<exp_of_e<2>()>(a.Eo[2], a.g, w.i, w.j, k, c, ez);
      }
    }
  }
}

// source time functions for this step: t = (n + 1/2) dt  (eq. 31)
__global__ void k_step_begin(DevState *st, const __grid_constant__ SourcesP src, double dt) {
  const int s = threadIdx.x;
  if (s >= src.count) return;
  // the time a source is evaluated at: soft E (n+1/2) dt (eq. 11), soft H n dt (the beginning of
  // the step), hard E / hard H (n+1) dt (after their updates)          (reading A25)
  const int kind = src.s[s].kind;
  const double t = ((double)st->steps + (kind == 0 ? 0.5 : (kind == 2 ? 0.0 : 1.0))) * dt;
  const double uu = (t - src.s[s].t0) / src.s[s].tp;
  st->src_amp[s] = src.s[s].amplitude * exp(-0.5 * uu * uu) * cos(2.0 * kPi * src.s[s].f0 * t);
}

// Hard E / soft H / hard H source number `idx` applied to field component F on its box
// (PAPER.md:100): F = amp * profile (hard) or F += dt * amp * profile (soft H).  Wall-tangential E
// edges and wall faces of H stay 0; periodic ghost images are refreshed.
struct BoxSrcArgs {
  GridP g;
  SourceP S;
  int idx;
  double *F;
  const DevState *st;
};
__global__ void k_box_source(const __grid_constant__ BoxSrcArgs a) {
  const SourceP &S = a.S;
  const int bx = S.hi[0] - S.lo[0], by = S.hi[1] - S.lo[1], bz = S.hi[2] - S.lo[2];
  const long long n = (long long)bx * by * bz;
  for (long long q = blockIdx.x * (long long)blockDim.x + threadIdx.x; q < n;
       q += (long long)gridDim.x * blockDim.x) {
    const int i = S.lo[0] + (int)(q % bx), j = S.lo[1] + (int)((q / bx) % by),
              k = S.lo[2] + (int)(q / ((long long)bx * by));
    const int idx[3] = {i, j, k};
    bool wall = false;
    if (S.kind == 1) {  // E edge: tangential to the walls of the two other axes
      for (int d = 0; d < 3; ++d)
        if (d != S.comp && a.g.wall[d] && idx[d] == 0) wall = true;
    } else {            // H face: the wall of its own axis
      wall = a.g.wall[S.comp] && idx[S.comp] == 0;
    }
    if (wall) continue;
    const double v = a.st->src_amp[a.idx] * (S.profile ? __ldg(S.profile + q) : 1.0);
    const int c = a.g.org + i + a.g.sy * j + a.g.sz * k;
    const double out = S.kind == 2 ? a.F[c] + a.g.dt * v : v;
    a.F[c] = out;
    if (S.kind == 1) {  // what the neighbouring slabs read of E: E_x, E_y of the first plane
      if (S.comp == 2) store_images_inl<EXP_NONE>(a.F, a.g, i, j, k, c, out);
      else store_images_inl<EXP_LO>(a.F, a.g, i, j, k, c, out);
    } else {            // of H: H_x, H_y of the last plane, H_z of the first
      if (S.comp == 2) store_images_inl<EXP_LO>(a.F, a.g, i, j, k, c, out);
      else store_images_inl<EXP_HI>(a.F, a.g, i, j, k, c, out);
    }
  }
}

// ------------------------------------------------------------------ open boundary (PML)
// PAPER.md:189 (reading A26): split-field PML with two-step time-centred multiplicative
// damping.  In the layer (the outermost cells of a PEC-backed axis) every component is the sum of
// two parts, one per term of the curl; each part is advanced by the macroscopic update (eq. 11
// with the local eps, sigma; eq. 21 with M = 0 and the local mu) between two multiplications by
// the square root g of its damping factor, g taken along the axis of the derivative in that term
// (dE: E parts at the nodes of that axis, one step; dH: H parts at the half positions, one half
// step).  These kernels run on the layer's slabs AFTER the regular update of the whole grid and
// overwrite the total fields there (every update is out of place, so they see the same inputs).
struct PmlArgs {
  GridP g;
  BoxP box;             // one slab of the layer
  const double *In[3];  // the OTHER field: H^{n+1/2} for the E update, E for the H half-step
  double *Out[3];       // total field of this update's result set
  double *P[6];         // split parts of the updated field: [2 * component + part]
  const double *d[3];   // sqrt damping factors along x, y, z (dE or dH), n[a] entries each
  const double *eps_r, *sigma, *mu_r;  // cell-centred arrays or nullptr (uniform)
  double eps_u, sigma_u, mu_u;
  SourcesP src;         // soft E sources (E update only)
  const DevState *st;
};

template <int D>
__device__ __forceinline__ double pml_e_edge(const PmlArgs &a, int c, const int idx[3], bool wall, double J) {
  constexpr int d1 = (D + 1) % 3, d2 = (D + 2) % 3;
  const int s1 = stride_of<d1>(a.g), s2 = stride_of<d2>(a.g);
  double eps = a.eps_u, sig = a.sigma_u;
  if (a.eps_r)
    eps = kEps0 * (0.25 * ((__ldg(a.eps_r + c) + __ldg(a.eps_r + c - s1)) +
                           (__ldg(a.eps_r + c - s2) + __ldg(a.eps_r + c - s1 - s2))));
  if (a.sigma)
    sig = 0.25 * ((__ldg(a.sigma + c) + __ldg(a.sigma + c - s1)) +
                  (__ldg(a.sigma + c - s2) + __ldg(a.sigma + c - s1 - s2)));
  const double t0 = (__ldg(a.In[d2] + c) - __ldg(a.In[d2] + c - s1)) * a.g.rd[d1];
  const double t1 = -(__ldg(a.In[d1] + c) - __ldg(a.In[d1] + c - s2)) * a.g.rd[d2];
  const double den = 0.5 * sig + eps / a.g.dt, keep = eps / a.g.dt - 0.5 * sig;
  const double g0 = __ldg(a.d[d1] + idx[d1]), g1 = __ldg(a.d[d2] + idx[d2]);
  double p0 = (t0 + keep * (g0 * a.P[2 * D][c]) - J) / den * g0;
  double p1 = (t1 + keep * (g1 * a.P[2 * D + 1][c])) / den * g1;
  if (wall) p0 = p1 = 0.0;
  a.P[2 * D][c] = p0;
  a.P[2 * D + 1][c] = p1;
  return p0 + p1;
}

template <int D>
__device__ __forceinline__ double pml_h_face(const PmlArgs &a, int c, const int idx[3], bool wall) {
  constexpr int d1 = (D + 1) % 3, d2 = (D + 2) % 3;
  const int s1 = stride_of<d1>(a.g), s2 = stride_of<d2>(a.g);
  double mu = a.mu_u;
  if (a.mu_r) mu = kMu0 * (0.5 * (__ldg(a.mu_r + c) + __ldg(a.mu_r + c - stride_of<D>(a.g))));
  const double t0 = (__ldg(a.In[d2] + c + s1) - __ldg(a.In[d2] + c)) * a.g.rd[d1];
  const double t1 = -(__ldg(a.In[d1] + c + s2) - __ldg(a.In[d1] + c)) * a.g.rd[d2];
  const double k = 0.5 * a.g.dt / mu;
  const double g0 = __ldg(a.d[d1] + idx[d1]), g1 = __ldg(a.d[d2] + idx[d2]);
  double p0 = (g0 * a.P[2 * D][c] - k * t0) * g0;
  double p1 = (g1 * a.P[2 * D + 1][c] - k * t1) * g1;
  if (wall) p0 = p1 = 0.0;
  a.P[2 * D][c] = p0;
  a.P[2 * D + 1][c] = p1;
  return p0 + p1;
}

template <bool IS_E>
__global__ void __launch_bounds__(NTHREADS) k_pml(const __grid_constant__ PmlArgs a) {
  for (int it = blockIdx.x; it < a.box.items; it += gridDim.x) {
    const Item w = decode_item(a.box, it);
    if (!w.active) continue;
    const Column col = make_column(a.g, w.i, w.j);
    int c = a.g.org + w.i + a.g.sy * w.j + a.g.sz * w.k0;
    for (int k = w.k0; k < w.k1; ++k, c += a.g.sz) {
      const int idx[3] = {w.i, w.j, k};
      const bool wk = wall_k(a.g, k);
      double v0, v1, v2;
      if (IS_E) {
        // soft E sources reach the layer through part 0 (source_term reads EArgs-like fields)
        double J0 = 0.0, J1 = 0.0, J2 = 0.0;
        for (int q = 0; q < a.src.count; ++q) {
          const SourceP &S = a.src.s[q];
          if (S.kind != 0) continue;
          if (w.i < S.lo[0] || w.i >= S.hi[0] || w.j < S.lo[1] || w.j >= S.hi[1] || k < S.lo[2] || k >= S.hi[2])
            continue;
          double pr = 1.0;
          if (S.profile) {
            const long long bx = S.hi[0] - S.lo[0], by = S.hi[1] - S.lo[1];
            pr = __ldg(S.profile + (w.i - S.lo[0]) + bx * ((w.j - S.lo[1]) + by * (long long)(k - S.lo[2])));
          }
          const double J = a.st->src_amp[q] * pr;
          if (S.comp == 0) J0 += J; else if (S.comp == 1) J1 += J; else J2 += J;
        }
        v0 = pml_e_edge<0>(a, c, idx, col.wall[1] || wk, J0);
        v1 = pml_e_edge<1>(a, c, idx, wk || col.wall[0], J1);
        v2 = pml_e_edge<2>(a, c, idx, col.wall[0] || col.wall[1], J2);
      } else {
        v0 = pml_h_face<0>(a, c, idx, col.wall[0]);
        v1 = pml_h_face<1>(a, c, idx, col.wall[1]);
        v2 = pml_h_face<2>(a, c, idx, wk);
      }
      a.Out[0][c] = v0;
      a.Out[1][c] = v1;
      a.Out[2][c] = v2;
      if (col.edge_ij || edge_k(a.g, k)) {
        store_images_inl<IS_E ? EXP_LO : EXP_HI>(a.Out[0], a.g, w.i, w.j, k, c, v0);
        store_images_inl<IS_E ? EXP_LO : EXP_HI>(a.Out[1], a.g, w.i, w.j, k, c, v1);
        store_images_inl<IS_E ? EXP_NONE : EXP_LO>(a.Out[2], a.g, w.i, w.j, k, c, v2);
      }
    }
  }
}

// ------------------------------------------------------------------ set-up kernels

__device__ __forceinline__ Cell make_cell(const GridP &g, int i, int j, int k) {
  Cell q;
  q.i = i; q.j = j; q.k = k;
  q.c = g.org + i + g.sy * j + g.sz * k;
  return q;
}
template <int D> __device__ __forceinline__ bool wall_face(const GridP &g, const Cell &q) {
  return g.wall[D] && (D == 0 ? q.i : (D == 1 ? q.j : q.k)) == 0;
}
template <int D> __device__ __forceinline__ bool wall_edge(const GridP &g, const Cell &q) {
  constexpr int t1 = (D + 1) % 3, t2 = (D + 2) % 3;
  const int v1 = t1 == 0 ? q.i : (t1 == 1 ? q.j : q.k), v2 = t2 == 0 ? q.i : (t2 == 1 ? q.j : q.k);
  return (g.wall[t1] && v1 == 0) || (g.wall[t2] && v2 == 0);
}

// ghost layer of one array: periodic axes mirror the opposite interior plane, PEC ghosts are 0;
// the ghost plane of a slab interface keeps what the caller put there (the neighbour's plane)
__global__ void k_fill_ghosts(double *__restrict__ a, const __grid_constant__ GridP g) {
  const long long px = g.n[0] + 2, py = g.n[1] + 2, pz = g.n[2] + 2;
  const long long total = px * py * pz;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const int idx[3] = {(int)(t % px) - 1, (int)((t / px) % py) - 1, (int)(t / (px * py)) - 1};
    int src[3];
    bool ghost = false, zero = false;
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      src[d] = idx[d];
      if (idx[d] < 0 || idx[d] >= g.n[d]) {
        if (d == 2 && g.ext[idx[d] < 0 ? 0 : 1]) continue;
        ghost = true;
        if (g.per[d]) src[d] = idx[d] < 0 ? g.n[d] - 1 : 0; else zero = true;
      }
    }
    if (!ghost) continue;
    const int dst = g.org + idx[0] + g.sy * idx[1] + g.sz * idx[2];
    a[dst] = zero ? 0.0 : a[g.org + src[0] + g.sy * src[1] + g.sz * src[2]];
  }
}

struct FieldsP {
  GridP g;
  double *E[3];
  double *H[3];
};

// zero tangential E and normal H on PEC walls
__global__ void k_enforce_walls(const __grid_constant__ FieldsP a) {
  // the ghost planes of slab interfaces hold the neighbours' values: the x / y walls cut them too
  const long long total = (long long)a.g.n[0] * a.g.n[1] * (a.g.n[2] + a.g.ext[0] + a.g.ext[1]);
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const Cell q = make_cell(a.g, (int)(t % a.g.n[0]), (int)((t / a.g.n[0]) % a.g.n[1]),
                             (int)(t / ((long long)a.g.n[0] * a.g.n[1])) - a.g.ext[0]);
    if (wall_edge<0>(a.g, q)) a.E[0][q.c] = 0.0;
    if (wall_edge<1>(a.g, q)) a.E[1][q.c] = 0.0;
    if (wall_edge<2>(a.g, q)) a.E[2][q.c] = 0.0;
    if (wall_face<0>(a.g, q)) a.H[0][q.c] = 0.0;
    if (wall_face<1>(a.g, q)) a.H[1][q.c] = 0.0;
    if (wall_face<2>(a.g, q)) a.H[2][q.c] = 0.0;
  }
}

struct InitMP {
  GridP g;
  const double *Mc[3];  // cell-centred initial M in the device layout, ghosts filled (nullptr = 0)
  double *M[9];         // face M out
  const double *Ms;     // array or nullptr
  double Ms_u;
  int enable_llg;
  DevState *st;
};

// cell-centred M averaged to faces; renormalised to the face's Ms (A11)
__global__ void k_init_m(const __grid_constant__ InitMP a) {
  const long long total = (long long)a.g.n[0] * a.g.n[1] * a.g.n[2];
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < total;
       t += (long long)gridDim.x * blockDim.x) {
    const Cell q = make_cell(a.g, (int)(t % a.g.n[0]), (int)((t / a.g.n[0]) % a.g.n[1]),
                             (int)(t / ((long long)a.g.n[0] * a.g.n[1])));
    const int st[3] = {1, a.g.sy, a.g.sz};
    const bool wall[3] = {wall_face<0>(a.g, q), wall_face<1>(a.g, q), wall_face<2>(a.g, q)};
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      double m[3] = {0.0, 0.0, 0.0};
      if (a.enable_llg && !wall[d]) {
        const int cm = q.c - st[d];
        double Msf = a.Ms_u;
        if (a.Ms) Msf = 0.5 * (a.Ms[q.c] + a.Ms[cm]);
        if (Msf > 0.0) {
          double v[3];
#pragma unroll
          for (int p = 0; p < 3; ++p) v[p] = a.Mc[p] ? 0.5 * (a.Mc[p][q.c] + a.Mc[p][cm]) : 0.0;
          const double nrm = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
          if (nrm > 0.0) {
            const double sc = Msf / nrm;
#pragma unroll
            for (int p = 0; p < 3; ++p) m[p] = v[p] * sc;
          } else {
            a.st->init_error = 1;
          }
        }
      }
#pragma unroll
      for (int p = 0; p < 3; ++p) a.M[3 * d + p][q.c] = m[p];
    }
  }
}

// min / max of a COMPACT user array: per-block partials, finished on the host
__global__ void k_minmax(const double *__restrict__ a, long long n, double *__restrict__ part) {
  double lo = INFINITY, hi = -INFINITY;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
       t += (long long)gridDim.x * blockDim.x) {
    const double v = a[t];
    lo = fmin(lo, v);
    hi = fmax(hi, v);
    if (v != v) { lo = v; hi = v; }
  }
  __shared__ double slo[256], shi[256];
  slo[threadIdx.x] = lo;
  shi[threadIdx.x] = hi;
  __syncthreads();
  for (int o = 128; o > 0; o >>= 1) {
    if ((int)threadIdx.x < o) {
      const double l2 = slo[threadIdx.x + o], h2 = shi[threadIdx.x + o];
      if (l2 != l2 || l2 < slo[threadIdx.x]) slo[threadIdx.x] = l2;
      if (h2 != h2 || h2 > shi[threadIdx.x]) shi[threadIdx.x] = h2;
    }
    __syncthreads();
  }
  if (threadIdx.x == 0) {
    part[2 * blockIdx.x] = slo[0];
    part[2 * blockIdx.x + 1] = shi[0];
  }
}

// bounding box and count of the cells with Ms > 0 (Ms in the device layout):
// box = {lo x,y,z, hi x,y,z (inclusive)}, count
__global__ void k_mag_box(const double *__restrict__ Ms, const __grid_constant__ GridP g, int *box,
                          unsigned long long *count) {
  // the neighbours' adjacent planes (ghost planes of slab interfaces) count for the box: their
  // magnetic cells make faces of this slab magnetic or read this slab's H (k = -1 and k = nz)
  const long long n = (long long)g.n[0] * g.n[1] * (g.n[2] + g.ext[0] + g.ext[1]);
  int lo[3] = {INT_MAX, INT_MAX, INT_MAX}, hi[3] = {INT_MIN, INT_MIN, INT_MIN};
  unsigned long long cnt = 0;
  bool any = false;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
       t += (long long)gridDim.x * blockDim.x) {
    const int i = (int)(t % g.n[0]), j = (int)((t / g.n[0]) % g.n[1]),
              k = (int)(t / ((long long)g.n[0] * g.n[1])) - g.ext[0];
    if (Ms[g.org + i + g.sy * j + g.sz * k] > 0.0) {
      lo[0] = min(lo[0], i); lo[1] = min(lo[1], j); lo[2] = min(lo[2], k);
      hi[0] = max(hi[0], i); hi[1] = max(hi[1], j); hi[2] = max(hi[2], k);
      any = true;
      if (k >= 0 && k < g.n[2]) ++cnt;   // the slab's own magnetic cells (statistics)
    }
  }
  if (any) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      atomicMin(box + d, lo[d]);
      atomicMax(box + 3 + d, hi[d]);
    }
    atomicAdd(count, cnt);
  }
}

}  // namespace fl
