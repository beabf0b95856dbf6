// kernels.cuh -- sm_100a device code of the coupled FDTD-LLG step (fp64, HBM-bound stencils).
//
// Citations are /root/reference/PAPER.md lines of arXiv 2103.12819.  Layout and staggering:
// include/fdtd_llg.h.  No ghost cells: periodic wrap and PEC walls are resolved per thread as
// neighbour OFFSETS with a validity bit (a read beyond a PEC wall is the constant 0).
//
// Kernels
//   k_h_update   Maxwell (H) half-step on every face OUTSIDE the LLG sweep box   eq. 21 with M = 0
//   k_hm_sweep   one Jacobi iterate r of the trapezoidal LLG solve + eq. 21 inside the sweep box
//   k_half_end   1 thread: iteration count / statistics from the residual words, re-arm them
//   k_canon      copies H^R into the canonical buffer when R is even
//   k_e_update   eq. 11 with in-kernel edge means of eps_r, sigma and the soft sources
//   k_step_begin source amplitudes g_s((n+1/2) dt) for this step
//   set-up: k_enforce_walls, k_init_m, k_minmax, k_mag_box
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

namespace fl {

constexpr int MAX_SOURCES = 8;
constexpr int BX = 32, BY = 4, BZ = 2;  // thread block = BX x BY x BZ cells, x fastest
constexpr int NTHREADS = BX * BY * BZ;

constexpr double kPi = 3.14159265358979323846;
constexpr double kMu0 = 4.0e-7 * kPi;
constexpr double kC0 = 299792458.0;
constexpr double kEps0 = 1.0 / (kMu0 * kC0 * kC0);

struct GridP {
  int n[3];        // nx, ny, nz
  int per[3];      // 1 = periodic, 0 = PEC
  long long s[3];  // element strides 1, nx, nx*ny
  double rd[3];    // 1/dx, 1/dy, 1/dz
  double dt;
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
  double resid_last;
  double src_amp[MAX_SOURCES];
};

struct SourceP {
  int comp;
  int lo[3], hi[3];
  const double *profile;  // device, box sized, or nullptr
  double amplitude, f0, t0, tp;
};

struct SourcesP {
  int count;
  SourceP s[MAX_SOURCES];
};

// per-thread neighbourhood: centre index, wrapped neighbour offsets and their validity
struct Stencil {
  int idx[3];
  long long c;
  long long m[3], p[3];  // offset (elements) to the -1 / +1 neighbour along each axis
  bool vm[3], vp[3];     // false: beyond a PEC wall (value 0)
};

__device__ __forceinline__ Stencil make_stencil(const GridP &g, int i, int j, int k) {
  Stencil st;
  st.idx[0] = i; st.idx[1] = j; st.idx[2] = k;
  st.c = (long long)i + g.s[1] * j + g.s[2] * k;
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    const int v = st.idx[d], n = g.n[d];
    st.vm[d] = (v > 0) || g.per[d];
    st.vp[d] = (v < n - 1) || g.per[d];
    st.m[d] = (v > 0) ? -g.s[d] : g.s[d] * (long long)(n - 1);
    st.p[d] = (v < n - 1) ? g.s[d] : -g.s[d] * (long long)(n - 1);
  }
  return st;
}

__device__ __forceinline__ double ldv(const double *__restrict__ a, long long at, bool ok) {
  return ok ? __ldg(a + at) : 0.0;
}

__device__ __forceinline__ bool wall_face(const GridP &g, const Stencil &st, int d) {
  return !g.per[d] && st.idx[d] == 0;
}
__device__ __forceinline__ bool wall_edge(const GridP &g, const Stencil &st, int d) {
  const int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  return (!g.per[t1] && st.idx[t1] == 0) || (!g.per[t2] && st.idx[t2] == 0);
}

// (curl E)_D at the D-face: forward differences (standard Yee)
template <int D>
__device__ __forceinline__ double curl_e(const GridP &g, const Stencil &st,
                                         const double *const *E) {
  constexpr int d1 = (D + 1) % 3, d2 = (D + 2) % 3;
  const double a0 = __ldg(E[d2] + st.c), a1 = ldv(E[d2], st.c + st.p[d1], st.vp[d1]);
  const double b0 = __ldg(E[d1] + st.c), b1 = ldv(E[d1], st.c + st.p[d2], st.vp[d2]);
  return (a1 - a0) * g.rd[d1] - (b1 - b0) * g.rd[d2];
}

// transverse component T of H at the D-face: four-point average
template <int D, int T>
__device__ __forceinline__ double avg4(const Stencil &st, const double *__restrict__ Ht) {
  const double v00 = __ldg(Ht + st.c);
  const double v10 = ldv(Ht, st.c + st.m[D], st.vm[D]);
  const double v01 = ldv(Ht, st.c + st.p[T], st.vp[T]);
  const double v11 = ldv(Ht, st.c + st.m[D] + st.p[T], st.vm[D] && st.vp[T]);
  return 0.25 * ((v00 + v10) + (v01 + v11));
}

// ------------------------------------------------------------------ Maxwell H half-step

struct HArgs {
  GridP g;
  const double *E[3];
  const double *Hn[3];
  double *Hc[3];
  const double *mu_r;  // cell-centred array or nullptr (uniform)
  double ch_uniform;   // dt / (2 mu0 mu_r) when uniform
  int has_box;
  int lo[3], hi[3];    // LLG sweep box (cells handled by k_hm_sweep), excluded here
};

template <int D, bool MU_ARR>
__device__ __forceinline__ void h_face(const HArgs &a, const Stencil &st) {
  if (wall_face(a.g, st, D)) return;  // stays 0
  double ch = a.ch_uniform;
  if (MU_ARR) {
    const double mu = 0.5 * (__ldg(a.mu_r + st.c) + __ldg(a.mu_r + st.c + st.m[D]));
    ch = a.g.dt / (2.0 * kMu0 * mu);
  }
  const double C = curl_e<D>(a.g, st, a.E);
  a.Hc[D][st.c] = __ldg(a.Hn[D] + st.c) - ch * C;  // eq. 21 with M = 0, local mu
}

template <bool MU_ARR>
__global__ void __launch_bounds__(NTHREADS) k_h_update(const __grid_constant__ HArgs a) {
  const int i = blockIdx.x * BX + threadIdx.x;
  const int j = blockIdx.y * BY + threadIdx.y;
  const int k = blockIdx.z * BZ + threadIdx.z;
  if (i >= a.g.n[0] || j >= a.g.n[1] || k >= a.g.n[2]) return;
  if (a.has_box && i >= a.lo[0] && i < a.hi[0] && j >= a.lo[1] && j < a.hi[1] && k >= a.lo[2] &&
      k < a.hi[2])
    return;
  const Stencil st = make_stencil(a.g, i, j, k);
  h_face<0, MU_ARR>(a, st);
  h_face<1, MU_ARR>(a, st);
  h_face<2, MU_ARR>(a, st);
}

// ------------------------------------------------------------------ LLG sweep

struct HMArgs {
  GridP g;
  const double *E[3];
  const double *Hn[3];  // H^n
  const double *Hp[3];  // H^{r-1}  (== Hn when FIRST)
  double *Hc[3];        // H^r
  const double *Mn[9];  // M^n      [face*3 + comp]
  double *Mr[9];        // M^{r-1} in, M^r out (same thread); FIRST: out only
  const double *Ms, *alpha, *gamma, *mu_r;  // cell-centred arrays or nullptr (uniform)
  double Ms_u, alpha_u, gamma_u, ch_uniform;
  double hb[3], hk, u[3];
  double tol;
  int lo[3], hi[3];
  unsigned long long *resid;  // [max_iter + 1] bit patterns of the residual of iterate r
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
__device__ __forceinline__ Vec3 h_em(const Stencil &st, const double *const *H) {
  Vec3 h;
  if (D == 0) {
    h.x = __ldg(H[0] + st.c); h.y = avg4<0, 1>(st, H[1]); h.z = avg4<0, 2>(st, H[2]);
  } else if (D == 1) {
    h.x = avg4<1, 0>(st, H[0]); h.y = __ldg(H[1] + st.c); h.z = avg4<1, 2>(st, H[2]);
  } else {
    h.x = avg4<2, 0>(st, H[0]); h.y = avg4<2, 1>(st, H[1]); h.z = __ldg(H[2] + st.c);
  }
  return h;
}

// One Jacobi iterate on the D-face of this thread's cell.  Returns the face's residual
// max_c |M^r_c - M^{r-1}_c| / Ms_f (0 on non-magnetic faces).
template <int D, bool FIRST, bool MS_ARR, bool AG_ARR, bool MU_ARR, bool ANISO>
__device__ __forceinline__ double hm_face(const HMArgs &a, const Stencil &st) {
  if (wall_face(a.g, st, D)) return 0.0;  // H = 0, M = 0 for ever (reading A13)
  const long long c = st.c, cm = st.c + st.m[D];
  double Msf = a.Ms_u;
  if (MS_ARR) Msf = 0.5 * (__ldg(a.Ms + c) + __ldg(a.Ms + cm));
  if (!(Msf > 0.0)) {
    // non-magnetic face inside the sweep box: Maxwell update at r = 1, copy afterwards so that
    // both Jacobi buffers hold it
    if (FIRST) {
      double ch = a.ch_uniform;
      if (MU_ARR) ch = a.g.dt / (2.0 * kMu0 * (0.5 * (__ldg(a.mu_r + c) + __ldg(a.mu_r + cm))));
      a.Hc[D][c] = __ldg(a.Hn[D] + c) - ch * curl_e<D>(a.g, st, a.E);
    } else {
      a.Hc[D][c] = __ldg(a.Hp[D] + c);
    }
    return 0.0;
  }
  double alf = a.alpha_u, gam = a.gamma_u;
  if (AG_ARR) {
    alf = 0.5 * (__ldg(a.alpha + c) + __ldg(a.alpha + cm));
    gam = 0.5 * (fabs(__ldg(a.gamma + c)) + fabs(__ldg(a.gamma + cm)));  // |gamma| (eqs. 19-20)
  }
  const double cf = kMu0 * gam * a.g.dt * 0.25;  // mu0 |gamma| dt / 4
  const double rMs = 1.0 / Msf;
  const Vec3 hb = {a.hb[0], a.hb[1], a.hb[2]};
  const Vec3 u = {a.u[0], a.u[1], a.u[2]};

  const Vec3 mn = {__ldg(a.Mn[3 * D + 0] + c), __ldg(a.Mn[3 * D + 1] + c),
                   __ldg(a.Mn[3 * D + 2] + c)};
  // H_eff^n = H_EM^n + H_bias + H_k (M^n.u / Ms) u            (A19)
  Vec3 hn = h_em<D>(st, a.Hn);
  hn.x += hb.x; hn.y += hb.y; hn.z += hb.z;
  if (ANISO) {
    const double p = a.hk * (dot(mn, u) * rMs);
    hn.x += p * u.x; hn.y += p * u.y; hn.z += p * u.z;
  }
  // H_eff^{r-1}, lagged; at r = 1 it is H_eff^n
  Vec3 he = hn, mp = mn;
  if (!FIRST) {
    mp = {a.Mr[3 * D + 0][c], a.Mr[3 * D + 1][c], a.Mr[3 * D + 2][c]};
    he = h_em<D>(st, a.Hp);
    he.x += hb.x; he.y += hb.y; he.z += hb.z;
    if (ANISO) {
      const double p = a.hk * (dot(mp, u) * rMs);
      he.x += p * u.x; he.y += p * u.y; he.z += p * u.z;
    }
  }
  // eqs. 18-20 in increment form (A24):  b = M^n + beta,  tau = a x M^n
  const Vec3 t0 = cross(mn, hn);
  const Vec3 beta = {-cf * t0.x, -cf * t0.y, -cf * t0.z};
  const Vec3 t1 = cross(mn, he);
  const Vec3 tau = {cf * t1.x, cf * t1.y, cf * t1.z};
  const double aM = alf * rMs;
  const Vec3 av = {-(cf * he.x + aM * mn.x), -(cf * he.y + aM * mn.y), -(cf * he.z + aM * mn.z)};  // (19)
  const Vec3 axt = cross(av, tau), axb = cross(av, beta);
  const double ab = dot(av, beta);
  const double rden = 1.0 / (1.0 + dot(av, av));
  const Vec3 De = {(beta.x - tau.x + axt.x + ab * av.x - axb.x) * rden,
                   (beta.y - tau.y + axt.y + ab * av.y - axb.y) * rden,
                   (beta.z - tau.z + axt.z + ab * av.z - axb.z) * rden};  // (18) - M^n
  // renormalisation N(M) applied to the increment
  const double x = (2.0 * dot(mn, De) + dot(De, De)) * (rMs * rMs);
  const double sq = sqrt(1.0 + x);
  const double sm1 = -x / (sq * (1.0 + sq));  // Ms/|M^n + Delta| - 1
  const Vec3 dM = {De.x + sm1 * (mn.x + De.x), De.y + sm1 * (mn.y + De.y),
                   De.z + sm1 * (mn.z + De.z)};
  const Vec3 mr = {mn.x + dM.x, mn.y + dM.y, mn.z + dM.z};
  a.Mr[3 * D + 0][c] = mr.x;
  a.Mr[3 * D + 1][c] = mr.y;
  a.Mr[3 * D + 2][c] = mr.z;
  // eq. 21, normal component:  H^r = H^n + M^n - M^r - (dt / 2 mu0) curl E
  const double C = curl_e<D>(a.g, st, a.E);
  a.Hc[D][c] = __ldg(a.Hn[D] + c) - comp<D>(dM) - (a.g.dt / (2.0 * kMu0)) * C;
  // stopping test of PAPER.md:154, per face; reduced by the caller
  const double e = fmax(fmax(fabs(mr.x - mp.x), fabs(mr.y - mp.y)), fabs(mr.z - mp.z));
  return e * rMs;
}

template <bool FIRST, bool MS_ARR, bool AG_ARR, bool MU_ARR, bool ANISO>
__global__ void __launch_bounds__(NTHREADS) k_hm_sweep(const __grid_constant__ HMArgs a) {
  // the whole grid takes the same decision: iterate r runs iff iterate r-1 was not converged
  if (!FIRST) {
    if (__longlong_as_double((long long)a.resid[a.r - 1]) < a.tol) return;
  }
  const int i = a.lo[0] + blockIdx.x * BX + threadIdx.x;
  const int j = a.lo[1] + blockIdx.y * BY + threadIdx.y;
  const int k = a.lo[2] + blockIdx.z * BZ + threadIdx.z;
  double res = 0.0;
  if (i < a.hi[0] && j < a.hi[1] && k < a.hi[2]) {
    const Stencil st = make_stencil(a.g, i, j, k);
    res = hm_face<0, FIRST, MS_ARR, AG_ARR, MU_ARR, ANISO>(a, st);
    res = fmax(res, hm_face<1, FIRST, MS_ARR, AG_ARR, MU_ARR, ANISO>(a, st));
    res = fmax(res, hm_face<2, FIRST, MS_ARR, AG_ARR, MU_ARR, ANISO>(a, st));
  }
  // convergence word: warp shuffles, then ONE atomic per block
#pragma unroll
  for (int o = 16; o > 0; o >>= 1) res = fmax(res, __shfl_xor_sync(0xffffffffu, res, o));
  __shared__ double wmax[NTHREADS / 32];
  const int tid = threadIdx.x + BX * (threadIdx.y + BY * threadIdx.z);
  if ((tid & 31) == 0) wmax[tid >> 5] = res;
  __syncthreads();
  if (tid == 0) {
    double m = wmax[0];
#pragma unroll
    for (int w = 1; w < NTHREADS / 32; ++w) m = fmax(m, wmax[w]);
    if (m > 0.0) atomicMax(a.resid + a.r, (unsigned long long)__double_as_longlong(m));
  }
}

// 1 thread: close an (H,M) half-step
__global__ void k_half_end(DevState *st, unsigned long long *resid, int max_iter, double tol,
                           int any_magnetic, int last_of_step) {
  if (any_magnetic) {
    int R = max_iter;
    for (int r = 1; r <= max_iter; ++r)
      if (__longlong_as_double((long long)resid[r]) < tol) { R = r; break; }
    const double res = __longlong_as_double((long long)resid[R]);
    if (!(res < tol)) st->nonconverged++;
    st->iters_last = R;
    st->iters_total += R;
    if (R > st->iters_max) st->iters_max = R;
    st->resid_last = res;
    st->last_R_even = ((R & 1) == 0);
    for (int r = 1; r <= max_iter; ++r) resid[r] = 0ull;
  } else {
    st->iters_last = 0;
    st->last_R_even = 0;
  }
  st->halfsteps++;
  if (last_of_step) st->steps++;
}

struct CanonArgs {
  GridP g;
  const double *src[3];
  double *dst[3];
  int lo[3], hi[3];
  const DevState *st;
};

__global__ void __launch_bounds__(NTHREADS) k_canon(const __grid_constant__ CanonArgs a) {
  if (!a.st->last_R_even) return;
  const int i = a.lo[0] + blockIdx.x * BX + threadIdx.x;
  const int j = a.lo[1] + blockIdx.y * BY + threadIdx.y;
  const int k = a.lo[2] + blockIdx.z * BZ + threadIdx.z;
  if (i >= a.hi[0] || j >= a.hi[1] || k >= a.hi[2]) return;
  const long long c = (long long)i + a.g.s[1] * j + a.g.s[2] * k;
#pragma unroll
  for (int d = 0; d < 3; ++d) a.dst[d][c] = __ldg(a.src[d] + c);
}

// ------------------------------------------------------------------ E update (eq. 11)

struct EArgs {
  GridP g;
  double *E[3];
  const double *H[3];
  const double *eps_r, *sigma;  // cell-centred arrays or nullptr (uniform)
  double eps_u, sigma_u;        // uniform values (eps_u is eps0*eps_r)
  SourcesP src;
  const DevState *st;
};

template <int D, bool EPS_ARR, bool SIG_ARR, bool HAS_SRC>
__device__ __forceinline__ void e_edge(const EArgs &a, const Stencil &st) {
  if (wall_edge(a.g, st, D)) return;  // tangential E on a PEC wall stays 0
  constexpr int d1 = (D + 1) % 3, d2 = (D + 2) % 3;
  const long long c = st.c;
  // (curl H)_D at the D-edge: backward differences
  const double h2 = __ldg(a.H[d2] + c), h2m = ldv(a.H[d2], c + st.m[d1], st.vm[d1]);
  const double h1 = __ldg(a.H[d1] + c), h1m = ldv(a.H[d1], c + st.m[d2], st.vm[d2]);
  const double curl = (h2 - h2m) * a.g.rd[d1] - (h1 - h1m) * a.g.rd[d2];
  // four-cell means of eps, sigma at the edge
  double eps = a.eps_u, sig = a.sigma_u;
  const long long c1 = c + st.m[d1], c2 = c + st.m[d2], c12 = c + st.m[d1] + st.m[d2];
  if (EPS_ARR)
    eps = kEps0 * (0.25 * ((__ldg(a.eps_r + c) + __ldg(a.eps_r + c1)) +
                           (__ldg(a.eps_r + c2) + __ldg(a.eps_r + c12))));
  if (SIG_ARR)
    sig = 0.25 * ((__ldg(a.sigma + c) + __ldg(a.sigma + c1)) +
                  (__ldg(a.sigma + c2) + __ldg(a.sigma + c12)));
  double J = 0.0;
  if (HAS_SRC) {
    for (int s = 0; s < a.src.count; ++s) {
      const SourceP &S = a.src.s[s];
      if (S.comp != D) continue;
      if (st.idx[0] < S.lo[0] || st.idx[0] >= S.hi[0] || st.idx[1] < S.lo[1] ||
          st.idx[1] >= S.hi[1] || st.idx[2] < S.lo[2] || st.idx[2] >= S.hi[2])
        continue;
      double p = 1.0;
      if (S.profile) {
        const long long bx = S.hi[0] - S.lo[0], by = S.hi[1] - S.lo[1];
        p = __ldg(S.profile + (st.idx[0] - S.lo[0]) +
                  bx * ((st.idx[1] - S.lo[1]) + by * (long long)(st.idx[2] - S.lo[2])));
      }
      J += a.st->src_amp[s] * p;
    }
  }
  const double edt = eps / a.g.dt, hs = 0.5 * sig;
  const double e0 = a.E[D][c];
  a.E[D][c] = (curl - (hs - edt) * e0 - J) / (hs + edt);  // eq. 11
}

template <bool EPS_ARR, bool SIG_ARR, bool HAS_SRC>
__global__ void __launch_bounds__(NTHREADS) k_e_update(const __grid_constant__ EArgs a) {
  const int i = blockIdx.x * BX + threadIdx.x;
  const int j = blockIdx.y * BY + threadIdx.y;
  const int k = blockIdx.z * BZ + threadIdx.z;
  if (i >= a.g.n[0] || j >= a.g.n[1] || k >= a.g.n[2]) return;
  const Stencil st = make_stencil(a.g, i, j, k);
  e_edge<0, EPS_ARR, SIG_ARR, HAS_SRC>(a, st);
  e_edge<1, EPS_ARR, SIG_ARR, HAS_SRC>(a, st);
  e_edge<2, EPS_ARR, SIG_ARR, HAS_SRC>(a, st);
}

// source time functions for this step: t = (n + 1/2) dt  (eq. 31)
__global__ void k_step_begin(DevState *st, const __grid_constant__ SourcesP src, double dt) {
  const int s = threadIdx.x;
  if (s >= src.count) return;
  const double t = ((double)st->steps + 0.5) * dt;
  const double uu = (t - src.s[s].t0) / src.s[s].tp;
  st->src_amp[s] = src.s[s].amplitude * exp(-0.5 * uu * uu) * cos(2.0 * kPi * src.s[s].f0 * t);
}

// ------------------------------------------------------------------ set-up kernels

struct FieldsP {
  GridP g;
  double *E[3];
  double *H[3];
};

// zero tangential E and normal H on PEC walls
__global__ void __launch_bounds__(NTHREADS) k_enforce_walls(const __grid_constant__ FieldsP a) {
  const int i = blockIdx.x * BX + threadIdx.x;
  const int j = blockIdx.y * BY + threadIdx.y;
  const int k = blockIdx.z * BZ + threadIdx.z;
  if (i >= a.g.n[0] || j >= a.g.n[1] || k >= a.g.n[2]) return;
  const Stencil st = make_stencil(a.g, i, j, k);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    if (wall_edge(a.g, st, d)) a.E[d][st.c] = 0.0;
    if (wall_face(a.g, st, d)) a.H[d][st.c] = 0.0;
  }
}

struct InitMP {
  GridP g;
  const double *Mc[3];  // cell-centred initial M (nullptr = 0)
  double *M[9];         // face M out
  const double *Ms;     // array or nullptr
  double Ms_u;
  int enable_llg;
  DevState *st;
};

// cell-centred M averaged to faces; renormalised to the face's Ms (A11)
__global__ void __launch_bounds__(NTHREADS) k_init_m(const __grid_constant__ InitMP a) {
  const int i = blockIdx.x * BX + threadIdx.x;
  const int j = blockIdx.y * BY + threadIdx.y;
  const int k = blockIdx.z * BZ + threadIdx.z;
  if (i >= a.g.n[0] || j >= a.g.n[1] || k >= a.g.n[2]) return;
  const Stencil st = make_stencil(a.g, i, j, k);
#pragma unroll
  for (int d = 0; d < 3; ++d) {
    double m[3] = {0.0, 0.0, 0.0};
    if (a.enable_llg && !wall_face(a.g, st, d)) {
      const long long cm = st.c + st.m[d];
      double Msf = a.Ms_u;
      if (a.Ms) Msf = 0.5 * (a.Ms[st.c] + a.Ms[cm]);
      if (Msf > 0.0) {
        double v[3];
#pragma unroll
        for (int q = 0; q < 3; ++q) v[q] = a.Mc[q] ? 0.5 * (a.Mc[q][st.c] + a.Mc[q][cm]) : 0.0;
        const double nrm = sqrt(v[0] * v[0] + v[1] * v[1] + v[2] * v[2]);
        if (nrm > 0.0) {
          const double sc = Msf / nrm;
#pragma unroll
          for (int q = 0; q < 3; ++q) m[q] = v[q] * sc;
        } else {
          a.st->init_error = 1;
        }
      }
    }
#pragma unroll
    for (int q = 0; q < 3; ++q) a.M[3 * d + q][st.c] = m[q];
  }
}

// min / max of an array: per-block partials, finished on the host
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

// bounding box and count of the cells with Ms > 0: out = {lo x,y,z, hi x,y,z (inclusive)}, count
__global__ void k_mag_box(const double *__restrict__ Ms, GridP g, int *box,
                          unsigned long long *count) {
  const long long n = (long long)g.n[0] * g.n[1] * g.n[2];
  int lo[3] = {INT_MAX, INT_MAX, INT_MAX}, hi[3] = {-1, -1, -1};
  unsigned long long cnt = 0;
  for (long long t = blockIdx.x * (long long)blockDim.x + threadIdx.x; t < n;
       t += (long long)gridDim.x * blockDim.x) {
    if (Ms[t] > 0.0) {
      const int i = (int)(t % g.n[0]), j = (int)((t / g.n[0]) % g.n[1]),
                k = (int)(t / ((long long)g.n[0] * g.n[1]));
      lo[0] = min(lo[0], i); lo[1] = min(lo[1], j); lo[2] = min(lo[2], k);
      hi[0] = max(hi[0], i); hi[1] = max(hi[1], j); hi[2] = max(hi[2], k);
      ++cnt;
    }
  }
  if (cnt) {
#pragma unroll
    for (int d = 0; d < 3; ++d) {
      atomicMin(box + d, lo[d]);
      atomicMax(box + 3 + d, hi[d]);
    }
    atomicAdd(count, cnt);
  }
}

}  // namespace fl
