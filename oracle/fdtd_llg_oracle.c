/*
 * fdtd_llg_oracle.c -- CPU ORACLE for the coupled FDTD-LLG time step.
 *
 * THIS FILE IS TEST INFRASTRUCTURE.  It is the plain, slow, obviously-correct
 * statement of what the hot path computes.  Only tests/, __graft_entry__.smoke()
 * and bench.py's cpu_baseline / --impl reference legs may build, load or call
 * it.  It shares no code, header, table or helper with the CUDA path under
 * paper_2103_12819_b200/csrc/ and neither includes the other.
 *
 * What it follows (citations are /root/reference/PAPER.md lines of
 * arXiv 2103.12819, Yao, Jambunathan, Zeng, Nonaka):
 *   - Yee staggering, M (all 3 components) on every face, four-point transverse
 *     averages, cell-centred materials averaged to edges/faces   PAPER.md:82-90 (S3.1)
 *   - step order  HM half-step -> E update -> HM half-step
 *   - E update, eq. 11
 *   - iterated trapezoidal LLG solve, eqs. 18-21, renormalisation N(M),
 *     global stopping test max|M^r - M^{r-1}|/Ms < tol
 *   - non-magnetic faces: eq. 21 with M = 0 and the local mu
 *   - periodic and PEC boundaries
 *   - soft current source J_src^{n+1/2} in eq. 11, envelope eq. 31
 * Readings of silent/ambiguous points are the A-numbers of DESIGN.md (S "Readings").
 *
 * Pins (tests/test_oracle_pins.py, all -m "not gpu"): exact Yee eigenmode /
 * numerical dispersion, exact leapfrog energy invariant, PEC cavity mode,
 * sigma recurrence, exact Cayley (trapezoidal) Larmor rotation, damping rate,
 * anisotropy rotation, |M| = Ms, div(H+M) invariant, eq. 15 residual,
 * second-order convergence rates of PAPER.md Tab. 2, PEC reflection = -1,
 * brute force on 8^3 against a structurally different numpy implementation.
 * Parity unpinned by the paper (oracle <-> GPU agreement only): A13 (M on PEC
 * wall faces), A15 (bandwidth -> T_p, source amplitude), A2 (norm of the stop
 * test), A4 (behaviour at the iteration cap), A11 (renormalising averaged M0).
 *
 * Two builds of this one file:
 *   default                      : REAL = double, LLG solve evaluated in the
 *                                  cancellation-free INCREMENT form (DESIGN.md
 *                                  reading A24) -- this is the parity reference.
 *   -DORACLE_LITERAL -DREAL="long double" -DORC_PREFIX=oracle_ld_ :
 *                                  eqs. 18-21 evaluated exactly as printed, state
 *                                  held in 80-bit -- the fidelity cross-check
 *                                  that the increment form is the paper's algorithm.
 *
 * Conventions.  nx*ny*nz cells, x fastest: idx = i + nx*(j + ny*k).  Entry
 * (i,j,k) of an array is the edge / face on the LOW side of cell (i,j,k):
 *   Ex (i+1/2,j,k)  Ey (i,j+1/2,k)  Ez (i,j,k+1/2)          edges
 *   Hx (i,j+1/2,k+1/2) Hy (i+1/2,j,k+1/2) Hz (i+1/2,j+1/2,k) faces
 *   M[d][c] : component c of M on the d-face, same place as H_d
 *   materials at cell centres (i+1/2,j+1/2,k+1/2).
 * Axis boundary bc[d]: 0 = PEC, 1 = periodic.  On a PEC axis index 0 is the
 * lower wall and index n (not stored) the upper wall; wall-tangential E,
 * wall-normal H and M on wall faces are 0 for ever (A12, A13), so a read
 * outside the stored range on a PEC axis returns 0.
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stddef.h>

#ifndef REAL
#define REAL double
#endif
#ifndef ORC_PREFIX
#define ORC_PREFIX oracle_
#endif
#define ORC_CAT2(a, b) a##b
#define ORC_CAT(a, b) ORC_CAT2(a, b)
#define ORC(name) ORC_CAT(ORC_PREFIX, name)

#define SQRT(x) ((REAL)sqrtl((long double)(x)))
#define FABS(x) ((REAL)fabsl((long double)(x)))

#define MAX_SOURCES 8

/* physical constants (paper silent on digits) */
static const long double PI_LD = 3.14159265358979323846264338327950288L;
#define MU0 ((REAL)(4.0L * PI_LD * 1e-7L))
#define C0 ((REAL)299792458.0L)
#define EPS0 ((REAL)(1.0L / (4.0L * PI_LD * 1e-7L * 299792458.0L * 299792458.0L)))

typedef struct {
  int kind;            /* 0 soft E (J in eq. 11), 1 hard E, 2 soft H, 3 hard H */
  int comp;            /* 0,1,2 = x,y,z component */
  int lo[3], hi[3];    /* edge-index box, lo inclusive, hi exclusive */
  REAL *profile;       /* box-sized, x fastest, or NULL = 1 */
  REAL amplitude, f0, t0, tp;
} source_t;

typedef struct {
  int n[3];
  REAL d[3], dt;
  int bc[3];
  int enable_llg;
  REAL hbias[3], hk, axis[3], tol;
  int max_iter;
  int scheme;          /* 0: second order, eqs. 15-21 (default); 1: first order, eqs. 6-9, 12-14 */
  /* open boundary: split-field PML with multiplicative damping (reading A26) */
  int has_pml, pml[3][2];          /* PML cells on the low / high side of each axis          */
  int pml_synced;                  /* split parts hold the present total fields              */
  REAL *pdE[3], *pdH[3];           /* sqrt of the damping factor of one update along each axis: */
                                   /* E parts (nodes, step dt), H parts (half positions, dt/2)   */
  REAL *Esp[3][2], *Hsp[3][2];     /* split parts: [component][0: d/d(d+1) term, 1: d/d(d+2)] */
  size_t ncell;
  REAL *eps_r, *sigma, *mu_r, *Ms, *alpha, *gamma; /* cell centred */
  REAL *E[3], *H[3], *M[3][3];
  /* work arrays of one HM half-step */
  REAL *C[3], *Hn[3], *Hp[3], *Hc[3], *Mn[3][3], *Mp[3][3];
  source_t src[MAX_SOURCES];
  int nsrc;
  /* statistics */
  long steps;
  long halfsteps;
  int iters_last;
  int iters_max;
  long iters_total;
  long nonconverged;
  REAL resid_last;
} oracle_t;

/* ---------------------------------------------------------------- indexing */

static size_t cidx(const oracle_t *o, int i, int j, int k) {
  return (size_t)i + (size_t)o->n[0] * ((size_t)j + (size_t)o->n[1] * (size_t)k);
}

/* boundary-aware read: wrap on periodic axes, 0 beyond a PEC wall */
static REAL rd(const oracle_t *o, const REAL *a, const int c[3]) {
  int q[3];
  for (int d = 0; d < 3; ++d) {
    int v = c[d];
    if (v < 0) {
      if (!o->bc[d]) return (REAL)0;
      v += o->n[d];
    } else if (v >= o->n[d]) {
      if (!o->bc[d]) return (REAL)0;
      v -= o->n[d];
    }
    q[d] = v;
  }
  return a[cidx(o, q[0], q[1], q[2])];
}

static REAL rd_off(const oracle_t *o, const REAL *a, const int c[3], int ax, int off) {
  int q[3] = {c[0], c[1], c[2]};
  q[ax] += off;
  return rd(o, a, q);
}

/* a d-face is a PEC wall face iff axis d is PEC and its index along d is 0 (A13) */
static int wall_face(const oracle_t *o, int d, const int c[3]) {
  return (!o->bc[d]) && c[d] == 0;
}

/* a d-edge is wall-tangential iff it lies in a PEC wall of a transverse axis */
static int wall_edge(const oracle_t *o, int d, const int c[3]) {
  int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  return ((!o->bc[t1]) && c[t1] == 0) || ((!o->bc[t2]) && c[t2] == 0);
}

/* mean of the two cells sharing the d-face at c  (A8) */
static REAL face_mean(const oracle_t *o, const REAL *a, int d, const int c[3]) {
  return (REAL)0.5 * (rd_off(o, a, c, d, -1) + rd(o, a, c));
}

/* mean of |.| of the two cells (gamma enters only as |gamma|, A1) */
static REAL face_mean_abs(const oracle_t *o, const REAL *a, int d, const int c[3]) {
  return (REAL)0.5 * (FABS(rd_off(o, a, c, d, -1)) + FABS(rd(o, a, c)));
}

/* mean of the four cells sharing the d-edge at c  (A8) */
static REAL edge_mean(const oracle_t *o, const REAL *a, int d, const int c[3]) {
  int t1 = (d + 1) % 3, t2 = (d + 2) % 3;
  REAL s = 0;
  for (int a1 = 0; a1 <= 1; ++a1)
    for (int a2 = 0; a2 <= 1; ++a2) {
      int q[3] = {c[0], c[1], c[2]};
      q[t1] -= a1;
      q[t2] -= a2;
      s += rd(o, a, q);
    }
  return (REAL)0.25 * s;
}

/* (curl E)_d at the d-face c: forward differences  (standard Yee) */
static REAL curl_E(const oracle_t *o, REAL *const E[3], int d, const int c[3]) {
  int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
  return (rd_off(o, E[d2], c, d1, +1) - rd(o, E[d2], c)) / o->d[d1] -
         (rd_off(o, E[d1], c, d2, +1) - rd(o, E[d1], c)) / o->d[d2];
}

/* (curl H)_d at the d-edge c: backward differences */
static REAL curl_H(const oracle_t *o, REAL *const H[3], int d, const int c[3]) {
  int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
  return (rd(o, H[d2], c) - rd_off(o, H[d2], c, d1, -1)) / o->d[d1] -
         (rd(o, H[d1], c) - rd_off(o, H[d1], c, d2, -1)) / o->d[d2];
}

/* transverse component t of H at the d-face c: "second-order four-point
 * average of the nearest values" (A7).  H_t sits at integer
 * position along t and half-integer along d, the d-face at integer d and
 * half-integer t: the nearest four are offsets {-1,0} along d and {0,+1} along t. */
static REAL avg4(const oracle_t *o, const REAL *Ht, int d, int t, const int c[3]) {
  REAL s = 0;
  for (int a = 0; a <= 1; ++a)
    for (int b = 0; b <= 1; ++b) {
      int q[3] = {c[0], c[1], c[2]};
      q[d] -= a;
      q[t] += b;
      s += rd(o, Ht, q);
    }
  return (REAL)0.25 * s;
}

/* ---------------------------------------------------------------- vectors */

static void cross(const REAL a[3], const REAL b[3], REAL out[3]) {
  out[0] = a[1] * b[2] - a[2] * b[1];
  out[1] = a[2] * b[0] - a[0] * b[2];
  out[2] = a[0] * b[1] - a[1] * b[0];
}
static REAL dot(const REAL a[3], const REAL b[3]) {
  return a[0] * b[0] + a[1] * b[1] + a[2] * b[2];
}

/* H_eff on the d-face c from the H arrays Hs and the face's own M vector m:
 * H_EM (own normal + two averages) + H_bias + uniaxial anisotropy
 * H_k (m.u/Ms_f) u   (A19, A20) */
static void h_eff(const oracle_t *o, REAL *const Hs[3], const REAL m[3], REAL Msf, int d,
                  const int c[3], REAL out[3]) {
  for (int t = 0; t < 3; ++t) {
    REAL h = (t == d) ? rd(o, Hs[d], c) : avg4(o, Hs[t], d, t, c);
    out[t] = h + o->hbias[t];
  }
  if (o->hk != (REAL)0) {
    REAL p = o->hk * (dot(m, o->axis) / Msf);
    for (int t = 0; t < 3; ++t) out[t] += p * o->axis[t];
  }
}

/* ------------------------------------------------------------- life cycle */

static REAL *alloc_fill(size_t n, const double *src, double dflt) {
  REAL *p = (REAL *)malloc(n * sizeof(REAL));
  if (!p) return NULL;
  for (size_t i = 0; i < n; ++i) p[i] = src ? (REAL)src[i] : (REAL)dflt;
  return p;
}

void ORC(destroy)(void *h);

/* Materials are host, cell-centred, nx*ny*nz, x fastest; NULL = eps_r 1,
 * sigma 0, mu_r 1, Ms 0, alpha 0, gamma 0.  bc[d]: 0 PEC, 1 periodic. */
void *ORC(create)(int nx, int ny, int nz, double dx, double dy, double dz, double dt,
                  const double *eps_r, const double *sigma, const double *mu_r,
                  const double *Ms, const double *alpha, const double *gamma, const int *bc,
                  int enable_llg, const double *hbias, double hk, const double *axis,
                  double tol, int max_iter) {
  if (nx < 1 || ny < 1 || nz < 1 || !(dx > 0) || !(dy > 0) || !(dz > 0) || !(dt > 0)) return NULL;
  if (enable_llg && (!(tol > 0) || max_iter < 1)) return NULL;
  oracle_t *o = (oracle_t *)calloc(1, sizeof(oracle_t));
  if (!o) return NULL;
  o->n[0] = nx; o->n[1] = ny; o->n[2] = nz;
  o->d[0] = (REAL)dx; o->d[1] = (REAL)dy; o->d[2] = (REAL)dz;
  o->dt = (REAL)dt;
  for (int d = 0; d < 3; ++d) {
    o->bc[d] = bc ? (bc[d] != 0) : 0;
    o->hbias[d] = hbias ? (REAL)hbias[d] : 0;
    o->axis[d] = axis ? (REAL)axis[d] : (REAL)(d == 2);
  }
  o->enable_llg = enable_llg;
  o->hk = (REAL)hk;
  o->tol = (REAL)tol;
  o->max_iter = max_iter;
  size_t n = (size_t)nx * ny * nz;
  o->ncell = n;
  o->eps_r = alloc_fill(n, eps_r, 1.0);
  o->sigma = alloc_fill(n, sigma, 0.0);
  o->mu_r = alloc_fill(n, mu_r, 1.0);
  o->Ms = alloc_fill(n, Ms, 0.0);
  o->alpha = alloc_fill(n, alpha, 0.0);
  o->gamma = alloc_fill(n, gamma, 0.0);
  int ok = o->eps_r && o->sigma && o->mu_r && o->Ms && o->alpha && o->gamma;
  for (int d = 0; d < 3 && ok; ++d) {
    o->E[d] = alloc_fill(n, NULL, 0.0);
    o->H[d] = alloc_fill(n, NULL, 0.0);
    o->C[d] = alloc_fill(n, NULL, 0.0);
    o->Hn[d] = alloc_fill(n, NULL, 0.0);
    o->Hp[d] = alloc_fill(n, NULL, 0.0);
    o->Hc[d] = alloc_fill(n, NULL, 0.0);
    ok = ok && o->E[d] && o->H[d] && o->C[d] && o->Hn[d] && o->Hp[d] && o->Hc[d];
    for (int c = 0; c < 3 && ok; ++c) {
      o->M[d][c] = alloc_fill(n, NULL, 0.0);
      o->Mn[d][c] = alloc_fill(n, NULL, 0.0);
      o->Mp[d][c] = alloc_fill(n, NULL, 0.0);
      ok = ok && o->M[d][c] && o->Mn[d][c] && o->Mp[d][c];
    }
  }
  for (size_t i = 0; i < n && ok; ++i)
    if (!(o->eps_r[i] > 0) || o->sigma[i] < 0 || !(o->mu_r[i] > 0) || o->Ms[i] < 0) ok = 0;
  if (!ok) {
    ORC(destroy)(o);
    return NULL;
  }
  return o;
}

void ORC(destroy)(void *h) {
  oracle_t *o = (oracle_t *)h;
  if (!o) return;
  free(o->eps_r); free(o->sigma); free(o->mu_r); free(o->Ms); free(o->alpha); free(o->gamma);
  for (int d = 0; d < 3; ++d) {
    free(o->E[d]); free(o->H[d]); free(o->C[d]); free(o->Hn[d]); free(o->Hp[d]); free(o->Hc[d]);
    for (int c = 0; c < 3; ++c) { free(o->M[d][c]); free(o->Mn[d][c]); free(o->Mp[d][c]); }
  }
  for (int s = 0; s < o->nsrc; ++s) free(o->src[s].profile);
  for (int a = 0; a < 3; ++a) {
    free(o->pdE[a]); free(o->pdH[a]);
    for (int q = 0; q < 2; ++q) { free(o->Esp[a][q]); free(o->Hsp[a][q]); }
  }
  free(o);
}

/* a d-face is magnetic iff LLG is on, Ms_face > 0 and it is not a PEC wall
 * face (A9, A13) */
static int magnetic_face(const oracle_t *o, int d, const int c[3], REAL *Msf) {
  if (!o->enable_llg || wall_face(o, d, c)) return 0;
  *Msf = face_mean(o, o->Ms, d, c);
  return *Msf > (REAL)0;
}

/* Initial fields.  E[3], H[3] directly on their Yee locations, Mc[3] the
 * initial magnetisation at CELL CENTRES, averaged to faces and renormalised to
 * the face's Ms (A11).  NULL = zero.  Wall-tangential E and
 * wall-normal H are forced to 0.  Returns 0, or -1 if a
 * magnetic face receives a zero averaged M (no direction to normalise). */
int ORC(set_fields)(void *h, const double *Ex, const double *Ey, const double *Ez,
                    const double *Hx, const double *Hy, const double *Hz, const double *Mcx,
                    const double *Mcy, const double *Mcz) {
  oracle_t *o = (oracle_t *)h;
  const double *Ein[3] = {Ex, Ey, Ez}, *Hin[3] = {Hx, Hy, Hz}, *Min[3] = {Mcx, Mcy, Mcz};
  int rc = 0;
  REAL *Mc[3];
  for (int c = 0; c < 3; ++c) {
    Mc[c] = alloc_fill(o->ncell, Min[c], 0.0);
    if (!Mc[c]) return -2;
  }
  for (int k = 0; k < o->n[2]; ++k)
    for (int j = 0; j < o->n[1]; ++j)
      for (int i = 0; i < o->n[0]; ++i) {
        int c[3] = {i, j, k};
        size_t id = cidx(o, i, j, k);
        for (int d = 0; d < 3; ++d) {
          o->E[d][id] = (Ein[d] && !wall_edge(o, d, c)) ? (REAL)Ein[d][id] : (REAL)0;
          o->H[d][id] = (Hin[d] && !wall_face(o, d, c)) ? (REAL)Hin[d][id] : (REAL)0;
          REAL Msf = 0;
          if (magnetic_face(o, d, c, &Msf)) {
            REAL m[3];
            for (int q = 0; q < 3; ++q) m[q] = face_mean(o, Mc[q], d, c);
            REAL nrm = SQRT(dot(m, m));
            if (!(nrm > 0)) {
              rc = -1;
              for (int q = 0; q < 3; ++q) o->M[d][q][id] = 0;
            } else {
              for (int q = 0; q < 3; ++q) o->M[d][q][id] = m[q] * (Msf / nrm);
            }
          } else {
            for (int q = 0; q < 3; ++q) o->M[d][q][id] = 0;
          }
        }
      }
  for (int c = 0; c < 3; ++c) free(Mc[c]);
  o->pml_synced = 0;
  return rc;
}

/* Soft current source entering eq. 11:
 * J_comp(t) = amplitude * exp(-(t-t0)^2/(2 tp^2)) * cos(2 pi f0 t) * profile
 * on the box lo <= index < hi of comp-edges; envelope of eq. 31 (A15). */
/* External excitations: "soft sources [are defined] in terms of the time-rate of
 * field change, and are applied at the beginning of the time step.  Hard sources are enforced
 * directly for the corresponding fields after their updates at each time step."  The paper prints
 * no formulas; the reading taken (A25), g(t) the envelope of eq. 31:
 *   kind 0  soft E: the current J_src^{n+1/2} of eq. 11, t = (n+1/2) dt
 *   kind 1  hard E: after the E update of step n, E_comp = A g((n+1) dt) profile on the box
 *   kind 2  soft H: before the first (H,M) half-step of step n, H_comp += dt A g(n dt) profile
 *   kind 3  hard H: after the second (H,M) half-step, H_comp = A g((n+1) dt) profile
 * Wall-tangential E edges and wall faces of H stay 0; M is never touched. */
int ORC(add_source)(void *h, int kind, int comp, const int *lo, const int *hi,
                    const double *profile, double amplitude, double f0, double t0, double tp) {
  oracle_t *o = (oracle_t *)h;
  if (kind < 0 || kind > 3) return -1;
  if (o->nsrc >= MAX_SOURCES || comp < 0 || comp > 2 || !(tp > 0)) return -1;
  source_t *s = &o->src[o->nsrc];
  size_t nb = 1;
  for (int d = 0; d < 3; ++d) {
    if (lo[d] < 0 || hi[d] > o->n[d] || lo[d] >= hi[d]) return -1;
    s->lo[d] = lo[d];
    s->hi[d] = hi[d];
    nb *= (size_t)(hi[d] - lo[d]);
  }
  s->kind = kind;
  s->comp = comp;
  s->profile = profile ? alloc_fill(nb, profile, 0.0) : NULL;
  s->amplitude = (REAL)amplitude;
  s->f0 = (REAL)f0;
  s->t0 = (REAL)t0;
  s->tp = (REAL)tp;
  o->nsrc++;
  return 0;
}

int ORC(set_source)(void *h, int comp, const int *lo, const int *hi, const double *profile,
                    double amplitude, double f0, double t0, double tp) {
  return ORC(add_source)(h, 0, comp, lo, hi, profile, amplitude, f0, t0, tp);
}

static REAL source_at(const oracle_t *o, int comp, const int c[3], REAL t) {
  REAL J = 0;
  for (int s = 0; s < o->nsrc; ++s) {
    const source_t *S = &o->src[s];
    if (S->kind != 0 || S->comp != comp) continue;
    int in = 1;
    for (int d = 0; d < 3; ++d) in = in && c[d] >= S->lo[d] && c[d] < S->hi[d];
    if (!in) continue;
    REAL u = (t - S->t0) / S->tp;
    REAL g = (REAL)expl((long double)(-(REAL)0.5 * u * u)) *
             (REAL)cosl((long double)((REAL)2 * (REAL)PI_LD * S->f0 * t));
    REAL p = 1;
    if (S->profile) {
      size_t bx = (size_t)(S->hi[0] - S->lo[0]), by = (size_t)(S->hi[1] - S->lo[1]);
      p = S->profile[(size_t)(c[0] - S->lo[0]) +
                     bx * ((size_t)(c[1] - S->lo[1]) + by * (size_t)(c[2] - S->lo[2]))];
    }
    J += S->amplitude * g * p;
  }
  return J;
}

/* ------------------------------------------------------------- E update */

/* eq. 11:
 * E^{n+1} = (sigma/2 + eps/dt)^-1 [ curl H^{n+1/2} - (sigma/2 - eps/dt) E^n - J_src^{n+1/2} ]
 * at every edge that is not wall-tangential; eps, sigma = four-cell means. */
/* ------------------------------------------------------------------ PML (open boundary)
 * "a perfectly matched layer (PML) first developed by Berenger ... damps out EM
 * waves using a non-physical conductivity in the guard cells ... field components E and H are
 * updated using macroscopic Maxwell's equations that account for spatially varying material
 * properties and then the updated field components are multiplied by the corresponding PML
 * damping coefficients".  The paper gives no formulas (it points to Shapoval et al. 2019); the
 * reading taken (A26):
 *  - the layer is the outermost pml[a][side] cells of the grid along axis a, backed by the PEC wall;
 *  - there every component is split in two parts, one per term of the curl (Berenger):
 *      F_d = F_d,0 + F_d,1,  part 0 <- d/d(d+1) term, part 1 <- d/d(d+2) term;
 *  - each part is advanced by the macroscopic update (eq. 11 for E with the local eps, sigma;
 *    eq. 21 with M = 0 and the local mu for H) with its own term of the curl, between two
 *    multiplications by the square root of its damping factor (two-step, time-centred: the
 *    "2SC" of the name): the factor is exp(-s_a dt) for E (one step) and exp(-s_a dt/2) for H
 *    (one half-step), a = the axis of the derivative in that term: the same decay RATE s_a for E
 *    and H, which is the matching condition sigma_a/eps = sigma*_a/mu in any medium;
 *  - s_a(u) = s_max (u/L)^m at depth u into a layer of thickness L, sampled at the nodes (E parts)
 *    and half positions (H parts) of axis a; s_max = -(m+1) c ln(R0) / (2 L), the textbook choice
 *    for a theoretical normal-incidence reflection R0;
 *  - no magnetic face inside the layer (future work in the paper too). */
static int in_pml(const oracle_t *o, const int c[3]) {
  for (int a = 0; a < 3; ++a)
    if (c[a] < o->pml[a][0] || c[a] >= o->n[a] - o->pml[a][1]) return 1;
  return 0;
}

static REAL pml_rate(const oracle_t *o, int a, long double x, long double r0, int order) {
  long double L, u;
  const long double len = (long double)o->n[a] * (long double)o->d[a];
  if (o->pml[a][0] > 0 && x < (L = o->pml[a][0] * (long double)o->d[a])) u = L - x;
  else if (o->pml[a][1] > 0 && x > len - (L = o->pml[a][1] * (long double)o->d[a])) u = x - (len - L);
  else return 0;
  long double smax = -(order + 1) * (long double)C0 * logl(r0) / (2 * L);
  return (REAL)(smax * powl(u / L, order));
}

int ORC(set_pml)(void *h, const int *pml, double r0, int order) {
  oracle_t *o = (oracle_t *)h;
  if (!(r0 > 0 && r0 < 1) || order < 1 || order > 6) return -1;
  for (int a = 0; a < 3; ++a)
    for (int sd = 0; sd < 2; ++sd) {
      int p = pml[2 * a + sd];
      if (p < 0 || (p > 0 && o->bc[a])) return -1; /* a PML axis ends on a PEC wall, not periodic */
      o->pml[a][sd] = p;
    }
  for (int a = 0; a < 3; ++a)
    if (o->pml[a][0] + o->pml[a][1] > o->n[a]) return -1;
  o->has_pml = 0;
  for (int a = 0; a < 3; ++a) o->has_pml |= (o->pml[a][0] | o->pml[a][1]) != 0;
  for (int a = 0; a < 3; ++a) {
    free(o->pdE[a]);
    free(o->pdH[a]);
    o->pdE[a] = (REAL *)malloc(sizeof(REAL) * (size_t)o->n[a]);
    o->pdH[a] = (REAL *)malloc(sizeof(REAL) * (size_t)o->n[a]);
    for (int i = 0; i < o->n[a]; ++i) {
      long double xe = i * (long double)o->d[a], xh = (i + 0.5L) * (long double)o->d[a];
      /* half of the damping of one update: exp(-s dt/2) for E (step dt), exp(-s dt/4) for H (dt/2) */
      o->pdE[a][i] = (REAL)expl(-(long double)pml_rate(o, a, xe, r0, order) * (long double)o->dt / 2);
      o->pdH[a][i] = (REAL)expl(-(long double)pml_rate(o, a, xh, r0, order) * (long double)o->dt / 4);
    }
    for (int q = 0; q < 2; ++q) {
      if (!o->Esp[a][q]) o->Esp[a][q] = alloc_fill(o->ncell, NULL, 0.0);
      if (!o->Hsp[a][q]) o->Hsp[a][q] = alloc_fill(o->ncell, NULL, 0.0);
    }
  }
  o->pml_synced = 0;
  /* no magnetic face may belong to a PML cell */
  for (int k = 0; k < o->n[2]; ++k)
    for (int j = 0; j < o->n[1]; ++j)
      for (int i = 0; i < o->n[0]; ++i) {
        int c[3] = {i, j, k};
        if (!in_pml(o, c)) continue;
        for (int d = 0; d < 3; ++d) {
          REAL Msf;
          if (magnetic_face(o, d, c, &Msf)) return -2;
        }
      }
  return 0;
}

/* one E edge of a PML cell: eq. 11 on each part, then the damping factors */
static REAL pml_e_edge(oracle_t *o, int d, const int c[3], size_t id, REAL J) {
  const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
  REAL eps = EPS0 * edge_mean(o, o->eps_r, d, c);
  REAL sig = edge_mean(o, o->sigma, d, c);
  REAL term0 = (rd(o, o->H[d2], c) - rd_off(o, o->H[d2], c, d1, -1)) / o->d[d1];
  REAL term1 = -(rd(o, o->H[d1], c) - rd_off(o, o->H[d1], c, d2, -1)) / o->d[d2];
  REAL den = sig / 2 + eps / o->dt, keep = -(sig / 2 - eps / o->dt);
  /* two-step, time-centred damping ("PML-2SC"): half of it before the update, half after */
  const REAL g0 = o->pdE[d1][c[d1]], g1 = o->pdE[d2][c[d2]];
  REAL p0 = (term0 + keep * (g0 * o->Esp[d][0][id]) - J) / den;
  REAL p1 = (term1 + keep * (g1 * o->Esp[d][1][id])) / den;
  p0 *= g0;
  p1 *= g1;
  o->Esp[d][0][id] = p0;
  o->Esp[d][1][id] = p1;
  return p0 + p1;
}

/* one H face of a PML cell over half a step: eq. 21 with M = 0 on each part, then the damping */
static REAL pml_h_face(oracle_t *o, int d, const int c[3], size_t id) {
  const int d1 = (d + 1) % 3, d2 = (d + 2) % 3;
  REAL mu = MU0 * face_mean(o, o->mu_r, d, c);
  REAL term0 = (rd_off(o, o->E[d2], c, d1, +1) - rd(o, o->E[d2], c)) / o->d[d1];
  REAL term1 = -(rd_off(o, o->E[d1], c, d2, +1) - rd(o, o->E[d1], c)) / o->d[d2];
  const REAL g0 = o->pdH[d1][c[d1]], g1 = o->pdH[d2][c[d2]];
  REAL p0 = g0 * o->Hsp[d][0][id] - (o->dt / 2 / mu) * term0;
  REAL p1 = g1 * o->Hsp[d][1][id] - (o->dt / 2 / mu) * term1;
  p0 *= g0;
  p1 *= g1;
  o->Hsp[d][0][id] = p0;
  o->Hsp[d][1][id] = p1;
  return p0 + p1;
}

static void e_update(oracle_t *o) {
  REAL t_half = ((REAL)o->steps + (REAL)0.5) * o->dt;
#pragma omp parallel for schedule(static)
  for (int k = 0; k < o->n[2]; ++k)
    for (int j = 0; j < o->n[1]; ++j)
      for (int i = 0; i < o->n[0]; ++i) {
        int c[3] = {i, j, k};
        size_t id = cidx(o, i, j, k);
        for (int d = 0; d < 3; ++d) {
          if (wall_edge(o, d, c)) continue; /* stays 0 */
          REAL eps = EPS0 * edge_mean(o, o->eps_r, d, c);
          REAL sig = edge_mean(o, o->sigma, d, c);
          REAL J = o->nsrc ? source_at(o, d, c, t_half) : (REAL)0;
          if (o->has_pml && in_pml(o, c)) {
            o->E[d][id] = pml_e_edge(o, d, c, id, J);
            continue;
          }
          REAL rhs = curl_H(o, o->H, d, c) - (sig / 2 - eps / o->dt) * o->E[d][id] - J;
          o->E[d][id] = rhs / (sig / 2 + eps / o->dt);
        }
      }
}

/* ------------------------------------------------------- H/M half-step */

/* One iterate of eqs. 18-21 on the magnetic d-face c.
 *   mn   = M^n            hn = H_eff^n (fixed during the iterations)
 *   he   = H_eff^{r-1}    (lagged)
 *   out: mr = M^r (renormalised), returns  M^n_d - M^r_d  (the term of eq. 21). */
static REAL llg_iterate(const REAL mn[3], const REAL hn[3], const REAL he[3], REAL cf,
                        REAL alpha_f, REAL Msf, int d, REAL mr[3]) {
  REAL a[3], t3[3];
#ifdef ORACLE_LITERAL
  /* exactly as printed: b (20), a (19), M^r (18), N(M) */
  REAL b[3], axb[3];
  cross(mn, hn, t3);
  for (int q = 0; q < 3; ++q) b[q] = mn[q] - cf * t3[q];
  for (int q = 0; q < 3; ++q) a[q] = -(cf * he[q] + (alpha_f / Msf) * mn[q]);
  cross(a, b, axb);
  REAL ab = dot(a, b), den = 1 + dot(a, a);
  for (int q = 0; q < 3; ++q) mr[q] = (b[q] + ab * a[q] - axb[q]) / den;
  REAL s = Msf / SQRT(dot(mr, mr));
  for (int q = 0; q < 3; ++q) mr[q] *= s;
  return mn[d] - mr[d];
#else
  /* increment form (A24): algebraically eq. 18 minus M^n, then the
   * renormalisation written for the increment; no O(Ms) cancellation. */
  REAL beta[3], tau[3], axt[3], axb[3], Delta[3];
  cross(mn, hn, t3);
  for (int q = 0; q < 3; ++q) beta[q] = -cf * t3[q];             /* b = M^n + beta (20) */
  cross(mn, he, t3);
  for (int q = 0; q < 3; ++q) tau[q] = cf * t3[q];               /* = a x M^n            */
  for (int q = 0; q < 3; ++q) a[q] = -(cf * he[q] + (alpha_f / Msf) * mn[q]); /* (19)   */
  cross(a, tau, axt);
  cross(a, beta, axb);
  REAL ab = dot(a, beta), den = 1 + dot(a, a);
  for (int q = 0; q < 3; ++q)
    Delta[q] = (beta[q] - tau[q] + axt[q] + ab * a[q] - axb[q]) / den; /* (18) - M^n    */
  REAL x = (2 * dot(mn, Delta) + dot(Delta, Delta)) / (Msf * Msf);
  REAL sq = SQRT(1 + x);
  REAL sm1 = -x / (sq * (1 + sq));                               /* Ms/|M^n+Delta| - 1  */
  REAL dM[3];
  for (int q = 0; q < 3; ++q) {
    dM[q] = Delta[q] + sm1 * (mn[q] + Delta[q]);
    mr[q] = mn[q] + dM[q];
  }
  return -dM[d];
#endif
}

/* First-order scheme, Step 1 / Step 3: forward Euler on eq. 6,
 *   M' = M + (dt/2) [ mu0 gamma_L (M x H_eff) + (alpha mu0 gamma_L / Ms) M x (M x H_eff) ],
 * gamma_L = gamma / (1 + alpha^2), then N(M').  The paper prints the step of eqs. 7 and 12 as
 * dt; both advance HALF a step (eqs. 8-9, 13-14 divide by dt/2), so dt/2 is used (DESIGN.md
 * A22).  gamma < 0 for the electron: mu0 gamma_L = -mu0 |gamma| / (1 + alpha^2).
 * Evaluated, like the second-order scheme, as an increment (A24).
 *   out: mr = M' (renormalised), returns M_d - M'_d  (the term of eqs. 9, 14). */
static REAL llg_euler(const REAL mn[3], const REAL hn[3], REAL gabs, REAL alpha_f, REAL Msf,
                      REAL half_dt, int d, REAL mr[3]) {
  REAL mxh[3], mxmxh[3], Delta[3], dM[3];
  const REAL gl = MU0 * gabs / (1 + alpha_f * alpha_f); /* mu0 |gamma_L| */
  cross(mn, hn, mxh);
  cross(mn, mxh, mxmxh);
  for (int q = 0; q < 3; ++q)
    Delta[q] = half_dt * (-gl * mxh[q] - (alpha_f * gl / Msf) * mxmxh[q]);
  REAL x = (2 * dot(mn, Delta) + dot(Delta, Delta)) / (Msf * Msf);
  REAL sq = SQRT(1 + x);
  REAL sm1 = -x / (sq * (1 + sq)); /* Ms/|M+Delta| - 1 */
  for (int q = 0; q < 3; ++q) {
    dM[q] = Delta[q] + sm1 * (mn[q] + Delta[q]);
    mr[q] = mn[q] + dM[q];
  }
  return -dM[d];
}

/* (H,M) advanced over dt/2 with curl E fixed. */
static void hm_half(oracle_t *o) {
  const int nx = o->n[0], ny = o->n[1], nz = o->n[2];
  const REAL half_dt = o->dt / 2;
  /* C = curl E on all faces; (H,M)^{r=0} = (H,M)^n */
#pragma omp parallel for schedule(static)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        int c[3] = {i, j, k};
        size_t id = cidx(o, i, j, k);
        for (int d = 0; d < 3; ++d) {
          o->C[d][id] = curl_E(o, o->E, d, c);
          o->Hn[d][id] = o->H[d][id];
          o->Hp[d][id] = o->H[d][id];
          for (int q = 0; q < 3; ++q) {
            o->Mn[d][q][id] = o->M[d][q][id];
            o->Mp[d][q][id] = o->M[d][q][id];
          }
        }
      }
  /* non-magnetic faces: eq. 21 with M = 0 and the local mu;
   * wall faces stay 0.  Their value is the same in every iterate. */
  long nmag = 0;
#pragma omp parallel for schedule(static) reduction(+ : nmag)
  for (int k = 0; k < nz; ++k)
    for (int j = 0; j < ny; ++j)
      for (int i = 0; i < nx; ++i) {
        int c[3] = {i, j, k};
        size_t id = cidx(o, i, j, k);
        for (int d = 0; d < 3; ++d) {
          REAL Msf = 0;
          if (magnetic_face(o, d, c, &Msf)) {
            nmag++;
            continue;
          }
          REAL v = 0;
          if (!wall_face(o, d, c)) {
            if (o->has_pml && in_pml(o, c)) {
              v = pml_h_face(o, d, c, id);
            } else {
              REAL mu = MU0 * face_mean(o, o->mu_r, d, c);
              v = o->Hn[d][id] - (half_dt / mu) * o->C[d][id];
            }
          }
          o->H[d][id] = v;
          o->Hc[d][id] = v; /* iterate r >= 1; Hp keeps H^{r=0} = H^n for the r = 1 sweep (A6) */
        }
      }
  o->halfsteps++;
  if (nmag == 0) {
    o->iters_last = 0;
    return;
  }

  int r = 0;
  REAL delta = 0;
  for (r = 1; r <= o->max_iter; ++r) {
    delta = 0;
#pragma omp parallel for schedule(static) reduction(max : delta)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          int c[3] = {i, j, k};
          size_t id = cidx(o, i, j, k);
          for (int d = 0; d < 3; ++d) {
            REAL Msf = 0;
            if (!magnetic_face(o, d, c, &Msf)) continue; /* Hc already final there */
            REAL alpha_f = face_mean(o, o->alpha, d, c);
            REAL cf = MU0 * face_mean_abs(o, o->gamma, d, c) * o->dt / 4;
            REAL mn[3], mp[3], mr[3], hn[3], he[3];
            for (int q = 0; q < 3; ++q) {
              mn[q] = o->Mn[d][q][id];
              mp[q] = o->Mp[d][q][id];
            }
            h_eff(o, o->Hn, mn, Msf, d, c, hn);
            h_eff(o, o->Hp, mp, Msf, d, c, he);
            REAL dMn = o->scheme == 1
                           ? llg_euler(mn, hn, face_mean_abs(o, o->gamma, d, c), alpha_f, Msf, half_dt, d, mr)
                           : llg_iterate(mn, hn, he, cf, alpha_f, Msf, d, mr);
            /* eq. 21: H^r = H^n + M^n - M^r - (dt/2mu0) curl E, normal component */
            o->Hc[d][id] = o->Hn[d][id] + dMn - (half_dt / MU0) * o->C[d][id];
            for (int q = 0; q < 3; ++q) {
              o->M[d][q][id] = mr[q];
              REAL e = FABS(mr[q] - mp[q]) / Msf;
              if (e > delta) delta = e;
            }
          }
        }
    /* iterate r becomes r-1 */
#pragma omp parallel for schedule(static)
    for (int k = 0; k < nz; ++k)
      for (int j = 0; j < ny; ++j)
        for (int i = 0; i < nx; ++i) {
          size_t id = cidx(o, i, j, k);
          for (int d = 0; d < 3; ++d) {
            o->Hp[d][id] = o->Hc[d][id];
            for (int q = 0; q < 3; ++q) o->Mp[d][q][id] = o->M[d][q][id];
          }
        }
    if (o->scheme == 1) { delta = 0; break; } /* explicit: one sweep, no stopping test */
    if (delta < o->tol) break;
  }
  if (r > o->max_iter) {
    r = o->max_iter;
    o->nonconverged++; /* A4: accept the last iterate */
  }
  for (int d = 0; d < 3; ++d) memcpy(o->H[d], o->Hc[d], o->ncell * sizeof(REAL));
  o->iters_last = r;
  o->iters_total += r;
  if (r > o->iters_max) o->iters_max = r;
  o->resid_last = delta;
}

/* n time steps:  HM half (curl E^n) ; E update ; HM half (curl E^{n+1}) */
/* fields given from outside (initial condition) enter the layer as part 0 of each component */
static void pml_sync(oracle_t *o) {
  if (!o->has_pml || o->pml_synced) return;
  for (int d = 0; d < 3; ++d)
    for (size_t i = 0; i < o->ncell; ++i) {
      o->Esp[d][0][i] = o->E[d][i]; o->Esp[d][1][i] = 0;
      o->Hsp[d][0][i] = o->H[d][i]; o->Hsp[d][1][i] = 0;
    }
  o->pml_synced = 1;
}

/* sources of one kind applied to E (kinds 1) or H (kinds 2, 3) at time t */
static void apply_field_sources(oracle_t *o, int kind, REAL t) {
  for (int q = 0; q < o->nsrc; ++q) {
    const source_t *S = &o->src[q];
    if (S->kind != kind) continue;
    REAL u = (t - S->t0) / S->tp;
    REAL g = (REAL)expl((long double)(-(REAL)0.5 * u * u)) *
             (REAL)cosl((long double)((REAL)2 * (REAL)PI_LD * S->f0 * t));
    REAL *F = (kind == 1) ? o->E[S->comp] : o->H[S->comp];
    size_t bx = (size_t)(S->hi[0] - S->lo[0]), by = (size_t)(S->hi[1] - S->lo[1]);
    for (int k = S->lo[2]; k < S->hi[2]; ++k)
      for (int j = S->lo[1]; j < S->hi[1]; ++j)
        for (int i = S->lo[0]; i < S->hi[0]; ++i) {
          int c[3] = {i, j, k};
          if (kind == 1 ? wall_edge(o, S->comp, c) : wall_face(o, S->comp, c)) continue;
          if (o->has_pml && in_pml(o, c)) continue; /* field sources act outside the layer only */
          REAL p = S->profile ? S->profile[(size_t)(i - S->lo[0]) +
                                           bx * ((size_t)(j - S->lo[1]) + by * (size_t)(k - S->lo[2]))]
                              : 1;
          REAL v = S->amplitude * g * p;
          size_t id = cidx(o, i, j, k);
          if (kind == 2) F[id] += o->dt * v;
          else F[id] = v;
        }
  }
}

int ORC(step)(void *h, int n) {
  oracle_t *o = (oracle_t *)h;
  pml_sync(o);
  for (int s = 0; s < n; ++s) {
    apply_field_sources(o, 2, (REAL)o->steps * o->dt);        /* soft H, beginning of the step */
    hm_half(o);
    e_update(o);
    apply_field_sources(o, 1, (REAL)(o->steps + 1) * o->dt);  /* hard E, after its update     */
    hm_half(o);
    apply_field_sources(o, 3, (REAL)(o->steps + 1) * o->dt);  /* hard H, after its update     */
    o->steps++;
  }
  return 0;
}

/* 0: second-order scheme (default); 1: first-order scheme of PAPER.md:102-150 */
int ORC(set_scheme)(void *h, int scheme) {
  if (scheme != 0 && scheme != 1) return -1;
  ((oracle_t *)h)->scheme = scheme;
  return 0;
}

/* test hook: ONE (H,M) half-step with the present E (no E update, no step count) */
int ORC(hm_half_step)(void *h) {
  pml_sync((oracle_t *)h);
  hm_half((oracle_t *)h);
  return 0;
}

/* out[15]: Ex,Ey,Ez, Hx,Hy,Hz, then M on x-faces (Mx,My,Mz), y-faces, z-faces;
 * each nx*ny*nz doubles or NULL to skip. */
int ORC(read_fields)(void *h, double *const *out) {
  oracle_t *o = (oracle_t *)h;
  for (int d = 0; d < 3; ++d) {
    if (out[d])
      for (size_t i = 0; i < o->ncell; ++i) out[d][i] = (double)o->E[d][i];
    if (out[3 + d])
      for (size_t i = 0; i < o->ncell; ++i) out[3 + d][i] = (double)o->H[d][i];
    for (int c = 0; c < 3; ++c)
      if (out[6 + 3 * d + c])
        for (size_t i = 0; i < o->ncell; ++i) out[6 + 3 * d + c][i] = (double)o->M[d][c][i];
  }
  return 0;
}

/* Overwrite the state directly on the Yee / face locations (no averaging, no
 * normalisation): used by tests that need a prescribed face M. in[15] as above. */
int ORC(write_fields)(void *h, const double *const *in) {
  oracle_t *o = (oracle_t *)h;
  for (int d = 0; d < 3; ++d) {
    if (in[d])
      for (size_t i = 0; i < o->ncell; ++i) o->E[d][i] = (REAL)in[d][i];
    if (in[3 + d])
      for (size_t i = 0; i < o->ncell; ++i) o->H[d][i] = (REAL)in[3 + d][i];
    for (int c = 0; c < 3; ++c)
      if (in[6 + 3 * d + c])
        for (size_t i = 0; i < o->ncell; ++i) o->M[d][c][i] = (REAL)in[6 + 3 * d + c][i];
  }
  o->pml_synced = 0;
  return 0;
}

/* out[8]: steps, time, iters_last, iters_max, iters_total, nonconverged, resid_last, halfsteps */
int ORC(get_stats)(void *h, double *out) {
  oracle_t *o = (oracle_t *)h;
  out[0] = (double)o->steps;
  out[1] = (double)((REAL)o->steps * o->dt);
  out[2] = (double)o->iters_last;
  out[3] = (double)o->iters_max;
  out[4] = (double)o->iters_total;
  out[5] = (double)o->nonconverged;
  out[6] = (double)o->resid_last;
  out[7] = (double)o->halfsteps;
  return 0;
}

/* physical constants as this build uses them (tests pin c = 1/sqrt(mu0 eps0)) */
void ORC(constants)(double *out) {
  out[0] = (double)MU0;
  out[1] = (double)EPS0;
  out[2] = (double)C0;
}
