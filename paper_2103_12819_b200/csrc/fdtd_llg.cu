// fdtd_llg.cu -- host side of the C ABI declared in include/fdtd_llg.h.
//
// Owns: workspace carve-up, material analysis (uniformity, magnetic bounding box), the static
// buffer rotation of the Jacobi iterates, and the CUDA Graph of one time step.  All arithmetic of
// the path is in kernels.cuh.  No device memory is allocated here: everything lives in the
// caller's workspace.
#include <algorithm>
#include <climits>
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/fdtd_llg.h"
#include "kernels.cuh"
#include "hm_stage.cuh"
#include "eh_stage.cuh"

using namespace fl;

namespace {

thread_local std::string g_create_error = "";

constexpr size_t ALIGN_D = 32;  // arrays start on 256-byte boundaries

size_t padded(size_t n) { return (n + ALIGN_D - 1) / ALIGN_D * ALIGN_D; }

// device layout of one array (kernels.cuh "DEVICE LAYOUT"): one ghost layer, 128-byte aligned rows
size_t row_pitch(int nx) { return ((size_t)PADL + nx + 1 + 15) / 16 * 16; }
size_t array_stride(int nx, int ny, int nz) {
  return padded(row_pitch(nx) * (size_t)(ny + 2) * (size_t)(nz + 2));
}

struct MatInfo {
  bool is_array = false;  // non-uniform: kept on the device
  double uniform = 0.0;   // value when uniform
  double maxv = 0.0;      // largest value of the map
  double *dev = nullptr;
};

}  // namespace

struct fdtd_llg {
  GridP g{};
  double d[3]{}, dt = 0;
  size_t ncell = 0, stride = 0;  // stride = array_stride(): doubles between consecutive arrays
  size_t ncell_user = 0;         // entries of a user array passed IN: ncell + the interface planes
  int num_sms = 148;
  fdtd_llg_options opt{};
  cudaStream_t stream = nullptr;
  char *ws = nullptr;
  size_t ws_bytes = 0;

  double *E[3]{};   // E set 0 (time n when host_steps is even)
  double *E2[3]{};  // E set 1: the E update is out of place, the two sets alternate
  double *Hset[3][3]{};  // three H sets (time-n, ping, pong), statically rotated per half-step
  double *Mset[2][9]{};  // two M sets
  MatInfo eps_r, sigma, mu_r, Ms, alpha, gamma;
  bool llg = false;  // LLG enabled AND at least one magnetic cell
  long long magnetic_cells = 0;
  int lo[3]{}, hi[3]{};  // sweep box (index triples), hi exclusive
  int lo0_unrounded = 0; // lo[0] before it was rounded down to an even index (kept odd next to a PML)
  BoxP box_llg{}, box_all{};
  int n_arrays = 0;  // arrays in the workspace tensor (4th TMA coordinate)
  bool staged = false;  // the LLG iterates run the staged sweep (hm_stage.cuh)
  StBox st_box{}, st_box_first{};  // work items of the iterates r >= 2 / of the r = 1 sweep
  CUtensorMap mapT{}, mapPM{};
  // staged Maxwell sweeps (eh_stage.cuh): the E update, fused with the merged H update outside the box
  bool eh_ok = false;        // tensor map built, kernels configured (no PML, kernel_path != 1)
  CUtensorMap mapEH{}, mapEF{};   // boxes of k_eh_stage (18 rows) and of k_eh_fused (17 rows)
  unsigned *work_eh = nullptr;  // [2][8] item counters: one per staged launch of a step, by step parity
  BoxP box_out[6]{};     // the complement of the sweep box, as slabs (merged H: within the interior)
  int n_out = 0;
  // merged H half-steps keep out of a margin at each side of the grid: the PML layer and thin boxes
  // of H sources at a boundary (their faces need H at integer time); cells from the side
  int um_lo[3]{}, um_hi[3]{};
  std::vector<BoxP> box_um;   // the margins minus the sweep box: plain half-steps
  // open boundary: split parts of E and H, damping tables, the layer's slabs
  bool has_pml = false;
  double *Esp[6]{}, *Hsp[6]{};   // [2 * component + part]
  double *pdE[3]{}, *pdH[3]{};   // sqrt damping factors along x, y, z (device)
  BoxP box_pml[6]{};
  int n_pml = 0;

  DevState *dstate = nullptr;
  unsigned long long *resid = nullptr;
  unsigned *work = nullptr;  // [max_iter + 1] item counters of the staged sweeps
  double *scratch = nullptr;  // 2*1024 doubles for reductions + 8 ints
  SourcesP src{};
  double *profile_pool = nullptr;
  size_t profile_cap = 0, profile_used = 0;

  // per-kernel timing of fdtd_llg_step_timed: an event pair around every launch
  struct ProfRec { cudaEvent_t a, b; int cls, half, r; };
  std::vector<ProfRec> *prof = nullptr;
  int prof_half = 0;
  int *r_hist = nullptr;  // device: iteration count R of half-step h at [h % R_HIST]

  cudaGraphExec_t graph[2] = {nullptr, nullptr};  // one captured step per E parity
  bool capturing = false;        // inside build_graph: the rarely needed iterates go into an IF node
  cudaStream_t aux = nullptr;    // captures the body of that node
  bool graph_valid[2] = {false, false};
  int launches_per_step = 0;
  long long kernel_launches = 0;
  long long host_steps = 0;
  // merged H half-steps (options.merge_h): outside the sweep box H lives at half-integer time
  bool merge = false;        // active for this handle (no PML, no H sources)
  bool primed = false;       // the outside faces have been advanced to t = dt/2 (first step taken)
  long long prime_at = 0;    // host_steps when that happened
  bool recon_valid = false;  // the integer-time H of the present state has been formed for reading
  // z-slab decomposition
  bool is_slab = false;      // any slab_ext side set
  int sub_next = 0;          // the sub-step fdtd_llg_substep expects next (FDTD_LLG_SUB_*)
  int sub_r = 0;             // last LLG iterate enqueued in the current half-step
  std::string err = "";
};

namespace {

constexpr int R_HIST = 4096;

// event pair around the launches between prof_begin and prof_end (no-ops outside step_timed)
void prof_begin(fdtd_llg *s, int cls, int r) {
  if (!s->prof) return;
  fdtd_llg::ProfRec p{};
  p.cls = cls; p.half = s->prof_half; p.r = r;
  cudaEventCreate(&p.a);
  cudaEventCreate(&p.b);
  cudaEventRecord(p.a, s->stream);
  s->prof->push_back(p);
}
void prof_end(fdtd_llg *s) {
  if (!s->prof) return;
  cudaEventRecord(s->prof->back().b, s->stream);
}

int fail(fdtd_llg *s, int code, const char *fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof buf, fmt, ap);
  va_end(ap);
  if (s) s->err = buf; else g_create_error = buf;
  return code;
}

#define CU(s, call)                                                                      \
  do {                                                                                   \
    cudaError_t e_ = (call);                                                             \
    if (e_ != cudaSuccess)                                                               \
      return fail((s), FDTD_LLG_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));         \
  } while (0)

// Work items: TX x TY columns marched over kz planes.  kz is as long as possible (amortises the
// cold first plane of the prefetch pipeline) while leaving >= 8 items per SM.
BoxP make_box(const fdtd_llg *s, const int lo[3], const int hi[3]) {
  BoxP b{};
  for (int d = 0; d < 3; ++d) { b.lo[d] = lo[d]; b.hi[d] = hi[d]; }
  // a box with fewer than TY rows (the paper's ny = 4 guides): tiles of 1, 2 or 4 rows, wider in x
  b.tyr = TY;
  while (b.tyr > 1 && b.tyr / 2 >= hi[1] - lo[1]) b.tyr /= 2;
  const int tw = TX * (TY / b.tyr);
  b.ntx = (hi[0] - lo[0] + tw - 1) / tw;
  b.nty = (hi[1] - lo[1] + b.tyr - 1) / b.tyr;
  const int ez = std::max(0, hi[2] - lo[2]);
  int kz = std::min(KZ_MAX, std::max(1, ez));
  while (kz > 1 && (long long)b.ntx * b.nty * ((ez + kz - 1) / kz) < 8LL * s->num_sms) kz = (kz + 1) / 2;
  b.kz = kz;
  b.items = b.ntx * b.nty * ((ez + kz - 1) / kz);
  return b;
}

// blocks_per_sm == 0: one block per work item (the hardware scheduler balances the load);
// otherwise a persistent grid of num_sms * blocks_per_sm blocks looping over the items
int grid_for(const fdtd_llg *s, const BoxP &b, int blocks_per_sm) {
  if (blocks_per_sm == 0) return std::max(1, b.items);
  const long long want = (long long)s->num_sms * blocks_per_sm;
  return (int)std::max(1LL, std::min<long long>(want, b.items));
}
int grid_1d(const fdtd_llg *s, long long n) {
  return (int)std::max(1LL, std::min<long long>((long long)s->num_sms * 8, (n + 255) / 256));
}

// strided copies between a user's compact array and the ghosted device layout
// (a slab's user arrays carry the neighbours' adjacent planes: k = -ext[0] .. nz - 1 + ext[1])
int copy_in(fdtd_llg *s, double *dev, const double *user, int mem_space) {
  cudaMemcpy3DParms p{};
  p.srcPtr = make_cudaPitchedPtr(const_cast<double *>(user), (size_t)s->g.n[0] * 8, (size_t)s->g.n[0] * 8, (size_t)s->g.n[1]);
  p.dstPtr = make_cudaPitchedPtr(dev, (size_t)s->g.sy * 8, (size_t)s->g.sy * 8, (size_t)s->g.n[1] + 2);
  p.dstPos = make_cudaPos((size_t)PADL * 8, 1, (size_t)(1 - s->g.ext[0]));
  p.extent = make_cudaExtent((size_t)s->g.n[0] * 8, (size_t)s->g.n[1], (size_t)(s->g.n[2] + s->g.ext[0] + s->g.ext[1]));
  p.kind = mem_space == FDTD_LLG_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
  cudaError_t e = cudaMemcpy3DAsync(&p, s->stream);
  if (e != cudaSuccess) { s->err = std::string("cudaMemcpy3DAsync (in): ") + cudaGetErrorString(e); return FDTD_LLG_ECUDA; }
  return FDTD_LLG_OK;
}
int copy_out(fdtd_llg *s, double *user, const double *dev, int mem_space) {
  cudaMemcpy3DParms p{};
  p.srcPtr = make_cudaPitchedPtr(const_cast<double *>(dev), (size_t)s->g.sy * 8, (size_t)s->g.sy * 8, (size_t)s->g.n[1] + 2);
  p.srcPos = make_cudaPos((size_t)PADL * 8, 1, 1);
  p.dstPtr = make_cudaPitchedPtr(user, (size_t)s->g.n[0] * 8, (size_t)s->g.n[0] * 8, (size_t)s->g.n[1]);
  p.extent = make_cudaExtent((size_t)s->g.n[0] * 8, (size_t)s->g.n[1], (size_t)s->g.n[2]);
  p.kind = mem_space == FDTD_LLG_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
  cudaError_t e = cudaMemcpy3DAsync(&p, s->stream);
  if (e != cudaSuccess) { s->err = std::string("cudaMemcpy3DAsync (out): ") + cudaGetErrorString(e); return FDTD_LLG_ECUDA; }
  return FDTD_LLG_OK;
}
int fill_ghosts(fdtd_llg *s, double *dev) {
  const long long total = (long long)(s->g.n[0] + 2) * (s->g.n[1] + 2) * (s->g.n[2] + 2);
  k_fill_ghosts<<<grid_1d(s, total), 256, 0, s->stream>>>(dev, s->g);
  cudaError_t e = cudaGetLastError();
  if (e != cudaSuccess) { s->err = std::string("k_fill_ghosts: ") + cudaGetErrorString(e); return FDTD_LLG_ECUDA; }
  return FDTD_LLG_OK;
}

bool valid_opts(const fdtd_llg_options *o, const char **why) {
  for (int d = 0; d < 3; ++d)
    if (o->bc[d] != FDTD_LLG_PEC && o->bc[d] != FDTD_LLG_PERIODIC) { *why = "bc must be 0 (PEC) or 1 (periodic)"; return false; }
  if (o->time_scheme != 0 && o->time_scheme != 1) { *why = "time_scheme must be 0 (second order) or 1 (first order)"; return false; }
  for (int a = 0; a < 3; ++a)
    for (int sd = 0; sd < 2; ++sd) {
      if (o->pml[2 * a + sd] < 0) { *why = "pml thickness must be >= 0"; return false; }
      if (o->pml[2 * a + sd] > 0 && o->bc[a] != FDTD_LLG_PEC) { *why = "a PML axis must be FDTD_LLG_PEC (the wall behind the layer)"; return false; }
    }
  if (o->pml[0] | o->pml[1] | o->pml[2] | o->pml[3] | o->pml[4] | o->pml[5]) {
    if (!(o->pml_r0 > 0 && o->pml_r0 < 1)) { *why = "pml_r0 must be in (0, 1)"; return false; }
    if (o->pml_order < 1 || o->pml_order > 6) { *why = "pml_order must be in 1..6"; return false; }
  }
  if (o->llg_max_iter < 1 || o->llg_max_iter > 1000) { *why = "llg_max_iter must be in 1..1000"; return false; }
  if (o->kernel_path != 0 && o->kernel_path != 1 && o->kernel_path != 5) { *why = "kernel_path must be 0, 1 or 5"; return false; }
  for (int sd = 0; sd < 2; ++sd) {
    if (o->slab_ext[sd] != 0 && o->slab_ext[sd] != 1) { *why = "slab_ext must be 0 or 1"; return false; }
    if (o->slab_ext[sd] && o->bc[2] != FDTD_LLG_PEC) { *why = "a slab interface needs bc[2] = FDTD_LLG_PEC (a periodic z axis is closed by connecting the end slabs)"; return false; }
    if (o->slab_ext[sd] && o->pml[4 + sd] > 0) { *why = "no PML on a slab interface"; return false; }
  }
  if (o->enable_llg) {
    if (!(o->llg_tol > 0) || !std::isfinite(o->llg_tol)) { *why = "llg_tol must be > 0"; return false; }
    if (o->ani_hk != 0.0) {
      double n2 = 0;
      for (int d = 0; d < 3; ++d) n2 += o->ani_axis[d] * o->ani_axis[d];
      if (!(std::fabs(n2 - 1.0) < 1e-9)) { *why = "ani_axis must be a unit vector"; return false; }
    }
    for (int d = 0; d < 3; ++d)
      if (!std::isfinite(o->h_bias[d])) { *why = "h_bias must be finite"; return false; }
  }
  return true;
}

size_t small_bytes(const fdtd_llg_options *o) {
  size_t b = 0;
  b += 4096;                                                  // DevState
  b += 2 * padded((size_t)(o->llg_max_iter + 2)) * 8 + 4096;  // residual words, item counters
  b += (2 * 1024 + 64) * 8;                                   // reduction scratch
  b += (size_t)1 << 20;                                       // source profiles pool (1 MiB)
  b += (size_t)R_HIST * sizeof(int);                          // iteration counts per half-step
  return (b + 255) / 256 * 256;
}

// min/max of a user array (host or device)
int array_minmax(fdtd_llg *s, const double *a, int mem_space, double *lo, double *hi) {
  const size_t n = s->ncell_user;
  if (mem_space == FDTD_LLG_HOST) {
    double l = INFINITY, h = -INFINITY;
    bool nan = false;
    for (size_t i = 0; i < n; ++i) {
      const double v = a[i];
      if (v != v) nan = true;
      if (v < l) l = v;
      if (v > h) h = v;
    }
    *lo = nan ? NAN : l;
    *hi = nan ? NAN : h;
    return FDTD_LLG_OK;
  }
  const int blocks = 1024;
  k_minmax<<<blocks, 256, 0, s->stream>>>(a, (long long)n, s->scratch);
  CU(s, cudaGetLastError());
  std::vector<double> part(2 * blocks);
  CU(s, cudaMemcpyAsync(part.data(), s->scratch, sizeof(double) * 2 * blocks,
                        cudaMemcpyDeviceToHost, s->stream));
  CU(s, cudaStreamSynchronize(s->stream));
  double l = INFINITY, h = -INFINITY;
  bool nan = false;
  for (int b = 0; b < blocks; ++b) {
    if (part[2 * b] != part[2 * b] || part[2 * b + 1] != part[2 * b + 1]) nan = true;
    l = std::fmin(l, part[2 * b]);
    h = std::fmax(h, part[2 * b + 1]);
  }
  *lo = nan ? NAN : l;
  *hi = nan ? NAN : h;
  return FDTD_LLG_OK;
}

// analyse one material: uniform -> scalar, else copy into the workspace slot
int take_material(fdtd_llg *s, MatInfo *m, const double *user, int mem_space, double dflt,
                  double **slot, const char *name, double min_allowed, bool strict_min,
                  unsigned bit) {
  m->is_array = false;
  m->uniform = dflt;
  m->dev = nullptr;
  if (!user) return FDTD_LLG_OK;
  double lo, hi;
  if (s->opt.scalar_material_mask & bit) {
    lo = hi = *user;  // one HOST double: the uniform value
  } else {
    int rc = array_minmax(s, user, mem_space, &lo, &hi);
    if (rc) return rc;
  }
  if (!(lo == lo) || !std::isfinite(lo) || !std::isfinite(hi))
    return fail(s, FDTD_LLG_EINVAL, "%s contains a non-finite value", name);
  if (strict_min ? !(lo > min_allowed) : !(lo >= min_allowed))
    return fail(s, FDTD_LLG_EINVAL, "%s must be %s %g everywhere (min is %g)", name,
                strict_min ? ">" : ">=", min_allowed, lo);
  m->maxv = hi;
  if (lo == hi) {
    m->uniform = lo;
    return FDTD_LLG_OK;
  }
  m->is_array = true;
  m->dev = *slot;
  *slot += s->stride;
  CU(s, cudaMemsetAsync(m->dev, 0, s->stride * sizeof(double), s->stream));
  int rc = copy_in(s, m->dev, user, mem_space);
  if (rc) return rc;
  return fill_ghosts(s, m->dev);
}

int find_sweep_box(fdtd_llg *s) {
  s->llg = false;
  s->magnetic_cells = 0;
  if (!s->opt.enable_llg) return FDTD_LLG_OK;
  int clo[3], chi[3];  // cell box, inclusive
  if (!s->Ms.is_array) {
    if (!(s->Ms.uniform > 0.0)) return FDTD_LLG_OK;
    for (int d = 0; d < 3; ++d) { clo[d] = 0; chi[d] = s->g.n[d] - 1; }
    clo[2] -= s->g.ext[0];   // a uniform map includes the neighbours' planes
    chi[2] += s->g.ext[1];
    s->magnetic_cells = (long long)s->ncell;
  } else {
    int *box = reinterpret_cast<int *>(s->scratch + 2 * 1024);
    unsigned long long *cnt = reinterpret_cast<unsigned long long *>(s->scratch + 2 * 1024 + 8);
    int init[6] = {INT_MAX, INT_MAX, INT_MAX, INT_MIN, INT_MIN, INT_MIN};
    unsigned long long zero = 0;
    CU(s, cudaMemcpyAsync(box, init, sizeof init, cudaMemcpyHostToDevice, s->stream));
    CU(s, cudaMemcpyAsync(cnt, &zero, sizeof zero, cudaMemcpyHostToDevice, s->stream));
    k_mag_box<<<grid_1d(s, (long long)s->ncell_user), 256, 0, s->stream>>>(s->Ms.dev, s->g, box, cnt);
    CU(s, cudaGetLastError());
    int out[6];
    unsigned long long c = 0;
    CU(s, cudaMemcpyAsync(out, box, sizeof out, cudaMemcpyDeviceToHost, s->stream));
    CU(s, cudaMemcpyAsync(&c, cnt, sizeof c, cudaMemcpyDeviceToHost, s->stream));
    CU(s, cudaStreamSynchronize(s->stream));
    if (out[3] == INT_MIN) return FDTD_LLG_OK;   // no magnetic cell, not even in a neighbour's plane
    for (int d = 0; d < 3; ++d) { clo[d] = out[d]; chi[d] = out[3 + d]; }
    s->magnetic_cells = (long long)c;
  }
  // A D-face at index p is magnetic iff cell p-1 or p is: p in clo..chi+1.  It reads its own H, and
  // through the four-point averages H at p-1, p along D and at t, t+1 along the
  // transverse axis (t in clo..chi): every H a magnetic face reads from the Jacobi buffers has its
  // index in clo-1..chi+1 on every axis.  That is the sweep box.  A box touching a periodic end
  // wraps: take the full axis there.
  for (int d = 0; d < 3; ++d) {
    int l = clo[d] - 1, h = chi[d] + 2;  // exclusive upper bound
    const int n = s->g.n[d];
    if (s->g.per[d] && (l < 0 || h > n)) { l = 0; h = n; }
    s->lo[d] = l < 0 ? 0 : l;
    s->hi[d] = h > n ? n : h;
    if (d == 0) {
      // even start in x for the staged sweeps (their TMA boxes then begin on 16-byte boundaries);
      // not when the extra column would lie in a PML (the layer has its own update there)
      s->lo0_unrounded = s->lo[d];
      if ((s->lo[d] & ~1) >= s->opt.pml[0]) s->lo[d] &= ~1;
    }
  }
  if (s->lo[2] >= s->hi[2]) return FDTD_LLG_OK;  // (cannot happen: a neighbour's magnetic plane reaches into the slab)
  s->llg = true;
  return FDTD_LLG_OK;
}

// outer \ inner as <= 6 disjoint boxes (inner inside outer, not empty): z slabs first (contiguous
// planes), then y, then x
template <class Emit>
void peel(const int olo[3], const int ohi[3], const int ilo[3], const int ihi[3], Emit emit) {
  int lo[3] = {olo[0], olo[1], olo[2]}, hi[3] = {ohi[0], ohi[1], ohi[2]};
  for (int d = 2; d >= 0; --d) {
    if (ilo[d] > lo[d]) {
      int l[3] = {lo[0], lo[1], lo[2]}, h[3] = {hi[0], hi[1], hi[2]};
      h[d] = ilo[d];
      emit(l, h);
    }
    if (ihi[d] < hi[d]) {
      int l[3] = {lo[0], lo[1], lo[2]}, h[3] = {hi[0], hi[1], hi[2]};
      l[d] = ihi[d];
      emit(l, h);
    }
    lo[d] = ilo[d];
    hi[d] = ihi[d];
  }
}
bool clip(const int alo[3], const int ahi[3], const int blo[3], const int bhi[3], int lo[3], int hi[3]) {
  bool any = true;
  for (int d = 0; d < 3; ++d) {
    lo[d] = std::max(alo[d], blo[d]);
    hi[d] = std::min(ahi[d], bhi[d]);
    any = any && lo[d] < hi[d];
  }
  return any;
}

// work decomposition: the sweep box, the whole grid, the complement of the box (within the interior
// when the H half-steps are merged) as <= 6 slabs, and the unmerged margins minus the box
void make_boxes(fdtd_llg *s) {
  const int zero[3] = {0, 0, 0};
  s->box_all = make_box(s, zero, s->g.n);
  s->n_out = 0;
  s->box_um.clear();
  if (s->llg) s->box_llg = make_box(s, s->lo, s->hi);
  int ilo[3] = {0, 0, 0}, ihi[3] = {s->g.n[0], s->g.n[1], s->g.n[2]};   // the interior
  if (s->merge)
    for (int d = 0; d < 3; ++d) { ilo[d] = s->um_lo[d]; ihi[d] = s->g.n[d] - s->um_hi[d]; }
  auto out = [&](const int *l, const int *h) { s->box_out[s->n_out++] = make_box(s, l, h); };
  auto um = [&](const int *l, const int *h) { s->box_um.push_back(make_box(s, l, h)); };
  int blo[3], bhi[3];
  if (s->llg && clip(ilo, ihi, s->lo, s->hi, blo, bhi)) peel(ilo, ihi, blo, bhi, out);
  else out(ilo, ihi);
  if (s->merge)
    peel(zero, s->g.n, ilo, ihi, [&](const int *l, const int *h) {   // the margins, each minus the box
      if (s->llg && clip(l, h, s->lo, s->hi, blo, bhi)) peel(l, h, blo, bhi, um);
      else um(l, h);
    });
}

// ---- tensor maps for the staged sweeps -------------------------------------------------------


typedef CUresult (*EncodeTiledFn)(CUtensorMap *, CUtensorMapDataType, cuuint32_t, void *,
                                  const cuuint64_t *, const cuuint64_t *, const cuuint32_t *,
                                  const cuuint32_t *, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

// cuTensorMapEncodeTiled through the runtime's driver entry point (no link against libcuda)
EncodeTiledFn encode_tiled_fn() {
  static EncodeTiledFn fn = nullptr;
  if (!fn) {
    void *p = nullptr;
    cudaDriverEntryPointQueryResult q;
    if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess &&
        q == cudaDriverEntryPointSuccess)
      fn = reinterpret_cast<EncodeTiledFn>(p);
  }
  return fn;
}

// tensor map over ALL arrays of the workspace: (x = row pitch, y = ny+2, z = nz+2, a = array),
// box = (bx, by, 1, ba) elements
int make_map(fdtd_llg *s, CUtensorMap *m, int bx, int by, int ba) {
  EncodeTiledFn enc = encode_tiled_fn();
  if (!enc) return fail(s, FDTD_LLG_ECUDA, "cuTensorMapEncodeTiled is not available");
  const cuuint64_t dims[4] = {(cuuint64_t)s->g.sy, (cuuint64_t)s->g.n[1] + 2, (cuuint64_t)s->g.n[2] + 2,
                              (cuuint64_t)s->n_arrays};
  const cuuint64_t strides[3] = {(cuuint64_t)s->g.sy * 8, (cuuint64_t)s->g.sz * 8, (cuuint64_t)s->stride * 8};
  const cuuint32_t box[4] = {(cuuint32_t)bx, (cuuint32_t)by, 1u, (cuuint32_t)ba};
  const cuuint32_t estr[4] = {1, 1, 1, 1};
  CUresult r = enc(m, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 4, s->E[0], dims, strides, box, estr,
                   CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                   CU_TENSOR_MAP_L2_PROMOTION_L2_128B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(s, FDTD_LLG_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  return FDTD_LLG_OK;
}

int array_index(const fdtd_llg *s, const double *p) { return (int)((p - s->E[0]) / (ptrdiff_t)s->stride); }

// ---- staged sweeps (hm_stage.cuh) ----------------------------------------------------------

// SW x by columns marched over ~kz_target planes; a persistent grid draws the items dynamically in
// the order x, y, z.  Short items keep the blocks that run at the same time on the same few planes
// (neighbouring tiles: their rims hit in L2, DRAM pages are shared) and balance the SMs; every
// item costs one extra stage.  Measured at 768^3: the iterates r >= 2 are fastest at 8-16 planes
// (14.1 ms at 97, 12.3 ms at 8), the r = 1 sweep at about 32.
StBox make_stbox(const int lo[3], const int hi[3], int by, int kz_target) {
  StBox b{};
  for (int d = 0; d < 3; ++d) { b.lo[d] = lo[d]; b.hi[d] = hi[d]; }
  b.ntx = (hi[0] - lo[0] + SW - 1) / SW;
  b.nty = (hi[1] - lo[1] + by - 1) / by;
  const int ez = std::max(1, hi[2] - lo[2]);
  const int nc = std::max(1, (ez + kz_target / 2) / kz_target);   // chunks of about kz_target planes
  b.kz = (ez + nc - 1) / nc;
  b.items = (int)((long long)b.ntx * b.nty * ((ez + b.kz - 1) / b.kz));
  return b;
}

template <bool FIRST>
int launch_hm_stage(fdtd_llg *s, const HMSArgs &p) {
  const bool ms = s->Ms.is_array, an = s->opt.ani_hk != 0.0;
  const int grid = std::max(1, std::min(p.tb.items, s->num_sms));   // one persistent block per SM
#define SK(MS, AN)                                                                          \
  if (ms == MS && an == AN) {                                                               \
    using L = StLayout<FIRST, MS>;                                                          \
    k_hm_stage<FIRST, MS, AN><<<grid, L::NTHREADS, L::SMEM_BYTES, s->stream>>>(p);          \
    return FDTD_LLG_OK;                                                                     \
  }
  SK(false, false) SK(false, true) SK(true, false) SK(true, true)
#undef SK
  return FDTD_LLG_OK;
}

int setup_hm_stage(fdtd_llg *s) {
#define SA(FIRST, MS, AN)                                                                   \
  CU(s, cudaFuncSetAttribute(k_hm_stage<FIRST, MS, AN>,                                     \
                             cudaFuncAttributeMaxDynamicSharedMemorySize,                   \
                             (int)StLayout<FIRST, MS>::SMEM_BYTES));
#define SA4(FIRST) SA(FIRST, false, false) SA(FIRST, false, true) SA(FIRST, true, false) SA(FIRST, true, true)
  SA4(true) SA4(false)
#undef SA4
#undef SA
  int rc;
  if ((rc = make_map(s, &s->mapT, SROW, SBY + 1, 1))) return rc;
  if ((rc = make_map(s, &s->mapPM, SW, SBY, 9))) return rc;
  s->st_box_first = make_stbox(s->lo, s->hi, SBY, 32);
  s->st_box = make_stbox(s->lo, s->hi, SBY, 8);
  // A sweep box that cannot give every SM an item (a thin slab, a small grid) is latency bound:
  // the direct-load kernels with their 32 x 8 x 16 blocks fill the GPU better there (32^3: 9 us
  // against 79 us per sweep; the bits are the same).
  if (s->opt.kernel_path == 0 && s->st_box.items < s->num_sms) s->staged = false;
  // ... and so is one whose 16-row tiles would be mostly empty (a box of a few rows: the paper's
  // ny = 4 guides): the direct-load kernels have 1-, 2- and 4-row tiles
  const int rows = s->hi[1] - s->lo[1], slots = (rows + SBY - 1) / SBY * SBY;
  if (s->opt.kernel_path == 0 && 5 * rows < 3 * slots) s->staged = false;
  return FDTD_LLG_OK;
}

// ---- staged Maxwell sweeps (eh_stage.cuh) ----------------------------------------------------

// Work items of a staged Maxwell sweep.  Long items amortise the two extra planes a fused item
// stages (k0-1 and k1) and its cold start; short ones balance the SMs when the region has few
// tiles and keep the blocks that run together on the same few planes.  Measured (k_eh_fused):
// 256^3 4.7-4.9 TB/s at 8-24 planes, 4.4 at 32, 3.8 at 64; 512x128x128 (two material arrays) 3.8 at
// 8, 4.0 at 12-24; 384^3 4.7 at 8, 5.0 at 12-16, 5.2-5.3 at 24-32: the longest of 32, 24, 16, 12
// planes that still gives every SM eight items.
StBox make_ehbox(const fdtd_llg *s, const int lo[3], const int hi[3], bool fuse) {
  const int by = fuse ? FBY : SBY;   // tile rows of k_eh_fused / k_eh_stage
  const int cand[4] = {32, 24, 16, 12};
  StBox b{};
  for (int q = 0; q < 4; ++q) {
    b = make_stbox(lo, hi, by, cand[q]);
    if (b.items >= 8 * s->num_sms) break;
  }
  return b;
}

template <bool FUSE>
int launch_eh_stage(fdtd_llg *s, const EHArgs &p) {
  const bool ea = s->eps_r.is_array, sa = s->sigma.is_array;
  bool hs = false;
  for (int q = 0; q < s->src.count; ++q) hs = hs || s->src.s[q].kind == FDTD_LLG_SRC_SOFT_E;
  const int grid = std::max(1, std::min(p.tb.items, s->num_sms));   // one persistent block per SM
#define EK(EA, SA, HS)                                                                          \
  if (ea == EA && sa == SA && hs == HS) {                                                       \
    if (FUSE) {                                                                                 \
      using L = EfLayout<EA, SA>;                                                               \
      k_eh_fused<EA, SA, HS><<<grid, L::NTHREADS, L::SMEM_BYTES, s->stream>>>(p);               \
    } else {                                                                                    \
      using L = EhLayout<EA, SA>;                                                               \
      k_eh_stage<EA, SA, HS><<<grid, L::NTHREADS, L::SMEM_BYTES, s->stream>>>(p);               \
    }                                                                                           \
    return FDTD_LLG_OK;                                                                         \
  }
  EK(false, false, false) EK(false, false, true) EK(false, true, false) EK(false, true, true)
  EK(true, false, false) EK(true, false, true) EK(true, true, false) EK(true, true, true)
#undef EK
  return FDTD_LLG_OK;
}

int setup_eh_stage(fdtd_llg *s) {
#define SA(EA, SA_, HS)                                                                         \
  CU(s, cudaFuncSetAttribute(k_eh_stage<EA, SA_, HS>,                                           \
                             cudaFuncAttributeMaxDynamicSharedMemorySize,                       \
                             (int)EhLayout<EA, SA_>::SMEM_BYTES));                              \
  CU(s, cudaFuncSetAttribute(k_eh_fused<EA, SA_, HS>,                                           \
                             cudaFuncAttributeMaxDynamicSharedMemorySize,                       \
                             (int)EfLayout<EA, SA_>::SMEM_BYTES));
  SA(false, false, false) SA(false, false, true) SA(false, true, false) SA(false, true, true)
  SA(true, false, false) SA(true, false, true) SA(true, true, false) SA(true, true, true)
#undef SA
  int rc = make_map(s, &s->mapEH, EW, EROWS, 1);
  if (rc) return rc;
  if ((rc = make_map(s, &s->mapEF, EW, FROWS, 1))) return rc;
  s->eh_ok = true;
  return FDTD_LLG_OK;
}

// ---- open boundary (A26) ---------------------------------------------

// decay rate s_a(x) of the layer on axis a at position x (host, long double)
long double pml_rate(const fdtd_llg *s, int a, long double x) {
  const long double dx = s->d[a], len = s->g.n[a] * dx;
  const int plo = s->opt.pml[2 * a], phi = s->opt.pml[2 * a + 1];
  long double L, u;
  if (plo > 0 && x < (L = plo * dx)) u = L - x;
  else if (phi > 0 && x > len - (L = phi * dx)) u = x - (len - L);
  else return 0.0L;
  const long double smax = -(s->opt.pml_order + 1) * (long double)kC0 * logl((long double)s->opt.pml_r0) / (2 * L);
  return smax * powl(u / L, s->opt.pml_order);
}

// split parts, damping tables and the slabs of the layer; *q = next free array of the workspace
int setup_pml(fdtd_llg *s, double **q) {
  const int *pm = s->opt.pml;
  s->has_pml = (pm[0] | pm[1] | pm[2] | pm[3] | pm[4] | pm[5]) != 0;
  if (!s->has_pml) return FDTD_LLG_OK;
  for (int a = 0; a < 3; ++a)
    if (pm[2 * a] + pm[2 * a + 1] > s->g.n[a]) return fail(s, FDTD_LLG_EINVAL, "the PML is thicker than the grid on axis %d", a);
  if (s->llg)  // the sweep box (magnetic cells + 1) must stay clear of the layer
    for (int a = 0; a < 3; ++a)
      if (s->lo[a] < pm[2 * a] || s->hi[a] > s->g.n[a] - pm[2 * a + 1])
        return fail(s, FDTD_LLG_EINVAL, "magnetic cells touch the PML on axis %d (PAPER.md:189: not supported)", a);
  const size_t abytes = s->stride * sizeof(double);
  for (int c = 0; c < 6; ++c) { s->Esp[c] = *q; *q += s->stride; }
  for (int c = 0; c < 6; ++c) { s->Hsp[c] = *q; *q += s->stride; }
  CU(s, cudaMemsetAsync(s->Esp[0], 0, 12 * abytes, s->stream));
  double *tab = *q;
  *q += s->stride;
  std::vector<double> host;
  for (int a = 0; a < 3; ++a) {
    s->pdE[a] = tab + host.size();
    for (int i = 0; i < s->g.n[a]; ++i)  // E parts: nodes of axis a, half the damping of one step dt
      host.push_back((double)expl(-pml_rate(s, a, i * (long double)s->d[a]) * (long double)s->dt / 2));
    s->pdH[a] = tab + host.size();
    for (int i = 0; i < s->g.n[a]; ++i)  // H parts: half positions, half the damping of dt/2
      host.push_back((double)expl(-pml_rate(s, a, (i + 0.5L) * (long double)s->d[a]) * (long double)s->dt / 4));
  }
  CU(s, cudaMemcpyAsync(tab, host.data(), host.size() * sizeof(double), cudaMemcpyHostToDevice, s->stream));
  CU(s, cudaStreamSynchronize(s->stream));
  // the layer = complement of the interior box, peeled into <= 6 disjoint slabs (z, then y, then x)
  int lo[3] = {0, 0, 0}, hi[3] = {s->g.n[0], s->g.n[1], s->g.n[2]};
  s->n_pml = 0;
  for (int d = 2; d >= 0; --d) {
    const int il = pm[2 * d], ih = s->g.n[d] - pm[2 * d + 1];
    if (il > lo[d]) {
      int l[3] = {lo[0], lo[1], lo[2]}, h[3] = {hi[0], hi[1], hi[2]};
      h[d] = il;
      s->box_pml[s->n_pml++] = make_box(s, l, h);
    }
    if (ih < hi[d]) {
      int l[3] = {lo[0], lo[1], lo[2]}, h[3] = {hi[0], hi[1], hi[2]};
      l[d] = ih;
      s->box_pml[s->n_pml++] = make_box(s, l, h);
    }
    lo[d] = il;
    hi[d] = ih;
  }
  return FDTD_LLG_OK;
}

// the layer's update of E (after k_e_update) or of H (after the H half-step): In = the other field
int enqueue_pml(fdtd_llg *s, bool is_e, double *const *In, double *const *Out, int *launches) {
  if (!s->has_pml) return FDTD_LLG_OK;
  PmlArgs a{};
  a.g = s->g;
  for (int d = 0; d < 3; ++d) {
    a.In[d] = In[d];
    a.Out[d] = Out[d];
    a.d[d] = is_e ? s->pdE[d] : s->pdH[d];
  }
  for (int c = 0; c < 6; ++c) a.P[c] = is_e ? s->Esp[c] : s->Hsp[c];
  a.eps_r = s->eps_r.is_array ? s->eps_r.dev : nullptr;
  a.sigma = s->sigma.is_array ? s->sigma.dev : nullptr;
  a.mu_r = s->mu_r.is_array ? s->mu_r.dev : nullptr;
  a.eps_u = kEps0 * s->eps_r.uniform;
  a.sigma_u = s->sigma.uniform;
  a.mu_u = kMu0 * s->mu_r.uniform;
  a.src = s->src;
  a.st = s->dstate;
  const dim3 blk(TX, TY, 1);
  for (int b = 0; b < s->n_pml; ++b) {
    a.box = s->box_pml[b];
    if (a.box.items == 0) continue;
    prof_begin(s, FDTD_LLG_K_OTHER, 0);
    if (is_e) k_pml<true><<<grid_for(s, a.box, 0), blk, 0, s->stream>>>(a);
    else k_pml<false><<<grid_for(s, a.box, 0), blk, 0, s->stream>>>(a);
    prof_end(s);
    ++*launches;
  }
  CU(s, cudaGetLastError());
  return FDTD_LLG_OK;
}

// ---- launching one step ----------------------------------------------------------------

template <bool FIRST>
int launch_sweep(fdtd_llg *s, const HMArgs &a, int grid) {
  const dim3 blk(TX, TY, 1);
  const bool ms = s->Ms.is_array, ag = s->alpha.is_array || s->gamma.is_array,
             mu = s->mu_r.is_array, an = s->opt.ani_hk != 0.0;
#define SW(MS, AG, MU, AN)                                                               \
  if (ms == MS && ag == AG && mu == MU && an == AN) {                                    \
    k_hm_sweep<FIRST, MS, AG, MU, AN><<<grid, blk, 0, s->stream>>>(a);                   \
    return FDTD_LLG_OK;                                                                  \
  }
  SW(false, false, false, false) SW(false, false, false, true) SW(false, false, true, false)
  SW(false, false, true, true) SW(false, true, false, false) SW(false, true, false, true)
  SW(false, true, true, false) SW(false, true, true, true) SW(true, false, false, false)
  SW(true, false, false, true) SW(true, false, true, false) SW(true, false, true, true)
  SW(true, true, false, false) SW(true, true, false, true) SW(true, true, true, false)
  SW(true, true, true, true)
#undef SW
  return FDTD_LLG_OK;
}

// The launches from here to end_cond_tail are captured into the body of an IF node of the step's
// graph; k_set_cond arms it when iterate r_next - 1 ran and missed the tolerance.
int begin_cond_tail(fdtd_llg *s, int r_next, cudaStream_t *outer) {
  cudaStreamCaptureStatus st;
  cudaGraph_t g = nullptr;
  const cudaGraphNode_t *deps = nullptr;
  size_t nd = 0;
  CU(s, cudaStreamGetCaptureInfo_v2(s->stream, &st, nullptr, &g, &deps, &nd));
  if (st != cudaStreamCaptureStatusActive || !g) return fail(s, FDTD_LLG_ESTATE, "begin_cond_tail outside a capture");
  cudaGraphConditionalHandle h;
  CU(s, cudaGraphConditionalHandleCreate(&h, g, 0, cudaGraphCondAssignDefault));
  k_set_cond<<<1, 1, 0, s->stream>>>(h, s->resid, s->opt.llg_tol, r_next);
  CU(s, cudaGetLastError());
  CU(s, cudaStreamGetCaptureInfo_v2(s->stream, &st, nullptr, &g, &deps, &nd));
  cudaGraphNodeParams np{};
  np.type = cudaGraphNodeTypeConditional;
  np.conditional.handle = h;
  np.conditional.type = cudaGraphCondTypeIf;
  np.conditional.size = 1;
  cudaGraphNode_t node;
  CU(s, cudaGraphAddNode(&node, g, deps, nd, &np));
  cudaGraph_t body = np.conditional.phGraph_out[0];
  CU(s, cudaStreamUpdateCaptureDependencies(s->stream, &node, 1, cudaStreamSetCaptureDependencies));
  CU(s, cudaStreamBeginCaptureToGraph(s->aux, body, nullptr, nullptr, 0, cudaStreamCaptureModeThreadLocal));
  *outer = s->stream;
  s->stream = s->aux;
  return FDTD_LLG_OK;
}

int end_cond_tail(fdtd_llg *s, cudaStream_t outer) {
  cudaGraph_t body = nullptr;
  cudaError_t e = cudaStreamEndCapture(s->aux, &body);
  s->stream = outer;
  if (e != cudaSuccess) return fail(s, FDTD_LLG_ECUDA, "cudaStreamEndCapture (IF body): %s", cudaGetErrorString(e));
  return FDTD_LLG_OK;
}

// ---- which H set holds what ------------------------------------
// Two half-steps everywhere (merge off): H^n in set 0, H^{n+1/2} in set 1, Jacobi buffer set 2.
// Merged H half-steps: the faces OUTSIDE the sweep box live at half-integer time and ping-pong
// between two sets, one read by the E update of even steps, the other by that of odd steps
// (every update stays out of place); the box uses the same set for its H^{n+1/2} and the other
// one as Jacobi buffer (disjoint regions).  With LLG storage these are sets 1 and 2 and the box's
// H^n stays in set 0; a Maxwell-only handle has two sets, 1 and 0.
int set_half(const fdtd_llg *s, int par) {
  if (!s->merge) return 1;
  return s->opt.enable_llg ? (par ? 2 : 1) : (par ? 0 : 1);
}
int set_tmp(const fdtd_llg *s, int par) {
  if (!s->merge) return 2;
  return s->opt.enable_llg ? (par ? 1 : 2) : 2;   // Maxwell-only: no sweep ever uses it
}
// Can the H half-steps be merged (options.merge_h), and outside which margins?  The PML layer takes
// two damped half-steps per step and an H source acts on H at integer time: their faces keep the
// plain half-steps.  An H source box must lie within 8 cells of a side of the grid (the paper's
// excitations sit on a wall plane), else nothing is merged.
constexpr int UM_MAX = 8;
bool decide_merge(fdtd_llg *s) {
  for (int d = 0; d < 3; ++d) { s->um_lo[d] = s->opt.pml[2 * d]; s->um_hi[d] = s->opt.pml[2 * d + 1]; }
  if (!s->opt.merge_h) return false;
  for (int q = 0; q < s->src.count; ++q) {
    const SourceP &S = s->src.s[q];
    if (S.kind != FDTD_LLG_SRC_SOFT_H && S.kind != FDTD_LLG_SRC_HARD_H) continue;
    int best = INT_MAX, bd = 0, bside = 0;
    for (int d = 0; d < 3; ++d) {
      // an interface to a neighbouring slab is not a side of the grid: the handle on the whole grid
      // would not see one there, and the slabs must decide as it does (bit-for-bit contract)
      const bool side_lo = !(d == 2 && s->g.ext[0]), side_hi = !(d == 2 && s->g.ext[1]);
      if (side_lo && S.hi[d] < best) { best = S.hi[d]; bd = d; bside = 0; }                         // from the low side
      if (side_hi && s->g.n[d] - S.lo[d] < best) { best = s->g.n[d] - S.lo[d]; bd = d; bside = 1; } // from the high side
    }
    if (best > std::max(UM_MAX, bside ? s->um_hi[bd] : s->um_lo[bd])) return false;
    if (bside) s->um_hi[bd] = std::max(s->um_hi[bd], best); else s->um_lo[bd] = std::max(s->um_lo[bd], best);
  }
  for (int d = 0; d < 3; ++d)
    if (s->um_lo[d] + s->um_hi[d] >= s->g.n[d]) return false;   // nothing left to merge
  return true;
}

// Maxwell update of the faces outside the sweep box (eq. 21 with M = 0):
// set `out` = set `in` - cmul (dt / 2 mu) curl E; cmul = 1: half a step, 2: two half-steps at once
// The E phase by regions.  The LLG sweep box and the slabs of its complement each get one launch:
//   staged  the TMA-fed sweep of eh_stage.cuh (else the direct-load kernel k_e_update);
//   fuse    the sweep also takes the merged H update of the region (merge_h): its faces are then
//           skipped by the second half-step's enqueue_outside.
struct ERegion {
  int lo[3], hi[3];
  bool staged, fuse;
  int kind;   // 0: a slab of the complement of the sweep box (merged H: of the interior), 1: a piece of
              // the unmerged margins, 2: the sweep box, 3: the whole grid (one direct-load launch)
};
constexpr int MAX_REG = 64;
enum { OUT_ALL = 0, OUT_LEFTOVER = 1, OUT_MARGINS = 2 };
int plan_e_regions(const fdtd_llg *s, ERegion *out);
bool fold_bookkeeping(const fdtd_llg *s);
int count_sources(const fdtd_llg *s, int kind);
// which = OUT_ALL: every slab of box_out; OUT_LEFTOVER: those whose merged update the E phase did not
// take along (not fused); OUT_MARGINS: the unmerged margins
int enqueue_outside(fdtd_llg *s, double *const *E, int in, int out, double cmul, bool exports, int *launches,
                    int which = OUT_ALL) {
  const dim3 blk(TX, TY, 1);
  HArgs h{};
  h.g = s->g;
  if (!exports) h.g.dlo = h.g.dhi = 0;
  for (int d = 0; d < 3; ++d) { h.E[d] = E[d]; h.Hn[d] = s->Hset[in][d]; h.Hc[d] = s->Hset[out][d]; }
  h.mu_r = s->mu_r.is_array ? s->mu_r.dev : nullptr;
  h.ch_uniform = s->dt / (2.0 * kMu0 * s->mu_r.uniform);
  h.cmul = cmul;
  std::vector<BoxP> boxes;
  if (which == OUT_MARGINS) {
    boxes = s->box_um;
  } else if (which == OUT_ALL) {
    boxes.assign(s->box_out, s->box_out + s->n_out);
  } else {
    ERegion reg[MAX_REG];
    const int nr = plan_e_regions(s, reg);
    if (nr == 1 && reg[0].kind == 3) {
      boxes.assign(s->box_out, s->box_out + s->n_out);
    } else {
      for (int r = 0; r < nr; ++r)
        if (reg[r].kind == 0 && !reg[r].fuse) boxes.push_back(make_box(s, reg[r].lo, reg[r].hi));
    }
  }
  for (size_t b = 0; b < boxes.size(); ++b) {
    h.box = boxes[b];
    if (h.box.items == 0) continue;
    const int grid = grid_for(s, h.box, 0);
    prof_begin(s, FDTD_LLG_K_H_UPDATE, 0);
    if (s->mu_r.is_array) k_h_update<true><<<grid, blk, 0, s->stream>>>(h);
    else k_h_update<false><<<grid, blk, 0, s->stream>>>(h);
    prof_end(s);
    ++*launches;
  }
  CU(s, cudaGetLastError());
  return FDTD_LLG_OK;
}

// (H,M) half-step, part 1: the faces outside the sweep box and the open-boundary layer.
// Merged H half-steps: nothing in the first half-step; in the second one (merged_to >= 0) the
// second half of this step and the first half of the next are taken at once, both with curl E^{n+1}
// (PAPER.md:94), from the set the E update read into the set the next E update will read.
int enqueue_half_pre(fdtd_llg *s, double *const *E, int in, int out, int merged_to, int *launches) {
  int rc = FDTD_LLG_OK;
  if (!s->merge) {
    rc = enqueue_outside(s, E, in, out, 1.0, true, launches);
  } else {
    // the margins (PML layer, H-source planes) take the plain half-step; in a Maxwell-only handle
    // `in` and `out` are the same set on odd steps: the update is pointwise, in place is fine
    rc = enqueue_outside(s, E, in, out, 1.0, true, launches, OUT_MARGINS);
    if (!rc && merged_to >= 0) rc = enqueue_outside(s, E, in, merged_to, 2.0, true, launches, OUT_LEFTOVER);
  }
  if (rc) return rc;
  return enqueue_pml(s, false, E, s->Hset[out], launches);
}

// (H,M) half-step, part 2: LLG iterate r on the sweep box.  Time-n set `in`, result in set `out`,
// `tmp` is the other Jacobi buffer (odd r writes `out`, even r `tmp`); M: time-n set `min`, iterate
// in set `mout`.
int enqueue_sweep(fdtd_llg *s, double *const *E, int in, int out, int tmp, int min, int mout, int r,
                  int *launches) {
  HMArgs a{};
  a.g = s->g;
  a.box = s->box_llg;
  for (int d = 0; d < 3; ++d) { a.E[d] = E[d]; a.Hn[d] = s->Hset[in][d]; }
  for (int q = 0; q < 9; ++q) { a.Mn[q] = s->Mset[min][q]; a.Mr[q] = s->Mset[mout][q]; }
  a.Ms = s->Ms.dev; a.alpha = s->alpha.dev; a.gamma = s->gamma.dev; a.mu_r = s->mu_r.dev;
  a.Ms_u = s->Ms.uniform; a.alpha_u = s->alpha.uniform; a.gamma_u = std::fabs(s->gamma.uniform);
  a.cf_u = kMu0 * a.gamma_u * s->dt * 0.25;   // the device expression, evaluated once
  a.kh = s->dt / (2.0 * kMu0);
  a.rMs_u = s->Ms.uniform > 0.0 ? 1.0 / s->Ms.uniform : 0.0;
  if (s->staged && s->Ms.is_array) {  // the most common face value and its reciprocal
    a.Ms_u = s->Ms.maxv;
    a.rMs_u = 1.0 / s->Ms.maxv;
  }
  a.ch_uniform = s->dt / (2.0 * kMu0 * s->mu_r.uniform);
  for (int d = 0; d < 3; ++d) { a.hb[d] = s->opt.h_bias[d]; a.u[d] = s->opt.ani_axis[d]; }
  a.hk = s->opt.ani_hk;
  a.tol = s->opt.llg_tol;
  a.euler = s->opt.time_scheme == 1;
  a.resid = s->resid;
  a.pipe_error = &s->dstate->pipe_error;
  // r <= 3 normally run: one block per item.  Later iterates almost never run: a small
  // persistent grid keeps their early exit at launch-latency cost.
  const int grid = grid_for(s, a.box, r <= 3 ? 0 : 4);
  // iterate r reads H^{r-1} and writes H^r: odd r -> `out`, even r -> `tmp`
  const int from = (r == 1) ? in : ((r & 1) ? tmp : out);
  const int to = (r & 1) ? out : tmp;
  for (int d = 0; d < 3; ++d) { a.Hp[d] = s->Hset[from][d]; a.Hc[d] = s->Hset[to][d]; }
  a.r = r;
  prof_begin(s, r == 1 ? FDTD_LLG_K_HM_FIRST : FDTD_LLG_K_HM_ITER, r);
  int rc;
  if (s->staged) {
    HMSArgs p{};
    p.a = a;
    p.tb = r == 1 ? s->st_box_first : s->st_box;
    p.mapT = s->mapT; p.mapM = s->mapPM;
    p.aE = array_index(s, a.E[0]); p.aHn = array_index(s, a.Hn[0]); p.aHp = array_index(s, a.Hp[0]);
    p.aMn = array_index(s, a.Mn[0]); p.aMp = array_index(s, a.Mr[0]);
    p.aMs = a.Ms ? array_index(s, a.Ms) : 0;
    p.work = s->work + r;
    p.cond = r > 1;
    rc = (r == 1) ? launch_hm_stage<true>(s, p) : launch_hm_stage<false>(s, p);
  } else {
    rc = (r == 1) ? launch_sweep<true>(s, a, grid) : launch_sweep<false>(s, a, grid);
  }
  prof_end(s);
  if (rc) return rc;
  ++*launches;
  CU(s, cudaGetLastError());
  return FDTD_LLG_OK;
}

// (H,M) half-step, part 3: iteration count and statistics from the residual words of the r_max
// iterates that were enqueued, the canonical H set
int enqueue_half_end(fdtd_llg *s, int out, int tmp, int r_max, bool last, int *launches) {
  if (fold_bookkeeping(s)) {   // done by the step's fused Maxwell launch
    if (s->prof) s->prof_half++;
    return FDTD_LLG_OK;
  }
  const dim3 blk(TX, TY, 1);
  prof_begin(s, FDTD_LLG_K_OTHER, 0);
  k_half_end<<<1, 1, 0, s->stream>>>(s->dstate, s->resid, s->work, s->work_eh, s->r_hist, r_max, s->opt.llg_max_iter,
                                     s->opt.llg_tol, s->llg ? 1 : 0, last ? 1 : 0);
  ++*launches;
  if (s->llg && r_max >= 2) {
    CanonArgs c{};
    c.g = s->g;
    c.box = s->box_llg;
    for (int d = 0; d < 3; ++d) { c.src[d] = s->Hset[tmp][d]; c.dst[d] = s->Hset[out][d]; }
    c.st = s->dstate;
    k_canon<<<grid_for(s, c.box, 8), blk, 0, s->stream>>>(c);
    ++*launches;
  }
  prof_end(s);
  if (s->prof) s->prof_half++;
  CU(s, cudaGetLastError());
  return FDTD_LLG_OK;
}

// the whole half-step as fdtd_llg_step enqueues it
int enqueue_half(fdtd_llg *s, double *const *E, int in, int out, int tmp, int min, int mout, bool last,
                 int merged_to, int *launches) {
  int rc = enqueue_half_pre(s, E, in, out, merged_to, launches);
  if (rc) return rc;
  if (s->llg) {
    cudaStream_t outer = nullptr;  // set while the launches go into the body of the IF node
    int body_launches = 0;
    int *cnt = launches;
    for (int r = 1; r <= s->opt.llg_max_iter && !rc; ++r) {
      // Iterates r >= 4 almost never run.  In the captured step they sit in ONE conditional (IF)
      // node armed on the device by k_set_cond, so the usual step does not even launch them.
      // (The node itself costs about as much as ten empty launches: only worth it for a long tail.)
      if (r == 4 && s->capturing && s->aux && s->opt.use_graph == 1 && s->opt.llg_max_iter >= 12) {
        rc = begin_cond_tail(s, r, &outer);
        if (rc) break;
        ++*launches;  // k_set_cond
        cnt = &body_launches;
      }
      rc = enqueue_sweep(s, E, in, out, tmp, min, mout, r, cnt);
    }
    if (outer) {  // on every exit: close the body capture, give the handle its stream back
      const int rc2 = end_cond_tail(s, outer);
      if (!rc) rc = rc2;
    }
    if (rc) return rc;
  }
  return enqueue_half_end(s, out, tmp, s->opt.llg_max_iter, last, launches);
}

int count_sources(const fdtd_llg *s, int kind) {
  int n = 0;
  for (int q = 0; q < s->src.count; ++q) n += s->src.s[q].kind == kind;
  return n;
}

// eq. 11 on one region of the grid with the direct-load kernel
int enqueue_e(fdtd_llg *s, double *const *Ein, double *const *Eout, int hset, const BoxP &box, int *launches) {
  const dim3 blk(TX, TY, 1);
  EArgs a{};
  a.g = s->g;
  a.box = box;
  for (int d = 0; d < 3; ++d) { a.E[d] = Ein[d]; a.Eo[d] = Eout[d]; a.H[d] = s->Hset[hset][d]; }
  a.eps_r = s->eps_r.dev; a.sigma = s->sigma.dev;
  a.eps_u = kEps0 * s->eps_r.uniform; a.sigma_u = s->sigma.uniform;
  a.rdt = 1.0 / s->dt;
  a.k_u = e_coef(a.eps_u, a.sigma_u, a.rdt);
  a.src = s->src;
  a.st = s->dstate;
  const int grid = grid_for(s, a.box, 0);
  const bool ea = s->eps_r.is_array, sa = s->sigma.is_array, hs = count_sources(s, FDTD_LLG_SRC_SOFT_E) > 0;
#define EK(EA, SA, HS)                                                        \
  if (ea == EA && sa == SA && hs == HS) k_e_update<EA, SA, HS><<<grid, blk, 0, s->stream>>>(a);
  prof_begin(s, FDTD_LLG_K_E_UPDATE, 0);
  EK(false, false, false) EK(false, false, true) EK(false, true, false) EK(false, true, true)
  EK(true, false, false) EK(true, false, true) EK(true, true, false) EK(true, true, true)
#undef EK
  prof_end(s);
  ++*launches;
  CU(s, cudaGetLastError());
  return FDTD_LLG_OK;
}

int plan_e_regions(const fdtd_llg *s, ERegion *out) {
  const int zero[3] = {0, 0, 0};
  auto put = [&](int n, const int *lo, const int *hi, bool staged, bool fuse, int kind) {
    for (int d = 0; d < 3; ++d) { out[n].lo[d] = lo[d]; out[n].hi[d] = hi[d]; }
    out[n].staged = staged;
    out[n].fuse = fuse;
    out[n].kind = kind;
    return n + 1;
  };
  // a staged box begins on a 16-byte boundary, and its tiles (15 or 16 rows) must not be mostly empty:
  // on a thin grid (the paper's ny = 4 guides) the direct-load kernels with their 1-, 2-, 4-row tiles do better
  auto stageable = [&](const int *lo, const int *hi, int by) {
    const int rows = hi[1] - lo[1], slots = (rows + by - 1) / by * by;
    return (lo[0] & 1) == 0 && 5 * rows >= 3 * slots;
  };
  const bool can_fuse = s->merge && !s->mu_r.is_array && count_sources(s, FDTD_LLG_SRC_HARD_E) == 0;
  int n = 0;
  long long items = 0;
  if (s->eh_ok) {
    for (int b = 0; b < s->n_out; ++b) {
      const BoxP &B = s->box_out[b];
      if (B.items == 0) continue;
      const bool fu = can_fuse && stageable(B.lo, B.hi, FBY);
      const bool st = fu || stageable(B.lo, B.hi, SBY);
      int hi[3] = {B.hi[0], B.hi[1], B.hi[2]};
      if (fu && s->g.ext[1] && hi[2] == s->g.n[2]) {
        // a slab's last plane needs E^{n+1} of the upper neighbour's first plane, which arrives with
        // that neighbour's E phase: its H update stays in the second half-step
        const int lo_top[3] = {B.lo[0], B.lo[1], std::max(B.lo[2], hi[2] - 1)};
        n = put(n, lo_top, hi, false, false, 0);
        hi[2] -= 1;
        if (hi[2] <= B.lo[2]) continue;
      }
      n = put(n, B.lo, hi, st, fu, 0);
      if (st) items += make_ehbox(s, B.lo, hi, fu).items;
    }
    for (size_t b = 0; b < s->box_um.size(); ++b)
      if (s->box_um[b].items) n = put(n, s->box_um[b].lo, s->box_um[b].hi, false, false, 1);
    if (s->llg) {
      const bool st = stageable(s->lo, s->hi, SBY);
      n = put(n, s->lo, s->hi, st, false, 2);
      if (st) items += make_ehbox(s, s->lo, s->hi, false).items;
    }
  }
  // a grid that cannot give every SM an item is latency bound: one direct-load launch serves it better
  if (!s->eh_ok || (items < s->num_sms && s->opt.kernel_path != 5)) return put(0, zero, s->g.n, false, false, 3);
  return n;
}

// A step without magnetic cells whose E phase is one fused launch over the whole grid: that launch
// also does the bookkeeping of the two H half-steps, and k_half_end is not launched (EHArgs::book)
bool fold_bookkeeping(const fdtd_llg *s) {
  // not on a slab: its residual words receive the other slabs' maxima and k_half_end must clear them
  // at the end of EVERY half-step, which one launch per step cannot do
  if (s->llg || s->has_pml || s->is_slab) return false;
  ERegion reg[MAX_REG];
  return plan_e_regions(s, reg) == 1 && reg[0].fuse;
}

int enqueue_e_regions(fdtd_llg *s, double *const *Ein, double *const *Eout, int hset, int hset_next, int par,
                      int *launches) {
  ERegion reg[MAX_REG];
  const int nr = plan_e_regions(s, reg);
  const bool fold = fold_bookkeeping(s);
  int widx = 8 * par;   // the staged launches of a step draw from the eight counters of its parity
  for (int r = 0; r < nr; ++r) {
    if (!reg[r].staged) {
      int rc = enqueue_e(s, Ein, Eout, hset, make_box(s, reg[r].lo, reg[r].hi), launches);
      if (rc) return rc;
      continue;
    }
    EHArgs p{};
    p.g = s->g;
    p.tb = make_ehbox(s, reg[r].lo, reg[r].hi, reg[r].fuse);
    p.map = reg[r].fuse ? s->mapEF : s->mapEH;
    p.aE = array_index(s, Ein[0]);
    p.aH = array_index(s, s->Hset[hset][0]);
    p.aEps = s->eps_r.is_array ? array_index(s, s->eps_r.dev) : 0;
    p.aSig = s->sigma.is_array ? array_index(s, s->sigma.dev) : 0;
    for (int d = 0; d < 3; ++d) { p.Eo[d] = Eout[d]; p.Ho[d] = s->Hset[hset_next][d]; }
    p.eps_u = kEps0 * s->eps_r.uniform;
    p.sigma_u = s->sigma.uniform;
    p.rdt = 1.0 / s->dt;
    p.k_u = e_coef(p.eps_u, p.sigma_u, p.rdt);
    p.chm = 2.0 * (s->dt / (2.0 * kMu0 * s->mu_r.uniform));   // cmul * ch of k_h_update, cmul = 2
    p.src = s->src;
    p.st = s->dstate;
    p.work = s->work_eh + widx++;
    p.pipe_error = &s->dstate->pipe_error;
    p.book = fold ? s->dstate : nullptr;
    p.work_other = s->work_eh + 8 * (par ^ 1);
    p.r_hist = s->r_hist;
    prof_begin(s, reg[r].fuse ? FDTD_LLG_K_EH_FUSED : FDTD_LLG_K_E_UPDATE, 0);
    int rc = reg[r].fuse ? launch_eh_stage<true>(s, p) : launch_eh_stage<false>(s, p);
    prof_end(s);
    if (rc) return rc;
    ++*launches;
  }
  CU(s, cudaGetLastError());
  return FDTD_LLG_OK;
}

// hard E / soft H / hard H sources of one kind: a small kernel per source on its box
int enqueue_box_sources(fdtd_llg *s, int kind, double *const *F, int *launches) {
  for (int q = 0; q < s->src.count; ++q) {
    const SourceP &S = s->src.s[q];
    if (S.kind != kind) continue;
    BoxSrcArgs a{};
    a.g = s->g;
    a.S = S;
    a.idx = q;
    a.F = F[S.comp];
    a.st = s->dstate;
    long long n = 1;
    for (int d = 0; d < 3; ++d) n *= S.hi[d] - S.lo[d];
    prof_begin(s, FDTD_LLG_K_OTHER, 0);
    k_box_source<<<grid_1d(s, n), 256, 0, s->stream>>>(a);
    prof_end(s);
    ++*launches;
  }
  CU(s, cudaGetLastError());
  return FDTD_LLG_OK;
}

// ---- the phases of one time step: HM half (curl E^n), E update, HM half
// (curl E^{n+1}).  par = parity of the step: E^n is in E set `par`, E^{n+1} goes to the other set.
// H sets: state in 0 -> half 1 result in set_half(par) -> half 2 result back in 0.  M: 0 -> 1 -> 0.
double *const *e_set(fdtd_llg *s, int par) { return par ? s->E2 : s->E; }

// merged H half-steps: the first step after set_fields takes the outside faces from t = 0 to dt/2
int enqueue_prime(fdtd_llg *s, int par, int *launches) {
  if (!s->merge || s->primed) return FDTD_LLG_OK;
  int rc = enqueue_outside(s, e_set(s, par), 0, set_half(s, par), 1.0, true, launches);
  if (rc) return rc;
  s->primed = true;
  s->prime_at = s->host_steps;
  return FDTD_LLG_OK;
}

int enqueue_begin(fdtd_llg *s, int *launches) {
  if (s->src.count > 0) {
    prof_begin(s, FDTD_LLG_K_OTHER, 0);
    k_step_begin<<<1, 32, 0, s->stream>>>(s->dstate, s->src, s->dt);
    prof_end(s);
    ++*launches;
  }
  return enqueue_box_sources(s, FDTD_LLG_SRC_SOFT_H, s->Hset[0], launches);  // beginning of the step
}

int enqueue_e_phase(fdtd_llg *s, int par, int *launches) {
  double *const *Ea = e_set(s, par), *const *Eb = e_set(s, par ^ 1);
  const int h1 = set_half(s, par);
  int rc = enqueue_e_regions(s, Ea, Eb, h1, set_half(s, par ^ 1), par, launches);
  if (rc) return rc;
  rc = enqueue_pml(s, true, s->Hset[h1], Eb, launches);
  if (rc) return rc;
  return enqueue_box_sources(s, FDTD_LLG_SRC_HARD_E, Eb, launches);            // after the E update
}

int enqueue_step(fdtd_llg *s, int par, int *launches) {
  *launches = 0;
  const int h1 = set_half(s, par), tmp = set_tmp(s, par);
  int rc = enqueue_begin(s, launches);
  if (rc) return rc;
  rc = enqueue_half(s, e_set(s, par), 0, h1, tmp, 0, 1, false, -1, launches);
  if (rc) return rc;
  rc = enqueue_e_phase(s, par, launches);
  if (rc) return rc;
  rc = enqueue_half(s, e_set(s, par ^ 1), h1, 0, tmp, 1, 0, true, set_half(s, par ^ 1), launches);
  if (rc) return rc;
  return enqueue_box_sources(s, FDTD_LLG_SRC_HARD_H, s->Hset[0], launches);    // after the H update
}

int build_graph(fdtd_llg *s, int par) {
  if (s->graph[par]) { cudaGraphExecDestroy(s->graph[par]); s->graph[par] = nullptr; }
  s->graph_valid[par] = false;
  cudaGraph_t g = nullptr;
  CU(s, cudaStreamBeginCapture(s->stream, cudaStreamCaptureModeThreadLocal));
  int launches = 0;
  s->capturing = true;
  int rc = enqueue_step(s, par, &launches);
  s->capturing = false;
  cudaError_t e = cudaStreamEndCapture(s->stream, &g);
  if (rc) { if (g) cudaGraphDestroy(g); return rc; }
  if (e != cudaSuccess) return fail(s, FDTD_LLG_ECUDA, "cudaStreamEndCapture: %s", cudaGetErrorString(e));
  e = cudaGraphInstantiate(&s->graph[par], g, 0);
  cudaGraphDestroy(g);
  if (e != cudaSuccess) return fail(s, FDTD_LLG_ECUDA, "cudaGraphInstantiate: %s", cudaGetErrorString(e));
  s->launches_per_step = launches;
  s->graph_valid[par] = true;
  return FDTD_LLG_OK;
}

// Merged H half-steps: form the integer-time H of the present state (time N) where it is kept at
// half-integer time: H^N = H^{N-1/2} - (dt / 2 mu) curl E^N, the half-step the paper's scheme takes
// (PAPER.md:94), from the set the last step read.  Returns the H set to read.
int reconstruct_h(fdtd_llg *s, int *read_set) {
  *read_set = 0;
  if (!s->merge || !s->primed) return FDTD_LLG_OK;
  const int par = (int)(s->host_steps & 1);       // parity of the NEXT step
  const int dead = set_half(s, par ^ 1);          // H^{N-1/2} outside the box, no longer needed
  const int target = s->opt.enable_llg ? 0 : dead;  // LLG storage: set 0 holds the box's H^N already
  *read_set = target;
  if (s->host_steps == s->prime_at) { *read_set = 0; return FDTD_LLG_OK; }  // set 0 still holds H^N
  if (s->recon_valid) return FDTD_LLG_OK;
  int launches = 0;
  int rc = enqueue_outside(s, e_set(s, par), dead, target, 1.0, false, &launches);
  if (rc) return rc;
  // the margins hold H^N in set 0; a Maxwell-only handle reads from `target`: copy them over
  // (the update with cmul = 0 is a copy)
  if (target != 0) rc = enqueue_outside(s, e_set(s, par), 0, target, 0.0, false, &launches, OUT_MARGINS);
  if (rc) return rc;
  s->recon_valid = true;
  return FDTD_LLG_OK;
}

// leave the merged mode (an H source was added, which needs H at integer time): the state goes
// back to set 0 at integer time
int unmerge(fdtd_llg *s) {
  if (!s->merge) return FDTD_LLG_OK;
  int rs = 0;
  int rc = reconstruct_h(s, &rs);
  if (rc) return rc;
  if (rs != 0)
    for (int d = 0; d < 3; ++d)
      CU(s, cudaMemcpyAsync(s->Hset[0][d], s->Hset[rs][d], s->stride * sizeof(double), cudaMemcpyDeviceToDevice, s->stream));
  s->merge = false;
  s->primed = false;
  s->recon_valid = false;
  s->graph_valid[0] = s->graph_valid[1] = false;
  make_boxes(s);
  return FDTD_LLG_OK;
}

// synchronise the stream and turn a pipeline time-out of a staged sweep into an error: the
// fields are only partly updated then
int check_pipe(fdtd_llg *s) {
  int pe = 0;
  CU(s, cudaMemcpyAsync(&pe, &s->dstate->pipe_error, sizeof pe, cudaMemcpyDeviceToHost, s->stream));
  CU(s, cudaStreamSynchronize(s->stream));
  if (pe) return fail(s, FDTD_LLG_ESTATE, "a TMA pipeline wait timed out (wait tag %d): results are invalid", pe);
  return FDTD_LLG_OK;
}

cudaMemcpyKind to_dev(int mem_space) {
  return mem_space == FDTD_LLG_HOST ? cudaMemcpyHostToDevice : cudaMemcpyDeviceToDevice;
}
cudaMemcpyKind from_dev(int mem_space) {
  return mem_space == FDTD_LLG_HOST ? cudaMemcpyDeviceToHost : cudaMemcpyDeviceToDevice;
}

}  // namespace

// ===================================================================================== C ABI

extern "C" {

void fdtd_llg_default_options(fdtd_llg_options *o) {
  if (!o) return;
  std::memset(o, 0, sizeof *o);
  o->bc[0] = o->bc[1] = o->bc[2] = FDTD_LLG_PEC;
  o->enable_llg = 1;
  o->ani_axis[2] = 1.0;
  o->llg_tol = 1e-6;
  o->llg_max_iter = 20;
  o->use_graph = 1;
  o->pml_r0 = 1e-6;
  o->pml_order = 3;
  o->merge_h = 1;
}

size_t fdtd_llg_workspace_bytes(int nx, int ny, int nz, const fdtd_llg_options *opt,
                                unsigned material_mask) {
  if (nx < 1 || ny < 1 || nz < 1 || !opt) return 0;
  if (opt->llg_max_iter < 1 || opt->llg_max_iter > 1000) return 0;
  const size_t stride = array_stride(nx, ny, nz);
  size_t arrays = 12;                      // two E sets, two H sets (every update is out of place)
  if (opt->enable_llg) arrays += 3 + 18;   // the Jacobi H buffer, two M sets
  for (unsigned b = 0; b < 6; ++b)
    if (material_mask & (1u << b)) ++arrays;
  if (opt->pml[0] | opt->pml[1] | opt->pml[2] | opt->pml[3] | opt->pml[4] | opt->pml[5])
    arrays += 13;                          // 12 split parts + one slot for the damping tables
  return arrays * stride * sizeof(double) + small_bytes(opt);
}

int fdtd_llg_create(fdtd_llg **out, int nx, int ny, int nz, double dx, double dy, double dz,
                    double dt, const double *eps_r, const double *sigma, const double *mu_r,
                    const double *Ms, const double *alpha, const double *gamma, int mem_space,
                    const fdtd_llg_options *opt, void *dev_workspace, size_t workspace_bytes,
                    void *cuda_stream) {
  if (!out) return fail(nullptr, FDTD_LLG_EINVAL, "out is NULL");
  *out = nullptr;
  if (nx < 1 || ny < 1 || nz < 1) return fail(nullptr, FDTD_LLG_EINVAL, "nx, ny, nz must be >= 1");
  if ((double)row_pitch(nx) * (ny + 2.0) * (nz + 2.0) > 2.0e9)
    return fail(nullptr, FDTD_LLG_EINVAL, "grid too large (> 2e9 elements per array with ghosts)");
  if (!(dx > 0) || !(dy > 0) || !(dz > 0) || !std::isfinite(dx) || !std::isfinite(dy) || !std::isfinite(dz))
    return fail(nullptr, FDTD_LLG_EINVAL, "dx, dy, dz must be finite and > 0");
  if (!(dt > 0) || !std::isfinite(dt)) return fail(nullptr, FDTD_LLG_EINVAL, "dt must be finite and > 0");
  if (!opt) return fail(nullptr, FDTD_LLG_EINVAL, "opt is NULL");
  if (mem_space != FDTD_LLG_HOST && mem_space != FDTD_LLG_DEVICE)
    return fail(nullptr, FDTD_LLG_EINVAL, "mem_space must be FDTD_LLG_HOST or FDTD_LLG_DEVICE");
  const char *why = "";
  if (!valid_opts(opt, &why)) return fail(nullptr, FDTD_LLG_EINVAL, "%s", why);
  if (!dev_workspace) return fail(nullptr, FDTD_LLG_EINVAL, "dev_workspace is NULL");
  if (reinterpret_cast<uintptr_t>(dev_workspace) % 256) return fail(nullptr, FDTD_LLG_EINVAL, "dev_workspace must be 256-byte aligned");
  unsigned mask = (eps_r ? 1u : 0) | (sigma ? 2u : 0) | (mu_r ? 4u : 0) | (Ms ? 8u : 0) | (alpha ? 16u : 0) | (gamma ? 32u : 0);
  mask &= ~opt->scalar_material_mask;
  const size_t need = fdtd_llg_workspace_bytes(nx, ny, nz, opt, mask);
  if (workspace_bytes < need)
    return fail(nullptr, FDTD_LLG_ENOMEM, "workspace too small: %zu bytes given, %zu needed", workspace_bytes, need);

  fdtd_llg *s = new (std::nothrow) fdtd_llg();
  if (!s) return fail(nullptr, FDTD_LLG_ENOMEM, "host allocation failed");
  s->g.n[0] = nx; s->g.n[1] = ny; s->g.n[2] = nz;
  s->g.sy = (int)row_pitch(nx);
  s->g.sz = s->g.sy * (ny + 2);
  s->g.org = PADL + s->g.sy + s->g.sz;
  s->d[0] = dx; s->d[1] = dy; s->d[2] = dz;
  for (int d = 0; d < 3; ++d) {
    s->g.per[d] = opt->bc[d] == FDTD_LLG_PERIODIC;
    s->g.wall[d] = opt->bc[d] == FDTD_LLG_PEC;
    s->g.wallhi[d] = s->g.wall[d];
    s->g.rd[d] = 1.0 / s->d[d];
  }
  // a slab interface is neither wall nor wrap; with one interface the other z side keeps its wall
  // (index 0 stays a wall face only if the LOW side is a real wall)
  s->g.ext[0] = opt->slab_ext[0];
  s->g.ext[1] = opt->slab_ext[1];
  if (s->g.ext[0]) s->g.wall[2] = 0;
  if (s->g.ext[1]) s->g.wallhi[2] = 0;
  s->is_slab = s->g.ext[0] || s->g.ext[1];
  s->g.dt = dt;
  s->dt = dt;
  s->ncell = (size_t)nx * ny * nz;
  s->ncell_user = (size_t)nx * ny * (size_t)(nz + s->g.ext[0] + s->g.ext[1]);
  s->stride = array_stride(nx, ny, nz);
  {
    int dev = 0, sms = 0;
    if (cudaGetDevice(&dev) == cudaSuccess &&
        cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev) == cudaSuccess && sms > 0)
      s->num_sms = sms;
  }
  s->opt = *opt;
  if (!opt->enable_llg) { s->opt.llg_max_iter = 1; s->opt.llg_tol = 1.0; }
  if (opt->time_scheme == 1) s->opt.llg_max_iter = 1;  // explicit: one sweep per half-step, no iteration
  s->stream = static_cast<cudaStream_t>(cuda_stream);
  if (cuda_stream && cudaStreamCreateWithFlags(&s->aux, cudaStreamNonBlocking) != cudaSuccess) s->aux = nullptr;
  if (!cuda_stream) s->opt.use_graph = 0;  // the legacy default stream cannot be captured
  s->ws = static_cast<char *>(dev_workspace);
  s->ws_bytes = workspace_bytes;

  auto bail = [&](int rc) { g_create_error = s->err; delete s; return rc; };
#define CUB(call)                                                                        \
  do {                                                                                   \
    cudaError_t e_ = (call);                                                             \
    if (e_ != cudaSuccess) {                                                             \
      fail(s, FDTD_LLG_ECUDA, "%s: %s", #call, cudaGetErrorString(e_));                  \
      return bail(FDTD_LLG_ECUDA);                                                       \
    }                                                                                    \
  } while (0)

  // carve the workspace: small state first, then the big arrays
  char *p = s->ws;
  s->dstate = reinterpret_cast<DevState *>(p); p += 4096;
  s->resid = reinterpret_cast<unsigned long long *>(p); p += padded((size_t)(s->opt.llg_max_iter + 2)) * 8;
  s->work = reinterpret_cast<unsigned *>(p); p += padded((size_t)(s->opt.llg_max_iter + 2)) * 8 + 4096;
  s->work_eh = s->work + 2 * padded((size_t)(s->opt.llg_max_iter + 2));   // in the 4 KB behind the sweeps' counters
  s->scratch = reinterpret_cast<double *>(p); p += (2 * 1024 + 64) * 8;
  s->profile_pool = reinterpret_cast<double *>(p); s->profile_cap = ((size_t)1 << 20) / 8; p += (size_t)1 << 20;
  s->r_hist = reinterpret_cast<int *>(p); p += (size_t)R_HIST * sizeof(int);
  p = s->ws + small_bytes(&s->opt);
  double *q = reinterpret_cast<double *>(p);
  for (int d = 0; d < 3; ++d) { s->E[d] = q; q += s->stride; }
  for (int d = 0; d < 3; ++d) { s->E2[d] = q; q += s->stride; }
  const int nh = opt->enable_llg ? 3 : 2;  // every update is out of place
  for (int h = 0; h < nh; ++h)
    for (int d = 0; d < 3; ++d) { s->Hset[h][d] = q; q += s->stride; }
  if (!opt->enable_llg)
    for (int d = 0; d < 3; ++d) s->Hset[2][d] = s->Hset[1][d];  // Maxwell only: no Jacobi buffer
  if (opt->enable_llg)
    for (int m = 0; m < 2; ++m)
      for (int c = 0; c < 9; ++c) { s->Mset[m][c] = q; q += s->stride; }
  const size_t state_arrays = 6 + 3 * nh + (opt->enable_llg ? 18 : 0);
  CUB(cudaMemsetAsync(s->ws, 0, small_bytes(&s->opt) + state_arrays * s->stride * sizeof(double), s->stream));

  int rc;
  if ((rc = take_material(s, &s->eps_r, eps_r, mem_space, 1.0, &q, "eps_r", 0.0, true, 1u))) return bail(rc);
  if ((rc = take_material(s, &s->sigma, sigma, mem_space, 0.0, &q, "sigma", 0.0, false, 2u))) return bail(rc);
  if ((rc = take_material(s, &s->mu_r, mu_r, mem_space, 1.0, &q, "mu_r", 0.0, true, 4u))) return bail(rc);
  if (opt->enable_llg) {
    if ((rc = take_material(s, &s->Ms, Ms, mem_space, 0.0, &q, "Ms", 0.0, false, 8u))) return bail(rc);
    if ((rc = take_material(s, &s->alpha, alpha, mem_space, 0.0, &q, "alpha", -INFINITY, false, 16u))) return bail(rc);
    if ((rc = take_material(s, &s->gamma, gamma, mem_space, 0.0, &q, "gamma", -INFINITY, false, 32u))) return bail(rc);
  }
  if ((rc = find_sweep_box(s))) return bail(rc);
  make_boxes(s);
  s->n_arrays = (int)((q - s->E[0]) / (ptrdiff_t)s->stride);
  if ((rc = setup_pml(s, &q))) return bail(rc);
  // the staged sweeps need uniform alpha, gamma, mu_r and an even first column (TMA boxes on 16-byte
  // boundaries); the direct-load kernels are the general path
  s->staged = s->llg && !s->alpha.is_array && !s->gamma.is_array && !s->mu_r.is_array &&
              (s->lo[0] & 1) == 0 && opt->kernel_path != 1;
  if (s->staged && (rc = setup_hm_stage(s))) return bail(rc);
  s->merge = decide_merge(s);
  make_boxes(s);   // again: the merged region keeps out of the margins
  if (!s->has_pml && opt->kernel_path != 1 && (rc = setup_eh_stage(s))) return bail(rc);
  CUB(cudaStreamSynchronize(s->stream));
#undef CUB
  *out = s;
  return FDTD_LLG_OK;
}

int fdtd_llg_set_fields(fdtd_llg *s, const double *const *E, const double *const *H,
                        const double *const *M_cell, int mem_space) {
  if (!s) return FDTD_LLG_EINVAL;
  if (mem_space != FDTD_LLG_HOST && mem_space != FDTD_LLG_DEVICE)
    return fail(s, FDTD_LLG_EINVAL, "mem_space must be FDTD_LLG_HOST or FDTD_LLG_DEVICE");
  const size_t abytes = s->stride * sizeof(double);
  int rc;
  for (int d = 0; d < 3; ++d) {
    CU(s, cudaMemsetAsync(s->E[d], 0, abytes, s->stream));
    CU(s, cudaMemsetAsync(s->Hset[0][d], 0, abytes, s->stream));
    if (E && E[d] && (rc = copy_in(s, s->E[d], E[d], mem_space))) return rc;
    if (H && H[d] && (rc = copy_in(s, s->Hset[0][d], H[d], mem_space))) return rc;
  }
  if (s->opt.enable_llg)
    for (int h = 1; h < 3; ++h)
      for (int d = 0; d < 3; ++d) CU(s, cudaMemsetAsync(s->Hset[h][d], 0, abytes, s->stream));
  FieldsP f{};
  f.g = s->g;
  for (int d = 0; d < 3; ++d) { f.E[d] = s->E[d]; f.H[d] = s->Hset[0][d]; }
  k_enforce_walls<<<grid_1d(s, (long long)s->ncell_user), 256, 0, s->stream>>>(f);
  CU(s, cudaGetLastError());
  for (int d = 0; d < 3; ++d) {
    if ((rc = fill_ghosts(s, s->E[d]))) return rc;
    if ((rc = fill_ghosts(s, s->Hset[0][d]))) return rc;
  }
  if (s->has_pml)  // fields given from outside enter the layer as part 0 of each component
    for (int d = 0; d < 3; ++d) {
      CU(s, cudaMemcpyAsync(s->Esp[2 * d], s->E[d], abytes, cudaMemcpyDeviceToDevice, s->stream));
      CU(s, cudaMemcpyAsync(s->Hsp[2 * d], s->Hset[0][d], abytes, cudaMemcpyDeviceToDevice, s->stream));
      CU(s, cudaMemsetAsync(s->Esp[2 * d + 1], 0, abytes, s->stream));
      CU(s, cudaMemsetAsync(s->Hsp[2 * d + 1], 0, abytes, s->stream));
    }
  // reset run state
  CU(s, cudaMemsetAsync(s->dstate, 0, sizeof(DevState), s->stream));
  CU(s, cudaMemsetAsync(s->resid, 0, (size_t)(s->opt.llg_max_iter + 2) * 8, s->stream));
  CU(s, cudaMemsetAsync(s->work, 0, padded((size_t)(s->opt.llg_max_iter + 2)) * 8 + 64, s->stream));
  if (s->opt.enable_llg) {
    InitMP a{};
    a.g = s->g;
    for (int c = 0; c < 3; ++c) {
      a.Mc[c] = nullptr;
      if (M_cell && M_cell[c]) {  // stage the cell-centred array, ghosted, in the second M set
        CU(s, cudaMemsetAsync(s->Mset[1][c], 0, abytes, s->stream));
        if ((rc = copy_in(s, s->Mset[1][c], M_cell[c], mem_space))) return rc;
        if ((rc = fill_ghosts(s, s->Mset[1][c]))) return rc;
        a.Mc[c] = s->Mset[1][c];
      }
    }
    for (int c = 0; c < 9; ++c) {
      CU(s, cudaMemsetAsync(s->Mset[0][c], 0, abytes, s->stream));
      a.M[c] = s->Mset[0][c];
    }
    a.Ms = s->Ms.dev;
    a.Ms_u = s->Ms.uniform;
    a.enable_llg = s->llg ? 1 : 0;
    a.st = s->dstate;
    k_init_m<<<grid_1d(s, (long long)s->ncell), 256, 0, s->stream>>>(a);
    CU(s, cudaGetLastError());
    for (int c = 0; c < 9; ++c) {
      if ((rc = fill_ghosts(s, s->Mset[0][c]))) return rc;
      CU(s, cudaMemsetAsync(s->Mset[1][c], 0, abytes, s->stream));
    }
    int err = 0;
    CU(s, cudaMemcpyAsync(&err, &s->dstate->init_error, sizeof(int), cudaMemcpyDeviceToHost, s->stream));
    CU(s, cudaStreamSynchronize(s->stream));
    if (err) return fail(s, FDTD_LLG_EINVAL, "a magnetic face received a zero averaged M (PAPER.md:90 needs a direction to normalise)");
  }
  CU(s, cudaStreamSynchronize(s->stream));
  s->host_steps = 0;
  s->kernel_launches = 0;
  s->primed = false;
  s->recon_valid = false;
  s->sub_next = FDTD_LLG_SUB_BEGIN;
  return FDTD_LLG_OK;
}

int fdtd_llg_set_source(fdtd_llg *s, int comp, const int *lo, const int *hi,
                        const double *profile, int mem_space, double amplitude, double f0,
                        double t0, double tp) {
  return fdtd_llg_add_source(s, FDTD_LLG_SRC_SOFT_E, comp, lo, hi, profile, mem_space, amplitude, f0, t0, tp);
}

int fdtd_llg_add_source(fdtd_llg *s, int kind, int comp, const int *lo, const int *hi,
                        const double *profile, int mem_space, double amplitude, double f0,
                        double t0, double tp) {
  if (!s) return FDTD_LLG_EINVAL;
  if (kind < FDTD_LLG_SRC_SOFT_E || kind > FDTD_LLG_SRC_HARD_H)
    return fail(s, FDTD_LLG_EINVAL, "kind must be one of FDTD_LLG_SRC_*");
  if (s->src.count >= MAX_SOURCES) return fail(s, FDTD_LLG_ESTATE, "at most %d sources", MAX_SOURCES);
  if (comp < 0 || comp > 2) return fail(s, FDTD_LLG_EINVAL, "comp must be 0, 1 or 2");
  if (!lo || !hi) return fail(s, FDTD_LLG_EINVAL, "lo / hi is NULL");
  if (!(tp > 0) || !std::isfinite(tp) || !std::isfinite(amplitude) || !std::isfinite(f0) || !std::isfinite(t0))
    return fail(s, FDTD_LLG_EINVAL, "tp must be > 0 and amplitude, f0, t0 finite");
  size_t nb = 1;
  for (int d = 0; d < 3; ++d) {
    if (lo[d] < 0 || hi[d] > s->g.n[d] || lo[d] >= hi[d])
      return fail(s, FDTD_LLG_EINVAL, "source box outside the grid or empty on axis %d", d);
    nb *= (size_t)(hi[d] - lo[d]);
  }
  if (s->has_pml && kind != FDTD_LLG_SRC_SOFT_E)
    for (int d = 0; d < 3; ++d)
      if (lo[d] < s->opt.pml[2 * d] || hi[d] > s->g.n[d] - s->opt.pml[2 * d + 1])
        return fail(s, FDTD_LLG_EINVAL, "hard / soft field sources must lie outside the PML");
  if (s->sub_next != FDTD_LLG_SUB_BEGIN) return fail(s, FDTD_LLG_ESTATE, "a time step is open (fdtd_llg_substep)");
  if (kind == FDTD_LLG_SRC_SOFT_H || kind == FDTD_LLG_SRC_HARD_H) {  // these act on H at integer time
    if (s->merge && (s->g.dlo != 0 || s->g.dhi != 0))
      return fail(s, FDTD_LLG_ESTATE, "an H source switches merge_h off, which all slabs of a grid must agree on: "
                  "add it before fdtd_llg_slab_connect (or create the slabs with options.merge_h = 0)");
    int rc = unmerge(s);
    if (rc) return rc;
  }
  SourceP &S = s->src.s[s->src.count];
  S.kind = kind;
  S.comp = comp;
  for (int d = 0; d < 3; ++d) { S.lo[d] = lo[d]; S.hi[d] = hi[d]; }
  S.amplitude = amplitude; S.f0 = f0; S.t0 = t0; S.tp = tp;
  S.profile = nullptr;
  if (profile) {
    if (mem_space != FDTD_LLG_HOST && mem_space != FDTD_LLG_DEVICE)
      return fail(s, FDTD_LLG_EINVAL, "mem_space must be FDTD_LLG_HOST or FDTD_LLG_DEVICE");
    if (s->profile_used + nb > s->profile_cap)
      return fail(s, FDTD_LLG_ENOMEM, "source profiles exceed the 1 MiB pool");
    double *dst = s->profile_pool + s->profile_used;
    CU(s, cudaMemcpyAsync(dst, profile, nb * sizeof(double), to_dev(mem_space), s->stream));
    CU(s, cudaStreamSynchronize(s->stream));
    S.profile = dst;
    s->profile_used += padded(nb);
  }
  s->src.count++;
  s->graph_valid[0] = s->graph_valid[1] = false;  // the step's kernel arguments changed
  if (kind == FDTD_LLG_SRC_SOFT_H || kind == FDTD_LLG_SRC_HARD_H) {
    // (the state is at integer time now: unmerge above) merge again outside the margin this source needs
    s->merge = decide_merge(s);
    make_boxes(s);
  }
  return FDTD_LLG_OK;
}

int fdtd_llg_step(fdtd_llg *s, int n) {
  if (!s) return FDTD_LLG_EINVAL;
  if (n < 0) return fail(s, FDTD_LLG_EINVAL, "n must be >= 0");
  if (n == 0) return FDTD_LLG_OK;
  if (s->sub_next != FDTD_LLG_SUB_BEGIN) return fail(s, FDTD_LLG_ESTATE, "a time step is open (fdtd_llg_substep)");
  if (s->g.dlo != 0 || s->g.dhi != 0)
    return fail(s, FDTD_LLG_ESTATE, "a connected slab is advanced with fdtd_llg_substep (the caller orders the slabs)");
  int rc = FDTD_LLG_OK, done = 0, extra = 0;
  rc = enqueue_prime(s, (int)(s->host_steps & 1), &extra);
  for (int t = 0; t < n && !rc; ++t) {
    const int par = (int)((s->host_steps + t) & 1);
    if (s->opt.use_graph) {
      if (!s->graph_valid[par]) rc = build_graph(s, par);
      if (!rc && cudaGraphLaunch(s->graph[par], s->stream) != cudaSuccess)
        rc = fail(s, FDTD_LLG_ECUDA, "cudaGraphLaunch: %s", cudaGetErrorString(cudaGetLastError()));
    } else {
      int launches = 0;
      rc = enqueue_step(s, par, &launches);
      if (!rc) s->launches_per_step = launches;
    }
    if (!rc) ++done;
  }
  // the steps that were enqueued count, also when a later one failed: the E-set parity and
  // fdtd_llg_read_fields follow the device
  s->host_steps += done;
  s->kernel_launches += (long long)done * s->launches_per_step + extra;
  if (done) s->recon_valid = false;
  return rc;
}

int fdtd_llg_step_timed(fdtd_llg *s, int n, double *ms_by_class, long long *launches_by_class) {
  if (!s) return FDTD_LLG_EINVAL;
  if (n < 1 || n > R_HIST / 2) return fail(s, FDTD_LLG_EINVAL, "n must be in 1..%d", R_HIST / 2);
  if (!ms_by_class || !launches_by_class) return fail(s, FDTD_LLG_EINVAL, "output array is NULL");
  if (s->sub_next != FDTD_LLG_SUB_BEGIN) return fail(s, FDTD_LLG_ESTATE, "a time step is open (fdtd_llg_substep)");
  if (s->g.dlo != 0 || s->g.dhi != 0) return fail(s, FDTD_LLG_ESTATE, "a connected slab is advanced with fdtd_llg_substep");
  std::vector<fdtd_llg::ProfRec> recs;
  DevState h0{};
  CU(s, cudaMemcpyAsync(&h0, s->dstate, sizeof h0, cudaMemcpyDeviceToHost, s->stream));
  CU(s, cudaStreamSynchronize(s->stream));
  int rc = FDTD_LLG_OK, done = 0, extra = 0;
  rc = enqueue_prime(s, (int)(s->host_steps & 1), &extra);
  s->prof = &recs;
  s->prof_half = 0;
  for (int t = 0; t < n && !rc; ++t) {
    int launches = 0;
    rc = enqueue_step(s, (int)((s->host_steps + t) & 1), &launches);
    if (!rc) { s->launches_per_step = launches; ++done; }
  }
  s->prof = nullptr;
  s->host_steps += done;
  s->kernel_launches += (long long)done * s->launches_per_step + extra;
  if (done) s->recon_valid = false;
  cudaError_t e = cudaStreamSynchronize(s->stream);
  std::vector<int> hist(R_HIST);
  if (e == cudaSuccess)
    e = cudaMemcpy(hist.data(), s->r_hist, sizeof(int) * R_HIST, cudaMemcpyDeviceToHost);
  for (int c = 0; c < FDTD_LLG_K_NCLASS; ++c) { ms_by_class[c] = 0.0; launches_by_class[c] = 0; }
  for (auto &p : recs) {
    float ms = 0.f;
    if (e == cudaSuccess && !rc) cudaEventElapsedTime(&ms, p.a, p.b);
    int cls = p.cls;
    // an LLG iterate beyond the half-step's iteration count exited on its first flag read
    if (cls == FDTD_LLG_K_HM_ITER && p.r > hist[(h0.halfsteps + p.half) % R_HIST]) cls = FDTD_LLG_K_HM_SKIPPED;
    else if (cls == FDTD_LLG_K_HM_ITER && p.r == 2) cls = FDTD_LLG_K_HM_SECOND;
    ms_by_class[cls] += ms;
    launches_by_class[cls]++;
    cudaEventDestroy(p.a);
    cudaEventDestroy(p.b);
  }
  if (rc) return rc;
  if (e != cudaSuccess) return fail(s, FDTD_LLG_ECUDA, "step_timed: %s", cudaGetErrorString(e));
  return check_pipe(s);
}

int fdtd_llg_read_fields(fdtd_llg *s, double *const *E, double *const *H, double *const *M,
                         int mem_space) {
  if (!s) return FDTD_LLG_EINVAL;
  if (mem_space != FDTD_LLG_HOST && mem_space != FDTD_LLG_DEVICE)
    return fail(s, FDTD_LLG_EINVAL, "mem_space must be FDTD_LLG_HOST or FDTD_LLG_DEVICE");
  if (s->sub_next != FDTD_LLG_SUB_BEGIN) return fail(s, FDTD_LLG_ESTATE, "a time step is open (fdtd_llg_substep)");
  const size_t bytes = s->ncell * sizeof(double);
  int rc, hset = 0;
  if (H && (H[0] || H[1] || H[2]) && (rc = reconstruct_h(s, &hset))) return rc;
  for (int d = 0; d < 3; ++d) {
    if (E && E[d] && (rc = copy_out(s, E[d], ((s->host_steps & 1) ? s->E2 : s->E)[d], mem_space))) return rc;
    if (H && H[d] && (rc = copy_out(s, H[d], s->Hset[hset][d], mem_space))) return rc;
  }
  if (M)
    for (int c = 0; c < 9; ++c)
      if (M[c]) {
        if (s->opt.enable_llg) { if ((rc = copy_out(s, M[c], s->Mset[0][c], mem_space))) return rc; }
        else if (mem_space == FDTD_LLG_HOST) std::memset(M[c], 0, bytes);
        else CU(s, cudaMemsetAsync(M[c], 0, bytes, s->stream));
      }
  return check_pipe(s);
}

int fdtd_llg_get_stats(fdtd_llg *s, fdtd_llg_stats *out) {
  if (!s || !out) return FDTD_LLG_EINVAL;
  DevState h{};
  CU(s, cudaMemcpyAsync(&h, s->dstate, sizeof h, cudaMemcpyDeviceToHost, s->stream));
  CU(s, cudaStreamSynchronize(s->stream));
  if (h.pipe_error)
    return fail(s, FDTD_LLG_ESTATE, "a TMA pipeline wait timed out (wait tag %d): results are invalid", h.pipe_error);
  std::memset(out, 0, sizeof *out);
  out->merged_h = s->merge ? 1 : 0;
  {
    ERegion reg[MAX_REG];
    const int nr = plan_e_regions(s, reg);
    for (int r = 0; r < nr; ++r)
      out->staged_maxwell = std::max(out->staged_maxwell, reg[r].fuse ? 2 : (reg[r].staged ? 1 : 0));
  }
  out->steps = h.steps;
  out->time = (double)h.steps * s->dt;
  out->iters_last = h.iters_last;
  out->iters_max = h.iters_max;
  out->iters_total = h.iters_total;
  out->nonconverged_halfsteps = h.nonconverged;
  out->resid_last = h.resid_last;
  out->halfsteps = h.halfsteps;
  const double lim = 1.0 / (kC0 * std::sqrt(1.0 / (s->d[0] * s->d[0]) + 1.0 / (s->d[1] * s->d[1]) + 1.0 / (s->d[2] * s->d[2])));
  out->courant = s->dt / lim;
  out->kernel_launches = s->kernel_launches;
  out->magnetic_cells = s->magnetic_cells;
  out->launches_per_step = s->launches_per_step;
  out->material_array_mask = (s->eps_r.is_array ? 1u : 0) | (s->sigma.is_array ? 2u : 0) |
                             (s->mu_r.is_array ? 4u : 0) | (s->Ms.is_array ? 8u : 0) |
                             (s->alpha.is_array ? 16u : 0) | (s->gamma.is_array ? 32u : 0);
  out->staged_sweeps = s->staged ? 1 : 0;
  out->sweep_cells = 0;
  if (s->llg) {
    out->sweep_cells = 1;
    for (int d = 0; d < 3; ++d) out->sweep_cells *= (long long)(s->hi[d] - s->lo[d]);
  }
  return FDTD_LLG_OK;
}

const char *fdtd_llg_last_error(const fdtd_llg *s) {
  return s ? s->err.c_str() : g_create_error.c_str();
}

void fdtd_llg_destroy(fdtd_llg *s) {
  if (!s) return;
  for (int p = 0; p < 2; ++p)
    if (s->graph[p]) cudaGraphExecDestroy(s->graph[p]);
  if (s->aux) cudaStreamDestroy(s->aux);
  delete s;
}

// ------------------------------------------------------------------------------- z-slabs

int fdtd_llg_get_slab_info(fdtd_llg *s, fdtd_llg_slab_info *out) {
  if (!s || !out) return FDTD_LLG_EINVAL;
  out->fields_offset = (unsigned long long)(reinterpret_cast<char *>(s->E[0]) - s->ws);
  out->array_stride = (unsigned long long)s->stride;
  out->nx = s->g.n[0]; out->ny = s->g.n[1]; out->nz = s->g.n[2];
  out->n_arrays = 6 + 3 * (s->opt.enable_llg ? 3 : 2) + (s->opt.enable_llg ? 18 : 0);
  out->merged_h = s->merge ? 1 : 0;
  return FDTD_LLG_OK;
}

int fdtd_llg_slab_connect(fdtd_llg *s, const fdtd_llg_slab_info *lo, void *lo_workspace,
                          const fdtd_llg_slab_info *hi, void *hi_workspace) {
  if (!s) return FDTD_LLG_EINVAL;
  if (s->sub_next != FDTD_LLG_SUB_BEGIN) return fail(s, FDTD_LLG_ESTATE, "a time step is open (fdtd_llg_substep)");
  fdtd_llg_slab_info me;
  fdtd_llg_get_slab_info(s, &me);
  const fdtd_llg_slab_info *nb[2] = {lo, hi};
  void *ws[2] = {lo_workspace, hi_workspace};
  long long delta[2] = {0, 0};
  for (int sd = 0; sd < 2; ++sd) {
    if (!nb[sd]) continue;
    if (!s->g.ext[sd]) return fail(s, FDTD_LLG_EINVAL, "side %d is not a slab interface (options.slab_ext)", sd);
    if (!ws[sd]) return fail(s, FDTD_LLG_EINVAL, "neighbour workspace is NULL");
    if (nb[sd]->nx != me.nx || nb[sd]->ny != me.ny || nb[sd]->nz != me.nz ||
        nb[sd]->array_stride != me.array_stride || nb[sd]->n_arrays != me.n_arrays)
      return fail(s, FDTD_LLG_EINVAL, "slabs must have the same nx, ny, nz and field storage (neighbour: %d x %d x %d, %d arrays)",
                  nb[sd]->nx, nb[sd]->ny, nb[sd]->nz, nb[sd]->n_arrays);
    if (nb[sd]->merged_h != me.merged_h)
      return fail(s, FDTD_LLG_EINVAL, "slabs disagree on merge_h (%d here, %d there): a PML or an H source switches it off for "
                  "one handle; create all slabs of the grid with options.merge_h = 0 then", me.merged_h, nb[sd]->merged_h);
    const char *theirs = static_cast<const char *>(ws[sd]) + nb[sd]->fields_offset;
    const long long base = (long long)(theirs - reinterpret_cast<const char *>(s->E[0]));
    const long long plane = 8LL * s->g.sz * s->g.n[2];
    // my (i,j,0) is their (i,j,nz); my (i,j,nz-1) is their (i,j,-1)
    delta[sd] = sd == 0 ? base + plane : base - plane;
    if (delta[sd] == 0) return fail(s, FDTD_LLG_EINVAL, "neighbour workspace overlaps this one");
  }
  s->g.dlo = delta[0];
  s->g.dhi = delta[1];
  s->graph_valid[0] = s->graph_valid[1] = false;
  return FDTD_LLG_OK;
}

int fdtd_llg_substep(fdtd_llg *s, int phase, int r) {
  if (!s) return FDTD_LLG_EINVAL;
  const bool hm = phase == FDTD_LLG_SUB_HM1 || phase == FDTD_LLG_SUB_HM2;
  // order: BEGIN, HM1 r = 1, 2, ..., HM1_END, E, HM2 r = 1, 2, ..., HM2_END
  const bool in_order = hm ? ((phase == s->sub_next && r == 1) || (phase + 1 == s->sub_next && r == s->sub_r + 1))
                           : phase == s->sub_next && (phase == FDTD_LLG_SUB_BEGIN || phase == FDTD_LLG_SUB_E || s->sub_r >= 1);
  if (phase < FDTD_LLG_SUB_BEGIN || phase > FDTD_LLG_SUB_HM2_END || !in_order)
    return fail(s, FDTD_LLG_ESTATE, "sub-step %d (r = %d) out of order: expected phase %d", phase, r, s->sub_next);
  if (hm && (r < 1 || r > s->opt.llg_max_iter)) return fail(s, FDTD_LLG_EINVAL, "r must be in 1..llg_max_iter");
  const int par = (int)(s->host_steps & 1);
  const int h1 = set_half(s, par), tmp = set_tmp(s, par);
  int launches = 0, rc = FDTD_LLG_OK;
  switch (phase) {
    case FDTD_LLG_SUB_BEGIN:
      rc = enqueue_prime(s, par, &launches);
      if (!rc) rc = enqueue_begin(s, &launches);
      s->sub_next = FDTD_LLG_SUB_HM1;
      s->sub_r = 0;
      break;
    case FDTD_LLG_SUB_HM1:
      if (r == 1) rc = enqueue_half_pre(s, e_set(s, par), 0, h1, -1, &launches);
      if (!rc && s->llg) rc = enqueue_sweep(s, e_set(s, par), 0, h1, tmp, 0, 1, r, &launches);
      s->sub_next = FDTD_LLG_SUB_HM1_END;
      s->sub_r = r;
      break;
    case FDTD_LLG_SUB_HM1_END:
      rc = enqueue_half_end(s, h1, tmp, s->sub_r, false, &launches);
      s->sub_next = FDTD_LLG_SUB_E;
      break;
    case FDTD_LLG_SUB_E:
      rc = enqueue_e_phase(s, par, &launches);
      s->sub_next = FDTD_LLG_SUB_HM2;
      s->sub_r = 0;
      break;
    case FDTD_LLG_SUB_HM2:
      if (r == 1) rc = enqueue_half_pre(s, e_set(s, par ^ 1), h1, 0, set_half(s, par ^ 1), &launches);
      if (!rc && s->llg) rc = enqueue_sweep(s, e_set(s, par ^ 1), h1, 0, tmp, 1, 0, r, &launches);
      s->sub_next = FDTD_LLG_SUB_HM2_END;
      s->sub_r = r;
      break;
    default:  // FDTD_LLG_SUB_HM2_END
      rc = enqueue_half_end(s, 0, tmp, s->sub_r, true, &launches);
      if (!rc) rc = enqueue_box_sources(s, FDTD_LLG_SRC_HARD_H, s->Hset[0], &launches);
      s->sub_next = FDTD_LLG_SUB_BEGIN;
      s->host_steps += 1;
      s->recon_valid = false;
      break;
  }
  s->kernel_launches += launches;
  return rc;
}

int fdtd_llg_residual_word(fdtd_llg *s, int r, void **dev_ptr) {
  if (!s || !dev_ptr) return FDTD_LLG_EINVAL;
  if (r < 0 || r > s->opt.llg_max_iter) return fail(s, FDTD_LLG_EINVAL, "r must be in 0..llg_max_iter");
  *dev_ptr = s->resid + r;
  return FDTD_LLG_OK;
}

int fdtd_llg_ipc_export(fdtd_llg *s, unsigned char *handle64, unsigned long long *offset) {
  if (!s || !handle64 || !offset) return FDTD_LLG_EINVAL;
  static_assert(sizeof(cudaIpcMemHandle_t) == 64, "CUDA IPC handle size");
  // the handle names the whole allocation the workspace was cut from (a caching allocator's block)
  typedef CUresult (*RangeFn)(CUdeviceptr *, size_t *, CUdeviceptr);
  void *fp = nullptr;
  cudaDriverEntryPointQueryResult q;
  if (cudaGetDriverEntryPoint("cuMemGetAddressRange", &fp, cudaEnableDefault, &q) != cudaSuccess ||
      q != cudaDriverEntryPointSuccess || !fp)
    return fail(s, FDTD_LLG_ECUDA, "cuMemGetAddressRange is not available");
  CUdeviceptr base = 0;
  size_t size = 0;
  if (reinterpret_cast<RangeFn>(fp)(&base, &size, (CUdeviceptr)(uintptr_t)s->ws) != CUDA_SUCCESS)
    return fail(s, FDTD_LLG_ECUDA, "cuMemGetAddressRange failed on the workspace");
  cudaIpcMemHandle_t h;
  CU(s, cudaIpcGetMemHandle(&h, reinterpret_cast<void *>((uintptr_t)base)));
  std::memcpy(handle64, &h, sizeof h);
  *offset = (unsigned long long)((uintptr_t)s->ws - (uintptr_t)base);
  return FDTD_LLG_OK;
}

int fdtd_llg_ipc_open(const unsigned char *handle64, unsigned long long offset, void **dev_ptr) {
  if (!handle64 || !dev_ptr) return fail(nullptr, FDTD_LLG_EINVAL, "NULL argument");
  cudaIpcMemHandle_t h;
  std::memcpy(&h, handle64, sizeof h);
  void *base = nullptr;
  cudaError_t e = cudaIpcOpenMemHandle(&base, h, cudaIpcMemLazyEnablePeerAccess);
  if (e != cudaSuccess) return fail(nullptr, FDTD_LLG_ECUDA, "cudaIpcOpenMemHandle: %s", cudaGetErrorString(e));
  *dev_ptr = static_cast<char *>(base) + offset;
  return FDTD_LLG_OK;
}

int fdtd_llg_ipc_close(void *dev_ptr, unsigned long long offset) {
  if (!dev_ptr) return FDTD_LLG_OK;
  cudaError_t e = cudaIpcCloseMemHandle(static_cast<char *>(dev_ptr) - offset);
  if (e != cudaSuccess) return fail(nullptr, FDTD_LLG_ECUDA, "cudaIpcCloseMemHandle: %s", cudaGetErrorString(e));
  return FDTD_LLG_OK;
}

}  // extern "C"

// ================================================================================================
// fdtd_llg_magnetic_box_static: the magnetic-cell scan for callers that cannot allocate
// (include/fdtd_llg.h "A QUERY THAT ALLOCATES NOTHING AT ALL" says who they are and why).
//
// The scan inside fdtd_llg_create (k_mag_box above) works in the handle's workspace: the map is first
// copied into the ghosted layout there and the box / count words it folds into with atomics live
// there too.  A caller without a handle has no workspace, and the callers this variant is for may not
// ask CUDA for one.  So the variant reads the caller's compact map directly and keeps its scratch --
// one partial box + count per thread block, and the ticket that tells the last block to finish -- in
// the fixed array below.  Array, kernel, address look-up and entry point sit in this one file because
// the array has internal linkage (static): only this translation unit can name it.
namespace {

constexpr int SB_THREADS = 256;
constexpr int SB_PER_THREAD = 64;
constexpr long long SB_CHUNK = (long long)SB_THREADS * SB_PER_THREAD;          // cells per block
constexpr long long SB_MAX_BLOCKS = FDTD_LLG_STATIC_MAX_CELLS / SB_CHUNK;      // 32768
struct SbPartial { int lo[3]; int hi[3]; unsigned long long count; };          // 32 bytes
constexpr size_t SB_HEAD = 256;   // the ticket word has the first 256 bytes to itself
static_assert(sizeof(SbPartial) == 32, "partial record");
static_assert(SB_HEAD + SB_MAX_BLOCKS * sizeof(SbPartial) == FDTD_LLG_STATIC_SCRATCH_BYTES,
              "the header states the size of the static scratch");

// The scratch.  Part of the library's device image: every GPU that loads the library holds these
// bytes until the process exits.  In HOST code this name is only a stand-in for the symbol, NOT a
// device address: handing it to a kernel makes the kernel fault or, where the GPU can reach host
// memory, scribble over the wrong bytes without a word.  Host code gets the real address from
// cudaGetSymbolAddress (static_scratch_address below) and passes that.
static __device__ __align__(256) unsigned char g_static_scratch[FDTD_LLG_STATIC_SCRATCH_BYTES];

// Block b scans cells [b * SB_CHUNK, (b + 1) * SB_CHUNK) of the compact map, leaves its partial in
// scratch and takes a ticket; the block that draws the last ticket folds all partials into out7 and
// puts the ticket word back to 0.  A partial is always written before it is read in the same launch,
// so what an earlier call left in the array is never seen.
__global__ void __launch_bounds__(SB_THREADS)
k_mag_box_static(const double *__restrict__ Ms, int nx, int ny, int nz, long long n,
                 unsigned char *scratch, long long *__restrict__ out7) {
  unsigned *ticket = reinterpret_cast<unsigned *>(scratch);
  SbPartial *part = reinterpret_cast<SbPartial *>(scratch + SB_HEAD);
  int lo[3] = {INT_MAX, INT_MAX, INT_MAX}, hi[3] = {INT_MIN, INT_MIN, INT_MIN};
  unsigned long long cnt = 0;

  // (i, j, k) of this thread's first cell by division, of the following ones by adding the
  // decomposition of the thread stride: 256 = si + nx * (sj + ny * sk)
  long long t = (long long)blockIdx.x * SB_CHUNK + threadIdx.x;
  int i = (int)(t % nx), j = (int)((t / nx) % ny), k = (int)(t / ((long long)nx * ny));
  const int si = SB_THREADS % nx, sj = (SB_THREADS / nx) % ny, sk = SB_THREADS / nx / ny;
  for (int m = 0; m < SB_PER_THREAD && t < n; ++m, t += SB_THREADS) {
    if (Ms[t] > 0.0) {   // the test of k_mag_box: a NaN is not magnetic
      lo[0] = min(lo[0], i); lo[1] = min(lo[1], j); lo[2] = min(lo[2], k);
      hi[0] = max(hi[0], i); hi[1] = max(hi[1], j); hi[2] = max(hi[2], k);
      ++cnt;
    }
    i += si;
    if (i >= nx) { i -= nx; ++j; }
    j += sj;
    if (j >= ny) { j -= ny; ++k; }
    k += sk;
  }

  __shared__ int s_lo[3][SB_THREADS / 32], s_hi[3][SB_THREADS / 32];
  __shared__ unsigned long long s_cnt[SB_THREADS / 32];
  __shared__ bool s_last;
  const int lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
  auto fold_block = [&]() {   // afterwards thread 0 holds the block's box and count
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
      for (int d = 0; d < 3; ++d) {
        lo[d] = min(lo[d], __shfl_xor_sync(0xffffffffu, lo[d], o));
        hi[d] = max(hi[d], __shfl_xor_sync(0xffffffffu, hi[d], o));
      }
      cnt += __shfl_xor_sync(0xffffffffu, cnt, o);
    }
    if (lane == 0) {
      for (int d = 0; d < 3; ++d) { s_lo[d][warp] = lo[d]; s_hi[d][warp] = hi[d]; }
      s_cnt[warp] = cnt;
    }
    __syncthreads();
    if (threadIdx.x == 0)
      for (int w = 1; w < SB_THREADS / 32; ++w) {
        for (int d = 0; d < 3; ++d) { lo[d] = min(lo[d], s_lo[d][w]); hi[d] = max(hi[d], s_hi[d][w]); }
        cnt += s_cnt[w];
      }
  };

  fold_block();
  if (threadIdx.x == 0) {
    SbPartial p;
    for (int d = 0; d < 3; ++d) { p.lo[d] = lo[d]; p.hi[d] = hi[d]; }
    p.count = cnt;
    part[blockIdx.x] = p;
    __threadfence();   // the partial is visible device-wide before the ticket is
    s_last = atomicAdd(ticket, 1u) == gridDim.x - 1;
  }
  __syncthreads();
  if (!s_last) return;

  __threadfence();     // all other blocks' partials are visible to this block
  for (int d = 0; d < 3; ++d) { lo[d] = INT_MAX; hi[d] = INT_MIN; }
  cnt = 0;
  for (unsigned b = threadIdx.x; b < gridDim.x; b += SB_THREADS) {
    const int4 a = __ldcg(reinterpret_cast<const int4 *>(part + b));       // lo x y z, hi x
    const int4 c = __ldcg(reinterpret_cast<const int4 *>(part + b) + 1);   // hi y z, count
    lo[0] = min(lo[0], a.x); lo[1] = min(lo[1], a.y); lo[2] = min(lo[2], a.z);
    hi[0] = max(hi[0], a.w); hi[1] = max(hi[1], c.x); hi[2] = max(hi[2], c.y);
    cnt += (unsigned long long)(unsigned)c.z | ((unsigned long long)(unsigned)c.w << 32);
  }
  __syncthreads();     // the shared arrays are reused
  fold_block();
  if (threadIdx.x == 0) {
    const int nn[3] = {nx, ny, nz};
    for (int d = 0; d < 3; ++d) {
      out7[d] = cnt ? lo[d] : nn[d];
      out7[3 + d] = cnt ? hi[d] : -1;
    }
    out7[6] = (long long)cnt;
    *ticket = 0u;      // as the next call expects it (the entry point clears it as well)
  }
}

// Device address of g_static_scratch on the CURRENT device: looked up on the first call per device
// and kept.  (Each device has its own instance of a __device__ variable, hence one address per
// device, asked for while that device is current.)
constexpr int SB_MAX_DEVICES = 64;
unsigned char *g_scratch_addr[SB_MAX_DEVICES] = {};
std::mutex g_scratch_mutex;

int static_scratch_address(unsigned char **out) {
  int dev = -1;
  CU(nullptr, cudaGetDevice(&dev));
  if (dev < 0 || dev >= SB_MAX_DEVICES)
    return fail(nullptr, FDTD_LLG_EINVAL, "device ordinal %d is beyond the %d this call keeps addresses for", dev, SB_MAX_DEVICES);
  std::lock_guard<std::mutex> lock(g_scratch_mutex);
  if (!g_scratch_addr[dev]) {
    void *p = nullptr;
    CU(nullptr, cudaGetSymbolAddress(&p, g_static_scratch));
    if (!p) return fail(nullptr, FDTD_LLG_ECUDA, "cudaGetSymbolAddress returned a NULL address");
    g_scratch_addr[dev] = static_cast<unsigned char *>(p);
  }
  *out = g_scratch_addr[dev];
  return FDTD_LLG_OK;
}

}  // namespace

extern "C" int fdtd_llg_magnetic_box_static(const double *Ms, int nx, int ny, int nz,
                                            long long *out7, void *cuda_stream) {
  if (!Ms || !out7) return fail(nullptr, FDTD_LLG_EINVAL, "Ms and out7 must be DEVICE pointers, not NULL");
  if (nx < 1 || ny < 1 || nz < 1) return fail(nullptr, FDTD_LLG_EINVAL, "nx, ny, nz must be >= 1");
  const long long n = (long long)nx * ny * nz;
  if (n > FDTD_LLG_STATIC_MAX_CELLS)
    return fail(nullptr, FDTD_LLG_EINVAL,
                "nx*ny*nz = %lld cells is more than the %lld the static scratch of this call is sized for "
                "(FDTD_LLG_STATIC_MAX_CELLS): scan the map in z ranges and merge the boxes",
                n, (long long)FDTD_LLG_STATIC_MAX_CELLS);
  unsigned char *scratch = nullptr;
  const int rc = static_scratch_address(&scratch);
  if (rc) return rc;
  cudaStream_t stream = static_cast<cudaStream_t>(cuda_stream);
  // the ticket must start at 0 whatever an earlier (perhaps aborted) call left behind
  CU(nullptr, cudaMemsetAsync(scratch, 0, SB_HEAD, stream));
  const unsigned blocks = (unsigned)((n + SB_CHUNK - 1) / SB_CHUNK);
  k_mag_box_static<<<blocks, SB_THREADS, 0, stream>>>(Ms, nx, ny, nz, n, scratch, out7);
  CU(nullptr, cudaGetLastError());
  return FDTD_LLG_OK;
}
