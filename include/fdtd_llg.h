/*
 * fdtd_llg.h -- C ABI of the B200-native coupled FDTD-LLG time stepper.
 *
 * The library advances the second-order coupled Maxwell / Landau-Lifshitz-Gilbert scheme of
 * Yao, Jambunathan, Zeng, Nonaka, arXiv 2103.12819 (citations: /root/reference/PAPER.md lines)
 * on ONE GPU (sm_100a), fp64:
 *
 *   per time step:   (H,M)^n -> (H,M)^{n+1/2}  with curl E^n       [S3.2.2 Step 1]
 *                                       E^n -> E^{n+1}            eq. 11              [S3.2.1 Step 2]
 *                                       (H,M)^{n+1/2} -> (H,M)^{n+1} with curl E^{n+1} [Step 3]
 *   each (H,M) half-step is the iterated trapezoidal LLG solve of eqs. 18-21
 *   with |M| = Ms renormalisation and the global stopping test of PAPER.md:154.
 *   Options add the first-order scheme, hard / soft sources of E and H
 *   (PAPER.md:100), the open boundary (PML) and the decomposition of the grid into
 *   z-slabs, one per GPU, with the halo exchange done by peer stores inside the update kernels
 *   (domain decomposition is the paper's parallelism; "Z-SLABS" below).
 *
 * Plain C types only: pointers (each argument says HOST or DEVICE), sizes, PODs.  No torch types.
 * Every step of the path runs in the library's own CUDA kernels; there is no CPU fallback.
 *
 * DATA LAYOUT (all arrays, user side and device side).  nx*ny*nz cells, x fastest, no ghost cells:
 *   idx = i + nx*(j + ny*k).  Entry (i,j,k) is the edge / face on the LOW side of cell (i,j,k):
 *     Ex (i+1/2,j,k)  Ey (i,j+1/2,k)  Ez (i,j,k+1/2)             tangential E on edges
 *     Hx (i,j+1/2,k+1/2)  Hy (i+1/2,j,k+1/2)  Hz (i+1/2,j+1/2,k)  normal H on faces
 *     M on the x-, y-, z-faces: all three components at every face (9 arrays)
 *     materials eps_r, sigma, mu_r, Ms, alpha, gamma at cell centres
 *   Boundaries per axis: FDTD_LLG_PEC or FDTD_LLG_PERIODIC; a PEC axis can carry
 *   an absorbing layer in front of its walls (options.pml).  On a PEC axis index 0
 *   is the lower wall, index n (not stored) the upper wall; wall-tangential E, wall-normal H and M on
 *   wall faces are identically 0.
 *
 * ERRORS.  Every call returns FDTD_LLG_OK (0) or a negative code; fdtd_llg_last_error() gives the
 * text (for a failed create: pass NULL).  Nothing is thrown, nothing aborts.
 *
 * THREADING.  A handle may be used by one host thread at a time.
 */
#ifndef FDTD_LLG_H
#define FDTD_LLG_H

#include <stddef.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fdtd_llg fdtd_llg; /* opaque */

enum {
  FDTD_LLG_OK = 0,
  FDTD_LLG_EINVAL = -1, /* bad argument (message says which)                       */
  FDTD_LLG_ENOMEM = -2, /* workspace too small / host allocation failed            */
  FDTD_LLG_ECUDA = -3,  /* a CUDA runtime call failed (message has the CUDA text)   */
  FDTD_LLG_ESTATE = -4  /* call not valid in this state                             */
};

enum { FDTD_LLG_PEC = 0, FDTD_LLG_PERIODIC = 1 };

/* where a user array lives */
enum { FDTD_LLG_HOST = 0, FDTD_LLG_DEVICE = 1 };

/* bits of `material_mask`: which material arrays are non-NULL */
enum {
  FDTD_LLG_MAT_EPS_R = 1, FDTD_LLG_MAT_SIGMA = 2, FDTD_LLG_MAT_MU_R = 4,
  FDTD_LLG_MAT_MS = 8, FDTD_LLG_MAT_ALPHA = 16, FDTD_LLG_MAT_GAMMA = 32
};

typedef struct {
  int bc[3];          /* per axis x,y,z: FDTD_LLG_PEC / FDTD_LLG_PERIODIC                        */
  int enable_llg;     /* 0: M = 0 everywhere, plain Maxwell                   */
  double h_bias[3];   /* uniform static bias H_0, A/m; enters H_eff only           */
  double ani_hk;      /* uniaxial anisotropy field H_k, A/m; 0 = off.  H_ani = H_k (M.u/Ms) u.
                         Not in the paper (future work); BASELINE config 4     */
  double ani_axis[3]; /* unit vector u                                                            */
  double llg_tol;     /* stop when max |M^r - M^{r-1}|/Ms < tol (paper uses 1e-6)   */
  int llg_max_iter;   /* iteration cap (the paper has none); at the cap the iterate is accepted   */
  int use_graph;      /* 1 (default): the step is captured once in a CUDA Graph and replayed, the LLG
                         iterates r >= 4 in a conditional node; 2: the same graph with plain kernel
                         nodes only (profilers do not look into conditional graphs); 0: no graph  */
  unsigned scalar_material_mask; /* FDTD_LLG_MAT_* bits: that material pointer addresses ONE double
                         in HOST memory, the uniform value (no nx*ny*nz array needed)            */
  int kernel_path;    /* which LLG sweep kernel runs (same arithmetic in all: bitwise-equal results).
                         0 (default): staged sweep, tile 32x16 (TMA-fed shared-memory ring for the
                         neighbour operands) where it applies (alpha, gamma, mu_r uniform) and the
                         sweep box gives every SM a work item, else the direct-load kernels;
                         1: direct-load kernels everywhere; 5: staged sweep whatever the box size
                         (1, 5: A/B checks of the two implementations)                           */
  int time_scheme;    /* 0 (default): the second-order scheme, iterated trapezoidal LLG;
                         1: the first-order scheme: one forward-Euler sweep of
                         eq. 7 / 12 per (H,M) half-step (advancing dt/2), N(M), then eq. 9 / 14;
                         llg_tol and llg_max_iter are not used                                   */
  int pml[6];         /* open boundary: cells of the PML on the x-low, x-high, y-low,
                         y-high, z-low, z-high side (0 = none).  The layer is part of the grid (its
                         outermost cells), the axis must be FDTD_LLG_PEC (the wall behind the layer)
                         and no magnetic cell may touch it.  Split-field Berenger layer with two-step
                         time-centred multiplicative damping, decay rate s(u) = s_max (u/L)^order,
                         s_max = -(order+1) c ln(pml_r0) / (2 L) (A26)                  */
  double pml_r0;      /* theoretical normal-incidence reflection of the layer (default 1e-6)       */
  int pml_order;      /* grading order m (default 3)                                               */
  int merge_h;        /* 1 (default): a face that no magnetic face reads (outside the LLG sweep box: the
                         whole grid of a Maxwell-only run) takes the second H half-step of step n and
                         the first of step n+1 -- the same curl E^{n+1}, PAPER.md:94 -- as ONE update:
                         H is kept at half-integer time there and the integer-time value (the mean
                         the paper's scheme holds) is formed when fields are read.  A third less
                         traffic; equal to the two half-steps up to rounding.  The PML layer and the
                         faces of an H source keep the plain half-steps: merging stops at a margin
                         on each side of the grid (the layer; an H-source box within 8 cells of a
                         side); an H source elsewhere switches it off.  0: two half-steps everywhere */
  int slab_ext[2];    /* z-low / z-high side of this grid is an INTERFACE to a neighbouring z-slab
                         (see Z-SLABS), neither wall nor periodic wrap; bc[2] must be FDTD_LLG_PEC
                         (it then describes the sides that are not interfaces)                    */
} fdtd_llg_options;

typedef struct {
  long long steps;                  /* time steps taken                                        */
  double time;                      /* steps * dt, s                                           */
  int iters_last;                   /* LLG iterations of the last (H,M) half-step              */
  int iters_max;                    /* largest iteration count of any half-step so far         */
  long long iters_total;            /* sum over all half-steps                                 */
  long long nonconverged_halfsteps; /* half-steps that hit llg_max_iter with residual >= tol   */
  double resid_last;                /* max |M^r - M^{r-1}|/Ms of the last executed iteration   */
  long long halfsteps;              /* (H,M) half-steps taken                                  */
  double courant;                   /* dt / vacuum Courant limit (>1 is allowed, not an error) */
  long long kernel_launches;        /* kernels this handle has launched in fdtd_llg_step       */
  long long magnetic_cells;         /* cells with Ms > 0 (0 when LLG is disabled)              */
  int launches_per_step;            /* kernel nodes one captured step launches (the LLG iterates
                                       r >= 4 sit in a conditional node and are not counted)   */
  long long sweep_cells;            /* cells of the LLG sweep box (bounding box of the magnetic
                                       cells + 1 halo cell), what one k_hm_sweep launch covers  */
  unsigned material_array_mask;     /* FDTD_LLG_MAT_* bits of the materials kept as device arrays
                                       (a uniform map is folded into a scalar)                  */
  int staged_sweeps;                /* 1: the LLG iterates r <= 3 run the staged kernel (hm_stage.cuh);
                                       0: the direct-load kernel (general materials, kernel_path 1,
                                       or a sweep box too small to give every SM a work item)   */
  int merged_h;                     /* 1: the H half-steps outside the sweep box are merged
                                       (options.merge_h and no H source far from the sides)     */
  int staged_maxwell;               /* the E phase runs the staged sweeps (eh_stage.cuh): 0 no (small
                                       grid, PML, kernel_path 1: k_e_update), 1 yes, 2 yes and fused
                                       with the merged H update outside the sweep box            */
} fdtd_llg_stats;

/* kernel classes of fdtd_llg_step_timed */
enum {
  FDTD_LLG_K_H_UPDATE = 0,   /* Maxwell H half-step outside the LLG sweep box (eq. 21, M = 0)   */
  FDTD_LLG_K_HM_FIRST = 1,   /* LLG iterate r = 1 (eqs. 18-21)                                  */
  FDTD_LLG_K_HM_ITER = 2,    /* LLG iterate r >= 3 that ran                                     */
  FDTD_LLG_K_HM_SKIPPED = 3, /* LLG iterate launched after convergence (exits on the flag)      */
  FDTD_LLG_K_E_UPDATE = 4,   /* eq. 11                                                          */
  FDTD_LLG_K_OTHER = 5,      /* source amplitudes, half-step bookkeeping, canonical-buffer copy */
  FDTD_LLG_K_HM_SECOND = 6,  /* LLG iterate r = 2 that ran                                       */
  FDTD_LLG_K_EH_FUSED = 7,   /* eq. 11 fused with the merged H update of the same faces (merge_h) */
  FDTD_LLG_K_NCLASS = 8
};

/* Fill *opt with the defaults: PEC x3, LLG on, no bias, no anisotropy (axis z), tol 1e-6
 * (PAPER.md:154), max 20 iterations, graph on, merge_h on, no slab interfaces. */
void fdtd_llg_default_options(fdtd_llg_options *opt);

/* Bytes of DEVICE workspace fdtd_llg_create needs for this grid.  `material_mask` = OR of the
 * FDTD_LLG_MAT_* bits of the material arrays that will be passed non-NULL (a uniform array costs
 * nothing once detected, so this is an upper bound).  Returns 0 on invalid arguments.
 * Budget: 12 doubles/cell for E,H (two sets each: every update is out of place); +21/cell when
 * enable_llg (the Jacobi H buffer, M and its time-n copy); +1/cell per material array; +13/cell
 * with a PML (12 split parts, the damping tables).  The same for a slab (its ghost planes exist
 * in every layout). */
size_t fdtd_llg_workspace_bytes(int nx, int ny, int nz, const fdtd_llg_options *opt,
                                unsigned material_mask);

/* Create a simulation (the user supplies CELL-CENTRED material maps).
 *   nx,ny,nz >= 1; dx,dy,dz,dt > 0 (SI).  dt above the Courant limit is allowed (stats.courant).
 *   eps_r, sigma, mu_r, Ms, alpha, gamma: nx*ny*nz doubles each, x fastest, in `mem_space`
 *     (HOST or DEVICE); NULL = uniform default 1, 0, 1, 0, 0, 0; with the material's bit set in
 *     opt->scalar_material_mask the pointer addresses one HOST double, the uniform value.  Read
 *     during the call, not retained.  Requirements: eps_r > 0, mu_r > 0, sigma >= 0, Ms >= 0 (else EINVAL).  gamma
 *     enters only as |gamma| (eqs. 19-20 use |gamma|).  Edge eps, sigma = mean of
 *     the 4 cells sharing the edge; face Ms, alpha, |gamma|, mu = mean of the 2 cells sharing the
 *     face, evaluated inside the kernels.  A face is magnetic iff enable_llg,
 *     Ms_face > 0 and it is not a PEC wall face.
 *   dev_workspace: DEVICE memory, >= fdtd_llg_workspace_bytes(), 256-byte aligned, owned by the
 *     caller and kept alive until fdtd_llg_destroy; the library allocates no device memory.
 *   cuda_stream: a cudaStream_t (NULL = default stream); all work is enqueued on it.
 * On success *out is the handle and all fields are zero. */
int fdtd_llg_create(fdtd_llg **out, int nx, int ny, int nz, double dx, double dy, double dz,
                    double dt, const double *eps_r, const double *sigma, const double *mu_r,
                    const double *Ms, const double *alpha, const double *gamma, int mem_space,
                    const fdtd_llg_options *opt, void *dev_workspace, size_t workspace_bytes,
                    void *cuda_stream);

/* Initial condition.  E[3], H[3]: values directly on their Yee locations; M_cell[3]:
 * magnetisation at CELL CENTRES, averaged to the faces (two-cell mean) and renormalised to the
 * face's Ms so that |M| = Ms holds discretely.  The array-of-pointers arguments are HOST arrays of
 * 3 pointers; the pointed-to data (nx*ny*nz doubles) lives in `mem_space`.  A NULL array or NULL
 * entry means zero.  Wall-tangential E and wall-normal H are forced to 0.
 * EINVAL if a magnetic face receives a zero averaged M.  Resets the step counter and statistics.
 * Synchronises the stream before returning. */
int fdtd_llg_set_fields(fdtd_llg *s, const double *const *E, const double *const *H,
                        const double *const *M_cell, int mem_space);

/* Add a soft current source to eq. 11, envelope of eq. 31:
 *   J_comp(t) = amplitude * exp(-(t-t0)^2 / (2 tp^2)) * cos(2 pi f0 t) * profile,  t = (n+1/2) dt,
 * on the comp-edges (comp 0,1,2 = Jx,Jy,Jz) with lo[d] <= index_d < hi[d].  profile: box-sized
 * ((hi-lo) doubles, x fastest) in `mem_space`, copied; NULL = 1.  Up to 8 sources. */
int fdtd_llg_set_source(fdtd_llg *s, int comp, const int *lo, const int *hi,
                        const double *profile, int mem_space, double amplitude, double f0,
                        double t0, double tp);

/* External excitations of both fields ("soft sources [are defined] in terms of the
 * time-rate of field change, and are applied at the beginning of the time step.  Hard sources are
 * enforced directly for the corresponding fields after their updates at each time step").  The
 * paper prints no formulas; the reading taken (A25), g(t) the envelope above:
 *   FDTD_LLG_SRC_SOFT_E  the current of fdtd_llg_set_source (A/m^2), t = (n+1/2) dt
 *   FDTD_LLG_SRC_HARD_E  after the E update of step n:   E_comp  = amplitude g((n+1) dt) profile
 *   FDTD_LLG_SRC_SOFT_H  before the first (H,M) half-step: H_comp += dt amplitude g(n dt) profile
 *   FDTD_LLG_SRC_HARD_H  after the second (H,M) half-step: H_comp = amplitude g((n+1) dt) profile
 * on the comp-edges (E) / comp-faces (H) of the box.  Wall-tangential E and wall-normal H stay 0;
 * M is never touched.  The 8 sources of a handle are shared by all kinds.  Other arguments and
 * errors as fdtd_llg_set_source (which is kind FDTD_LLG_SRC_SOFT_E). */
enum { FDTD_LLG_SRC_SOFT_E = 0, FDTD_LLG_SRC_HARD_E = 1, FDTD_LLG_SRC_SOFT_H = 2, FDTD_LLG_SRC_HARD_H = 3 };
int fdtd_llg_add_source(fdtd_llg *s, int kind, int comp, const int *lo, const int *hi,
                        const double *profile, int mem_space, double amplitude, double f0,
                        double t0, double tp);

/* Advance n >= 0 time steps.  Asynchronous: only enqueues work on the stream (n graph launches). */
int fdtd_llg_step(fdtd_llg *s, int n);

/* Advance n time steps (1 <= n <= 2048) with plain launches (no graph) and a CUDA-event pair
 * around every kernel launch; returns, per kernel class FDTD_LLG_K_*, the summed device time in
 * milliseconds (ms_by_class[FDTD_LLG_K_NCLASS], HOST) and the number of launches
 * (launches_by_class[FDTD_LLG_K_NCLASS], HOST).  Same arithmetic as fdtd_llg_step.  Synchronises
 * the stream.  This is the measurement hook of bench.py's roofline block. */
int fdtd_llg_step_timed(fdtd_llg *s, int n, double *ms_by_class, long long *launches_by_class);

/* Copy the present fields out.  E[3], H[3], M[9] are HOST arrays of pointers (or NULL); each
 * non-NULL entry receives nx*ny*nz doubles in `mem_space`.  M order: x-face (Mx,My,Mz), y-face
 * (Mx,My,Mz), z-face (Mx,My,Mz).  Synchronises the stream before returning. */
int fdtd_llg_read_fields(fdtd_llg *s, double *const *E, double *const *H, double *const *M,
                         int mem_space);

/* Statistics so far (synchronises the stream). */
int fdtd_llg_get_stats(fdtd_llg *s, fdtd_llg_stats *out);

/* Text of the last error on this handle; with s == NULL, of the last failed fdtd_llg_create (or
 * other call that takes no handle) on this thread.  Never NULL. */
const char *fdtd_llg_last_error(const fdtd_llg *s);

/* Release the handle (host memory, graph).  The workspace stays the caller's.  NULL is a no-op. */
void fdtd_llg_destroy(fdtd_llg *s);

/* ------------------------------------------------------------------------------------ Z-SLABS
 * Domain decomposition (one grid per rank, ghost cells exchanged "after each
 * variable advancement routine"; in the paper that exchange went through the MPI hosts and was 60 %
 * of the GPU run time).  Here the global grid is cut into slabs along z, one
 * handle (one GPU) each, every slab nx x ny x nz with the SAME nx, ny, nz.  A handle created with
 * options.slab_ext[side] = 1 treats that z side as an interface:
 *   - every array passed to fdtd_llg_create and fdtd_llg_set_fields then carries the neighbour's
 *     adjacent plane on that side: planes k = -1 (if slab_ext[0]) .. nz (if slab_ext[1]), i.e.
 *     nx*ny*(nz + slab_ext[0] + slab_ext[1]) doubles, lowest plane first (the caller cuts them out
 *     of the global arrays; for a globally periodic z axis the planes wrap around).  A material
 *     given as one scalar (scalar_material_mask) stays one scalar.  fdtd_llg_read_fields returns
 *     the slab's own nz planes; source boxes are in slab coordinates (0 <= index < nz).
 *   - after fdtd_llg_slab_connect, the kernel that writes a value of the slab's first / last plane
 *     also stores it into the neighbour's ghost plane (E_x, E_y, H_z of plane 0 go down, H_x, H_y
 *     of plane nz-1 go up: what the curls and the four-point averages read across the cut), with
 *     plain stores to the neighbour's workspace, which must be mapped in this process (same
 *     process, or fdtd_llg_ipc_open + peer access over NVLink).  No separate exchange step exists.
 * The caller drives the step with fdtd_llg_substep and orders the slabs:
 *   RULE: a sub-step may be enqueued on a slab only after BOTH neighbours have completed the
 *   previous sub-step (it reads ghost planes they wrote and overwrites ghost planes they read), and
 *   the residual word of LLG iterate r (fdtd_llg_residual_word) must hold the MAXIMUM over all
 *   slabs before iterate r+1 or the closing sub-step is enqueued anywhere (the
 *   stopping test is over the entire domain).  A max-allreduce of that one word on the slabs'
 *   streams (NCCL) is both the merge and the barrier; one host thread driving several handles on one
 *   stream gets the order for free.  Nothing here needs a host synchronisation.
 * The slabs then hold, bit for bit, what a single handle on the global grid holds (every update
 * is a Jacobi sweep: independent of the order in which faces are visited). */
typedef struct {
  unsigned long long fields_offset; /* bytes from the workspace start to the first field array */
  unsigned long long array_stride;  /* doubles between consecutive arrays                        */
  int nx;
  int ny;
  int nz;
  int n_arrays;                     /* field arrays at that stride (E, H, M sets)                */
  int merged_h;                     /* the handle's merge_h state: all slabs of a grid must agree (a
                                       PML or an H source switches it off for the handle that has it:
                                       create the other slabs with options.merge_h = 0 then)       */
} fdtd_llg_slab_info;

/* Layout facts a neighbour needs (HOST struct out). */
int fdtd_llg_get_slab_info(fdtd_llg *s, fdtd_llg_slab_info *out);

/* Connect the interfaces.  lo / hi: the lower / upper neighbour's info (NULL on a side that is not
 * an interface), lo_workspace / hi_workspace: DEVICE address of that neighbour's workspace as seen
 * from this process and this GPU.  EINVAL if the shapes or the merge_h states differ.  Sources of H
 * (which switch merge_h off) must be added before connecting.  Invalidates the captured step. */
int fdtd_llg_slab_connect(fdtd_llg *s, const fdtd_llg_slab_info *lo, void *lo_workspace,
                          const fdtd_llg_slab_info *hi, void *hi_workspace);

/* The sub-steps of one time step, in the order they must be enqueued: */
enum {
  FDTD_LLG_SUB_BEGIN = 0,   /* source amplitudes, soft H sources                      */
  FDTD_LLG_SUB_HM1 = 1,     /* first (H,M) half-step, LLG iterate r (argument): r = 1 also advances
                               the faces outside the sweep box; r >= 2 exits on the device if iterate
                               r-1 met the tolerance                                               */
  FDTD_LLG_SUB_HM1_END = 2, /* closes the half-step: iteration count, canonical H set              */
  FDTD_LLG_SUB_E = 3,       /* eq. 11, then the hard E sources                                     */
  FDTD_LLG_SUB_HM2 = 4,     /* second (H,M) half-step, iterate r (r = 1: also the merged H update
                               of the faces outside the sweep box, see merge_h)                    */
  FDTD_LLG_SUB_HM2_END = 5  /* closes it; hard H sources; the step counter advances                */
};
/* Enqueue one sub-step (asynchronous, plain launches).  r is used by the two HM phases only
 * (1 <= r <= llg_max_iter; without magnetic cells only r = 1 does anything).  ESTATE when called out
 * of order.  Works on any handle (a handle without interfaces: the same result as fdtd_llg_step). */
int fdtd_llg_substep(fdtd_llg *s, int phase, int r);

/* DEVICE address of the 8-byte residual word of LLG iterate r (1..llg_max_iter): the bit pattern
 * of the double max |M^r - M^{r-1}|/Ms over this slab's magnetic faces, >= 0, re-armed to 0 by the
 * closing sub-step.  r = 0: a scratch word the library never reads (for barriers). */
int fdtd_llg_residual_word(fdtd_llg *s, int r, void **dev_ptr);

/* Sharing a workspace between processes (one process per GPU): export gives the CUDA IPC handle
 * (64 bytes, HOST) of the allocation that holds this handle's workspace and the workspace's offset
 * in it; open maps it in another process (peer access is enabled as needed) and returns the
 * workspace's DEVICE address there; close unmaps (pass what open returned and the same offset). */
int fdtd_llg_ipc_export(fdtd_llg *s, unsigned char *handle64, unsigned long long *offset);
int fdtd_llg_ipc_open(const unsigned char *handle64, unsigned long long offset, void **dev_ptr);
int fdtd_llg_ipc_close(void *dev_ptr, unsigned long long offset);

/* --------------------------------------------------------- A QUERY THAT ALLOCATES NOTHING AT ALL
 * Where the magnet is, asked BEFORE a handle exists: the bounding box of the cells with Ms > 0 and
 * their number -- what fdtd_llg_create finds out for itself (stats.magnetic_cells; stats.sweep_cells
 * is this box plus the one-cell halo of the four-point averages) and what a caller
 * wants earlier: to cut the grid into slabs that share the magnetic cells, to see whether a workload
 * has an LLG part at all (+21 doubles per cell of workspace), to size the workspace it is about to
 * reserve.
 *
 * WHO THIS IS FOR.  Everything else in this library works inside the workspace the caller hands to
 * fdtd_llg_create, so it needs no allocation either -- but a caller with no handle yet has no
 * workspace to lend, and some callers cannot get device memory on the spot: a host application that
 * gave the whole GPU to its own memory pool at start-up (arena allocators of AMR frameworks such as the
 * one the paper's code is built on; the caching allocators of ML runtimes), where a
 * cudaMalloc from a library fails or fragments the pool; a time loop or a server thread that must not
 * stall, for which cudaMalloc / cudaFree are off limits because they may wait for all work in flight on
 * the device; code under a fixed memory budget that must not fail half-way.  For those callers this
 * one entry point keeps its scratch (one partial result per thread block and a ticket word) in a
 * fixed array that is part of the library's device image: FDTD_LLG_STATIC_SCRATCH_BYTES (1 MiB + 256 B)
 * on every GPU that loads the library, from load to process exit, used by nothing else.  It calls no
 * cudaMalloc, no cudaFree and no library routine that allocates device memory.
 *
 *   Ms    DEVICE, nx*ny*nz doubles, x fastest (the cell-centred map fdtd_llg_create takes), read only
 *   nx, ny, nz >= 1 with nx*ny*nz <= FDTD_LLG_STATIC_MAX_CELLS (2^29: a 768^3 grid fits, 1024^3 does
 *         not); beyond that EINVAL with a message that says so -- take the map in z ranges then and
 *         merge the boxes
 *   out7  DEVICE, 7 long long, written by the kernel: lo_x, lo_y, lo_z, hi_x, hi_y, hi_z (cell
 *         indices, hi INCLUSIVE), count.  No magnetic cell: lo = (nx, ny, nz), hi = (-1, -1, -1), 0.
 *         A NaN in the map is not magnetic (NaN > 0 is false), as in fdtd_llg_create's own scan
 *   cuda_stream  a cudaStream_t of the CURRENT device (NULL = default stream); the call only enqueues
 *         (one 256-byte memset of the ticket word and one kernel) and returns; out7 is valid once that
 *         work has completed on the stream.
 * Errors: EINVAL (NULL pointer, bad extent, too many cells), ECUDA; text through
 * fdtd_llg_last_error(NULL) (the per-thread message of the handle-free calls).
 *
 * RULES THAT COME WITH A SHARED, FIXED ARRAY.
 *  - The FIRST call on each device looks up the array's device address (once per device, under a
 *    lock, with that device current); it may load the library's device code.  Make that first call
 *    during set-up, before any stream capture is begun on the calling thread.
 *  - Every call on a device uses the same array, and the array keeps what the previous call left.
 *    The call clears the ticket word itself and overwrites every partial it later reads, so calls
 *    one after the other -- on one stream, or ordered by events -- need no clean-up by the caller.
 *    Two calls of one process that can be in flight on one GPU at the same time (streams without an
 *    ordering between them, two host threads) RACE on the array and both results are garbage:
 *    serialise them.  Separate processes do not share it: each has its own copy on the device.
 *  - The stream's device must be the current device (as for any kernel launch). */
#define FDTD_LLG_STATIC_MAX_CELLS (1LL << 29)
#define FDTD_LLG_STATIC_SCRATCH_BYTES ((1 << 20) + 256)
int fdtd_llg_magnetic_box_static(const double *Ms, int nx, int ny, int nz, long long *out7,
                                 void *cuda_stream);

#ifdef __cplusplus
}
#endif
#endif /* FDTD_LLG_H */
