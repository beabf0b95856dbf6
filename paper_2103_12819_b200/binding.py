"""Thin ctypes binding of the C ABI in ``include/fdtd_llg.h`` -- argument marshalling only.

Same names as the C entry points (``fdtd_llg_create`` ...), plus :class:`FdtdLlg`, a small
convenience wrapper that owns the torch workspace tensor and the stream.  PyTorch is used for
device memory and streams, nothing else: every step of the path runs in the library's kernels.
There is NO fallback: if ``libfdtd_llg.so`` is missing or does not load, importing a symbol from
it raises.
"""
from __future__ import annotations

import ctypes as C
import subprocess
from pathlib import Path

_HERE = Path(__file__).resolve().parent
LIB_PATH = _HERE / "libfdtd_llg.so"
_lib = None

OK, EINVAL, ENOMEM, ECUDA, ESTATE = 0, -1, -2, -3, -4
PEC, PERIODIC = 0, 1
HOST, DEVICE = 0, 1
MAT_BITS = {"eps_r": 1, "sigma": 2, "mu_r": 4, "Ms": 8, "alpha": 16, "gamma": 32}
MAT_ORDER = ("eps_r", "sigma", "mu_r", "Ms", "alpha", "gamma")
FIELD_NAMES = ("Ex", "Ey", "Ez", "Hx", "Hy", "Hz",
               "Mxx", "Mxy", "Mxz", "Myx", "Myy", "Myz", "Mzx", "Mzy", "Mzz")


class Options(C.Structure):
    _fields_ = [("bc", C.c_int * 3), ("enable_llg", C.c_int), ("h_bias", C.c_double * 3),
                ("ani_hk", C.c_double), ("ani_axis", C.c_double * 3), ("llg_tol", C.c_double),
                ("llg_max_iter", C.c_int), ("use_graph", C.c_int),
                ("scalar_material_mask", C.c_uint), ("kernel_path", C.c_int),
                ("time_scheme", C.c_int), ("pml", C.c_int * 6), ("pml_r0", C.c_double),
                ("pml_order", C.c_int), ("merge_h", C.c_int), ("slab_ext", C.c_int * 2)]


class Stats(C.Structure):
    _fields_ = [("steps", C.c_longlong), ("time", C.c_double), ("iters_last", C.c_int),
                ("iters_max", C.c_int), ("iters_total", C.c_longlong),
                ("nonconverged_halfsteps", C.c_longlong), ("resid_last", C.c_double),
                ("halfsteps", C.c_longlong), ("courant", C.c_double),
                ("kernel_launches", C.c_longlong), ("magnetic_cells", C.c_longlong),
                ("launches_per_step", C.c_int), ("sweep_cells", C.c_longlong),
                ("material_array_mask", C.c_uint), ("staged_sweeps", C.c_int),
                ("merged_h", C.c_int), ("staged_maxwell", C.c_int)]

    def as_dict(self):
        return {k: getattr(self, k) for k, _ in self._fields_}


class SlabInfo(C.Structure):
    _fields_ = [("fields_offset", C.c_ulonglong), ("array_stride", C.c_ulonglong),
                ("nx", C.c_int), ("ny", C.c_int), ("nz", C.c_int), ("n_arrays", C.c_int),
                ("merged_h", C.c_int)]

    def as_tuple(self):
        return tuple(getattr(self, k) for k, _ in self._fields_)

    @classmethod
    def from_tuple(cls, t):
        return cls(*t)


EXPORTS = ("fdtd_llg_default_options", "fdtd_llg_workspace_bytes", "fdtd_llg_create",
           "fdtd_llg_set_fields", "fdtd_llg_set_source", "fdtd_llg_add_source", "fdtd_llg_step", "fdtd_llg_step_timed",
           "fdtd_llg_read_fields",
           "fdtd_llg_get_stats", "fdtd_llg_last_error", "fdtd_llg_destroy",
           "fdtd_llg_get_slab_info", "fdtd_llg_slab_connect", "fdtd_llg_substep",
           "fdtd_llg_residual_word", "fdtd_llg_ipc_export", "fdtd_llg_ipc_open", "fdtd_llg_ipc_close",
           "fdtd_llg_magnetic_box_static")

# limits of fdtd_llg_magnetic_box_static (fdtd_llg.h)
STATIC_MAX_CELLS = 1 << 29
STATIC_SCRATCH_BYTES = (1 << 20) + 256

# sub-steps of one time step (fdtd_llg.h FDTD_LLG_SUB_*)
SUB_BEGIN, SUB_HM1, SUB_HM1_END, SUB_E, SUB_HM2, SUB_HM2_END = range(6)

KERNEL_CLASSES = ("h_update", "hm_first", "hm_iter", "hm_skipped", "e_update", "other", "hm_second",
                  "eh_fused")

_VP = C.c_void_p
_PP = C.POINTER(C.c_void_p)


def build_library(extra_flags=()) -> Path:
    """Compile ``csrc/fdtd_llg.cu`` for sm_100a into ``libfdtd_llg.so`` (in-tree)."""
    subprocess.run(["sh", str(_HERE / "csrc" / "build.sh"), *extra_flags], check=True)
    return LIB_PATH


def lib() -> C.CDLL:
    """The loaded library.  Raises (loudly) when it is not built -- there is no other path."""
    global _lib
    if _lib is None:
        if not LIB_PATH.exists():
            raise RuntimeError(
                f"{LIB_PATH} is missing: build it with __graft_entry__.build() "
                "(nvcc, sm_100a).  This package has no CPU or PyTorch fallback.")
        L = C.CDLL(str(LIB_PATH))
        L.fdtd_llg_default_options.argtypes = [C.POINTER(Options)]
        L.fdtd_llg_default_options.restype = None
        L.fdtd_llg_workspace_bytes.argtypes = [C.c_int] * 3 + [C.POINTER(Options), C.c_uint]
        L.fdtd_llg_workspace_bytes.restype = C.c_size_t
        L.fdtd_llg_create.argtypes = ([C.POINTER(_VP)] + [C.c_int] * 3 + [C.c_double] * 4
                                      + [_VP] * 6 + [C.c_int, C.POINTER(Options), _VP,
                                                     C.c_size_t, _VP])
        L.fdtd_llg_create.restype = C.c_int
        L.fdtd_llg_set_fields.argtypes = [_VP, _PP, _PP, _PP, C.c_int]
        L.fdtd_llg_set_fields.restype = C.c_int
        L.fdtd_llg_set_source.argtypes = [_VP, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int),
                                          _VP, C.c_int] + [C.c_double] * 4
        L.fdtd_llg_set_source.restype = C.c_int
        L.fdtd_llg_add_source.argtypes = [_VP, C.c_int, C.c_int, C.POINTER(C.c_int), C.POINTER(C.c_int),
                                          _VP, C.c_int] + [C.c_double] * 4
        L.fdtd_llg_add_source.restype = C.c_int
        L.fdtd_llg_step.argtypes = [_VP, C.c_int]
        L.fdtd_llg_step.restype = C.c_int
        L.fdtd_llg_step_timed.argtypes = [_VP, C.c_int, C.POINTER(C.c_double),
                                          C.POINTER(C.c_longlong)]
        L.fdtd_llg_step_timed.restype = C.c_int
        L.fdtd_llg_read_fields.argtypes = [_VP, _PP, _PP, _PP, C.c_int]
        L.fdtd_llg_read_fields.restype = C.c_int
        L.fdtd_llg_get_stats.argtypes = [_VP, C.POINTER(Stats)]
        L.fdtd_llg_get_stats.restype = C.c_int
        L.fdtd_llg_last_error.argtypes = [_VP]
        L.fdtd_llg_last_error.restype = C.c_char_p
        L.fdtd_llg_destroy.argtypes = [_VP]
        L.fdtd_llg_destroy.restype = None
        L.fdtd_llg_get_slab_info.argtypes = [_VP, C.POINTER(SlabInfo)]
        L.fdtd_llg_get_slab_info.restype = C.c_int
        L.fdtd_llg_slab_connect.argtypes = [_VP, C.POINTER(SlabInfo), _VP, C.POINTER(SlabInfo), _VP]
        L.fdtd_llg_slab_connect.restype = C.c_int
        L.fdtd_llg_substep.argtypes = [_VP, C.c_int, C.c_int]
        L.fdtd_llg_substep.restype = C.c_int
        L.fdtd_llg_residual_word.argtypes = [_VP, C.c_int, C.POINTER(_VP)]
        L.fdtd_llg_residual_word.restype = C.c_int
        L.fdtd_llg_ipc_export.argtypes = [_VP, C.POINTER(C.c_ubyte), C.POINTER(C.c_ulonglong)]
        L.fdtd_llg_ipc_export.restype = C.c_int
        L.fdtd_llg_ipc_open.argtypes = [C.POINTER(C.c_ubyte), C.c_ulonglong, C.POINTER(_VP)]
        L.fdtd_llg_ipc_open.restype = C.c_int
        L.fdtd_llg_ipc_close.argtypes = [_VP, C.c_ulonglong]
        L.fdtd_llg_ipc_close.restype = C.c_int
        L.fdtd_llg_magnetic_box_static.argtypes = [_VP, C.c_int, C.c_int, C.c_int, _VP, _VP]
        L.fdtd_llg_magnetic_box_static.restype = C.c_int
        _lib = L
    return _lib


# ---- the C entry points under their own names (pointers as ints / ctypes objects) -----------

def fdtd_llg_default_options() -> Options:
    o = Options()
    lib().fdtd_llg_default_options(C.byref(o))
    return o


def fdtd_llg_workspace_bytes(nx, ny, nz, opt: Options, material_mask: int) -> int:
    return lib().fdtd_llg_workspace_bytes(nx, ny, nz, C.byref(opt), material_mask)


def fdtd_llg_last_error(handle=None) -> str:
    return lib().fdtd_llg_last_error(handle).decode()


class FdtdLlgError(RuntimeError):
    def __init__(self, code, msg):
        super().__init__(f"fdtd_llg error {code}: {msg}")
        self.code = code


def _check(rc, handle):
    if rc != OK:
        raise FdtdLlgError(rc, fdtd_llg_last_error(handle))


def _ptr(t):
    """Data pointer of a torch tensor / numpy array (contiguous float64), or None."""
    if t is None:
        return None
    if hasattr(t, "data_ptr"):
        return t.data_ptr()
    return t.ctypes.data


def _ptr_array(items, n):
    arr = (C.c_void_p * n)()
    for q in range(n):
        arr[q] = _ptr(items[q]) if items is not None and items[q] is not None else None
    return arr


class FdtdLlg:
    """One simulation.  ``materials``: dict name -> array (torch CPU/CUDA tensor or numpy array,
    float64, nx*ny*nz, x fastest) or missing for the default.  All arrays passed in one call must
    live in the same memory space."""

    def __init__(self, nx, ny, nz, dx, dy, dz, dt, *, materials=None, bc=(PEC, PEC, PEC),
                 enable_llg=True, h_bias=(0.0, 0.0, 0.0), ani_hk=0.0, ani_axis=(0.0, 0.0, 1.0),
                 llg_tol=1e-6, llg_max_iter=20, use_graph=True, device="cuda:0", stream=None,
                 kernel_path=0, time_scheme=0, pml=None, pml_r0=None, pml_order=None,
                 merge_h=True, slab_ext=(0, 0)):
        import torch
        self._torch = torch
        self.shape = (nz, ny, nx)
        self.n = nx * ny * nz
        # a slab's input arrays carry the neighbours' adjacent planes (fdtd_llg.h "Z-SLABS")
        self.slab_ext = (int(bool(slab_ext[0])), int(bool(slab_ext[1])))
        self.n_in = nx * ny * (nz + sum(self.slab_ext))
        self.device = torch.device(device)
        self._h = None
        L = lib()
        opt = fdtd_llg_default_options()
        for d in range(3):
            opt.bc[d] = int(bc[d])
            opt.h_bias[d] = float(h_bias[d])
            opt.ani_axis[d] = float(ani_axis[d])
        opt.enable_llg = int(bool(enable_llg))
        opt.ani_hk = float(ani_hk)
        opt.llg_tol = float(llg_tol)
        opt.llg_max_iter = int(llg_max_iter)
        opt.use_graph = 2 if use_graph == 2 else int(bool(use_graph))   # 2: graph without the conditional node
        opt.kernel_path = int(kernel_path)
        opt.time_scheme = int(time_scheme)
        if pml is not None:
            for q in range(6):
                opt.pml[q] = int(pml[q])
        if pml_r0 is not None:
            opt.pml_r0 = float(pml_r0)
        if pml_order is not None:
            opt.pml_order = int(pml_order)
        opt.merge_h = int(bool(merge_h))
        opt.slab_ext[0], opt.slab_ext[1] = self.slab_ext
        self.options = opt
        materials = {k: v for k, v in (materials or {}).items() if v is not None}
        scalars = {k: C.c_double(float(v)) for k, v in materials.items()
                   if isinstance(v, (int, float))}
        opt.scalar_material_mask = sum(MAT_BITS[k] for k in scalars)
        mats = [None if k in scalars else self._prep(materials.get(k)) for k in MAT_ORDER]
        mask = sum(MAT_BITS[k] for k in MAT_ORDER if k in materials and k not in scalars)
        space = self._space([m for m in mats if m is not None])
        nbytes = fdtd_llg_workspace_bytes(nx, ny, nz, opt, mask)
        if nbytes == 0:
            raise FdtdLlgError(EINVAL, "fdtd_llg_workspace_bytes rejected the grid/options")
        with torch.cuda.device(self.device):
            self.stream = stream if stream is not None else torch.cuda.Stream(self.device)
            self.workspace = torch.empty(nbytes, dtype=torch.uint8, device=self.device)
            h = C.c_void_p()
            # make allocations of the current stream visible to ours
            self.stream.wait_stream(torch.cuda.current_stream(self.device))
            rc = L.fdtd_llg_create(C.byref(h), nx, ny, nz, dx, dy, dz, dt,
                                   *[C.addressof(scalars[k]) if k in scalars else _ptr(m)
                                     for k, m in zip(MAT_ORDER, mats)], space, C.byref(opt),
                                   self.workspace.data_ptr(), nbytes, self.stream.cuda_stream)
        if rc != OK:
            raise FdtdLlgError(rc, fdtd_llg_last_error(None))
        self._h = h

    # -- helpers ------------------------------------------------------------------------------
    def _prep(self, a):
        if a is None:
            return None
        torch = self._torch
        if isinstance(a, torch.Tensor):
            t = a.detach().to(torch.float64).contiguous()
        else:
            import numpy as np
            t = torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64))
        if t.numel() != self.n_in:
            raise ValueError(f"array has {t.numel()} entries, expected {self.n_in}")
        return t

    @staticmethod
    def _space(tensors):
        kinds = {t.is_cuda for t in tensors}
        if len(kinds) > 1:
            raise ValueError("all arrays of one call must live in the same memory space")
        return DEVICE if kinds == {True} else HOST

    def _sync_in(self):
        self.stream.wait_stream(self._torch.cuda.current_stream(self.device))

    # -- the C calls --------------------------------------------------------------------------
    def set_fields(self, E=None, H=None, M_cell=None):
        E = [self._prep(a) for a in (E or (None,) * 3)]
        H = [self._prep(a) for a in (H or (None,) * 3)]
        M = [self._prep(a) for a in (M_cell or (None,) * 3)]
        space = self._space([t for t in (*E, *H, *M) if t is not None])
        self._sync_in()
        with self._torch.cuda.device(self.device):
            rc = lib().fdtd_llg_set_fields(self._h, _ptr_array(E, 3), _ptr_array(H, 3),
                                           _ptr_array(M, 3), space)
        _check(rc, self._h)

    def set_source(self, comp, lo, hi, profile=None, amplitude=1.0, f0=0.0, t0=0.0, tp=1.0, kind=0):
        """kind: 0 soft E (the current of eq. 11), 1 hard E, 2 soft H, 3 hard H (fdtd_llg_add_source)."""
        prof = None
        if profile is not None:
            torch = self._torch
            prof = (profile.detach().to(torch.float64).contiguous()
                    if isinstance(profile, torch.Tensor) else self._prep_any(profile))
        space = DEVICE if (prof is not None and prof.is_cuda) else HOST
        self._sync_in()
        with self._torch.cuda.device(self.device):
            rc = lib().fdtd_llg_add_source(self._h, int(kind), int(comp), (C.c_int * 3)(*lo),
                                           (C.c_int * 3)(*hi), _ptr(prof), space,
                                           float(amplitude), float(f0), float(t0), float(tp))
        _check(rc, self._h)

    def _prep_any(self, a):
        import numpy as np
        return self._torch.from_numpy(np.ascontiguousarray(a, dtype=np.float64))

    def step(self, n=1):
        with self._torch.cuda.device(self.device):
            rc = lib().fdtd_llg_step(self._h, int(n))
        _check(rc, self._h)

    def step_timed(self, n=1) -> dict:
        """n steps with an event pair around every launch: {class: (ms, launches)}."""
        ms = (C.c_double * len(KERNEL_CLASSES))()
        cnt = (C.c_longlong * len(KERNEL_CLASSES))()
        with self._torch.cuda.device(self.device):
            rc = lib().fdtd_llg_step_timed(self._h, int(n), ms, cnt)
        _check(rc, self._h)
        return {k: (ms[q], cnt[q]) for q, k in enumerate(KERNEL_CLASSES)}

    def read_fields(self, names=None, device=None, out=None) -> dict:
        """Fields as torch tensors shaped (nz, ny, nx).  ``device=None``: pinned host memory."""
        torch = self._torch
        names = FIELD_NAMES if names is None else tuple(names)
        if out is None:
            if device is None:
                out = {nm: torch.empty(self.shape, dtype=torch.float64).pin_memory() for nm in names}
            else:
                out = {nm: torch.empty(self.shape, dtype=torch.float64, device=device) for nm in names}
        space = self._space(list(out.values()))
        ptrs = [out.get(nm) for nm in FIELD_NAMES]
        self._sync_in()
        with torch.cuda.device(self.device):
            rc = lib().fdtd_llg_read_fields(self._h, _ptr_array(ptrs[0:3], 3),
                                            _ptr_array(ptrs[3:6], 3), _ptr_array(ptrs[6:15], 9),
                                            space)
        _check(rc, self._h)
        return out

    # -- z-slabs (fdtd_llg.h "Z-SLABS") -------------------------------------------------------
    def slab_info(self) -> SlabInfo:
        info = SlabInfo()
        _check(lib().fdtd_llg_get_slab_info(self._h, C.byref(info)), self._h)
        return info

    def connect(self, lo=None, hi=None):
        """lo / hi: (SlabInfo, device address of that neighbour's workspace in this process) or None."""
        a = [(C.byref(x[0]), C.c_void_p(x[1])) if x is not None else (None, None) for x in (lo, hi)]
        with self._torch.cuda.device(self.device):
            rc = lib().fdtd_llg_slab_connect(self._h, a[0][0], a[0][1], a[1][0], a[1][1])
        _check(rc, self._h)

    def substep(self, phase, r=0):
        with self._torch.cuda.device(self.device):
            rc = lib().fdtd_llg_substep(self._h, int(phase), int(r))
        _check(rc, self._h)

    def residual_word(self, r):
        """Zero-copy view (1 float64) of the residual word of LLG iterate r inside the workspace."""
        p = C.c_void_p()
        _check(lib().fdtd_llg_residual_word(self._h, int(r), C.byref(p)), self._h)
        off = p.value - self.workspace.data_ptr()
        return self.workspace[off:off + 8].view(self._torch.float64)

    def ipc_export(self):
        """(64-byte CUDA IPC handle, offset) of the workspace, for fdtd_llg_ipc_open in another process."""
        h = (C.c_ubyte * 64)()
        off = C.c_ulonglong()
        _check(lib().fdtd_llg_ipc_export(self._h, h, C.byref(off)), self._h)
        return bytes(h), int(off.value)

    def stats(self) -> dict:
        st = Stats()
        with self._torch.cuda.device(self.device):
            rc = lib().fdtd_llg_get_stats(self._h, C.byref(st))
        _check(rc, self._h)
        return st.as_dict()

    def close(self):
        if self._h is not None:
            self.stream.synchronize()
            lib().fdtd_llg_destroy(self._h)
            self._h = None
            self.workspace = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass


def fdtd_llg_ipc_open(handle: bytes, offset: int) -> int:
    """Map another process's workspace; returns its device address here."""
    h = (C.c_ubyte * 64).from_buffer_copy(handle)
    p = C.c_void_p()
    rc = lib().fdtd_llg_ipc_open(h, C.c_ulonglong(offset), C.byref(p))
    if rc != OK:
        raise FdtdLlgError(rc, fdtd_llg_last_error(None))
    return p.value


def fdtd_llg_ipc_close(ptr: int, offset: int) -> None:
    rc = lib().fdtd_llg_ipc_close(C.c_void_p(ptr), C.c_ulonglong(offset))
    if rc != OK:
        raise FdtdLlgError(rc, fdtd_llg_last_error(None))


def fdtd_llg_magnetic_box_static(Ms, out7, stream=None) -> None:
    """Bounding box and number of the cells with Ms > 0, for callers that must not allocate device
    memory (a GPU handed over to the application's own memory pool, a loop that cannot afford the
    device-wide wait an allocation may cost, a fixed memory budget): the kernel's scratch is a fixed
    array inside the library, so neither the library nor this wrapper allocates anything.

    ``Ms``: CUDA float64 tensor shaped (nz, ny, nx), contiguous, at most ``STATIC_MAX_CELLS`` cells;
    ``out7``: CUDA int64 tensor of 7 entries on the same device, supplied by the caller, filled with
    lo_x, lo_y, lo_z, hi_x, hi_y, hi_z (inclusive), count -- or (nx, ny, nz), (-1, -1, -1), 0 when no
    cell is magnetic; ``stream``: a torch stream (default: the current one).  Only enqueues: read
    ``out7`` in stream order.  Calls share the library's one scratch array per GPU: calls that could
    run at the same time on one GPU race, keep them on one stream or order them.  The first call on
    a device does a one-time address look-up; make it during set-up, before any stream capture."""
    import torch
    if not (isinstance(Ms, torch.Tensor) and Ms.is_cuda and Ms.dtype == torch.float64
            and Ms.dim() == 3 and Ms.is_contiguous()):
        raise ValueError("Ms must be a contiguous CUDA float64 tensor shaped (nz, ny, nx)")
    if not (isinstance(out7, torch.Tensor) and out7.device == Ms.device and out7.dtype == torch.int64
            and out7.numel() == 7 and out7.is_contiguous()):
        raise ValueError("out7 must be a contiguous CUDA int64 tensor of 7 entries on Ms's device")
    nz, ny, nx = Ms.shape
    with torch.cuda.device(Ms.device):
        st = stream if stream is not None else torch.cuda.current_stream(Ms.device)
        rc = lib().fdtd_llg_magnetic_box_static(Ms.data_ptr(), nx, ny, nz, out7.data_ptr(),
                                                st.cuda_stream)
    if rc != OK:
        raise FdtdLlgError(rc, fdtd_llg_last_error(None))


def from_workload(w, device="cuda:0", use_graph=True, stream=None, fields_device=None,
                  kernel_path=0, time_scheme=0, merge_h=True, slab_ext=None) -> FdtdLlg:
    """Create a simulation from a :class:`workloads.Workload` and load its initial state.
    Arrays are passed in whatever memory space the workload's tensors live in."""
    sim = FdtdLlg(w.nx, w.ny, w.nz, w.dx, w.dy, w.dz, w.dt, materials=w.materials, bc=w.bc,
                  enable_llg=w.enable_llg, h_bias=w.h_bias, ani_hk=w.ani_hk, ani_axis=w.ani_axis,
                  llg_tol=w.llg_tol, llg_max_iter=w.llg_max_iter, use_graph=use_graph,
                  device=device, stream=stream, kernel_path=kernel_path,
                  time_scheme=time_scheme, pml=getattr(w, "pml", None),
                  pml_r0=getattr(w, "pml_r0", None), pml_order=getattr(w, "pml_order", None),
                  merge_h=merge_h,
                  slab_ext=slab_ext if slab_ext is not None else getattr(w, "slab_ext", (0, 0)))
    sim.set_fields(w.E, w.H, w.M_cell)
    for s in w.sources:
        sim.set_source(s.comp, s.lo, s.hi, s.profile, s.amplitude, s.f0, s.t0, s.tp,
                       kind=getattr(s, "kind", 0))
    return sim
