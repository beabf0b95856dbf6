"""z-slab decomposition of the coupled FDTD-LLG step over several GPUs (fdtd_llg.h "Z-SLABS").

Domain decomposition is the paper's parallelism: one grid per rank, ghost cells
exchanged after each variable advancement, plus the global maximum of the LLG stopping test
(PAPER.md:154).  Here the cut is along z, one slab (one ``fdtd_llg`` handle, one GPU) per rank:

* the halo exchange is part of the update kernels: the thread that writes a value of a slab's
  first / last plane also stores it into the neighbour's ghost plane (peer-mapped memory, NVLink);
* what the slabs still need from each other is ORDER (a sub-step may start only after the
  neighbours finished the previous one) and the max of the residual word of every LLG iterate:
  one 8-byte max-allreduce per sub-step on the slabs' streams gives both (``merge``).

This module holds the host logic only: the partition plan, cutting a workload into slab inputs,
and the sequence of sub-steps.  No arithmetic of the method lives here.
"""
from __future__ import annotations

import copy
from dataclasses import dataclass
from typing import Optional

from .binding import (SUB_BEGIN, SUB_E, SUB_HM1, SUB_HM1_END, SUB_HM2, SUB_HM2_END, FdtdLlg,
                      SlabInfo, fdtd_llg_ipc_close, fdtd_llg_ipc_open, from_workload)

PEC, PERIODIC = 0, 1


# ----------------------------------------------------------------------------- the plan

@dataclass(frozen=True)
class SlabPlan:
    rank: int
    world: int
    k0: int                 # first global plane of the slab
    k1: int                 # one past its last plane
    lo: Optional[int]       # rank of the lower neighbour (None: the global z-low boundary)
    hi: Optional[int]       # rank of the upper neighbour

    @property
    def nz(self) -> int:
        return self.k1 - self.k0

    @property
    def ext(self) -> tuple:
        return (int(self.lo is not None), int(self.hi is not None))


def plan_slabs(nz_global: int, world: int, periodic_z: bool) -> list:
    """Equal slabs along z (the kernels address a neighbour's ghost plane with one offset for all
    arrays, which needs equal shapes).  A periodic z axis is closed by making the end slabs
    neighbours; with one slab there is no interface at all (the handle wraps by itself)."""
    if world < 1 or nz_global % world:
        raise ValueError(f"nz = {nz_global} is not a multiple of {world} slabs")
    nz = nz_global // world
    plans = []
    for r in range(world):
        lo = r - 1 if r > 0 else (world - 1 if periodic_z and world > 1 else None)
        hi = r + 1 if r < world - 1 else (0 if periodic_z and world > 1 else None)
        plans.append(SlabPlan(r, world, r * nz, (r + 1) * nz, lo, hi))
    return plans


def _planes(plan: SlabPlan, nz_global: int) -> list:
    """Global planes a slab's input arrays hold: its own and the neighbours' adjacent ones."""
    ks = list(range(plan.k0, plan.k1))
    if plan.lo is not None:
        ks.insert(0, (plan.k0 - 1) % nz_global)
    if plan.hi is not None:
        ks.append(plan.k1 % nz_global)
    return ks


def cut_workload(w, plan: SlabPlan):
    """The slab-local workload: every array cut to the slab's planes plus the neighbours' adjacent
    planes, source boxes clipped to the slab (slab coordinates), the z boundary type kept only
    where the slab touches the global boundary."""
    import torch
    if plan.world == 1:
        return w
    ks = _planes(plan, w.nz)
    contiguous = ks == list(range(ks[0], ks[0] + len(ks)))

    def cut(t):
        if t is None or isinstance(t, (int, float)):
            return t
        if contiguous:
            return t[ks[0]:ks[-1] + 1].contiguous()
        return t.index_select(0, torch.tensor(ks, device=t.device)).contiguous()

    s = copy.copy(w)
    s.name = f"{w.name}[slab {plan.rank}/{plan.world}]"
    s.nz = plan.nz
    s.bc = (w.bc[0], w.bc[1], PEC)
    s.slab_ext = plan.ext
    s.materials = {k: cut(v) for k, v in w.materials.items()}
    s.E = [cut(t) for t in w.E]
    s.H = [cut(t) for t in w.H]
    s.M_cell = [cut(t) for t in w.M_cell]
    s.sources = []
    for q in w.sources:
        z0, z1 = max(q.lo[2], plan.k0), min(q.hi[2], plan.k1)
        if z0 >= z1:
            continue
        c = copy.copy(q)
        c.lo = (q.lo[0], q.lo[1], z0 - plan.k0)
        c.hi = (q.hi[0], q.hi[1], z1 - plan.k0)
        if q.profile is not None:
            c.profile = q.profile[z0 - q.lo[2]:z1 - q.lo[2]].contiguous()
        s.sources.append(c)
    if getattr(w, "pml", None) is not None:
        p = list(w.pml)
        if plan.lo is not None:
            p[4] = 0
        if plan.hi is not None:
            p[5] = 0
        if p[4] > plan.nz or p[5] > plan.nz:
            raise ValueError("the z PML does not fit in the end slab")
        s.pml = tuple(p)
    return s


def stack_copies(w, plan: SlabPlan):
    """Weak-scaling input: the global grid is `world` copies of workload w stacked along z
    (PAPER.md:209 grows its base case in z the same way), walls only at the global ends.  The
    material maps and the initial magnetisation of every second copy are MIRRORED in z, so that
    like meets like at the interfaces (a magnet continues across one interface, vacuum across the
    next): every rank then has the same sweep box, i.e. the same work.  The E and H arrays are the
    copy's own everywhere (seeded noise or zero in the configs).  The slab of rank r is one copy;
    its neighbours' adjacent planes are cut from the neighbouring copies."""
    import torch
    if plan.world == 1:
        return w
    if w.bc[2] == PERIODIC:
        raise ValueError("stack_copies: a periodic z axis has no ends to stack on")

    def copy_of(t, rank, mirrored_kind):
        return t.flip(0) if (mirrored_kind and rank % 2 == 1) else t

    def ext(t, mirrored_kind):
        if t is None or isinstance(t, (int, float)):
            return t
        parts = [copy_of(t, plan.rank, mirrored_kind)]
        if plan.lo is not None:
            parts.insert(0, copy_of(t, plan.lo, mirrored_kind)[-1:])
        if plan.hi is not None:
            parts.append(copy_of(t, plan.hi, mirrored_kind)[:1])
        return torch.cat(parts, 0).contiguous()

    s = copy.copy(w)
    s.name = f"{w.name}[copy {plan.rank} of {plan.world} stacked in z]"
    s.slab_ext = plan.ext
    s.materials = {k: ext(v, True) for k, v in w.materials.items()}
    s.E = [ext(t, False) for t in w.E]
    s.H = [ext(t, False) for t in w.H]
    s.M_cell = [ext(t, True) for t in w.M_cell]
    if plan.rank % 2 == 1:      # the sources go with the structure
        s.sources = []
        for q in w.sources:
            c = copy.copy(q)
            c.lo = (q.lo[0], q.lo[1], w.nz - q.hi[2])
            c.hi = (q.hi[0], q.hi[1], w.nz - q.lo[2])
            if q.profile is not None:
                c.profile = q.profile.flip(0).contiguous()
            s.sources.append(c)
    if getattr(w, "pml", None) is not None:
        p = list(w.pml)
        if plan.rank % 2 == 1:
            p[4], p[5] = p[5], p[4]
        if plan.lo is not None:
            p[4] = 0
        if plan.hi is not None:
            p[5] = 0
        s.pml = tuple(p)
    return s


# ----------------------------------------------------------------------------- the sub-step sequence

class SlabStepper:
    """Sequence of sub-steps of one time step over the slabs this process drives (``self.sims``).

    Subclasses provide ``merge(r)``: afterwards the residual word r of every slab holds the maximum
    over ALL slabs, and every slab has completed the sub-step enqueued before it (stream order).
    ``converged(r)`` reads that word on the host -- the only host synchronisation, once per
    half-step in the usual case (``check_from``), never per iterate."""

    check_from = 3      # LLG iterations per half-step observed at tol 1e-12
    check_every = 3

    def __init__(self, sims, any_llg: bool, max_iter: int, tol: float):
        self.sims = list(sims)
        self.any_llg = bool(any_llg)
        self.max_iter = int(max_iter)
        self.tol = float(tol)
        self.merges = 0
        self.host_checks = 0

    def merge(self, r: int) -> None:
        raise NotImplementedError

    def converged(self, r: int) -> bool:
        raise NotImplementedError

    def _all(self, phase, r=0):
        for s in self.sims:
            s.substep(phase, r)

    def _half(self, phase, end):
        r = 0
        while True:
            r += 1
            self._all(phase, r)
            self.merge(r)
            if not self.any_llg or r >= self.max_iter:
                break
            if r >= self.check_from and (r - self.check_from) % self.check_every == 0:
                self.host_checks += 1
                if self.converged(r):
                    break
        self._all(end)
        self.merge(0)

    def step(self, n: int = 1) -> None:
        for _ in range(int(n)):
            self._all(SUB_BEGIN)
            self.merge(0)
            self._half(SUB_HM1, SUB_HM1_END)
            self._all(SUB_E)
            self.merge(0)
            self._half(SUB_HM2, SUB_HM2_END)


class LocalSlabs(SlabStepper):
    """All slabs of a grid on ONE device, driven by one host thread on one stream: the stream orders
    the sub-steps, the residual words are merged by a tiny elementwise max.  This is the one-GPU
    check of the decomposition (the same kernels, the same peer stores -- the 'peer' is local)."""

    def __init__(self, w, world: int, device="cuda:0", kernel_path=0, merge_h=True, time_scheme=0):
        import torch
        self.torch = torch
        self.plans = plan_slabs(w.nz, world, w.bc[2] == PERIODIC)
        self.stream = torch.cuda.Stream(device)
        def make(merge):
            return [from_workload(cut_workload(w, p), device=device, stream=self.stream, use_graph=False,
                                  kernel_path=kernel_path, merge_h=merge, time_scheme=time_scheme,
                                  slab_ext=p.ext) for p in self.plans]
        sims = make(merge_h)
        # merge_h is a property of the whole grid: a handle whose H source cannot be kept in a margin
        # switches it off for itself; then nobody merges (fdtd_llg_slab_connect refuses a mismatch)
        if len({s.stats()["merged_h"] for s in sims}) > 1:
            for s in sims:
                s.close()
            sims = make(False)
        for p, s in zip(self.plans, sims):
            nb = [None if q is None else (sims[q].slab_info(), sims[q].workspace.data_ptr())
                  for q in (p.lo, p.hi)]
            if world > 1:
                s.connect(nb[0], nb[1])
        any_llg = any(s.stats()["sweep_cells"] > 0 for s in sims)
        # the first-order scheme takes one explicit sweep per half-step (no iteration)
        super().__init__(sims, any_llg, w.llg_max_iter if (w.enable_llg and not time_scheme) else 1, w.llg_tol)
        self._words = {}

    def _word(self, r):
        if r not in self._words:
            self._words[r] = [s.residual_word(r) for s in self.sims]
        return self._words[r]

    def merge(self, r):
        self.merges += 1
        if r == 0 or len(self.sims) == 1:
            return                      # one stream: already ordered
        ws = self._word(r)
        with self.torch.cuda.stream(self.stream):
            m = ws[0].clone()
            for x in ws[1:]:
                m = self.torch.maximum(m, x)
            for x in ws:
                x.copy_(m)

    def converged(self, r):
        # the word is written on self.stream (a non-blocking stream the default stream does not wait
        # for): read it in that stream's order, or the host sees the re-armed 0 of a GPU that lags
        with self.torch.cuda.stream(self.stream):
            return float(self._word(r)[0].item()) < self.tol

    def read_fields(self, names=None) -> dict:
        """The global fields, slabs concatenated along z (host numpy arrays)."""
        import numpy as np
        parts = [{k: v.numpy() for k, v in s.read_fields(names).items()} for s in self.sims]
        return {k: np.concatenate([p[k] for p in parts], 0) for k in parts[0]}


class SlabSetupError(RuntimeError):
    """Raised on EVERY rank when the slabs of a grid could not be created and connected."""


class DistSlab(SlabStepper):
    """One slab per rank of a ``torch.distributed`` group, one process per GPU.  The neighbours'
    workspaces are mapped with CUDA IPC (peer access over NVLink); ``merge`` is an 8-byte
    max-allreduce on the slab's stream (NCCL), which is also the barrier the peer stores need.
    With ``backend == 'gloo'`` (tests: two processes sharing one GPU) the word goes through the
    host, which synchronises every sub-step; the kernels never wait on one another either way."""

    def __init__(self, slab_workload, plan: SlabPlan, device, group=None, kernel_path=0,
                 merge_h=True, time_scheme=0):
        import torch
        import torch.distributed as dist
        self.torch, self.dist, self.group = torch, dist, group
        self.plan = plan
        self.device = torch.device(device)
        self.stream = torch.cuda.Stream(self.device)
        w = slab_workload
        self.sim, self._mapped = None, {}
        # Set-up in lockstep: every step that can fail locally (creating the handle, exporting its
        # workspace, mapping a neighbour's) is followed by a collective in which ALL ranks learn
        # whether it worked, so that a failure on one rank raises SlabSetupError on every rank
        # instead of leaving the others in a collective.
        err, mine, everyone = None, None, [None] * plan.world
        for merge in ((True, False) if merge_h else (False,)):
            # merge_h is a property of the whole grid: if the slabs come out disagreeing (an H source
            # that cannot be kept in a margin switches it off on the handle that has it), all are
            # created again without it
            try:
                if self.sim is not None:
                    self.sim.close()
                self.sim = from_workload(w, device=self.device, stream=self.stream, use_graph=False,
                                         kernel_path=kernel_path, merge_h=merge, time_scheme=time_scheme,
                                         slab_ext=plan.ext)
                if plan.world > 1:
                    mine = (self.sim.slab_info().as_tuple(),) + self.sim.ipc_export()
            except Exception as e:          # noqa: BLE001  (reported to all ranks below)
                err, mine = e, None
            if plan.world == 1:
                break
            dist.all_gather_object(everyone, mine, group=group)
            states = {x[0][-1] for x in everyone if x is not None}     # SlabInfo.merged_h of every slab
            if len(states) <= 1 or any(x is None for x in everyone):
                break
        if plan.world > 1:
            if err is None:
                try:
                    nb = []
                    for q in (plan.lo, plan.hi):
                        if q is None:
                            nb.append(None)
                            continue
                        if everyone[q] is None:
                            raise RuntimeError(f"rank {q} could not create or export its slab")
                        info, handle, off = everyone[q]
                        if q not in self._mapped:
                            with torch.cuda.device(self.device):
                                self._mapped[q] = (fdtd_llg_ipc_open(handle, off), off)
                        nb.append((SlabInfo.from_tuple(info), self._mapped[q][0]))
                    self.sim.connect(nb[0], nb[1])
                except Exception as e:  # noqa: BLE001
                    err = e
            ok = torch.tensor([0.0 if err is not None else 1.0], dtype=torch.float64,
                              device="cpu" if self._gloo() else self.device)
            dist.all_reduce(ok, op=dist.ReduceOp.MIN, group=group)
            if float(ok.item()) == 0.0:
                self._release()
                raise SlabSetupError(repr(err) if err is not None else "the slab set-up failed on another rank")
        elif err is not None:
            raise err
        sim = self.sim
        flag = torch.tensor([float(sim.stats()["sweep_cells"] > 0)], dtype=torch.float64,
                            device="cpu" if self._gloo() else self.device)
        if plan.world > 1:
            dist.all_reduce(flag, op=dist.ReduceOp.MAX, group=group)
        super().__init__([sim], bool(flag.item() > 0),
                         w.llg_max_iter if (w.enable_llg and not time_scheme) else 1, w.llg_tol)
        self._words = {}
        if plan.world > 1:
            dist.barrier(group=group)

    def _release(self):
        for p, off in self._mapped.values():
            try:
                fdtd_llg_ipc_close(p, off)
            except Exception:           # noqa: BLE001
                pass
        self._mapped = {}
        if self.sim is not None:
            self.sim.close()
            self.sim = None

    def _gloo(self):
        return self.dist.get_backend(self.group) == "gloo"

    def _word(self, r):
        if r not in self._words:
            self._words[r] = self.sim.residual_word(r)
        return self._words[r]

    def merge(self, r):
        self.merges += 1
        if self.plan.world == 1:
            return
        w = self._word(r)
        if self._gloo():
            self.stream.synchronize()
            h = w.cpu()
            self.dist.all_reduce(h, op=self.dist.ReduceOp.MAX, group=self.group)
            with self.torch.cuda.stream(self.stream):
                w.copy_(h)
            self.stream.synchronize()
        else:
            with self.torch.cuda.stream(self.stream):
                self.dist.all_reduce(w, op=self.dist.ReduceOp.MAX, group=self.group)

    def converged(self, r):
        with self.torch.cuda.stream(self.stream):
            return float(self._word(r).item()) < self.tol

    def close(self):
        self.stream.synchronize()
        if self.plan.world > 1:
            self.dist.barrier(group=self.group)      # nobody still stores into a workspace that goes away
        self._release()
