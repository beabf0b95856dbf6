"""Host logic of the z-slab decomposition (paper_2103_12819_b200/slabs.py) on CPU: the partition
plan, cutting a workload into slab inputs, and -- two gloo processes, world_size 2 -- the
residual-word max-allreduce / stopping decisions of the sub-step sequence with a scripted stand-in
for the device library (the CUDA side of the same sequence is tests/test_slabs_gpu.py)."""
import os
import socket

import numpy as np
import pytest
import torch
import torch.multiprocessing as mp

from paper_2103_12819_b200 import workloads as wl
from paper_2103_12819_b200.slabs import (PERIODIC, SlabStepper, cut_workload, plan_slabs, stack_copies)
from paper_2103_12819_b200.binding import SUB_BEGIN, SUB_E, SUB_HM1, SUB_HM1_END, SUB_HM2, SUB_HM2_END


def test_plan_neighbours_and_ranges():
    p = plan_slabs(24, 4, False)
    assert [(q.k0, q.k1, q.lo, q.hi) for q in p] == [(0, 6, None, 1), (6, 12, 0, 2), (12, 18, 1, 3), (18, 24, 2, None)]
    assert [q.ext for q in p] == [(0, 1), (1, 1), (1, 1), (1, 0)]
    p = plan_slabs(24, 3, True)
    assert [(q.lo, q.hi) for q in p] == [(2, 1), (0, 2), (1, 0)]       # periodic z closed over the ends
    assert plan_slabs(24, 1, True)[0].ext == (0, 0)                      # one slab wraps by itself
    with pytest.raises(ValueError):
        plan_slabs(25, 4, False)


@pytest.mark.parametrize("cfg,world", [(5, 3), (4, 5), (2, 4)])
def test_cut_workload_carries_the_neighbours_planes_and_clips_sources(cfg, world):
    shape = {5: (10, 8, 12), 4: (12, 10, 40), 2: (8, 6, 12)}[cfg]
    w = wl.make_config(cfg, shape=shape)
    plans = plan_slabs(w.nz, world, w.bc[2] == PERIODIC)
    slabs = [cut_workload(w, p) for p in plans]
    glob = [t for t in (*w.E, *w.H, *w.M_cell, *w.materials.values()) if isinstance(t, torch.Tensor)]
    assert glob
    for p, s in zip(plans, slabs):
        assert s.nz == p.nz and s.slab_ext == p.ext and s.bc[2] == 0
        loc = [t for t in (*s.E, *s.H, *s.M_cell, *s.materials.values()) if isinstance(t, torch.Tensor)]
        for g, l in zip(glob, loc):
            assert l.shape[0] == p.nz + sum(p.ext)
            own = l[p.ext[0]:p.ext[0] + p.nz]
            assert torch.equal(own, g[p.k0:p.k1])
            if p.lo is not None:
                assert torch.equal(l[0], g[(p.k0 - 1) % w.nz])
            if p.hi is not None:
                assert torch.equal(l[-1], g[p.k1 % w.nz])
        for q in s.sources:
            assert 0 <= q.lo[2] < q.hi[2] <= p.nz
    # every source plane lands in exactly one slab
    for q in w.sources:
        n = sum((c.hi[2] - c.lo[2]) for s in slabs for c in s.sources if c.comp == q.comp)
        assert n == q.hi[2] - q.lo[2]
    # scalars stay scalars
    if cfg == 5:
        assert all(s.materials["alpha"] == 0.01 for s in slabs)


def test_stack_copies_mirrors_every_second_copy_so_that_like_meets_like():
    w = wl.make_config(5, shape=(10, 8, 12))
    plans = plan_slabs(3 * w.nz, 3, False)
    Ms = w.materials["Ms"]
    low, mid, top = (stack_copies(w, p) for p in plans)
    assert mid.slab_ext == (1, 1) and mid.nz == w.nz
    # copy 0 as it is (magnet in the lower half), copy 1 mirrored (magnet in the upper half), copy 2 as it is
    assert torch.equal(low.materials["Ms"][:-1], Ms) and torch.equal(mid.materials["Ms"][1:-1], Ms.flip(0))
    # interface 0|1: vacuum on both sides; interface 1|2: magnet on both sides
    assert float(low.materials["Ms"][-2].max()) == 0.0 and float(low.materials["Ms"][-1].max()) == 0.0
    assert float(mid.materials["Ms"][-2].min()) > 0.0 and float(mid.materials["Ms"][-1].min()) > 0.0
    # the ghost planes are the neighbours' edge planes
    assert torch.equal(low.materials["Ms"][-1], mid.materials["Ms"][1])
    assert torch.equal(mid.materials["Ms"][0], low.materials["Ms"][-2])
    assert torch.equal(mid.materials["Ms"][-1], top.materials["Ms"][1])
    assert torch.equal(mid.M_cell[2][-1], top.M_cell[2][1]) and torch.equal(top.M_cell[2][0], mid.M_cell[2][-2])
    # fields are the copy's own
    assert torch.equal(mid.E[0][0], w.E[0][-1]) and torch.equal(mid.E[0][-1], w.E[0][0])
    assert stack_copies(w, plans[0]).E[0].shape[0] == w.nz + 1


class _FakeSim:
    """Stands for one slab handle: records the sub-steps and 'computes' a scripted residual."""

    def __init__(self, script):
        self.script, self.calls, self.half, self.word = script, [], 0, {}

    def substep(self, phase, r=0):
        self.calls.append((phase, r))
        if phase in (SUB_HM1, SUB_HM2):
            res = self.script[self.half % len(self.script)]
            self.word[r] = res[r - 1] if r <= len(res) else 0.0
        if phase in (SUB_HM1_END, SUB_HM2_END):
            self.half += 1


class _GlooStepper(SlabStepper):
    def __init__(self, sim, max_iter, tol):
        super().__init__([sim], True, max_iter, tol)
        self.sim = sim

    def merge(self, r):
        import torch.distributed as dist
        self.merges += 1
        t = torch.tensor([self.sim.word.get(r, 0.0) if r else 0.0], dtype=torch.float64)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        if r:
            self.sim.word[r] = float(t[0])

    def converged(self, r):
        return self.sim.word[r] < self.tol


def _free_port():
    with socket.socket() as s:
        s.bind(("127.0.0.1", 0))
        return s.getsockname()[1]


def _worker(rank, world, port, q):
    import torch.distributed as dist
    os.environ["MASTER_ADDR"] = "127.0.0.1"
    os.environ["MASTER_PORT"] = str(port)
    dist.init_process_group("gloo", rank=rank, world_size=world)
    tol = 1e-12
    # residual of iterate r per half-step: rank 0 converges at r = 2, rank 1 needs 3 in the first
    # half-step and 5 in the second (its slab holds the slow faces): everybody must follow rank 1
    script = ([(1e-3, 1e-13, 0.0)], [(1e-3, 1e-8, 1e-13), (1e-2, 1e-5, 1e-8, 1e-10, 1e-13)])[rank]
    sim = _FakeSim(script)
    st = _GlooStepper(sim, 20, tol)
    st.step(2)
    q.put((rank, sim.calls, st.merges, st.host_checks, dict(sim.word)))
    dist.destroy_process_group()


def test_two_gloo_ranks_take_the_same_stopping_decisions():
    world, port = 2, _free_port()
    ctx = mp.get_context("spawn")
    q = ctx.Queue()
    procs = [ctx.Process(target=_worker, args=(r, world, port, q)) for r in range(world)]
    for p in procs:
        p.start()
    got = sorted(q.get(timeout=120) for _ in range(world))
    for p in procs:
        p.join(timeout=60)
        assert p.exitcode == 0
    (_, calls0, merges0, checks0, words0), (_, calls1, merges1, checks1, words1) = got
    assert calls0 == calls1 and merges0 == merges1 and checks0 == checks1
    # per step: BEGIN, HM1 r = 1..3 (checked at 3: converged), END, E, HM2 r = 1..6 (checked at 3: no,
    # at 6: iterate 6 found 5 converged and wrote nothing), END
    one = ([(SUB_BEGIN, 0)] + [(SUB_HM1, r) for r in (1, 2, 3)] + [(SUB_HM1_END, 0), (SUB_E, 0)]
           + [(SUB_HM2, r) for r in (1, 2, 3, 4, 5, 6)] + [(SUB_HM2_END, 0)])
    assert calls0 == one + one
    assert checks0 == 2 * 3 and merges0 == 2 * (1 + 3 + 1 + 1 + 6 + 1)
    assert words0 == words1                      # the merged words are the maxima over the ranks
    assert words0[3] == 1e-8 and words0[5] == 1e-13
