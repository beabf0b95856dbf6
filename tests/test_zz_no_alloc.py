"""``fdtd_llg_magnetic_box_static``: the one entry point for callers that cannot allocate.

Some users of this library may not call cudaMalloc when they need an answer: an application that
handed the whole GPU to its own memory pool at start-up (the arena of an AMR framework, the caching
allocator of an ML runtime), a time loop or server thread for which the device-wide wait that an
allocation or a free may cost is not acceptable, a job under a fixed memory budget.  Everything else
here lives in the workspace the caller lends to ``fdtd_llg_create``; this query is asked before a
handle (and hence a workspace) exists, so its scratch is a fixed 1 MiB array inside the library.

What is checked: the answer equals the one the existing path gives -- ``fdtd_llg_create``'s own scan
of the same Ms map, read back through ``stats`` (``magnetic_cells`` exactly; ``sweep_cells`` = the
box plus the one-cell halo, rebuilt here from the box) -- and a plain numpy scan, bit for bit (these
are integers: the suite's tolerance for index work is zero), on calls issued back to back on one
stream, where the later call must not see what the earlier one left in the shared array.

This file sorts last on purpose: ``pytest -x`` stops at the first failure, and a failure here must
not hide the parity tests.  It does not depend on them: it passes alone in a fresh process too.
"""
import ctypes as C

import numpy as np
import pytest


def _numpy_box(ms):
    """(lo_x, lo_y, lo_z, hi_x, hi_y, hi_z, count) of ms > 0; ms shaped (nz, ny, nx)."""
    nz, ny, nx = ms.shape
    k, j, i = np.nonzero(ms > 0)
    if i.size == 0:
        return [nx, ny, nz, -1, -1, -1, 0]
    return [int(i.min()), int(j.min()), int(k.min()), int(i.max()), int(j.max()), int(k.max()), int(i.size)]


def _sweep_cells_from_box(box, shape):
    """The LLG sweep box of a PEC grid without PML, as fdtd_llg_create builds it from the cell box
    (fdtd_llg.h stats.sweep_cells): one halo cell below, two index planes above (faces of the last
    cell + halo), clipped to the grid, x start rounded down to an even index."""
    nz, ny, nx = shape
    if box[6] == 0:
        return 0
    cells = 1
    for d, n in enumerate((nx, ny, nz)):
        lo = max(box[d] - 1, 0)
        if d == 0:
            lo &= ~1
        hi = min(box[3 + d] + 2, n)
        cells *= hi - lo
    return cells


def _maps():
    """Seeded Ms maps, (name, array (nz, ny, nx)): several thread blocks with a ragged tail, rows
    shorter and longer than the 256-cell thread stride, an empty map, a full one, single cells in
    the corners of the index space, a NaN (not magnetic)."""
    rng = np.random.default_rng(20260611)
    out = []
    a = np.zeros((90, 150, 200))                    # 2.7 M cells: 165 blocks, the last one ragged
    a[20:61, 33:100, 41:160] = 1.4e5                # a ferrite slab ...
    a[20:61, 33:100, 41:160] *= rng.random((41, 67, 119)) > 0.3   # ... with holes
    a[77, 3, 197] = 1.0                             # and two stray cells
    a[5, 140, 2] = 2.0
    out.append(("slab_with_holes_200x150x90", a))
    from paper_2103_12819_b200 import workloads as wl
    w4 = wl.make_config(4, shape=wl.SMALL_SHAPES[4])
    out.append(("config4_small", w4.materials["Ms"].numpy().reshape(w4.nz, w4.ny, w4.nx).copy()))
    b = np.zeros((70, 4, 1024))                     # the paper's thin guides: ny = 4
    b[30:50, 1:3, 500:700] = 8.0e4
    out.append(("thin_1024x4x70", b))
    c = np.zeros((3001, 5, 3))                      # rows far shorter than the thread stride
    c[1234, 2, 1] = 1.0
    c[2999, 4, 2] = 1.0
    c[17, 0, 0] = np.nan                            # NaN > 0 is false: not magnetic
    out.append(("needle_3x5x3001", c))
    out.append(("empty_50x40x30", np.zeros((30, 40, 50))))
    out.append(("full_33x17x9", np.full((9, 17, 33), 1.0e5)))
    e = np.zeros((6, 7, 1000))                      # rows longer than the thread stride
    e[0, 0, 0] = 1.0
    e[5, 6, 999] = 1.0
    out.append(("corners_1000x7x6", e))
    return out


@pytest.mark.gpu
def test_static_scratch_scan_matches_create_and_numpy_on_calls_in_a_row():
    import torch
    from paper_2103_12819_b200 import binding as B

    dev = torch.device("cuda:0")
    maps = _maps()
    ms_dev = [torch.from_numpy(m).to(dev) for _, m in maps]
    # outputs are the caller's: allocated here, before the calls, poisoned so that a skipped write shows
    outs = [torch.full((7,), -777, dtype=torch.int64, device=dev) for _ in range(2 * len(maps))]
    torch.cuda.synchronize(dev)

    # the first call on a device does the one-time address look-up (set-up, may load device code)
    B.fdtd_llg_magnetic_box_static(ms_dev[0], outs[0])
    torch.cuda.synchronize(dev)
    free_before = torch.cuda.mem_get_info(dev)[0]

    # all maps back to back on one stream, no synchronisation in between, big before small and small
    # before big: each call shares the array with the one before it
    order = list(range(len(maps))) + list(reversed(range(len(maps))))
    for slot, q in enumerate(order):
        B.fdtd_llg_magnetic_box_static(ms_dev[q], outs[slot])
    torch.cuda.synchronize(dev)
    free_after = torch.cuda.mem_get_info(dev)[0]
    assert free_after >= free_before, "the calls took device memory"

    for slot, q in enumerate(order):
        name, m = maps[q]
        got = outs[slot].cpu().tolist()
        assert got == _numpy_box(m), (name, slot, got)

    # the existing path: fdtd_llg_create's own scan of the same map (in the handle's workspace)
    for (name, m), t in zip(maps, ms_dev):
        nz, ny, nx = m.shape
        if not np.all(np.isfinite(m)):
            continue                                 # create refuses a non-finite map
        sim = B.FdtdLlg(nx, ny, nz, 1e-6, 1e-6, 1e-6, 1e-15,
                        materials={"Ms": t.reshape(-1), "alpha": 0.01, "gamma": -1.759e11})
        st = sim.stats()
        sim.close()
        out = torch.full((7,), -777, dtype=torch.int64, device=dev)
        B.fdtd_llg_magnetic_box_static(t, out)      # once more, after create's kernels ran
        got = out.cpu().tolist()
        assert got[6] == st["magnetic_cells"], name
        assert _sweep_cells_from_box(got, m.shape) == st["sweep_cells"], name


@pytest.mark.gpu
def test_static_scratch_scan_on_a_side_stream_and_a_large_map():
    """256^3 (1024 thread blocks, 16.8 M cells) on a non-default stream, twice, against torch's own
    reductions on the device."""
    import torch
    from paper_2103_12819_b200 import binding as B

    dev = torch.device("cuda:0")
    g = torch.Generator(device=dev).manual_seed(7)
    ms = (torch.rand((256, 256, 256), generator=g, device=dev, dtype=torch.float64) > 0.999).double()
    ms[:40] = 0
    ms[:, 250:] = 0
    ms[:, :, :3] = 0
    k, j, i = torch.nonzero(ms > 0, as_tuple=True)
    ref = [int(i.min()), int(j.min()), int(k.min()), int(i.max()), int(j.max()), int(k.max()), int(i.numel())]
    out = torch.zeros((2, 7), dtype=torch.int64, device=dev)
    s = torch.cuda.Stream(dev)
    s.wait_stream(torch.cuda.current_stream(dev))
    B.fdtd_llg_magnetic_box_static(ms, out[0], stream=s)
    B.fdtd_llg_magnetic_box_static(ms, out[1], stream=s)
    s.synchronize()
    assert out[0].cpu().tolist() == ref and out[1].cpu().tolist() == ref


def test_static_scratch_call_rejects_what_it_cannot_hold():
    """Argument checks come before anything touches a device (this runs on a box without a GPU):
    a map beyond FDTD_LLG_STATIC_MAX_CELLS is refused with a message that names the limit."""
    from paper_2103_12819_b200 import binding as B
    if not B.LIB_PATH.exists():
        B.build_library()
    L = B.lib()
    fake = C.c_void_p(4096)   # never dereferenced: the checks fail first
    assert L.fdtd_llg_magnetic_box_static(fake, 1024, 1024, 1024, fake, None) == B.EINVAL
    msg = B.fdtd_llg_last_error(None)
    assert "FDTD_LLG_STATIC_MAX_CELLS" in msg and str(1024 ** 3) in msg and str(B.STATIC_MAX_CELLS) in msg
    assert L.fdtd_llg_magnetic_box_static(fake, 1024, 1024, 513, fake, None) == B.EINVAL
    assert L.fdtd_llg_magnetic_box_static(None, 8, 8, 8, fake, None) == B.EINVAL
    assert L.fdtd_llg_magnetic_box_static(fake, 8, 8, 8, None, None) == B.EINVAL
    assert L.fdtd_llg_magnetic_box_static(fake, 0, 8, 8, fake, None) == B.EINVAL
    assert L.fdtd_llg_magnetic_box_static(fake, 8, -1, 8, fake, None) == B.EINVAL
    # the header's figures are the binding's
    hdr = (B._HERE.parent / "include" / "fdtd_llg.h").read_text()
    assert "#define FDTD_LLG_STATIC_MAX_CELLS (1LL << 29)" in hdr
    assert "#define FDTD_LLG_STATIC_SCRATCH_BYTES ((1 << 20) + 256)" in hdr
    assert B.STATIC_SCRATCH_BYTES == (1 << 20) + 256
