"""CPU-side checks of the boundary: the C-ABI library loads here (no GPU) and exports every symbol
``include/*.h`` declares; the argument validation that needs no device answers with error codes."""
import ctypes as C
import re
from pathlib import Path

import pytest

ROOT = Path(__file__).resolve().parent.parent


@pytest.fixture(scope="module")
def B():
    from paper_2103_12819_b200 import binding
    if not binding.LIB_PATH.exists():
        binding.build_library()
    return binding


def _declared_symbols():
    names = set()
    for h in (ROOT / "include").glob("*.h"):
        txt = re.sub(r"/\*.*?\*/", "", h.read_text(), flags=re.S)
        names |= set(re.findall(r"\b(fdtd_llg_[a-z_]+)\s*\(", txt))
    return names


def test_library_exports_every_declared_symbol(B):
    declared = _declared_symbols()
    assert declared == set(B.EXPORTS)          # the binding knows them all, and nothing else
    L = C.CDLL(str(B.LIB_PATH))
    for name in declared:
        assert hasattr(L, name), name


def test_header_structs_match_binding(B):
    """Field names of the ctypes mirrors follow the header, in order."""
    txt = (ROOT / "include" / "fdtd_llg.h").read_text()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    for cname, mirror in (("fdtd_llg_options", B.Options), ("fdtd_llg_stats", B.Stats),
                          ("fdtd_llg_slab_info", B.SlabInfo)):
        body = re.search(r"typedef struct \{([^{}]*)\} %s;" % cname, txt).group(1)
        fields = re.findall(r"\b([a-z_][a-z_0-9]*)(?:\[\d\])?\s*;", body)
        assert fields == [f for f, _ in mirror._fields_], cname


def test_struct_layout_as_the_c_compiler_sees_it(B, tmp_path):
    """A C translation unit includes the header and prints sizeof / offsetof; the ctypes mirrors
    must agree byte for byte (a mismatch would otherwise only show as wrong numbers on the GPU)."""
    import subprocess
    exe = tmp_path / "abi_layout"
    subprocess.run(["gcc", "-std=c99", "-Wall", "-Werror", "-I", str(ROOT / "include"),
                    str(ROOT / "tests" / "abi_layout.c"), "-o", str(exe)], check=True)
    out = subprocess.run([str(exe)], check=True, capture_output=True, text=True).stdout
    mirrors = {"fdtd_llg_options": B.Options, "fdtd_llg_stats": B.Stats, "fdtd_llg_slab_info": B.SlabInfo}
    seen = {k: set() for k in mirrors}
    for line in out.splitlines():
        t = line.split()
        if t[0] == "sizeof":
            assert C.sizeof(mirrors[t[1]]) == int(t[2]), line
        elif t[0] == "offsetof":
            assert getattr(mirrors[t[1]], t[2]).offset == int(t[3]), line
            seen[t[1]].add(t[2])
        elif t[:2] == ["enum", "SUB"]:
            assert [int(v) for v in t[2:]] == [B.SUB_BEGIN, B.SUB_HM1, B.SUB_HM1_END, B.SUB_E, B.SUB_HM2, B.SUB_HM2_END]
        elif t[:2] == ["enum", "K_NCLASS"]:
            assert int(t[2]) == len(B.KERNEL_CLASSES)
    for name, m in mirrors.items():
        assert seen[name] == {f for f, _ in m._fields_}, name      # every field was checked


def test_defaults_and_workspace_budget(B):
    o = B.fdtd_llg_default_options()
    assert list(o.bc) == [0, 0, 0] and o.enable_llg == 1 and o.llg_max_iter == 20
    assert o.llg_tol == 1e-6 and o.use_graph == 1 and list(o.ani_axis) == [0.0, 0.0, 1.0]
    # device layout: one ghost layer, rows padded to 128-byte alignment (kernels.cuh)
    n = ((16 + 64 + 1 + 15) // 16 * 16) * (48 + 2) * (40 + 2)
    full = B.fdtd_llg_workspace_bytes(64, 48, 40, o, 0)
    assert 33 * n * 8 <= full < 33 * n * 8 + (4 << 20)       # E 2x3 + H 3x3 + M 2x9
    assert B.fdtd_llg_workspace_bytes(64, 48, 40, o, 8 | 1) - full == n * 8 * 2
    o.enable_llg = 0
    assert B.fdtd_llg_workspace_bytes(64, 48, 40, o, 0) < 12 * n * 8 + (4 << 20)  # E 2x3 + H 2x3
    assert B.fdtd_llg_workspace_bytes(0, 48, 40, o, 0) == 0
    # config 5 (768^3, Ms array) fits a 180 GB B200 with room for the inputs
    o.enable_llg = 1
    assert B.fdtd_llg_workspace_bytes(768, 768, 768, o, 8) < 130e9


def test_create_validates_before_touching_the_device(B):
    L = B.lib()
    o = B.fdtd_llg_default_options()
    h = C.c_void_p()

    def create(nx=8, ny=8, nz=8, dx=1e-6, dt=1e-15, ws=256, nbytes=1 << 40, opt=o, space=0):
        return L.fdtd_llg_create(C.byref(h), nx, ny, nz, dx, dx, dx, dt, None, None, None, None,
                                 None, None, space, C.byref(opt), ws, nbytes, None)

    assert create(nx=0) == B.EINVAL and "nx" in B.fdtd_llg_last_error(None)
    assert create(dx=-1.0) == B.EINVAL
    assert create(dt=float("nan")) == B.EINVAL and "dt" in B.fdtd_llg_last_error(None)
    assert create(ws=None) == B.EINVAL
    assert create(ws=8) == B.EINVAL and "aligned" in B.fdtd_llg_last_error(None)
    assert create(nbytes=1024) == B.ENOMEM and "workspace" in B.fdtd_llg_last_error(None)
    assert create(space=7) == B.EINVAL
    bad = B.fdtd_llg_default_options()
    bad.llg_tol = 0.0
    assert create(opt=bad) == B.EINVAL and "tol" in B.fdtd_llg_last_error(None)
    bad = B.fdtd_llg_default_options()
    bad.bc[1] = 3
    assert create(opt=bad) == B.EINVAL
    bad = B.fdtd_llg_default_options()
    bad.ani_hk, bad.ani_axis[2] = 1e3, 0.5
    assert create(opt=bad) == B.EINVAL and "unit" in B.fdtd_llg_last_error(None)
    assert h.value is None
    # NULL handles are rejected, never dereferenced
    assert L.fdtd_llg_step(None, 1) == B.EINVAL
    assert L.fdtd_llg_get_stats(None, None) == B.EINVAL
    L.fdtd_llg_destroy(None)


def test_missing_library_fails_loudly(B, monkeypatch, tmp_path):
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "LIB_PATH", tmp_path / "nope.so")
    with pytest.raises(RuntimeError, match="no CPU or PyTorch fallback"):
        B.lib()


def test_product_path_never_touches_the_oracle():
    """The package must not import, read or run anything under oracle/ (and vice versa)."""
    pat = re.compile(r"(^|\s)(import|from)\s+oracle\b|liboracle|oracle_create|oracle/|#include\s+.*oracle", re.M)
    for p in (ROOT / "paper_2103_12819_b200").rglob("*"):
        if p.suffix in (".py", ".cu", ".cuh", ".h", ".sh"):
            assert not pat.search(p.read_text()), p
    for p in (ROOT / "oracle").glob("*"):
        if p.suffix in (".py", ".c", ".h"):
            txt = p.read_text()
            assert "import paper_2103_12819_b200" not in txt and "from paper_2103_12819_b200" not in txt
            assert "csrc" not in txt.replace("paper_2103_12819_b200/csrc/", "")
