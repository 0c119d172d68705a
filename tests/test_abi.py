"""CPU-only checks of the C-ABI boundary: the library builds, loads, exports every symbol that
include/md_b200.h declares, and its host-side argument validation works without a GPU."""
import ctypes as C
import re
from pathlib import Path

import numpy as np
import pytest

import workloads as W

ROOT = Path(__file__).resolve().parent.parent
HEADER = ROOT / "include" / "md_b200.h"


@pytest.fixture(scope="module")
def lib():
    from paper_1401_4350_b200.build import build
    build()
    from paper_1401_4350_b200 import load_library
    return load_library()


def declared_symbols():
    text = re.sub(r"/\*.*?\*/", "", HEADER.read_text(), flags=re.S)
    return sorted(set(re.findall(r"\b(md_[a-z_]+)\s*\(", text)))


def test_header_symbols_exported(lib):
    from paper_1401_4350_b200 import EXPORTED_SYMBOLS
    decl = declared_symbols()
    assert len(decl) >= 15
    assert sorted(EXPORTED_SYMBOLS) == decl          # the binding wraps exactly what the header declares
    for name in decl:
        assert hasattr(lib, name), name


def test_no_torch_types_in_header():
    text = HEADER.read_text()
    sigs = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    assert "at::" not in sigs and "Tensor" not in sigs and "std::" not in sigs
    assert 'extern "C"' in sigs


def _ws(lib, N, box, rcut, skin, pot, max_neigh, f32_box=True):
    from paper_1401_4350_b200.binding import make_potential
    p = make_potential(pot)
    b = np.ascontiguousarray(box, dtype=np.float64)
    if f32_box:
        b = b.astype(np.float32).astype(np.float64)      # S:Q7: boxes exactly representable in fp32
    n = C.c_size_t(0)
    rc = lib.md_workspace_bytes(N, b.ctypes.data_as(C.POINTER(C.c_double)), rcut, skin, C.byref(p), max_neigh, C.byref(n))
    return rc, n.value


def test_workspace_bytes_and_validation(lib):
    pot = W.lj_potential(2.5)
    rc, n1 = _ws(lib, 2048, [13.68] * 3, 2.5, 0.3, pot, 116)
    assert rc == 0 and n1 > 2048 * 116 * 4
    rc, n2 = _ws(lib, 4096, [13.68, 13.68, 27.36], 2.5, 0.3, pot, 116)
    assert rc == 0 and n2 > n1
    assert _ws(lib, 0, [13.68] * 3, 2.5, 0.3, pot, 116)[0] == -1            # N <= 0
    assert _ws(lib, 2048, [5.0] * 3, 2.5, 0.3, pot, 116)[0] == -1           # box < 2 (rcut + 2 skin)
    assert _ws(lib, 2048, [13.68] * 3, -1.0, 0.3, pot, 116)[0] == -1
    assert _ws(lib, 2 ** 22, [200.0] * 3, 2.5, 0.3, pot, 1024)[0] == -1     # N * max_neigh >= 2^31
    assert _ws(lib, 2048, [13.68] * 3, 2.5, 0.3, pot, 480)[0] == 0
    assert _ws(lib, 2048, [13.68] * 3, 2.5, 0.3, pot, 481)[0] == -1          # max_neigh > 480 (md_b200.h)
    # a box that fp32 cannot hold would give the fp32 minimum image and the fp64 predicates different boxes
    assert _ws(lib, 2048, [13.68] * 3, 2.5, 0.3, pot, 116, f32_box=False)[0] == -1
    assert _ws(lib, 2048, [13.5, 14.25, 16.0], 2.5, 0.3, pot, 116, f32_box=False)[0] == 0
    bad = dict(W.patchy_potential())
    bad["patch_dir"] = bad["patch_dir"] * 1.1                               # non-unit patch vectors
    assert _ws(lib, 2048, [20.0] * 3, 1.5, 0.3, bad, 40)[0] == -1
    rc, n3 = _ws(lib, 2048, [20.0] * 3, 1.5, 0.3, W.patchy_potential(), 40)
    assert rc == 0 and n3 > 0


def test_create_rejects_bad_workspace_without_gpu(lib):
    from paper_1401_4350_b200.binding import make_potential
    p = make_potential(W.lj_potential(2.5))
    b = np.array([13.68] * 3).astype(np.float32).astype(np.float64)
    h = C.c_void_p(None)
    rc = lib.md_create(C.byref(h), 2048, b.ctypes.data_as(C.POINTER(C.c_double)), 2.5, 0.3, C.byref(p), 116,
                       None, 0, None)
    assert rc == -1 and not h.value
    assert lib.md_forces(None, 0, 0) == -1
    assert lib.md_launch_count(None) == 0
    assert lib.md_last_error(None) == b"null handle"


def test_product_does_not_import_oracle():
    """The product path never touches oracle/ (and vice versa)."""
    pkg = ROOT / "paper_1401_4350_b200"
    for f in list(pkg.rglob("*.py")) + list(pkg.rglob("*.cu")) + list(pkg.rglob("*.cuh")) + [HEADER]:
        t = f.read_text()
        assert "import oracle" not in t and "from oracle" not in t and "md_oracle" not in t, f
    for f in (ROOT / "oracle").glob("*"):
        if f.suffix in (".py", ".c"):
            t = f.read_text()
            assert "md_b200" not in t and "import paper_1401_4350_b200" not in t, f


def test_missing_library_fails_loudly(monkeypatch, tmp_path):
    import paper_1401_4350_b200.binding as B
    monkeypatch.setattr(B, "_lib", None)
    monkeypatch.setattr(B, "_LIB_PATH", tmp_path / "nope.so")
    with pytest.raises(ImportError):
        B.load_library()
