"""No-GPU checks: the C-ABI library builds for sm_100a, loads, and exports every symbol include/arche.h declares."""
import ctypes
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    src = open(os.path.join(ROOT, "include", "arche.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(arche_[a-z0-9_]+)\s*\(", src)))


def test_library_exports_every_declared_symbol():
    import paper_2606_13283_b200 as pk
    lib = pk.load()
    names = _declared()
    assert len(names) >= 15
    for n in names:
        assert hasattr(lib, n), n
    assert sorted(pk.SYMBOLS) == names


def test_workspace_query_needs_no_gpu():
    import paper_2606_13283_b200 as pk
    lib = pk.load()
    P = pk.Params()
    P.cell[:] = [10.0, 10.0, 10.0]; P.grid[:] = [32, 32, 32]; P.n_ions = 0; P.kT = 0.3; P.n_electrons = 4.0
    n = lib.arche_workspace_bytes(ctypes.byref(P))
    assert n >= 136 * 32 ** 3          # 5 real + 6 complex fields
    P.grid[:] = [30, 32, 32]           # 30 = 2*3*5 is not supported
    assert lib.arche_workspace_bytes(ctypes.byref(P)) == 0


def test_product_does_not_import_oracle():
    for dirpath, _, files in os.walk(os.path.join(ROOT, "paper_2606_13283_b200")):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "import oracle" not in txt and "arche_oracle" not in txt and "liboracle" not in txt, f
