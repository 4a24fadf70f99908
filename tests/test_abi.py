"""not gpu: the C-ABI library builds, loads and exports every symbol include/psdns.h declares."""
import os
import re

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def test_library_exports_every_declared_symbol():
    from paper_2406_01322_b200 import build as B
    B.build()
    import paper_2406_01322_b200 as P
    hdr = open(os.path.join(ROOT, "include", "psdns.h")).read()
    declared = set(re.findall(r"\b(psdns_[a-z_]+)\s*\(", hdr))
    assert {"psdns_init", "psdns_set_state", "psdns_step", "psdns_get_state",
            "psdns_transform_roundtrip", "psdns_workspace_bytes", "psdns_destroy"} <= declared
    sym = P.exported_symbols()
    for name in declared:
        assert sym.get(name, False) or hasattr(P.load_library(), name), name


def test_workspace_bytes_host_logic():
    import ctypes as C
    from paper_2406_01322_b200.binding import load_library, psdns_grid, psdns_params
    lib = load_library()
    p = psdns_params(3000, 40, .025, 1, 2e-5, 0, 1.0, 1, 1)
    sizes = [lib.psdns_workspace_bytes(C.byref(psdns_grid(*n, 12.566, 6.283)), C.byref(p))
             for n in [(32, 32, 33), (128, 128, 129), (1024, 512, 513)]]
    assert 0 < sizes[0] < sizes[1] < sizes[2] < 180 * 2 ** 30
    for bad in [(24, 32, 33), (32, 32, 34), (2048, 32, 33), (32, 32, 5)]:
        assert lib.psdns_workspace_bytes(C.byref(psdns_grid(*bad, 1.0, 1.0)), C.byref(p)) == 0
    pbad = psdns_params(3000, 40, .025, 1, -1.0, 0, 1.0, 1, 1)
    assert lib.psdns_workspace_bytes(C.byref(psdns_grid(32, 32, 33, 1.0, 1.0)), C.byref(pbad)) == 0


def test_no_oracle_import_in_product():
    pkg = os.path.join(ROOT, "paper_2406_01322_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dirpath, f)).read()
                assert "psdns_oracle" not in txt and "isosurface_oracle" not in txt and "import oracle" not in txt, f
    orc = open(os.path.join(ROOT, "oracle", "psdns_oracle.py")).read()
    assert "paper_2406_01322_b200" not in orc.replace("`paper_2406_01322_b200`", "")
