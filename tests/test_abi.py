"""CPU-only checks of the boundary: the C-ABI library builds for sm_100a, loads,
exports every symbol include/md.h declares, and its host-side argument checks
return the documented error codes (no kernel is launched here)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def B():
    from paper_1912_04232_b200 import build
    build.build()
    from paper_1912_04232_b200 import binding
    binding.lib()
    return binding


def declared_symbols():
    text = open(os.path.join(ROOT, "include", "md.h")).read()
    text = re.sub(r"/\*.*?\*/", "", text, flags=re.S)
    return sorted(set(re.findall(r"\b(md_[a-z_0-9]+)\s*\(", text)))


def test_library_exports_every_declared_symbol(B):
    names = declared_symbols()
    assert {"md_cell_list_build", "md_neighbor_list_build", "md_needs_rebuild",
            "md_pair_energy_force", "md_nve_step"} <= set(names)       # north_star's five calls
    L = B.lib()
    for name in names:
        assert hasattr(L, name), name
    assert sorted(B.SYMBOLS) == names


def test_no_torch_types_in_the_abi():
    text = open(os.path.join(ROOT, "include", "md.h")).read()
    assert "torch" not in text and "at::" not in text and "#include <cuda" not in text


def test_workspace_bytes_and_config_errors(B):
    cfg = B.make_config(3, [10.0775776] * 3, 2.5, 0.3, 128)
    b = B.md_workspace_bytes(cfg, 864)
    assert b > 864 * (16 * 3 + 4 * 5) and b % 256 == 0
    assert B.md_workspace_bytes(cfg, 256000) > b

    def code(cfg, n=864):
        with pytest.raises(B.MdError) as e:
            B.md_workspace_bytes(cfg, n)
        assert B.md_last_error() != ""
        return e.value.code

    assert code(cfg, 0) == B.MD_EINVAL
    assert code(B.make_config(4, [10.0] * 3, 2.5, 0.3, 128)) == B.MD_EINVAL
    assert code(B.make_config(3, [10.0] * 3, 2.5, 0.3, 0)) == B.MD_EINVAL
    assert code(B.make_config(3, [10.0] * 3, 2.5, 0.3, 126)) == B.MD_EINVAL
    assert code(B.make_config(3, [10.0] * 3, -1.0, 0.3, 128)) == B.MD_EINVAL
    assert code(B.make_config(3, [10.0] * 3, 2.5, -0.1, 128)) == B.MD_EINVAL
    # fewer than 3 cells per side: 8.0 / 2.8 = 2.86
    assert code(B.make_config(3, [8.0, 10.0, 10.0], 2.5, 0.3, 128)) == B.MD_EBOX
    # cell side equal to R: margin rule
    assert code(B.make_config(2, [8.4, 8.4], 2.5, 0.3, 128)) == B.MD_EBOX
    # 2-D ignores box[2]
    assert B.md_workspace_bytes(B.make_config(2, [9.0, 9.0, 0.0], 2.5, 0.3, 32), 100) > 0


def test_create_rejects_bad_workspace_before_touching_cuda(B):
    cfg = B.make_config(3, [10.0775776] * 3, 2.5, 0.3, 128)
    h = C.c_void_p(None)
    rc = B.lib().md_create(C.byref(cfg), 864, None, 0, C.byref(h))
    assert rc == B.MD_EWORKSPACE and h.value is None
    rc = B.lib().md_create(C.byref(cfg), 864, 256 + 8, 1 << 30, C.byref(h))   # unaligned
    assert rc == B.MD_EWORKSPACE
    rc = B.lib().md_create(C.byref(cfg), 864, 256, 1024, C.byref(h))          # too small
    assert rc == B.MD_EWORKSPACE
    assert "workspace" in B.md_last_error()
    assert B.lib().md_destroy(None) == B.MD_OK


def test_product_does_not_import_the_oracle():
    """The product path must not route through oracle/ (or any CPU fallback)."""
    pkg = os.path.join(ROOT, "paper_1912_04232_b200")
    for dirpath, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                text = open(os.path.join(dirpath, f)).read()
                assert "md_oracle" not in text, f
                for line in text.splitlines():
                    code = line.strip()
                    if code.startswith(("import ", "from ", "#include")):
                        assert "oracle" not in code, (f, line)
    orc = (open(os.path.join(ROOT, "oracle", "md_oracle.py")).read()
           + open(os.path.join(ROOT, "oracle", "md_oracle.c")).read())
    assert "paper_1912_04232_b200 import" not in orc and "import paper_1912" not in orc
    assert "md_kernels" not in orc and '"md.h"' not in orc
