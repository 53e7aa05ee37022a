"""Host-side checks that need no GPU: the C-ABI library builds, loads and exports every symbol that
include/mop.h declares; creation fails loudly without a device (no CPU fallback)."""
import ctypes as C
import os
import re

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


def _declared():
    txt = open(os.path.join(ROOT, "include", "mop.h")).read()
    txt = re.sub(r"/\*.*?\*/", "", txt, flags=re.S)
    return sorted(set(re.findall(r"\b(mop_[a-z0-9_]+)\s*\(", txt)))


def test_header_declares_the_north_star_entry_points():
    names = _declared()
    for n in ("mop_create", "mop_set_topology", "mop_eval_veff_grad", "mop_step", "mop_destroy"):
        assert n in names


def test_library_builds_loads_and_exports_every_declared_symbol():
    from paper_2501_11962_b200 import binding
    L = binding.load()
    for n in _declared():
        assert hasattr(L, n), "libmop_b200.so does not export %s" % n
    assert sorted(binding.EXPORTS) == _declared()


def test_struct_layouts_match_the_header():
    """ctypes mirrors of mop_params / mop_topology have the C layout (sizes on LP64)."""
    from paper_2501_11962_b200 import binding
    assert C.sizeof(binding.mop_params) == 72
    assert C.sizeof(binding.mop_topology) == 112


def test_no_cpu_fallback():
    """Without a CUDA device creating a context must fail (status MOP_ERR_CUDA), not fall back."""
    import torch
    if torch.cuda.is_available():
        pytest.skip("a GPU is present")
    from paper_2501_11962_b200 import binding, workloads
    with pytest.raises(RuntimeError):
        binding.Mop(workloads.config1(n_beads=2), 2)
    L = binding.load()
    p = binding.mop_params()
    p.n_atoms, p.n_beads = 8, 2
    p.box[0] = p.box[1] = p.box[2] = 3.0
    p.r_cut, p.dt_path, p.nu = 1.0, 0.002, 50.0
    ctx = C.c_void_p()
    assert L.mop_create(C.byref(ctx), C.byref(p)) == 5
    assert b"no CPU fallback" in L.mop_last_error(None)
    L.mop_destroy(None)  # NULL-safe


def test_product_never_imports_the_oracle():
    """The package (binding, build, workloads, csrc) must not reference oracle/."""
    pkg = os.path.join(ROOT, "paper_2501_11962_b200")
    for dp, _, files in os.walk(pkg):
        for f in files:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                txt = open(os.path.join(dp, f)).read()
                assert "import oracle" not in txt and "from oracle" not in txt and "mop_oracle" not in txt, f
