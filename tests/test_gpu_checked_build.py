"""The checked build on the GPU (sanitizers; compute-sanitizer is closed on this pool, see
profiles/r02_sanitizers.md): the library compiled with -DMOP_CHECK -- device-side bounds assertions on every index that
is derived from list data -- under its own file name, taken through the tour of tests/sanitizer_target.py in a process of
its own, so that the product library and this pytest process are not touched.  A fired assertion traps the kernel and the
tour exits non-zero."""
import os
import subprocess
import sys

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.mark.gpu
def test_checked_build_runs_the_tour_without_an_assertion():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device: the library has no CPU fallback")
    from paper_2501_11962_b200 import build
    before = os.path.getmtime(build.build())
    r = subprocess.run([sys.executable, os.path.join(ROOT, "tests", "sanitizer_target.py"), "--checked"], capture_output=True,
                       text=True, timeout=1500, cwd=ROOT)
    assert r.returncode == 0, (r.stdout[-1500:], r.stderr[-3000:])
    assert "checked build (-DMOP_CHECK): no assertion fired" in r.stdout
    assert os.path.exists(build.CHECKED_LIB) and os.path.getmtime(build.LIB) == before    # the product was not rebuilt
