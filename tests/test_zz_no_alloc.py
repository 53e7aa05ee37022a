"""mop_eta_spring_noalloc: the one entry point of the library that allocates no device memory.

It exists for callers that cannot let a library call cudaMalloc: host programs that own all device memory through a pool
of their own and forbid later driver allocations, processes in which something else has already taken almost all of HBM,
and stepping loops that cannot afford the device-wide synchronisation cudaMalloc / cudaFree bring.  Its working memory is
a fixed array inside the library image, shared by all calls on a GPU and never cleared between them, so the things to
check are: (1) it gives what the context path gives (stage S4: eta^n and E_spring) within the bars the other GPU tests
use; (2) a call is not affected by what the previous call left in that array -- hence two calls in a row, the second one
smaller than the first, then the first again; (3) a problem beyond the stated limit is refused with a message, not run.

This file sorts last on purpose (pytest -x stops at the first failure): it must pass after all other tests have used the
library in the same process, and on its own in a fresh process, where its first call is also the first use of the GPU.
"""
import ctypes as C

import numpy as np
import pytest

from paper_2501_11962_b200 import workloads as W

TOL_V = 1e-6      # the V_eff bar of tests/test_gpu_parity.py (relative)
TOL_RMS = 1e-4    # the RMS bar for force-like arrays there (G14)


def _existing_path(binding, s, R):
    """F, eta (original atom order) and E_spring of the context path for the path R."""
    m = binding.Mop(s, R.shape[0])
    m.mop_eval_veff_grad(R, want_grad=False)
    F, eta, es = m.mop_debug_get("F"), m.mop_debug_get("eta"), m.mop_get_stats()["E_spring"]
    m.close()
    return F, eta, es


@pytest.mark.gpu
def test_no_alloc_entry_point_matches_the_context_path_on_calls_in_a_row():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device: the library has no CPU fallback")
    from paper_2501_11962_b200 import binding
    from tests import helpers as H
    dev = torch.device("cuda", 0)
    s = W.water_box(10, 3.2, seed=5, n_beads=6, name="noalloc_water")    # 3,000 atoms: 59 thread blocks and a ragged tail
    m = binding.Mop(s, 6)
    R = W.brownian_path(s, 6, lambda X: m.mop_force_hvp(X)[0].cpu().numpy().astype(np.float64), seed=1).astype(np.float32)
    m.close()
    cases = [R, R[2:5].copy(), R]                                        # large, small (stale partials beyond it), large again
    ref = {id(c): _existing_path(binding, s, c) for c in cases[:2]}
    ref[id(cases[2])] = ref[id(cases[0])]
    mass = torch.as_tensor(np.asarray(s.mass, np.float32), device=dev)
    energies = []
    for k, Rk in enumerate(cases):
        F_ref, eta_ref, es_ref = ref[id(Rk)]
        N = Rk.shape[0]
        # the caller owns inputs AND outputs; poison the outputs so that an unwritten element shows
        Rd, Fd = torch.as_tensor(Rk, device=dev), torch.as_tensor(F_ref[:N - 1], device=dev)
        eta = torch.full((N - 1, s.n_atoms, 3), float("nan"), dtype=torch.float32, device=dev)
        es = torch.full((1,), float("nan"), dtype=torch.float64, device=dev)
        free_before = torch.cuda.mem_get_info(dev)[0]
        binding.mop_eta_spring_noalloc(Rd, Fd, mass, s.dt_path, s.nu, eta, es)
        torch.cuda.synchronize(dev)
        assert torch.cuda.mem_get_info(dev)[0] >= free_before or k == 0, "device memory shrank during call %d" % k
        H.assert_close(eta.cpu().numpy(), eta_ref[:N - 1], TOL_RMS)
        assert np.array_equal(eta.cpu().numpy(), eta_ref[:N - 1]), "same FP32 operations: eta should agree bit for bit"
        e = float(es.item())
        assert abs(e - es_ref) <= TOL_V * abs(es_ref), (k, e, es_ref)
        energies.append(e)
    assert energies[0] == energies[2], "the sum has a fixed order: equal inputs must give equal bits"
    assert energies[1] != energies[0]


@pytest.mark.gpu
def test_no_alloc_entry_point_refuses_what_its_fixed_array_cannot_hold():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device: the library has no CPU fallback")
    from paper_2501_11962_b200 import binding
    L = binding.load()
    dev = torch.device("cuda", 0)
    small = torch.zeros(64, dtype=torch.float32, device=dev)
    e = torch.zeros(1, dtype=torch.float64, device=dev)
    err = C.create_string_buffer(512)
    p = C.c_void_p(small.data_ptr())
    # one (atom, bead) pair over the limit: refused before anything is launched (the pointers are never followed)
    Q = binding.MOP_NOALLOC_MAX_ATOM_BEADS // 4 + 1
    st = L.mop_eta_spring_noalloc(0, None, Q, 5, 0.002, 50.0, p, p, p, p, C.c_void_p(e.data_ptr()), err, len(err))
    assert st == 1 and b"MOP_NOALLOC_MAX_ATOM_BEADS" in err.value, err.value
    for args in ((4, 1), (0, 2)):                                        # N = 1 has no eta; Q = 0
        st = L.mop_eta_spring_noalloc(0, None, args[0], args[1], 0.002, 50.0, p, p, p, p, C.c_void_p(e.data_ptr()), err, len(err))
        assert st == 1 and err.value
    st = L.mop_eta_spring_noalloc(0, None, 4, 2, 0.002, 50.0, p, None, p, p, C.c_void_p(e.data_ptr()), err, len(err))
    assert st == 1 and b"NULL" in err.value
    torch.cuda.synchronize(dev)
    assert float(e.item()) == 0.0                                        # nothing ran


def test_no_alloc_limit_is_checked_before_any_cuda_call():
    """No GPU needed: the size check comes first, so the refusal (and its message) can be seen on any machine."""
    from paper_2501_11962_b200 import binding
    L = binding.load()
    err = C.create_string_buffer(512)
    dummy = C.c_void_p(256)
    st = L.mop_eta_spring_noalloc(0, None, binding.MOP_NOALLOC_MAX_ATOM_BEADS + 1, 2, 0.002, 50.0, dummy, dummy, dummy, dummy,
                                  dummy, err, len(err))
    assert st == 1 and b"exceeds MOP_NOALLOC_MAX_ATOM_BEADS = 33554432" in err.value, err.value
    hdr = open(__file__.rsplit("/tests/", 1)[0] + "/include/mop.h").read()
    assert "#define MOP_NOALLOC_MAX_ATOM_BEADS %d" % binding.MOP_NOALLOC_MAX_ATOM_BEADS in hdr
