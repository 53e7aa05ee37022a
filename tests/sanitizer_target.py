"""A short tour of the CUDA path for compute-sanitizer: run as

    compute-sanitizer --tool memcheck  python tests/sanitizer_target.py
    compute-sanitizer --tool racecheck python tests/sanitizer_target.py
    python tests/sanitizer_target.py --checked      (where compute-sanitizer is not available: builds the library with
                                                     -DMOP_CHECK, device-side bounds assertions, as libmop_b200_checked.so
                                                     and runs the tour on that; tests/test_gpu_checked_build.py does this)

on a B200 (one tool per gpurun call).  Small systems only -- the sanitizer slows kernels by two orders of magnitude:
__graft_entry__.smoke(), then config 1 (512 LJ atoms, N = 16) through the device and host entry points, mop_step with a
bias and hills, the Langevin thermostat, the finite-difference form, the buffered list, a forced list overflow with
regrow, two bead blocks, and the tiny bonded chain (exclusion rows, bonded kernels on the side stream)."""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)


def main():
    checked = "--checked" in sys.argv
    if checked:   # the library with -DMOP_CHECK: device-side bounds assertions on every index derived from list data,
        # built under its own file name and loaded instead of the product library, which is not touched
        from paper_2501_11962_b200 import binding, build
        binding.load(path=build.build(extra=["-DMOP_CHECK"], out=build.CHECKED_LIB))
    tour()
    print("checked build (-DMOP_CHECK): no assertion fired" if checked else "plain build")


def tour():
    import torch
    import __graft_entry__ as G
    from oracle import oracle as O
    from paper_2501_11962_b200 import binding as B, workloads as W
    from tests import helpers as H
    G.smoke()
    s = W.config1(n_beads=16)
    o = O.OracleSystem(s)
    R = W.brownian_path(s, 16, lambda X: O.bead(o, X, geom=0)["F"], seed=0)
    m = B.Mop(s, 16)
    v, g = m.mop_eval_veff_grad(R)
    v2, g2 = m.mop_eval_veff_grad(R)                          # CUDA-graph replay
    Rh, Gh = torch.as_tensor(R).pin_memory(), torch.empty(R.shape).pin_memory()
    vh = m.mop_eval_veff_grad_host(Rh, Gh)                    # split copies
    assert abs(vh - v) <= 1e-7 * abs(v)
    m.mop_eval_veff_grad_fd(R, 0.01)
    m.mop_debug_pairs(0)
    m.mop_debug_count_inrange(2)
    Rg, Vg = torch.tensor(R, device="cuda"), torch.zeros(R.shape, device="cuda")
    m.mop_set_bias(np.arange(0, 40), np.arange(200, 260), 0.01, 1.0, pace=2)
    m.mop_step(Rg, Vg, 0.0005, 4)
    m.mop_step_continue(Rg, Vg, 0.0005, 2)
    m.mop_step_langevin(Rg, Vg, 0.0005, 3, 250.0, 120.0, seed=3)
    m.mop_get_bias()
    m.mop_set_bias([], [], 1.0, 0.0)
    st = m.mop_get_stats()
    m.mop_debug_set_list_capacity(entries=max(64, int(st["entries"] // 3)))
    try:
        m.mop_eval_veff_grad(R)
        raise SystemExit("expected MOP_ERR_OOM")
    except B.MopError as e:
        assert e.status == 4
    m.mop_eval_veff_grad(R)
    m.close()
    mb = B.Mop(s, 16, r_buf=0.05)
    mb.mop_eval_veff_grad(R)
    mb.mop_eval_veff_grad(R)
    mb.close()
    a, b = B.Mop(s, 8, block=(0, 16)), B.Mop(s, 8, block=(8, 16))
    Rg = torch.tensor(R, device="cuda")
    keta = torch.zeros((s.n_atoms, 3), device="cuda")
    a.mop_block_pass1(Rg[:8], Rg[8].contiguous(), keta)
    b.mop_block_pass1(Rg[8:])
    a.mop_block_pass2(Rg[:8]), b.mop_block_pass2(Rg[8:])
    va, _ = a.mop_block_assemble(None)
    vb, _ = b.mop_block_assemble(keta)
    assert abs(va + vb - v) <= 1e-7 * abs(v)
    a.close(), b.close()
    sc = H.tiny_chain()
    oc = O.OracleSystem(sc)
    Rc = W.brownian_path(sc, 6, lambda X: O.bead(oc, X, geom=0, brute=True)["F"], seed=0)
    mc = B.Mop(sc, 6)
    vc, gc = mc.mop_eval_veff_grad(Rc)
    vr, gr = O.veff_grad(oc, Rc.astype(np.float64), geom=1, brute=True)
    assert abs(vc - vr) <= 1e-6 * abs(vr) and H.rms_rel(gc.cpu().numpy(), gr) <= 1e-4
    mc.close()
    # the membrane-shaped system: scaled-down always, the 150,000-atom bench workload with --big (library forces for its path)
    for sm in [W.small_membrane(n_beads=3)] + ([W.config4(seed=0, n_beads=8)] if "--big" in sys.argv else []):
        m1 = B.Mop(sm, 1)
        Rm = W.brownian_path(sm, sm.n_beads, lambda X: m1.mop_force_hvp(X)[0].double().cpu().numpy(), seed=0)
        m1.close()
        mm = B.Mop(sm, sm.n_beads)
        vm, _ = mm.mop_eval_veff_grad(Rm)
        vm2 = mm.mop_eval_veff_grad_host(torch.as_tensor(Rm).pin_memory(), torch.empty(Rm.shape).pin_memory())
        assert np.isfinite(vm) and abs(vm2 - vm) <= 1e-7 * abs(vm)
        mm.close()
    torch.cuda.synchronize()
    print("sanitizer target finished: V_eff(config 1) = %.6f" % v)


if __name__ == "__main__":
    main()
