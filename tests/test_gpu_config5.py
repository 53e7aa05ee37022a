"""GPU parity on the 150,000-atom membrane-protein-shaped system (BASELINE.json configs[3] and the bead-count sweep
configs[4]: N = 1, 4, 8, 16, 64, 128), in the launch configuration bench.py times.  All tests need a B200 (-m gpu).

One 16-bead Brownian path over the system is generated once with the ORACLE's force (never the CUDA path's) and
shared by all tests of this module: the recursion is sequential, so its first N beads are the N-bead path of the same
seed.  For N = 64 and 128 the recursion itself would cost 8 and 16 minutes of oracle time, so those paths walk the 16
beads back and forth (1..16, 15..1, 2..16, ...): every consecutive pair of beads is still one Brownian step apart
(taken forwards or backwards), the path is image-consistent, and any path is a valid argument of eq. (3).  At those
sizes the oracle checks sampled beads one by one -- eqs (5)-(7) are local: G^n depends on beads n-1, n, n+1 only, so
the oracle's gradient of the 3-bead sub-path (R^{n-1}, R^n, R^{n+1}) on its middle bead IS G^n of the long path -- and
V_eff by a full, unsampled oracle evaluation at N = 64; at N = 128 V_eff is checked through the additivity of eq. (3)
over consecutive bead pairs, each pair's term coming from the oracle (a full evaluation would take several minutes).
"""
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

from paper_2501_11962_b200 import workloads as W
from tests import helpers as H

pytestmark = pytest.mark.gpu

TOL_V = 1e-6
TOL_RMS = 1e-4


@pytest.fixture(scope="module")
def B():
    import torch
    if not torch.cuda.is_available():
        pytest.fail("gpu tests need a CUDA device: the library has no CPU fallback")
    from paper_2501_11962_b200 import binding
    binding.load()
    return binding


@pytest.fixture(scope="module")
def big(oracle):
    s = W.config4(seed=0, n_beads=16)
    o = oracle.OracleSystem(s)
    R16 = W.brownian_path(s, 16, lambda X: oracle.bead(o, X, geom=0)["F"], seed=0)
    return s, o, R16


def zigzag(R16, N):
    """Bead indices 0..15, 14..0, 1..15, ... (N of them) into the 16-bead path."""
    period = list(range(16)) + list(range(14, 0, -1))
    idx = [period[k % len(period)] for k in range(N)]
    return np.ascontiguousarray(R16[idx]), idx


def momentum_ok(arr):
    a = arr.astype(np.float64)
    return np.abs(a.sum(1)).max() <= 1e-4 * np.abs(a).sum(1).max()


def test_config4_full_size_bench_configuration(B, oracle, big):
    """BASELINE.json configs[3] at full size (150,000 atoms, N = 8: the workload and launch configuration bench.py
    times).  V_eff and the whole gradient against the oracle; the in-range pair COUNT of every force bead -- from the
    pair walker and from the production kernel's own decisions --, the pair SET restricted to a sample of atoms,
    bit-exact; momentum conservation (P6) on the GPU's F and H.eta at this size."""
    s, o, R16 = big
    R = R16[:8]
    m = B.Mop(s, 8)
    v, g = m.mop_eval_veff_grad(R)
    v_ref, g_ref, parts = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=False, want_parts=True)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    H.assert_close(g.cpu().numpy(), g_ref, TOL_RMS)
    F, Heta = m.mop_debug_get("F"), m.mop_debug_get("Heta")
    H.assert_close(F, parts["F"], TOL_RMS)
    H.assert_close(m.mop_debug_get("eta"), parts["eta"], TOL_RMS)
    H.assert_close(Heta, parts["Heta"], TOL_RMS)
    assert momentum_ok(F) and momentum_ok(Heta)
    ref = oracle.pairs(o, R[0].astype(np.float64), geom=1, brute=False)
    got, cnt = m.mop_debug_pairs(0)
    assert cnt == len(ref), "pair count differs on bead 0: %d vs %d" % (cnt, len(ref))
    pick = lambda P: P[(P[:, 0] % 97 == 0) | (P[:, 1] % 97 == 0)]
    assert np.array_equal(pick(got), pick(ref)), "sampled pair set differs on bead 0"
    with ThreadPoolExecutor(6) as ex:
        n_ref = list(ex.map(lambda n: oracle.bead(o, R[n].astype(np.float64), geom=1, want_force=False)["npairs"], range(1, 7)))
    n_ref = [len(ref)] + n_ref
    assert sum(n_ref) == parts["npairs"]
    for n in range(1, m.nf):
        assert m.mop_debug_pairs(n, cap=0)[1] == n_ref[n], "pair count differs on bead %d" % n
    assert m.mop_debug_pair_hash(0) == (n_ref[0], H.pair_set_fingerprint([(0, ref)], s.n_atoms))   # the production kernel's own pair SET
    assert m.mop_debug_count_inrange(1) == sum(n_ref[1:])
    m.close()


@pytest.mark.parametrize("N", [1, 4, 16])
def test_config5_sweep_full_parity(B, oracle, big, N):
    """BASELINE.json configs[4], N = 1, 4, 16: V_eff and the whole gradient against a full oracle evaluation."""
    s, o, R16 = big
    R = R16[:N]
    m = B.Mop(s, N)
    v, g = m.mop_eval_veff_grad(R)
    v_ref, g_ref, parts = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=False, want_parts=True)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    H.assert_close(g.cpu().numpy(), g_ref, TOL_RMS)
    H.assert_close(m.mop_debug_get("F"), parts["F"], TOL_RMS)
    if N > 1:
        H.assert_close(m.mop_debug_get("Heta"), parts["Heta"], TOL_RMS)
    assert m.mop_debug_count_inrange(2) == parts["npairs"]
    m.close()


@pytest.mark.parametrize("N", [64, 128])
def test_config5_sweep_sampled_beads(B, oracle, big, N):
    """BASELINE.json configs[4], N = 64, 128 (zig-zag path, see the module docstring): F, eta, H.eta and the gradient
    of the first bead, two interior beads and the last bead against the oracle's sub-path evaluations; momentum
    conservation of every bead's F and H.eta; the production kernel's in-range count; V_eff (see docstring)."""
    s, o, R16 = big
    R, idx = zigzag(R16, N)
    m = B.Mop(s, N)
    v, g = m.mop_eval_veff_grad(R)
    g = g.cpu().numpy()
    F, eta, Heta = m.mop_debug_get("F"), m.mop_debug_get("eta"), m.mop_debug_get("Heta")
    assert momentum_ok(F) and momentum_ok(Heta)
    Rd = R.astype(np.float64)

    def sub(lo, hi):
        return oracle.veff_grad(o, Rd[lo:hi], geom=1, brute=False, want_parts=True)

    interior = [N // 3, (2 * N) // 3 + 1]
    jobs = [(0, 2)] + [(n - 1, n + 2) for n in interior] + [(N - 2, N)]
    with ThreadPoolExecutor(len(jobs)) as ex:
        res = list(ex.map(lambda j: sub(*j), jobs))
    # first bead: G^1 and F, eta, H.eta of force bead 0
    _, g_ref, p = res[0]
    H.assert_close(g[0], g_ref[0], TOL_RMS)
    H.assert_close(F[0], p["F"][0], TOL_RMS)
    H.assert_close(eta[0], p["eta"][0], TOL_RMS)
    H.assert_close(Heta[0], p["Heta"][0], TOL_RMS)
    for n, (_, g_ref, p) in zip(interior, res[1:3]):
        H.assert_close(g[n], g_ref[1], TOL_RMS)
        H.assert_close(F[n], p["F"][1], TOL_RMS)
        H.assert_close(eta[n], p["eta"][1], TOL_RMS)
        H.assert_close(Heta[n], p["Heta"][1], TOL_RMS)
    # last bead: G^N = K eta^{N-1}, and the last force bead
    _, g_ref, p = res[3]
    H.assert_close(g[N - 1], g_ref[1], TOL_RMS)
    H.assert_close(F[N - 2], p["F"][0], TOL_RMS)
    H.assert_close(Heta[N - 2], p["Heta"][0], TOL_RMS)
    if N == 64:
        v_ref, g_full, parts = oracle.veff_grad(o, Rd, geom=1, brute=False, want_parts=True)
        assert abs(v - v_ref) <= TOL_V * abs(v_ref)
        H.assert_close(g, g_full, TOL_RMS)
        assert m.mop_debug_count_inrange(2) == parts["npairs"]
    else:
        # eq. (3) is a sum over consecutive bead pairs: V_eff = U(R^1) + sum_n E_spring(R^n, R^{n+1}); the zig-zag path
        # holds 30 distinct ordered pairs (15 forwards, 15 backwards), each term from a 2-bead oracle evaluation
        pairs = sorted({(idx[n], idx[n + 1]) for n in range(N - 1)})
        with ThreadPoolExecutor(16) as ex:
            terms = list(ex.map(lambda ab: oracle.veff_grad(o, R16[[ab[0], ab[1]]].astype(np.float64), geom=1, brute=False,
                                                            want_parts=True)[2], pairs))
        e_spring = dict(zip(pairs, [t["E_spring"] for t in terms]))
        npairs = dict(zip(pairs, [t["npairs"] for t in terms]))
        v_ref = res[0][2]["U1"] + sum(e_spring[(idx[n], idx[n + 1])] for n in range(N - 1))
        assert abs(v - v_ref) <= TOL_V * abs(v_ref)
        assert m.mop_debug_count_inrange(2) == sum(npairs[(idx[n], idx[n + 1])] for n in range(N - 1))
    m.close()


def test_config4_bead_blocks_reproduce_the_whole_path(B, oracle, big):
    """NEXT-4 on the bench workload: beads [0,4) and [4,8) in two contexts on this one GPU against the whole-path
    evaluation (V_eff 1e-8, gradient 1e-6 RMS)."""
    from tests.test_gpu_blocks import run_blocks
    s, o, R16 = big
    R = np.ascontiguousarray(R16[:8])
    m = B.Mop(s, 8)
    v0, g0 = m.mop_eval_veff_grad(R)
    g0 = g0.cpu().numpy()
    m.close()
    v, g = run_blocks(B, s, R, [(0, 4), (4, 4)])
    assert abs(v - v0) <= 1e-8 * abs(v0)
    assert H.rms_rel(g, g0) <= 1e-6
