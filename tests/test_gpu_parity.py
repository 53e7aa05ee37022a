"""GPU parity: the CUDA path (through the C-ABI binding) against the FP64 oracle, element by element, on the
same seeded inputs.  Bars (BASELINE.json north_star): neighbour sets bit-exact, V_eff relative error <= 1e-6,
RMS relative error (G14) <= 1e-4 for forces and gradient.  All tests here need a B200 (-m gpu).
"""
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


_CACHE = {}


def case(oracle, name):
    """(system, OracleSystem, path R float32 [N][Q][3]) for a named parity case (seeded, cached)."""
    if name in _CACHE:
        return _CACHE[name]
    if name == "c1":
        s = W.config1(n_beads=16)
    elif name == "c2":
        s = W.config2(n_beads=8)          # config 2 at N=8 (the N=64 form runs in test_config2_full)
    elif name == "c2_full":
        s = W.config2(n_beads=64)
    elif name == "chain":
        s = H.tiny_chain()
        s.n_beads = 6
    elif name == "c3":
        s = W.config3(n_beads=3)
    elif name == "c3_full":
        s = W.config3(n_beads=32)         # BASELINE.json configs[2] at its stated bead count
    elif name == "c2_n1":
        s = W.config2(n_beads=1)
    elif name == "chain_n1":
        s = H.tiny_chain()
        s.n_beads = 1
    elif name == "memb":
        s = W.small_membrane(n_beads=3)
    elif name == "lj_n1":
        s = W.config1(n_beads=1)
    elif name == "lj_n2":
        s = W.config1(n_beads=2)
    else:
        raise KeyError(name)
    o = oracle.OracleSystem(s)
    R = W.brownian_path(s, s.n_beads, lambda X: oracle.bead(o, X, geom=0)["F"], seed=0)
    _CACHE[name] = (s, o, R)
    return _CACHE[name]


# --------------------------------------------------------------------------- S0: cell ids + stable sort
@pytest.mark.parametrize("name", ["c1", "c2", "chain", "memb"])
def test_cell_ids_and_stable_sort_bit_exact(B, oracle, name):
    s, o, R = case(oracle, name)
    m = B.Mop(s, s.n_beads)
    m.mop_eval_veff_grad(R, want_grad=False)
    d = m.dims()
    dims = [d["nx"], d["ny"], d["nz"]]
    assert dims == oracle.grid_dims(s.n_atoms, o.box, d["cluster"], d["bin_z"])
    cell = m.mop_debug_get("cell")
    perm = m.mop_debug_get("perm")
    xq = m.mop_debug_get("xq")
    ncell = dims[0] * dims[1] * dims[2]
    for n in range(m.nf):
        xw = oracle.wrap(R[n], o.box)
        c_ref = oracle.cell_ids(xw, o.box, dims)
        assert np.array_equal(cell[n], c_ref), "cell ids differ on bead %d" % n
        p_ref = oracle.stable_sort_by_cell(c_ref, ncell)
        real = perm[n] >= 0
        assert np.array_equal(perm[n][real], p_ref), "stable permutation differs on bead %d" % n
        # sorted coordinates are the wrapped ones, bit for bit; charges ride along
        assert np.array_equal(xq[n][real][:, :3], xw[p_ref])
        assert np.array_equal(xq[n][real][:, 3], np.asarray(s.charge, np.float32)[p_ref])
        # padding only at column ends: inside a column the real slots come first, columns start at multiples of 8
        col = c_ref[p_ref] // dims[2]
        slots = np.flatnonzero(real)
        for cc in np.unique(col)[:50]:
            sl = slots[col == cc]
            assert sl[0] % d["cluster"] == 0 and np.array_equal(sl, np.arange(sl[0], sl[0] + len(sl)))
    m.close()


# --------------------------------------------------------------------------- O1: neighbour sets
@pytest.mark.parametrize("name,brute", [("c1", True), ("c2", True), ("chain", True), ("c3", False), ("memb", False)])
def test_neighbour_sets_bit_exact(B, oracle, name, brute):
    s, o, R = case(oracle, name)
    m = B.Mop(s, s.n_beads)
    m.mop_eval_veff_grad(R, want_grad=False)
    beads = range(m.nf) if s.n_atoms <= 3000 else [0, m.nf - 1]
    for n in beads:
        ref = oracle.pairs(o, R[n].astype(np.float64), geom=1, brute=brute)
        got, cnt = m.mop_debug_pairs(n)
        assert cnt == len(ref), "pair count differs on bead %d: %d vs %d" % (n, cnt, len(ref))
        assert np.array_equal(got, ref), "pair set differs on bead %d" % n
    m.close()


# --------------------------------------------------------------------------- O2/O3: force and H.s of one bead
@pytest.mark.parametrize("name", ["c1", "c2", "chain", "memb"])
def test_force_and_hvp_single_bead(B, oracle, name):
    s, o, R = case(oracle, name)
    rng = np.random.default_rng(5)
    sv = rng.normal(0, 1e-3, (s.n_atoms, 3)).astype(np.float32)
    m = B.Mop(s, 1)
    X = R[min(1, len(R) - 1)]
    F, Hs = m.mop_force_hvp(X, sv)
    ref = oracle.bead(o, X.astype(np.float64), geom=1, brute=s.n_atoms <= 3000, s=sv.astype(np.float64))
    H.assert_close(F.cpu().numpy(), ref["F"], TOL_RMS)
    H.assert_close(Hs.cpu().numpy(), ref["Hs"], TOL_RMS)
    # invariants on the GPU output itself: Newton's third law (P6)
    Fn = F.double().cpu().numpy()
    assert np.abs(Fn.sum(0)).max() <= 1e-5 * np.abs(Fn).sum(0).max()
    m.close()


# --------------------------------------------------------------------------- O4/O5: V_eff and its gradient
@pytest.mark.parametrize("name", ["c1", "c2", "chain", "c3", "memb", "lj_n1", "lj_n2"])
def test_veff_and_gradient(B, oracle, name):
    s, o, R = case(oracle, name)
    m = B.Mop(s, s.n_beads)
    v, g = m.mop_eval_veff_grad(R)
    v_ref, g_ref, parts = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=s.n_atoms <= 3000, want_parts=True)
    st = m.mop_get_stats()
    # per stage, so that a failure localises
    H.assert_close(m.mop_debug_get("F"), parts["F"], TOL_RMS)
    if s.n_beads > 1:
        H.assert_close(m.mop_debug_get("eta"), parts["eta"], TOL_RMS)
        H.assert_close(m.mop_debug_get("Heta"), parts["Heta"], TOL_RMS)
    assert abs(st["U1"] - parts["U1"]) <= TOL_V * max(abs(parts["U1"]), abs(v_ref))
    assert abs(st["E_spring"] - parts["E_spring"]) <= TOL_V * abs(v_ref)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    H.assert_close(g.cpu().numpy(), g_ref, TOL_RMS)
    m.close()


def test_config2_full_64_beads(B, oracle):
    s, o, R = case(oracle, "c2_full")
    m = B.Mop(s, 64)
    v, g = m.mop_eval_veff_grad(R)
    v_ref, g_ref = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=False)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    H.assert_close(g.cpu().numpy(), g_ref, TOL_RMS)
    m.close()


def test_config3_full_32_beads(B, oracle):
    """BASELINE.json configs[2] at its stated size: 23,000 atoms, N = 32 beads."""
    s, o, R = case(oracle, "c3_full")
    m = B.Mop(s, 32)
    v, g = m.mop_eval_veff_grad(R)
    v_ref, g_ref, parts = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=False, want_parts=True)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    H.assert_close(g.cpu().numpy(), g_ref, TOL_RMS)
    H.assert_close(m.mop_debug_get("F"), parts["F"], TOL_RMS)
    H.assert_close(m.mop_debug_get("Heta"), parts["Heta"], TOL_RMS)
    assert m.mop_debug_count_inrange(2) == parts["npairs"]
    m.close()


@pytest.mark.parametrize("name", ["c2_n1", "chain_n1", "lj_n1"])
def test_energy_terms_of_a_single_bead(B, oracle, name):
    """N = 1: V_eff = U(R^1).  Each term of U (LJ, reaction field, bonds, angles) is held to 1e-6 of |U(R^1)| on its
    own, so that no term hides behind a larger one."""
    s, o, R = case(oracle, name)
    m = B.Mop(s, 1)
    v, g = m.mop_eval_veff_grad(R)
    ref = oracle.bead(o, R[0].astype(np.float64), geom=1, brute=True)
    st = m.mop_get_stats()
    u1 = float(ref["U"].sum())
    assert abs(v - u1) <= TOL_V * abs(u1)
    for key, val in zip(("U_lj", "U_coul", "U_bond", "U_angle"), ref["U"]):
        assert abs(st[key] - val) <= TOL_V * abs(u1), (key, st[key], val)
    H.assert_close(g.cpu().numpy()[0], -ref["F"], TOL_RMS)
    m.close()


# --------------------------------------------------------------------------- the production kernel's own decisions
@pytest.mark.parametrize("name", ["c1", "c2", "chain", "memb"])
def test_production_kernel_inrange_count_equals_oracle_pair_count(B, oracle, name):
    """The bit-exact neighbour-set claim for the PRODUCTION force kernel (not the scalar pair walker): its counting
    instance -- the same code plus a population count of its own per-pair decisions (G8 predicate AND exclusion bit) --
    must count exactly the oracle's in-range, non-excluded pairs, bead 1 and the other force beads separately, and its
    fingerprint of the decided pairs (a 64-bit hash of (bead, i, j) summed over them) must equal the fingerprint of the
    oracle's pair lists: the same set, not only the same size."""
    s, o, R = case(oracle, name)
    m = B.Mop(s, s.n_beads)
    m.mop_eval_veff_grad(R, want_grad=False)
    P = [oracle.pairs(o, R[n].astype(np.float64), geom=1, brute=s.n_atoms <= 3000) for n in range(m.nf)]
    n_ref = [len(p) for p in P]
    assert m.mop_debug_count_inrange(0) == n_ref[0]
    assert m.mop_debug_count_inrange(1) == sum(n_ref[1:])
    # ... and the SET: the kernel's order-independent 64-bit fingerprint of (bead, i, j) over its own decisions
    assert m.mop_debug_pair_hash(2) == (sum(n_ref), H.pair_set_fingerprint(list(enumerate(P)), s.n_atoms))
    assert m.mop_debug_pair_hash(0) == (n_ref[0], H.pair_set_fingerprint([(0, P[0])], s.n_atoms))
    m.close()


# --------------------------------------------------------------------------- NEXT-1: the paper's finite-difference form
TOL_FD = 1e-3   # FP32 force rounding (~1e-6 |F|, see BASELINE.md parity rows) enters twice and is divided by 4 eps:
                # sqrt(2) 1e-6 |F|_rms / (4 eps |G|_rms) ~ 4e-5 at eps = 0.01 with |F| ~ |G|; 1e-3 leaves room for the
                # few coordinates whose FP32 displaced position rounds differently from FP64 eta (1 ulp)


@pytest.mark.parametrize("name", ["c1", "c2", "chain", "memb", "lj_n1"])
def test_fd_form_matches_oracle_fd_form(B, oracle, name):
    """mop_eval_veff_grad_fd (eqs 5-7 as printed, three force passes) against the oracle's own FD form at the same
    eps, and -- loosely -- against the analytic form (they differ by O(eps^2) and by pairs crossing r_c, G9)."""
    s, o, R = case(oracle, name)
    eps = 0.01
    m = B.Mop(s, s.n_beads)
    v, g = m.mop_eval_veff_grad_fd(R, eps)
    v_ref, g_ref = oracle.veff_grad_fd(o, R.astype(np.float64), float(np.float32(eps)), geom=1, brute=s.n_atoms <= 3000)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    assert H.rms_rel(g.cpu().numpy(), g_ref) <= TOL_FD
    v2, g2 = m.mop_eval_veff_grad(R)
    assert abs(v - v2) <= 1e-7 * abs(v2)
    assert H.rms_rel(g.cpu().numpy(), g2.cpu().numpy()) <= 5e-2
    m.close()


def test_async_eval_matches_sync_and_repeats(B, oracle):
    """veff_out = NULL leaves the value in the context; repeated evaluations agree to float-atomic noise."""
    s, o, R = case(oracle, "c2")
    m = B.Mop(s, s.n_beads)
    v1, g1 = m.mop_eval_veff_grad(R)
    _, g2 = m.mop_eval_veff_grad(R, sync=False)
    v2 = m.mop_get_stats()["veff"]
    assert abs(v1 - v2) <= 1e-7 * abs(v1)   # float-atomic order noise in F -> eta -> E_spring
    assert H.rms_rel(g2.cpu().numpy(), g1.cpu().numpy()) <= 1e-5
    m.close()


# --------------------------------------------------------------------------- O6: velocity Verlet
@pytest.mark.parametrize("name", ["c1", "chain"])
def test_step_matches_oracle(B, oracle, name):
    import torch
    s, o, R = case(oracle, name)
    rng = np.random.default_rng(11)
    sd = np.sqrt(W.KB * s.temperature / s.mass.astype(np.float64))
    V0 = (rng.normal(0, 1, R.shape) * sd[None, :, None]).astype(np.float32)
    m = B.Mop(s, s.n_beads)
    Rg = torch.tensor(R, device="cuda")
    Vg = torch.tensor(V0, device="cuda")
    nst, dt = 5, 0.001
    m.mop_step(Rg, Vg, dt, nst)
    R_ref, V_ref, en = oracle.step(o, R.astype(np.float64), V0.astype(np.float64), dt, nst, geom=1, brute=True)
    dR_ref = R_ref - R.astype(np.float64)
    dR = Rg.cpu().numpy().astype(np.float64) - R.astype(np.float64)
    # FP32 positions: each update rounds at ulp(R) ~ 2e-7 nm against displacements of ~5e-3 nm
    assert H.rms_rel(dR, dR_ref) <= 2e-3
    assert H.rms_rel(Vg.cpu().numpy(), V_ref) <= 1e-4
    ek = m.mop_get_stats()["E_kin"]
    assert abs(ek - en[-1, 1]) <= 1e-4 * en[-1, 1]
    m.close()


def test_step_continue_equals_one_longer_call(B, oracle):
    """mop_step(n1) + mop_step_continue(n2) (no evaluation at the start of the second call) lands where
    mop_step(n1 + n2) does, up to float-atomic ordering noise; without a held gradient it is refused."""
    import torch
    s, o, R = case(oracle, "chain")
    rng = np.random.default_rng(13)
    sd = np.sqrt(W.KB * s.temperature / s.mass.astype(np.float64))
    V0 = (rng.normal(0, 1, R.shape) * sd[None, :, None]).astype(np.float32)
    out = []
    for split in (False, True):
        m = B.Mop(s, s.n_beads)
        Rg, Vg = torch.tensor(R, device="cuda"), torch.tensor(V0, device="cuda")
        if split:
            with pytest.raises(B.MopError):
                m.mop_step_continue(Rg, Vg, 0.001, 1)
            m.mop_step(Rg, Vg, 0.001, 3)
            l0 = m.mop_get_stats()["launches"]
            m.mop_step_continue(Rg, Vg, 0.001, 4)
            l1 = m.mop_get_stats()["launches"]
        else:
            m.mop_step(Rg, Vg, 0.001, 7)
        out.append((Rg.cpu().numpy(), Vg.cpu().numpy(), m.mop_get_stats()))
        m.close()
    assert H.rms_rel(out[1][0] - R, out[0][0] - R) <= 1e-5
    assert H.rms_rel(out[1][1], out[0][1]) <= 1e-5
    assert abs(out[1][2]["veff"] - out[0][2]["veff"]) <= 1e-6 * abs(out[0][2]["veff"])
    # the continued call ran 4 evaluations, not 5
    m = B.Mop(s, s.n_beads)
    Rg, Vg = torch.tensor(R, device="cuda"), torch.tensor(V0, device="cuda")
    la = m.mop_get_stats()["launches"]
    m.mop_step(Rg, Vg, 0.001, 4)
    lb = m.mop_get_stats()["launches"]
    m.close()
    assert (l1 - l0) < (lb - la)


def test_nve_energy_conservation(B, oracle):
    """Fig. 4a analogue: total energy V_eff + E_kin of the polymer is conserved by mop_step."""
    import torch
    s, o, R = case(oracle, "c1")
    rng = np.random.default_rng(12)
    sd = np.sqrt(W.KB * s.temperature / s.mass.astype(np.float64))
    m = B.Mop(s, s.n_beads)
    Rg = torch.tensor(R, device="cuda")
    Vg = torch.tensor((rng.normal(0, 1, R.shape) * sd[None, :, None]).astype(np.float32), device="cuda")
    tot = []
    for _ in range(6):
        m.mop_step(Rg, Vg, 0.0005, 20)
        st = m.mop_get_stats()
        tot.append(st["veff"] + st["E_kin"])
    ekin = st["E_kin"]
    assert max(tot) - min(tot) <= 2e-3 * ekin
    m.close()


# --------------------------------------------------------------------------- NEXT-2: Langevin thermostat (G19)
def test_thermostat_noise_bits_bit_exact(B, oracle):
    s = W.config1(n_beads=2)
    m = B.Mop(s, 2)
    for seed, step in ((0, 0), (7, 3), (2 ** 63 + 5, 2 ** 40)):
        got = m.mop_debug_noise_bits(seed, step, 4096)
        ref = np.array([oracle.noise_bits(seed, step, i) for i in range(4096)], dtype=np.uint64)
        assert np.array_equal(got, ref)
    m.close()


@pytest.mark.parametrize("name", ["c1", "chain"])
def test_langevin_step_matches_oracle(B, oracle, name):
    import torch
    s, o, R = case(oracle, name)
    rng = np.random.default_rng(21)
    sd = np.sqrt(W.KB * s.temperature / s.mass.astype(np.float64))
    V0 = (rng.normal(0, 1, R.shape) * sd[None, :, None]).astype(np.float32)
    m = B.Mop(s, s.n_beads)
    Rg, Vg = torch.tensor(R, device="cuda"), torch.tensor(V0, device="cuda")
    nst, dt, gamma = 5, 0.001, 250.0          # the paper's damping: 0.25 fs^-1 = 250 ps^-1
    m.mop_step_langevin(Rg, Vg, dt, nst, gamma, s.temperature, seed=9, step0=100)
    R_ref, V_ref, en = oracle.step_langevin(o, R.astype(np.float64), V0.astype(np.float64), dt, nst, gamma,
                                            s.temperature, seed=9, step0=100, geom=1, brute=True)
    dR_ref = R_ref - R.astype(np.float64)
    dR = Rg.cpu().numpy().astype(np.float64) - R.astype(np.float64)
    assert H.rms_rel(dR, dR_ref) <= 2e-3        # FP32 positions, as in test_step_matches_oracle
    assert H.rms_rel(Vg.cpu().numpy(), V_ref) <= 1e-4
    ek = m.mop_get_stats()["E_kin"]
    assert abs(ek - en[-1, 1]) <= 1e-4 * en[-1, 1]
    # gamma = 0 is mop_step
    Ra, Va = torch.tensor(R, device="cuda"), torch.tensor(V0, device="cuda")
    Rb, Vb = torch.tensor(R, device="cuda"), torch.tensor(V0, device="cuda")
    m.mop_step(Ra, Va, dt, 2)
    m.mop_step_langevin(Rb, Vb, dt, 2, 0.0, s.temperature)
    assert H.rms_rel(Vb.cpu().numpy(), Va.cpu().numpy()) <= 1e-5 and H.rms_rel(Rb.cpu().numpy(), Ra.cpu().numpy()) <= 1e-7
    m.close()


def test_nvt_temperature_stays_at_target(B, oracle):
    """Fig. 4b analogue: kinetic temperature of the polymer under the thermostat, from rest."""
    import torch
    s, o, R = case(oracle, "c1")
    m = B.Mop(s, s.n_beads)
    Rg = torch.tensor(R, device="cuda")
    Vg = torch.zeros_like(Rg)
    T, dt, gamma = s.temperature, 0.0005, 100.0
    m.mop_step_langevin(Rg, Vg, dt, 150, gamma, T, seed=1)
    tk, done = [], 150
    for _ in range(12):
        m.mop_step_langevin(Rg, Vg, dt, 25, gamma, T, seed=1, step0=done)
        done += 25
        tk.append(2.0 * m.mop_get_stats()["E_kin"] / (R.size * W.KB))
    assert abs(np.mean(tk) / T - 1.0) < 0.03      # 24,576 degrees of freedom, 12 samples
    m.close()


# --------------------------------------------------------------------------- NEXT-3: the MoP bias on S_e2e
def test_mop_bias_matches_oracle(B, oracle):
    """CV, V(S) and the bias gradient on beads 1 and N against the oracle (same FP32 path, explicit hills)."""
    s, o, R = case(oracle, "chain")
    ga, gb = np.arange(0, 10), np.arange(10, 19)          # the chain against the three waters: both whole
    m = B.Mop(s, s.n_beads)
    v0, g0 = m.mop_eval_veff_grad(R)
    m.mop_set_bias(ga, gb, 0.002, 3.0)
    Rd = R.astype(np.float64)
    _, _, (S_ref, s1_ref, sN_ref) = oracle.bias(o, Rd, ga, gb, [], 0.002, 3.0)
    hills = [S_ref + 0.001, S_ref - 0.003, S_ref + 0.0004]
    for h in hills:
        m.mop_add_hill(h)
    v1, g1 = m.mop_eval_veff_grad(R)
    vb_ref, gb_ref, _ = oracle.bias(o, Rd, ga, gb, hills, 0.002, 3.0)
    st = m.mop_get_bias()
    assert v1 == pytest.approx(v0, rel=1e-7)                                  # veff_out is eq. (3) without V(S)
    assert st["n_hills"] == 3 and np.array_equal(st["hills"], np.asarray(hills))
    assert abs(st["s1"] - s1_ref) <= 1e-12 and abs(st["sN"] - sN_ref) <= 1e-12 and abs(st["S"] - S_ref) <= 1e-12
    assert st["V"] == pytest.approx(vb_ref, rel=1e-10)
    dg = (g1 - g0).cpu().numpy().astype(np.float64)
    # interior beads: untouched by the bias; two evaluations differ by the order of the float atomics only (FP32 rounding of
    # a gradient component, relative to the largest component of that bead block).  Measured on a B200: 200 repeated
    # evaluations of this path, with and without the bias, differ from the first by at most 4.9e-8 max|G|; the bar is 20 x that
    assert np.abs(dg[1:-1]).max() <= 1e-6 * np.abs(g0[1:-1].cpu().numpy()).max()
    scale = np.abs(gb_ref).max()
    assert np.abs(dg[0] - gb_ref[0]).max() <= 2e-3 * scale and np.abs(dg[-1] - gb_ref[-1]).max() <= 2e-3 * scale
    #   (g1 - g0 is a difference of two FP32 gradients of size ~|G|; the bias part itself is exact to FP32 rounding)
    m.mop_set_bias([], [], 1.0, 0.0)
    v2, g2 = m.mop_eval_veff_grad(R)
    assert H.rms_rel(g2.cpu().numpy(), g0.cpu().numpy()) <= 1e-5
    m.close()


def test_mop_hills_are_deposited_every_pace_steps(B, oracle):
    import torch
    s, o, R = case(oracle, "c1")
    m = B.Mop(s, s.n_beads)
    m.mop_set_bias(np.arange(0, 40), np.arange(200, 260), 0.01, 1.0, pace=3)
    Rg = torch.tensor(R, device="cuda")
    Vg = torch.zeros_like(Rg)
    m.mop_step(Rg, Vg, 0.001, 7)
    assert m.mop_get_bias()["n_hills"] == 2
    m.mop_step_langevin(Rg, Vg, 0.001, 2, 50.0, s.temperature, seed=3, step0=7)   # step 9 deposits the third hill
    st = m.mop_get_bias()
    assert st["n_hills"] == 3 and st["hills"][2] == st["S"]
    _, _, (S_ref, _, _) = oracle.bias(o, Rg.cpu().numpy().astype(np.float64), np.arange(0, 40), np.arange(200, 260), [], 0.01, 1.0)
    assert abs(st["S"] - S_ref) <= 1e-9
    with pytest.raises(B.MopError):
        m.mop_set_bias([0], [s.n_atoms], 0.01, 1.0)
    m.close()


# --------------------------------------------------------------------------- degenerate inputs and errors
def test_edge_cases(B, oracle):
    # two atoms, one pair; then out of range
    for r, npair in ((0.5, 1), (1.05, 0)):
        s = H.two_atoms(r, q=(0.3, -0.3), lj_shift=1)
        o = oracle.OracleSystem(s)
        m = B.Mop(s, 1)
        v, g = m.mop_eval_veff_grad(s.R1[None].astype(np.float32))
        v_ref, g_ref = oracle.veff_grad(o, s.R1[None].astype(np.float32).astype(np.float64), geom=1, brute=True)
        assert m.mop_debug_pairs(0)[1] == npair
        assert abs(v - v_ref) <= 1e-6 * max(abs(v_ref), 1e-3)
        assert np.allclose(g.cpu().numpy(), g_ref, rtol=1e-4, atol=1e-4)
        m.close()
    # one atom: no pairs at all, zero energy and gradient
    s = H.make_system("one", [3.0] * 3, [[1.0, 1.0, 1.0]], [12.0], [0.5], [0], [0.3], [0.5])
    m = B.Mop(s, 3)
    R = np.tile(np.float32(s.R1), (3, 1, 1)) + np.float32([[[0.0]], [[0.001]], [[0.003]]])
    v, g = m.mop_eval_veff_grad(R)
    K = 12.0 * 50.0 / (2 * 0.002)
    assert v == pytest.approx(0.5 * K * 3 * (0.001 ** 2 + 0.002 ** 2), rel=1e-3)
    m.close()


def test_box_barely_above_twice_the_cutoff(B, oracle):
    """min(box) = 2.0001 r_c: every cluster pair is listed under several periodic shifts (up to 27 work units per
    i-cluster); the in-range image of an atom pair is still unique.  Also a rectangular box with one tight side."""
    for box in ([2.0001] * 3, [2.0001, 3.3, 2.6]):
        s = H.lj_cluster(64, L=2.0001, r_cut=1.0)
        if box[1] != box[0]:
            # a jittered 4 x 6 x 4 lattice (uniformly random positions would put atoms 0.02 nm apart, where r^-13 forces
            # amplify the 1e-7 nm resolution of FP32 coordinates beyond any parity bar)
            rng = np.random.default_rng(4)
            g = np.stack(np.meshgrid(np.arange(4), np.arange(6), np.arange(4), indexing="ij"), -1).reshape(-1, 3)
            X = (g + 0.5) * (np.asarray(box) / [4, 6, 4]) + rng.normal(0, 0.04, (96, 3))
            s = H.make_system("rect", box, X, np.full(96, 39.948), rng.normal(0, 0.2, 96), np.zeros(96, int), [0.2],
                              [0.3], r_cut=1.0, eps_rf=78.0, lj_shift=1, T=120.0)
        s.n_beads = 3
        o = oracle.OracleSystem(s)
        R = W.brownian_path(s, 3, lambda X: oracle.bead(o, X, geom=0, brute=True)["F"], seed=0)
        m = B.Mop(s, 3)
        v, g = m.mop_eval_veff_grad(R)
        for n in range(m.nf):
            ref = oracle.pairs(o, R[n].astype(np.float64), geom=1, brute=True)
            got, cnt = m.mop_debug_pairs(n)
            assert cnt == len(ref) and np.array_equal(got, ref)
        v_ref, g_ref = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=True)
        assert abs(v - v_ref) <= TOL_V * abs(v_ref)
        H.assert_close(g.cpu().numpy(), g_ref, TOL_RMS)
        m.close()


def test_buffered_list_reuse(B, oracle):
    """r_buf > 0: the list survives displacements below r_buf/2 (stats count the reuses), a larger move rebuilds it, and
    every evaluation still matches the oracle on the moved coordinates (the r_c test is per atom pair)."""
    s, o, R = case(oracle, "c2")
    m = B.Mop(s, s.n_beads, r_buf=0.08)
    rng = np.random.default_rng(31)
    Rk = R.copy()
    for k in range(4):
        v, g = m.mop_eval_veff_grad(Rk)
        v_ref, g_ref = oracle.veff_grad(o, Rk.astype(np.float64), geom=1, brute=False)
        assert abs(v - v_ref) <= TOL_V * abs(v_ref), k
        assert H.rms_rel(g.cpu().numpy(), g_ref) <= TOL_RMS, k   # RMS only: a pair within rounding of r_c may differ (force jump, G9)
        ref = oracle.pairs(o, Rk[0].astype(np.float64), geom=1, brute=True)
        assert abs(m.mop_debug_pairs(0, cap=0)[1] - len(ref)) <= 2        # same pairs up to FP32 rounding of r^2 at r_c
        st = m.mop_get_stats()
        assert (st["rebuilds"], st["reuses"]) == ((1, k) if k < 3 else (2, 2)), (k, st["rebuilds"], st["reuses"])
        step = 0.008 if k < 2 else 0.06                                   # the third move exceeds r_buf / 2 = 0.04
        Rk = (Rk + rng.uniform(-1, 1, Rk.shape).astype(np.float32) * np.float32(step / np.sqrt(3))).astype(np.float32)
    # atoms that cross a box face keep their image: shift everything by 0.03 nm along x twice
    m2 = B.Mop(s, s.n_beads, r_buf=0.08)
    for k in range(2):
        Rs = (R + np.float32([0.03 * k, 0, 0])).astype(np.float32)
        v, g = m2.mop_eval_veff_grad(Rs)
        v_ref, g_ref = oracle.veff_grad(o, Rs.astype(np.float64), geom=1, brute=False)
        assert abs(v - v_ref) <= TOL_V * abs(v_ref) and H.rms_rel(g.cpu().numpy(), g_ref) <= TOL_RMS
    assert m2.mop_get_stats()["reuses"] == 1
    m.close()
    m2.close()


def test_many_beads(B, oracle):
    """N = 130 beads of the 512-atom LJ system (more beads than the largest sweep point): V_eff, gradient, and the
    neighbour sets of the first and last force bead."""
    s = W.config1(n_beads=130)
    o = oracle.OracleSystem(s)
    R = W.brownian_path(s, 130, lambda X: oracle.bead(o, X, geom=0)["F"], seed=0)
    m = B.Mop(s, 130)
    v, g = m.mop_eval_veff_grad(R)
    v_ref, g_ref = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=False)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    H.assert_close(g.cpu().numpy(), g_ref, TOL_RMS)
    for n in (0, m.nf - 1):
        ref = oracle.pairs(o, R[n].astype(np.float64), geom=1, brute=True)
        got, cnt = m.mop_debug_pairs(n)
        assert cnt == len(ref) and np.array_equal(got, ref)
    m.close()


def test_maximum_number_of_types(B, oracle):
    """n_types = 64 (the header's maximum; 59 KB of dynamic shared memory for the LJ tables) with several all-zero
    LJ rows (the reaction-field-only body) and charges; 65 types are rejected."""
    rng = np.random.default_rng(12)
    n, nt = 300, 64
    box = [2.7, 2.9, 3.1]
    g = np.stack(np.meshgrid(np.arange(6), np.arange(7), np.arange(8), indexing="ij"), -1).reshape(-1, 3)[:n]
    X = (g + 0.5) * (np.asarray(box) / [6, 7, 8]) + rng.normal(0, 0.02, (n, 3))
    sig = rng.uniform(0.25, 0.36, nt)
    eps = rng.uniform(0.2, 1.0, nt)
    eps[::5] = 0.0                                   # every fifth type has no LJ at all
    typ = rng.integers(0, nt, n)
    q = rng.normal(0, 0.3, n)
    s = H.make_system("types64", box, X, rng.uniform(5, 40, n), q - q.mean(), typ, list(sig), list(eps), r_cut=1.0,
                      eps_rf=78.0, lj_shift=1, T=200.0)
    s.n_beads = 3
    o = oracle.OracleSystem(s)
    R = W.brownian_path(s, 3, lambda Y: oracle.bead(o, Y, geom=0, brute=True)["F"], seed=0)
    m = B.Mop(s, 3)
    v, g_ = m.mop_eval_veff_grad(R)
    v_ref, g_ref = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=True)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    H.assert_close(g_.cpu().numpy(), g_ref, TOL_RMS)
    ref = oracle.pairs(o, R[0].astype(np.float64), geom=1, brute=True)
    got, cnt = m.mop_debug_pairs(0)
    assert cnt == len(ref) and np.array_equal(got, ref)
    m.close()
    s2 = H.make_system("types65", box, X, rng.uniform(5, 40, n), q - q.mean(), typ, list(sig) + [0.3], list(eps) + [0.5])
    with pytest.raises(B.MopError) as e:
        B.Mop(s2, 2)
    assert e.value.status == 1


def test_atoms_outside_the_box_and_on_faces(B, oracle):
    """Caller coordinates are never wrapped per bead; atoms far outside [0,L) and exactly on faces."""
    s, o, R = case(oracle, "c1")
    R2 = R.copy()
    R2[:, ::3, 0] += np.float32(2.88) * 3     # whole images away, consistently along the path
    R2[:, 1::5, 1] -= np.float32(2.88) * 2
    R2[0, 0] = [0.0, 2.88, 5.76]
    R2[1:, 0] = R2[0, 0] + (R[1:, 0] - R[0, 0])
    m = B.Mop(s, s.n_beads)
    v, g = m.mop_eval_veff_grad(R2)
    for n in (0, m.nf - 1):
        ref = oracle.pairs(o, R2[n].astype(np.float64), geom=1, brute=True)
        got, cnt = m.mop_debug_pairs(n)
        assert cnt == len(ref) and np.array_equal(got, ref)
    v_ref, g_ref = oracle.veff_grad(o, R2.astype(np.float64), geom=1, brute=True)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    H.assert_close(g.cpu().numpy(), g_ref, TOL_RMS)
    m.close()


def test_host_buffer_entry_point_matches_device_one(B, oracle):
    """mop_eval_veff_grad_host (pinned host buffers in and out: the end-to-end form bench.py times) gives the device
    entry point's numbers."""
    import torch
    s, o, R = case(oracle, "c2")
    m = B.Mop(s, s.n_beads)
    v, g = m.mop_eval_veff_grad(R)
    Rh = torch.as_tensor(R).pin_memory()
    Gh = torch.empty_like(Rh).pin_memory()
    vh = m.mop_eval_veff_grad_host(Rh, Gh)
    assert abs(vh - v) <= 1e-7 * abs(v)
    assert H.rms_rel(Gh.numpy(), g.cpu().numpy()) <= 1e-5
    m.close()


def test_one_context_different_paths_in_turn(B, oracle):
    """One context evaluates two different paths alternately, through the device and the host entry point (CUDA graphs,
    split copies, bonded kernels on the side stream): nothing may survive from the previous evaluation -- a bonded
    kernel that ran before the new sort would scatter through the old slot map and still pass a repeat of the SAME path."""
    import torch
    s, o, R = case(oracle, "c2")
    rng = np.random.default_rng(17)
    R2 = (R[::-1] + rng.normal(0, 0.004, R.shape)).astype(np.float32).copy()     # another path over the same system
    ref = [oracle.veff_grad(o, X.astype(np.float64), geom=1, brute=False) for X in (R, R2)]
    m = B.Mop(s, s.n_beads)
    Gh = torch.empty(R.shape, dtype=torch.float32).pin_memory()
    for k in range(6):
        X, (v_ref, g_ref) = (R, R2)[k % 2], ref[k % 2]
        if k < 3:
            v, g = m.mop_eval_veff_grad(X)
            g = g.cpu().numpy()
        else:
            v = m.mop_eval_veff_grad_host(torch.as_tensor(X).pin_memory(), Gh)
            g = Gh.numpy().copy()
        assert abs(v - v_ref) <= TOL_V * abs(v_ref), k
        H.assert_close(g, g_ref, TOL_RMS)
    m.close()


@pytest.mark.parametrize("name", ["lj_n1", "lj_n2", "chain", "c3"])
def test_graph_replay_and_host_entry_point_at_small_bead_counts(B, oracle, name):
    """The first evaluation of a context takes the plain launch sequence (it checks the list capacities); later ones replay
    the CUDA graphs, and the host entry point splits its copies only when there are at least two H.eta beads: N = 1, 2, 3
    and 6 through all three forms against the oracle."""
    import torch
    s, o, R = case(oracle, name)
    v_ref, g_ref = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=s.n_atoms <= 3000)
    m = B.Mop(s, s.n_beads)
    Rh, Gh = torch.as_tensor(R).pin_memory(), torch.empty(R.shape, dtype=torch.float32).pin_memory()
    for form in ("first", "graphs", "graphs", "host", "host"):
        if form == "host":
            v = m.mop_eval_veff_grad_host(Rh, Gh)
            g = Gh.numpy().copy()
        else:
            v, g = m.mop_eval_veff_grad(R)
            g = g.cpu().numpy()
        assert abs(v - v_ref) <= TOL_V * abs(v_ref), form
        H.assert_close(g, g_ref, TOL_RMS)
    m.close()


def test_topology_can_be_replaced(B, oracle):
    """mop_set_topology again on a live context (here: all charges zero): captured graphs and lists follow."""
    import copy
    s, o, R = case(oracle, "c2")
    m = B.Mop(s, s.n_beads)
    v0, _ = m.mop_eval_veff_grad(R)
    v0b, _ = m.mop_eval_veff_grad(R)                      # graph replay
    s2 = copy.copy(s)
    s2.charge = np.zeros_like(s.charge)
    m.mop_set_topology(s2)
    v1, g1 = m.mop_eval_veff_grad(R)
    v1b, g1b = m.mop_eval_veff_grad(R)
    v_ref, g_ref = oracle.veff_grad(oracle.OracleSystem(s2), R.astype(np.float64), geom=1, brute=False)
    assert abs(v0 - v0b) <= 1e-7 * abs(v0) and abs(v1 - v_ref) <= TOL_V * abs(v_ref) and abs(v1b - v_ref) <= TOL_V * abs(v_ref)
    assert abs(v1 - v0) > 1e-3 * abs(v0)
    H.assert_close(g1b.cpu().numpy(), g_ref, TOL_RMS)
    m.close()


def test_argument_errors_of_the_added_entry_points(B):
    import torch
    s = W.config1(n_beads=1)
    m = B.Mop(s, 1)
    with pytest.raises(B.MopError) as e:          # the end-to-end CV needs two beads
        m.mop_set_bias([0], [1], 0.01, 1.0)
    assert e.value.status == 1
    R = torch.tensor(np.float32(s.R1)[None], device="cuda")
    V = torch.zeros_like(R)
    with pytest.raises(B.MopError):
        m.mop_step_langevin(R, V, 0.001, 1, -1.0, 300.0)
    with pytest.raises(B.MopError):
        m.mop_eval_veff_grad_fd(R, 0.0)
    with pytest.raises(B.MopError):
        m.mop_add_hill(0.0)                       # no bias set
    v, g = m.mop_eval_veff_grad_fd(R, 0.01)       # N = 1: plain -F
    v2, g2 = m.mop_eval_veff_grad(R)
    assert v == pytest.approx(v2, rel=1e-7) and H.rms_rel(g.cpu().numpy(), g2.cpu().numpy()) <= 1e-5
    m.close()


def test_error_codes(B):
    s = W.config1(n_beads=2)
    s.box = np.asarray([1.9, 2.88, 2.88], np.float32)
    with pytest.raises(B.MopError) as e:
        B.Mop(s, 2)
    assert e.value.status == 3
    s = W.config1(n_beads=2)
    s.mass = s.mass.copy()
    s.mass[7] = 0.0
    with pytest.raises(B.MopError) as e:
        B.Mop(s, 2)
    assert e.value.status == 1
    s = W.config2(n_beads=2)
    s.excl_list = s.excl_list.copy()
    s.excl_list[0] = 5          # asymmetric exclusion
    with pytest.raises(B.MopError) as e:
        B.Mop(s, 2)
    assert e.value.status == 1


# --------------------------------------------------------------------------- list capacity and runaway coordinates
def _blob_system(n=1500, L=12.0, spacing=0.36, seed=5):
    rng = np.random.default_rng(seed)
    k = int(np.ceil(n ** (1 / 3)))
    g = np.stack(np.meshgrid(*[np.arange(k)] * 3, indexing="ij"), -1).reshape(-1, 3)[:n]
    Xb = (g - (k - 1) / 2.0) * spacing + rng.normal(0, 0.02, (n, 3))
    s = H.make_system("blob", [L] * 3, Xb, np.full(n, 39.948), np.zeros(n), np.zeros(n, int), [0.34], [0.996],
                      r_cut=1.0, eps_rf=0.0, lj_shift=1, T=120.0)
    return s, Xb


def test_inhomogeneous_system_cluster_on_the_box_corner(B, oracle):
    """A dense cluster in a large vacuum box (local density far above Q/V), centred on the box corner so that every
    periodic shift is in use, and in the middle of the box."""
    s, Xb = _blob_system()
    o = oracle.OracleSystem(s)
    for centre in (0.0, 6.0):
        X = (Xb + centre).astype(np.float32)
        m = B.Mop(s, 1)
        v, g = m.mop_eval_veff_grad(X[None])
        ref = oracle.bead(o, X.astype(np.float64), geom=1, brute=False)
        assert abs(v - ref["U"].sum()) <= TOL_V * abs(ref["U"].sum())
        H.assert_close(g.cpu().numpy()[0], -ref["F"], TOL_RMS)
        assert m.mop_debug_count_inrange(2) == ref["npairs"]
        m.close()


@pytest.mark.parametrize("which", ["entries", "units", "masks"])
def test_pair_list_overflow_is_reported_and_regrown(B, oracle, which):
    """Each pair-list buffer made too small on purpose (mop_debug_set_list_capacity): the evaluation returns MOP_ERR_OOM
    -- no memory fault, nothing written past the buffers --, the buffers have been regrown from the builder's own counts,
    and the repeated call matches the oracle.  Also through mop_step (an overflow in a build no synchronising call
    follows immediately is still reported by the next one: the flag is sticky on the device)."""
    import torch
    s, o, R = case(oracle, "c2")
    m = B.Mop(s, s.n_beads)
    v0, g0 = m.mop_eval_veff_grad(R)
    st = m.mop_get_stats()
    small = {"entries": dict(entries=max(64, int(st["entries"] // 3))), "units": dict(units=max(64, int(st["units"] // 3))),
             "masks": dict(masks=max(64, int(st["masks"] // 3)))}[which]
    m.mop_debug_set_list_capacity(**small)
    with pytest.raises(B.MopError) as e:
        m.mop_eval_veff_grad(R)
    assert e.value.status == 4
    v, g = m.mop_eval_veff_grad(R)                     # buffers were regrown: the repeated call succeeds
    v_ref, g_ref = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=False)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    H.assert_close(g.cpu().numpy(), g_ref, TOL_RMS)
    # asynchronous calls: the overflow of a mop_step build surfaces at the next synchronising call
    m.mop_debug_set_list_capacity(**small)
    Rg, Vg = torch.tensor(R, device="cuda"), torch.zeros(R.shape, device="cuda")
    m.mop_step(Rg, Vg, 0.0005, 2)
    with pytest.raises(B.MopError) as e:
        m.mop_get_stats()
    assert e.value.status == 4
    v, g = m.mop_eval_veff_grad(R)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    m.close()


def test_overflow_in_a_middle_build_only_still_grows_the_buffer(B):
    """The overflow word is sticky across the builds of one call, the builder's counts are those of the LAST build only.
    Here a dense configuration (all atoms in one octant of the box) overflows the entry buffer and a sparse one (the same
    atoms spread over the whole box), built right after it without a synchronising call in between, fits with more than
    the regrow margin to spare.  The flagged buffer must grow all the same, otherwise repeating the sequence meets the
    same overflow for ever."""
    s = H.lj_cluster(n=512, L=5.0, seed=4)                            # lattice spacing 0.625 nm: a thin gas
    rng = np.random.default_rng(11)
    RB = (s.R1[None] + rng.normal(0, 0.002, (4, s.n_atoms, 3))).astype(np.float32)
    RA = (0.5 * RB).astype(np.float32)                                # spacing 0.31 nm: 8 x the density, in one octant
    m = B.Mop(s, 4)
    vA, gA = m.mop_eval_veff_grad(RA)
    nA = m.mop_get_stats()["entries"]
    m.mop_eval_veff_grad(RB)
    nB = m.mop_get_stats()["entries"]
    assert nA > 1.45 * nB, (nA, nB)                                   # the premise: 1.3 x the last count is below the capacity
    m.mop_debug_set_list_capacity(entries=int(1.4 * nB))              # holds RB with > 1.3 x to spare, not RA
    for attempt in range(8):
        m.mop_eval_veff_grad(RA, sync=False)                          # overflows (or not any more)
        m.mop_eval_veff_grad(RB, sync=False)                          # fits; its counts are the ones a regrow sees
        try:
            m.mop_get_stats()
            break
        except B.MopError as e:
            assert e.status == 4
    else:
        pytest.fail("the entry buffer never grew: the same overflow after 8 repeats (entries %d vs %d)" % (nA, nB))
    assert attempt >= 1                                               # the first round did overflow
    v, g = m.mop_eval_veff_grad(RA)                                   # and the dense path now evaluates as it did before
    assert abs(v - vA) <= 1e-8 * abs(vA) and H.rms_rel(g.cpu().numpy(), gA.cpu().numpy()) <= 1e-6
    m.close()


def test_create_refuses_sizes_beyond_the_index_arithmetic(B):
    """mop_create checks what the kernels' packed indices assume (24-bit j-octet index in a list entry, 32-bit element
    offsets bead * S + slot) before it allocates anything."""
    import ctypes as C
    L = B.load()
    for Q, N, box, word in ((140_000_000, 1, (300.0, 300.0, 300.0), b"octets"), (1000, 1_000_000, (1000.0, 1000.0, 2.5), b"2^31")):
        p = B.mop_params()
        p.n_atoms, p.n_beads = Q, N
        p.box[0], p.box[1], p.box[2] = box
        p.r_cut, p.dt_path, p.nu = 1.0, 0.002, 50.0
        ctx = C.c_void_p()
        assert L.mop_create(C.byref(ctx), C.byref(p)) == 1
        assert word in L.mop_last_error(None), L.mop_last_error(None)
        assert not ctx.value


@pytest.mark.parametrize("bad", [1.0e12, -3.0e30, float("inf"), float("nan")])
def test_runaway_coordinates_are_reported_not_faulted(B, oracle, bad):
    """A coordinate the wrap cannot bring back into the box (|x| >~ 1e7 L, Inf, NaN) -- what a diverging trajectory
    passes through -- gives MOP_ERR_NONFINITE, never an out-of-bounds cell index; the device stays usable."""
    import torch
    s, o, R = case(oracle, "c1")
    R2 = R.copy()
    R2[3, 17, 1] = bad
    m = B.Mop(s, s.n_beads)
    with pytest.raises(B.MopError) as e:
        m.mop_eval_veff_grad(R2)
    assert e.value.status == 6
    m.close()
    torch.cuda.synchronize()
    m = B.Mop(s, s.n_beads)
    v, g = m.mop_eval_veff_grad(R)
    v_ref, _ = oracle.veff_grad(o, R.astype(np.float64), geom=1, brute=True)
    assert abs(v - v_ref) <= TOL_V * abs(v_ref)
    m.close()
