"""Pins of the FP64 oracle against what the paper and the mathematics fix (no GPU).

P1..P13 follow SURVEY.md section 8(c).  The paper prints no numeric worked example, so the
pins are closed forms (tests/golden/closed_forms.txt), finite differences, invariants, special
cases and brute force, chosen so that a dropped term, a wrong sign/index or a transposed operand
in oracle/mop_oracle.c fails at least one of them.
"""
import os

import numpy as np
import pytest

from paper_2501_11962_b200 import workloads as W
from tests import helpers as H

KE = 138.935458
GOLD = {}
with open(os.path.join(os.path.dirname(__file__), "golden", "closed_forms.txt")) as f:
    for line in f:
        if not line.startswith("#"):
            k, v = line.split()
            GOLD[k] = float(v)


# ---------------------------------------------------------------- P1 / P2 closed forms
@pytest.mark.parametrize("r", [0.30, 0.34, 0.40, 0.55, 0.90])
def test_P1_lj_two_atom_closed_form(oracle, r):
    """LJ 12-6 energy and force of an isolated pair vs the textbook closed form."""
    for axis in range(3):
        s = H.two_atoms(r, axis=axis)
        o = oracle.OracleSystem(s)
        for geom in (0, 1):
            res = oracle.bead(o, s.R1, geom=geom, brute=True)
            assert res["npairs"] == 1
            # geom 1 first rounds the coordinates to float32 (relative 6e-8 on r, x13 on the force)
            tol = 3e-6 if geom == 0 else 1e-4
            assert res["U"][0] == pytest.approx(GOLD["lj_u_r=%.2f" % r], rel=tol, abs=tol)
            F = res["F"]
            # atom 1 sits at +r along `axis`: repulsive force pushes it towards +axis
            assert F[1, axis] == pytest.approx(GOLD["lj_F_r=%.2f" % r], rel=tol)
            assert F[0, axis] == pytest.approx(-GOLD["lj_F_r=%.2f" % r], rel=tol)
            off = [a for a in range(3) if a != axis]
            assert np.abs(F[:, off]).max() < 1e-9


def test_P1_lj_minimum_and_curvature(oracle):
    rstar = GOLD["lj_rstar"]
    s = H.two_atoms(rstar)
    o = oracle.OracleSystem(s)
    sv = np.zeros((2, 3))
    sv[1] = [1.0, 0.0, 0.0]
    res = oracle.bead(o, s.R1, geom=0, brute=True, s=sv)
    assert res["U"][0] == pytest.approx(GOLD["lj_u_at_rstar"], rel=1e-6)
    assert np.abs(res["F"]).max() < 2e-4          # zero force at the minimum (c6/c12 are float32)
    # along-axis curvature u''(r*) = 72 eps/(2^(1/3) sigma^2); transverse u'/r = 0
    assert res["Hs"][1, 0] == pytest.approx(GOLD["lj_upp_at_rstar"], rel=1e-5)
    assert res["Hs"][0, 0] == pytest.approx(-GOLD["lj_upp_at_rstar"], rel=1e-5)
    sv[1] = [0.0, 1.0, 0.0]
    res = oracle.bead(o, s.R1, geom=0, brute=True, s=sv)
    assert np.abs(res["Hs"]).max() < 2e-3


def test_P1_lj_potential_shift(oracle):
    """lj_shift=1 makes U_LJ(r_c) = 0 and leaves the force unchanged."""
    r = 0.9999999
    a = oracle.bead(oracle.OracleSystem(H.two_atoms(r, lj_shift=1)), H.two_atoms(r).R1, geom=0, brute=True)
    b = oracle.bead(oracle.OracleSystem(H.two_atoms(r, lj_shift=0)), H.two_atoms(r).R1, geom=0, brute=True)
    assert abs(a["U"][0]) < 1e-8
    assert abs(b["U"][0]) > 1e-3
    assert np.allclose(a["F"], b["F"], rtol=0, atol=1e-14)
    # beyond the cutoff: no pair
    c = oracle.bead(oracle.OracleSystem(H.two_atoms(1.0000001)), H.two_atoms(1.0000001).R1, geom=0, brute=True)
    assert c["npairs"] == 0 and np.abs(c["F"]).max() == 0.0


@pytest.mark.parametrize("r", [0.25, 0.50, 0.90])
def test_P2_reaction_field_closed_form(oracle, r):
    s = H.two_atoms(r, eps=0.0, q=(-0.82, 0.41))
    o = oracle.OracleSystem(s)
    res = oracle.bead(o, s.R1, geom=0, brute=True)
    qs = float(np.float32(-0.82)) * float(np.float32(0.41)) / (-0.82 * 0.41)   # float32 charges
    assert res["U"][1] == pytest.approx(GOLD["rf_u_r=%.2f" % r] * qs, rel=1e-9)
    assert res["F"][1, 0] == pytest.approx(GOLD["rf_F_r=%.2f" % r] * qs, rel=1e-9)
    assert res["U"][0] == 0.0


def test_P2_reaction_field_at_cutoff(oracle):
    r = 1.0 - 1e-10
    s = H.two_atoms(r, eps=0.0, q=(-0.82, 0.41))
    res = oracle.bead(oracle.OracleSystem(s), s.R1, geom=0, brute=True)
    qs = float(np.float32(-0.82)) * float(np.float32(0.41)) / (-0.82 * 0.41)
    assert abs(res["U"][1]) < 1e-7                                   # u(r_c) = 0
    assert res["F"][1, 0] == pytest.approx(GOLD["rf_F_at_rc"] * qs, rel=1e-7)
    # eps_rf <= 0 means infinity: k_rf = 1/(2 rc^3), force vanishes at r_c
    s2 = H.two_atoms(r, eps=0.0, q=(-0.82, 0.41), eps_rf=0.0)
    res2 = oracle.bead(oracle.OracleSystem(s2), s2.R1, geom=0, brute=True)
    assert abs(res2["F"][1, 0]) < 1e-6 and abs(res2["U"][1]) < 1e-7


# ---------------------------------------------------------------- P3 HVP vs finite differences
def _clear_of_cutoff(make, tol=2e-4):
    """G9: FD pins need configurations with no pair at the cutoff; take the first seed that has none."""
    for seed in range(1, 50):
        s = make(seed)
        if H.pairs_near_cutoff(s, s.R1, tol) == 0:
            return s
    raise RuntimeError("no seed without a pair at the cutoff")


def _systems():
    return [_clear_of_cutoff(lambda sd: H.lj_cluster(32, seed=sd)),
            _clear_of_cutoff(lambda sd: H.tiny_water(seed=sd)),
            _clear_of_cutoff(lambda sd: H.tiny_chain(seed=sd)),
            _clear_of_cutoff(lambda sd: H.lj_cluster(27, seed=sd, masses=np.linspace(5, 40, 27)))]


@pytest.mark.parametrize("idx", range(3))
def test_P3_hvp_vs_central_difference_of_forces(oracle, idx):
    s = _systems()[idx]
    assert H.pairs_near_cutoff(s, s.R1, 2e-4) == 0, "G9: move the seed, a pair sits at the cutoff"
    o = oracle.OracleSystem(s)
    rng = np.random.default_rng(5)
    sv = rng.normal(0, 1, (s.n_atoms, 3))
    res = oracle.bead(o, s.R1, geom=0, brute=True, s=sv)
    eps = 1e-6
    Fp = oracle.bead(o, s.R1 + eps * sv, geom=0, brute=True)["F"]
    Fm = oracle.bead(o, s.R1 - eps * sv, geom=0, brute=True)["F"]
    Hs_fd = -(Fp - Fm) / (2 * eps)
    assert H.rms_rel(res["Hs"], Hs_fd) < 2e-7
    # each term type separately has to be there: zero direction on all but one atom
    sv1 = np.zeros_like(sv)
    sv1[3] = [0.3, -0.2, 0.9]
    r1 = oracle.bead(o, s.R1, geom=0, brute=True, s=sv1)["Hs"]
    Fp = oracle.bead(o, s.R1 + eps * sv1, geom=0, brute=True)["F"]
    Fm = oracle.bead(o, s.R1 - eps * sv1, geom=0, brute=True)["F"]
    assert H.rms_rel(r1, -(Fp - Fm) / (2 * eps)) < 2e-7


def test_P3_force_is_minus_gradient_of_energy(oracle):
    """F = -dU/dR by central differences of the oracle's own energy."""
    for s in _systems()[:3]:
        o = oracle.OracleSystem(s)
        F = oracle.bead(o, s.R1, geom=0, brute=True)["F"]
        rng = np.random.default_rng(11)
        for _ in range(6):
            i, a = int(rng.integers(s.n_atoms)), int(rng.integers(3))
            e = 1e-6
            Xp, Xm = s.R1.copy(), s.R1.copy()
            Xp[i, a] += e
            Xm[i, a] -= e
            up = oracle.bead(o, Xp, geom=0, brute=True)["U"].sum()
            um = oracle.bead(o, Xm, geom=0, brute=True)["U"].sum()
            assert F[i, a] == pytest.approx(-(up - um) / (2 * e), rel=2e-6, abs=2e-5)


# ---------------------------------------------------------------- P4 / P5 gradient of V_eff
def _tiny_path(oracle, s, N, seed=0, noise=True):
    o = oracle.OracleSystem(s)
    R = W.brownian_path(s, N, lambda X: oracle.bead(o, X, geom=0, brute=True)["F"], seed=seed, noise=noise,
                        dtype=np.float64)
    return o, R


@pytest.mark.parametrize("idx", [2, 3])
def test_P4_gradient_vs_finite_difference_of_veff(oracle, idx):
    s = _systems()[idx]
    o, R = _tiny_path(oracle, s, 5)
    v, G = oracle.veff_grad(o, R, geom=0, brute=True)
    rng = np.random.default_rng(3)
    e = 2e-7
    worst = 0.0
    for _ in range(40):
        n, i, a = int(rng.integers(R.shape[0])), int(rng.integers(s.n_atoms)), int(rng.integers(3))
        Rp, Rm = R.copy(), R.copy()
        Rp[n, i, a] += e
        Rm[n, i, a] -= e
        fd = (oracle.veff_grad(o, Rp, geom=0, brute=True)[0] - oracle.veff_grad(o, Rm, geom=0, brute=True)[0]) / (2 * e)
        worst = max(worst, abs(fd - G[n, i, a]) / max(abs(G[n, i, a]), 1.0))
    assert worst < 5e-6


def test_P5_paper_equations_5_6_7(oracle):
    """-grad equals eqs (5),(6),(7) of the paper with the bracket evaluated by central differences."""
    s = _systems()[3]                     # unequal masses
    o, R = _tiny_path(oracle, s, 5)
    v, G, parts = oracle.veff_grad(o, R, geom=0, brute=True, want_parts=True)
    N = R.shape[0]
    m = s.mass.astype(float)[:, None]
    K = m * s.nu / (2 * s.dt_path)
    a = s.dt_path / (m * s.nu)
    force = lambda X: oracle.bead(o, X, geom=0, brute=True)["F"]
    F = [force(R[n]) for n in range(N)]
    eps = 1e-4

    def bracket(n):
        eta = R[n + 1] - R[n] - a * F[n]
        sc = eps / np.abs(eta).max()
        return (force(R[n] + sc * eta) - force(R[n] - sc * eta)) / (4 * sc)

    Feff = np.zeros_like(R)
    Feff[0] = 0.5 * F[0] + K * (R[1] - R[0]) + bracket(0)                                   # eq. (6)
    for n in range(1, N - 1):
        Feff[n] = -K * (2 * R[n] - R[n - 1] - R[n + 1]) + 0.5 * (F[n - 1] - F[n]) + bracket(n)  # eq. (5)
    Feff[N - 1] = -K * (R[N - 1] - R[N - 2]) + 0.5 * F[N - 2]                               # eq. (7)
    assert H.rms_rel(-G, Feff) < 1e-6
    for n in range(N):
        assert H.rms_rel(-G[n], Feff[n]) < 5e-6


def test_P5b_fd_form_of_the_oracle(oracle):
    """veff_grad_fd is eqs (5),(6),(7) as printed.  Pinned two ways: (i) against the equations retyped here with
    the oracle's plain force (no shared arithmetic beyond F); (ii) against the analytic gradient, from which it may
    differ only by the O(eps^2) truncation of the central difference (and by pairs crossing r_c, G9: none here)."""
    s = _systems()[3]
    o, R = _tiny_path(oracle, s, 5)
    N = R.shape[0]
    m = s.mass.astype(float)[:, None]
    K = m * s.nu / (2 * s.dt_path)
    a = s.dt_path / (m * s.nu)
    force = lambda X: oracle.bead(o, X, geom=0, brute=True)["F"]
    F = [force(R[n]) for n in range(N)]
    eps = 0.02
    Feff = np.zeros_like(R)
    for n in range(N - 1):
        eta = R[n + 1] - R[n] - a * F[n]
        br = (force(R[n] + eps * eta) - force(R[n] - eps * eta)) / (4 * eps)
        Feff[n] = (0.5 * F[0] + K * (R[1] - R[0]) + br) if n == 0 else \
            (-K * (2 * R[n] - R[n - 1] - R[n + 1]) + 0.5 * (F[n - 1] - F[n]) + br)
    Feff[N - 1] = -K * (R[N - 1] - R[N - 2]) + 0.5 * F[N - 2]
    v_fd, G_fd = oracle.veff_grad_fd(o, R, eps, geom=0, brute=True)
    v, G = oracle.veff_grad(o, R, geom=0, brute=True)
    assert v_fd == pytest.approx(v, rel=1e-13)
    assert H.rms_rel(-G_fd, Feff) < 1e-12
    assert H.rms_rel(G_fd, G) < 1e-8      # eps |eta| ~ 1e-4 nm: truncation ~1e-12, and no pair crosses r_c here (G9)
    # N = 1: plain force
    v1, G1 = oracle.veff_grad_fd(o, R[:1], eps, geom=0, brute=True)
    assert np.allclose(G1[0], -F[0], rtol=1e-13, atol=1e-13)


# ---------------------------------------------------------------- P6 / P7 invariants
@pytest.mark.parametrize("idx", range(3))
def test_P6_newton_third_law_and_translation(oracle, idx):
    s = _systems()[idx]
    o = oracle.OracleSystem(s)
    rng = np.random.default_rng(9)
    sv = rng.normal(0, 1, (s.n_atoms, 3))
    res = oracle.bead(o, s.R1, geom=0, brute=True, s=sv)
    scale = np.abs(res["F"]).max()
    assert np.abs(res["F"].sum(0)).max() < 1e-11 * scale
    assert np.abs(res["Hs"].sum(0)).max() < 1e-10 * np.abs(res["Hs"]).max()
    t = np.tile([[0.3, -1.0, 0.7]], (s.n_atoms, 1))
    Ht = oracle.bead(o, s.R1, geom=0, brute=True, s=t)["Hs"]
    assert np.abs(Ht).max() < 1e-9 * np.abs(res["Hs"]).max()


@pytest.mark.parametrize("idx", range(3))
def test_P7_hessian_symmetry(oracle, idx):
    s = _systems()[idx]
    o = oracle.OracleSystem(s)
    rng = np.random.default_rng(10)
    a = rng.normal(0, 1, (s.n_atoms, 3))
    b = rng.normal(0, 1, (s.n_atoms, 3))
    Ha = oracle.bead(o, s.R1, geom=0, brute=True, s=a)["Hs"]
    Hb = oracle.bead(o, s.R1, geom=0, brute=True, s=b)["Hs"]
    assert (b * Ha).sum() == pytest.approx((a * Hb).sum(), rel=1e-10)


# ---------------------------------------------------------------- P8 / P9 / P10 the path
def test_P8_equipartition_on_generated_path(oracle):
    """On a Brownian path E_spring/(3Q(N-1)) = kT/2 (pins K, L^n scale and reading G1)."""
    s = W.config1()
    o = oracle.OracleSystem(s)
    N = 6
    R = W.brownian_path(s, N, lambda X: oracle.bead(o, X, geom=0)["F"], seed=0, dtype=np.float64)
    v, G, parts = oracle.veff_grad(o, R, geom=0, want_parts=True)
    dof = 3 * s.n_atoms * (N - 1)
    ratio = parts["E_spring"] / dof / (0.5 * W.KB * s.temperature)
    assert abs(ratio - 1.0) < 4.0 * np.sqrt(2.0 / dof)
    assert v == pytest.approx(parts["U1"] + parts["E_spring"], rel=1e-14)


def test_P9_noise_free_euler_path(oracle):
    s = H.tiny_chain()
    o, R = _tiny_path(oracle, s, 5, noise=False)
    v, G, parts = oracle.veff_grad(o, R, geom=0, brute=True, want_parts=True)
    F1 = oracle.bead(o, R[0], geom=0, brute=True)
    assert parts["E_spring"] < 1e-18
    assert np.abs(parts["eta"]).max() < 1e-15
    assert v == pytest.approx(F1["U"].sum(), rel=1e-13)
    assert H.rms_rel(G[0], -F1["F"]) < 1e-9
    assert np.abs(G[1:]).max() < 1e-8 * np.abs(G[0]).max()


def test_P10_special_cases_N1_N2(oracle):
    s = H.tiny_chain()
    o, R = _tiny_path(oracle, s, 2)
    b = oracle.bead(o, R[0], geom=0, brute=True)
    v1, G1 = oracle.veff_grad(o, R[:1], geom=0, brute=True)
    assert v1 == pytest.approx(b["U"].sum(), rel=1e-14)
    assert np.allclose(G1[0], -b["F"], rtol=0, atol=1e-12 * np.abs(b["F"]).max())
    v2, G2, p2 = oracle.veff_grad(o, R, geom=0, brute=True, want_parts=True)
    m = s.mass.astype(float)[:, None]
    K = m * s.nu / (2 * s.dt_path)
    eta = R[1] - R[0] - s.dt_path / (m * s.nu) * b["F"]
    assert np.allclose(G2[1], K * eta, rtol=1e-12, atol=1e-9)
    assert v2 == pytest.approx(b["U"].sum() + (0.5 * K * eta ** 2).sum(), rel=1e-13)


def test_P11_zero_length_harmonic_dimer(oracle):
    """b0 = 0: U = k|r1-r2|^2/2, H = k[[I,-I],[-I,I]] constant; V_eff is a homogeneous quadratic form in
    the bead coordinates, hence x . grad V_eff = 2 V_eff (Euler) and grad is linear in x."""
    k = 1234.5
    X = np.array([[1.0, 1.0, 1.0], [1.13, 0.95, 1.08]])
    s = H.make_system("dimer", [5.0] * 3, X, [12.0, 3.0], [0, 0], [0, 0], [0.3], [0.0], bonds=[[0, 1]],
                      bpar=[[0.0, k]], r_cut=1.0)
    o = oracle.OracleSystem(s)
    rng = np.random.default_rng(4)
    sv = rng.normal(0, 1, (2, 3))
    res = oracle.bead(o, X, geom=0, brute=True, s=sv)
    assert np.allclose(res["Hs"][0], k * (sv[0] - sv[1]), rtol=1e-12)
    assert np.allclose(res["Hs"][1], -k * (sv[0] - sv[1]), rtol=1e-12)
    assert res["U"][2] == pytest.approx(0.5 * k * ((X[0] - X[1]) ** 2).sum(), rel=1e-13)
    N = 4
    R = rng.normal(0, 0.05, (N, 2, 3)) + 1.0
    c = np.array([1.0, 1.0, 1.0])          # V_eff depends on r1-r2 and bead differences only
    v, G = oracle.veff_grad(o, R, geom=0, brute=True)
    assert ((R - c) * G).sum() == pytest.approx(2.0 * v, rel=1e-11)
    v3, G3 = oracle.veff_grad(o, c + 3.0 * (R - c), geom=0, brute=True)
    assert v3 == pytest.approx(9.0 * v, rel=1e-11)
    assert np.allclose(G3, 3.0 * G, rtol=1e-10, atol=1e-9)


def _rotation(seed):
    """A proper rotation matrix from a seeded QR (so that no closed-form pin is axis-aligned by accident)."""
    q, r = np.linalg.qr(np.random.default_rng(seed).normal(size=(3, 3)))
    q = q * np.sign(np.diag(r))
    if np.linalg.det(q) < 0:
        q[:, 0] = -q[:, 0]
    return q


@pytest.mark.parametrize("rot", [None, 1, 2])
def test_P16_harmonic_bond_closed_form(oracle, rot):
    """Two bonded atoms, b0 = 0.125 nm, k_b = 1e5, r = 0.140625 nm (all exact in FP32; values from
    tests/golden/make_golden.py, formulas only): U = k_b/2 (r-b0)^2 = 12.207, |F| = k_b (r-b0) = 1562.5 along the bond
    and attractive, curvature k_b along the bond and
    k_b (1 - b0/r) across it.  Fixes b0, k_b, their order in the parameter pair, and the sign of the force."""
    Q = np.eye(3) if rot is None else _rotation(rot)
    u = Q @ np.array([1.0, 0.0, 0.0])
    t = Q @ np.array([0.0, 1.0, 0.0])
    X = np.array([[2.0, 2.0, 2.0], [2.0, 2.0, 2.0] + 0.140625 * u])
    s = H.make_system("bond", [5.0] * 3, X, [12.0, 3.0], [0, 0], [0, 0], [0.3], [0.0], bonds=[[0, 1]],
                      bpar=[[0.125, 1.0e5]], r_cut=1.0)
    o = oracle.OracleSystem(s)
    sv = np.zeros((2, 3))
    sv[0] = u
    res = oracle.bead(o, X, geom=0, brute=True, s=sv)
    assert res["U"][2] == pytest.approx(GOLD["bond_U"], rel=1e-12) and res["U"][0] == 0 and res["U"][1] == 0
    assert np.allclose(res["F"][0], GOLD["bond_F"] * u, rtol=1e-10, atol=1e-9)      # atom 0 is pulled towards atom 1
    assert np.allclose(res["F"][1], -GOLD["bond_F"] * u, rtol=1e-10, atol=1e-9)
    assert np.allclose(res["Hs"][0], GOLD["bond_kpar"] * u, rtol=1e-10, atol=1e-6)  # displacement along the bond
    assert np.allclose(res["Hs"][1], -GOLD["bond_kpar"] * u, rtol=1e-10, atol=1e-6)
    sv[0] = t
    res = oracle.bead(o, X, geom=0, brute=True, s=sv)
    assert np.allclose(res["Hs"][0], GOLD["bond_kperp"] * t, rtol=1e-10, atol=1e-6)  # displacement across the bond
    # compressed bond: repulsive, same magnitude law
    X2 = np.array([[2.0, 2.0, 2.0], [2.0, 2.0, 2.0] + 0.109375 * u])
    res = oracle.bead(o, X2, geom=0, brute=True)
    assert np.allclose(res["F"][0], -1.0e5 * 0.015625 * u, rtol=1e-9, atol=1e-8)
    assert res["U"][2] == pytest.approx(0.5 * 1.0e5 * 0.015625 ** 2, rel=1e-10)


@pytest.mark.parametrize("deg", [90, 150])
@pytest.mark.parametrize("rot", [None, 3])
def test_P16_harmonic_angle_closed_form(oracle, deg, rot):
    """Three atoms i-j-k, j central, |a| = 0.1, |b| = 0.15, theta0 = 1.875 rad (107.43 deg, exact in FP32), k_theta = 383, at
    theta = 90 deg (opens) and 150 deg (closes): U = k/2 (theta-theta0)^2, F_i perpendicular to a in the plane with
    |F_i| = k |theta-theta0| / |a|, F_k likewise with |b|, F_j = -F_i - F_k (tests/golden/make_golden.py, formulas
    only).  Fixes theta0, k_theta, which atom is central, the angle convention (not its supplement) and the signs."""
    Q = np.eye(3) if rot is None else _rotation(rot)
    th = np.deg2rad(deg)
    rj = np.array([2.0, 2.2, 1.9])
    ri = rj + Q @ (0.1 * np.array([1.0, 0.0, 0.0]))
    rk = rj + Q @ (0.15 * np.array([np.cos(th), np.sin(th), 0.0]))
    gold = {n: Q @ np.array([GOLD["angle%d_%s%s" % (deg, n, ax)] for ax in "xyz"]) for n in ("Fi", "Fj", "Fk")}
    for order in ((0, 1, 2), (2, 1, 0)):        # (i, j, k) and the same angle named (k, j, i): identical physics
        X = np.zeros((3, 3))
        X[order[0]], X[order[1]], X[order[2]] = ri, rj, rk
        s = H.make_system("angle", [5.0] * 3, X, [12.0, 3.0, 5.0], [0, 0, 0], [0, 0, 0], [0.3], [0.0],
                          angles=[[order[0], order[1], order[2]]], apar=[[1.875, 383.0]], r_cut=1.0,
                          excl=W.exclusions_from_bonds(3, [[0, 1], [1, 2]]))
        o = oracle.OracleSystem(s)
        res = oracle.bead(o, X, geom=0, brute=True)
        assert res["U"][3] == pytest.approx(GOLD["angle%d_U" % deg], rel=1e-12)
        assert res["U"][0] == 0 and res["U"][1] == 0 and res["U"][2] == 0
        for n, idx in (("Fi", order[0]), ("Fj", order[1]), ("Fk", order[2])):
            assert np.allclose(res["F"][idx], gold[n], rtol=1e-10, atol=1e-8), (n, res["F"][idx], gold[n])
    # the force on i does no work along a (pure rotation) and opens (90 deg) or closes (150 deg) the angle
    assert abs(gold["Fi"] @ (ri - rj)) < 1e-9
    assert np.sign(gold["Fi"] @ (rk - rj)) == (1.0 if deg == 150 else -1.0)


def test_G13_grid_dimensions_and_cell_ids_by_hand(oracle):
    """Search-grid dimensions and cell ids on a hand-sized case: box 3 x 4 x 5, Q = 1000, cluster 8, z bins 0.125:
    side = cbrt(8 * 60 / 1000) = 0.78297..., nx = floor(3 / side) = 3, ny = floor(4 / side) = 5, nz = floor(5 / 0.125) = 40;
    cell = (cx ny + cy) nz + cz with c = floor(x n / L)."""
    box = np.array([3.0, 4.0, 5.0], np.float32)
    assert oracle.grid_dims(1000, box, 8, 0.125) == [3, 5, 40]
    assert oracle.grid_dims(125, box, 8, 0.125)[:2] == [1, 2]          # side = cbrt(3.84) = 1.566: floor(3/1.566), floor(4/1.566)
    X = np.array([[0.1, 0.1, 0.1], [2.9, 3.9, 4.9], [1.5, 2.0, 2.5], [2.1, 0.7, 0.2]], np.float32)
    cell = oracle.cell_ids(X, box, [3, 5, 40])
    #            (0,0,0)   (2,4,39)               (1,2,20)               (2,0,1)
    assert cell.tolist() == [0, (2 * 5 + 4) * 40 + 39, (1 * 5 + 2) * 40 + 20, (2 * 5 + 0) * 40 + 1]


# ---------------------------------------------------------------- P12 integrator
def test_P12_velocity_verlet_invariants(oracle):
    s = H.lj_cluster(32)
    o, R = _tiny_path(oracle, s, 4)
    rng = np.random.default_rng(8)
    V = rng.normal(0, 1, R.shape) * np.sqrt(W.KB * 120.0 / s.mass.astype(float))[None, :, None]
    dt = 0.001
    R1, V1, e1 = oracle.step(o, R, V, dt, 200, geom=0, brute=True)
    R2, V2, e2 = oracle.step(o, R, V, dt / 2, 400, geom=0, brute=True)
    fl1 = np.std(e1[:, 2])
    fl2 = np.std(e2[::2, 2])
    assert fl1 < 2e-2 * np.std(e1[:, 1])                  # total energy conserved vs kinetic swings
    assert 2.5 < fl1 / fl2 < 6.0                          # fluctuation ~ dt^2
    assert abs(e1[-1, 2] - e1[0, 2]) < 5 * fl1 + 1e-9     # no drift
    # time reversal
    Rb, Vb, _ = oracle.step(o, R1, -V1, dt, 200, geom=0, brute=True)
    assert np.abs(Rb - R).max() < 1e-9
    assert np.abs(Vb + V).max() < 1e-6


# ---------------------------------------------------------------- P14 Langevin thermostat (NEXT-2, reading G19)
def test_P14_noise_generator_statistics(oracle):
    """The counter-based generator: unbiased bits, N(0,1) moments, no correlation along idx or step."""
    bits = np.array([oracle.noise_bits(7, 3, i) for i in range(20000)], dtype=np.uint64)
    for b in (0, 1, 17, 31, 32, 47, 63):
        assert abs(float(((bits >> np.uint64(b)) & np.uint64(1)).mean()) - 0.5) < 0.012
    assert len(np.unique(bits)) == len(bits)
    x = np.array([[oracle.noise_normal(11, st, i) for i in range(20000)] for st in range(3)])
    assert abs(x.mean()) < 0.015 and abs(x.var() - 1.0) < 0.02
    assert abs((x ** 4).mean() - 3.0) < 0.15 and abs((x ** 3).mean()) < 0.05
    assert abs(np.mean(x[0, :-1] * x[0, 1:])) < 0.02 and abs(np.mean(x[0] * x[1])) < 0.02
    assert oracle.noise_normal(11, 0, 5) != oracle.noise_normal(12, 0, 5)          # the seed matters
    assert oracle.noise_normal(11, 2, 5) == x[2, 5]                                # and it is a pure function


def test_P14_gamma_zero_is_velocity_verlet(oracle):
    s = H.lj_cluster(32)
    o, R = _tiny_path(oracle, s, 3)
    V = np.random.default_rng(4).normal(0, 0.3, R.shape)
    R1, V1, e1 = oracle.step(o, R, V, 0.001, 7, geom=0, brute=True)
    R2, V2, e2 = oracle.step_langevin(o, R, V, 0.001, 7, 0.0, 120.0, seed=5, geom=0, brute=True)
    assert np.array_equal(R1, R2) and np.array_equal(V1, V2) and np.array_equal(e1, e2)


def test_P14_free_particles_follow_the_exact_ornstein_uhlenbeck_law(oracle):
    """No forces (eps = 0, q = 0, N = 1, so V_eff = 0): v_n is an exact OU chain with c = exp(-gamma dt):
    Var(v_n) = (kT/m)(1 - c^(2n)) from rest, lag-1 correlation c in the stationary state."""
    n = 1500
    rng = np.random.default_rng(1)
    m = np.linspace(4.0, 40.0, n)
    s = H.make_system("free", [6.0] * 3, rng.uniform(0, 6, (n, 3)), m, np.zeros(n), np.zeros(n, int), [0.3], [0.0],
                      r_cut=1.0, eps_rf=0.0, T=300.0)
    o = oracle.OracleSystem(s)
    R0, V0 = s.R1[None].astype(float), np.zeros((1, n, 3))
    T, dt, gamma = 300.0, 0.001, 200.0
    c = np.exp(-gamma * dt)
    kT_m = oracle.KB * T / m[None, :, None]
    R1, V1, _ = oracle.step_langevin(o, R0, V0, dt, 3, gamma, T, seed=2, geom=0, brute=False)
    r = (V1 ** 2 / kT_m).mean()
    assert abs(r - (1 - c ** 6)) < 4 * (1 - c ** 6) * np.sqrt(2.0 / (3 * n))
    Ra, Va, _ = oracle.step_langevin(o, R0, V0, dt, 40, gamma, T, seed=2, geom=0, brute=False)        # 8 relaxation times
    Rb, Vb, _ = oracle.step_langevin(o, Ra, Va, dt, 1, gamma, T, seed=2, step0=40, geom=0, brute=False)
    assert abs((Va ** 2 / kT_m).mean() - 1.0) < 4 * np.sqrt(2.0 / (3 * n))
    assert abs((Va * Vb / kT_m).mean() - c) < 4 / np.sqrt(3 * n)
    # continuing with step0 replays the same stream as one longer call
    Rc, Vc, _ = oracle.step_langevin(o, R0, V0, dt, 41, gamma, T, seed=2, geom=0, brute=False)
    assert np.allclose(Vc, Vb, rtol=0, atol=1e-12) and np.allclose(Rc, Rb, rtol=0, atol=1e-12)


def test_P14_nvt_temperature_of_an_interacting_path(oracle):
    """Fig. 4b analogue: the kinetic temperature of the polymer under the thermostat stays at T."""
    s = H.lj_cluster(32)
    o, R = _tiny_path(oracle, s, 4)
    T = 120.0
    V = np.zeros_like(R)
    Ra, Va, _ = oracle.step_langevin(o, R, V, 0.0005, 300, 100.0, T, seed=3, geom=0, brute=True)     # equilibrate
    Rb, Vb, en = oracle.step_langevin(o, Ra, Va, 0.0005, 1500, 100.0, T, seed=3, step0=300, geom=0, brute=True)
    dof = R.size
    t_kin = 2.0 * en[:, 1] / (dof * oracle.KB)
    assert abs(t_kin.mean() / T - 1.0) < 0.04


# ---------------------------------------------------------------- P15 MoP bias (NEXT-3)
def test_P15_bias_closed_forms_and_gradient(oracle):
    """(i) two single-atom groups: s is their distance, S_e2e the difference between last and first bead, one hill
    at S gives V = w and zero force; (ii) dV/dR against central differences of V; (iii) the bias force on each end
    bead sums to zero (translation invariance) and vanishes on interior beads."""
    s = H.lj_cluster(32, masses=np.linspace(5, 40, 32))
    o = oracle.OracleSystem(s)
    rng = np.random.default_rng(6)
    R = s.R1[None] + rng.normal(0, 0.02, (4, 32, 3))
    box = np.asarray(s.box, float)
    mi = lambda d: d - box * np.round(d / box)            # minimum image of the COM difference
    d1 = np.linalg.norm(mi(R[0, 3] - R[0, 17]))
    dN = np.linalg.norm(mi(R[3, 3] - R[3, 17]))
    v, g, (S, s1, sN) = oracle.bias(o, R, [3], [17], [dN - d1], 0.05, 2.5)
    assert s1 == pytest.approx(d1, rel=1e-14) and sN == pytest.approx(dN, rel=1e-14) and S == pytest.approx(dN - d1, abs=1e-14)
    assert v == pytest.approx(2.5, rel=1e-12) and np.abs(g).max() < 1e-9
    v, g, (S, s1, sN) = oracle.bias(o, R, [3], [17], [S + 0.03], 0.05, 2.5)
    assert v == pytest.approx(2.5 * np.exp(-0.5 * 0.36), rel=1e-10)
    ga, gb = np.arange(0, 9), np.arange(20, 32)
    hills = [0.01, -0.04, 0.08]
    v, g, (S, s1, sN) = oracle.bias(o, R, ga, gb, hills, 0.05, 2.5)
    M = s.mass.astype(float)
    com = lambda X, idx: (M[idx, None] * X[idx]).sum(0) / M[idx].sum()
    assert s1 == pytest.approx(np.linalg.norm(mi(com(R[0], ga) - com(R[0], gb))), rel=1e-13)
    assert np.abs(g[1:3]).max() == 0.0 and np.abs(g[0]).max() > 0 and np.abs(g[3]).max() > 0
    assert np.abs(g[0].sum(0)).max() < 1e-12 * np.abs(g[0]).max() and np.abs(g[3].sum(0)).max() < 1e-12 * np.abs(g[3]).max()
    e = 1e-6
    for n, i, a in ((0, 2, 0), (0, 25, 2), (3, 7, 1), (3, 30, 0), (3, 15, 1)):
        Rp, Rm = R.copy(), R.copy()
        Rp[n, i, a] += e
        Rm[n, i, a] -= e
        fd = (oracle.bias(o, Rp, ga, gb, hills, 0.05, 2.5)[0] - oracle.bias(o, Rm, ga, gb, hills, 0.05, 2.5)[0]) / (2 * e)
        assert fd == pytest.approx(g[n, i, a], rel=1e-6, abs=1e-9)
    # periodic images of a whole group do not change s
    R2 = R.copy()
    R2[:, gb] += np.asarray(s.box, float) * [1, -2, 0]
    assert oracle.bias(o, R2, ga, gb, hills, 0.05, 2.5)[0] == pytest.approx(v, rel=1e-10)


# ---------------------------------------------------------------- P13 + G8 neighbour sets
@pytest.mark.parametrize("mk", ["c1", "c2", "tiny", "edge"])
def test_P13_cell_list_equals_brute_force(oracle, mk):
    if mk == "c1":
        s = W.config1()
    elif mk == "c2":
        s = W.config2()
    elif mk == "tiny":
        s = H.tiny_chain()
    else:
        s = H.lj_cluster(64, L=2.0001, r_cut=1.0)       # box barely above 2 r_c
    o = oracle.OracleSystem(s)
    rng = np.random.default_rng(1)
    X = s.R1 + rng.integers(-2, 3, (s.n_atoms, 1)) * np.asarray(s.box, float)   # unwrapped images
    for geom in (0, 1):
        pb = oracle.pairs(o, X, geom=geom, brute=True)
        pc = oracle.pairs(o, X, geom=geom, brute=False)
        assert pb.shape == pc.shape and (pb == pc).all()
    # FP32-contract set differs from the FP64 set only by pairs at the cutoff / the float rounding of X
    p0 = oracle.pairs(o, s.R1.astype(np.float32).astype(np.float64), geom=0)
    p1 = oracle.pairs(o, s.R1, geom=1)
    a = set(map(tuple, p0.tolist()))
    b = set(map(tuple, p1.tolist()))
    assert len(a ^ b) <= max(2, len(a) // 100000)
    # no excluded pair is ever listed
    ex = {(i, int(j)) for i in range(s.n_atoms) for j in s.excl_list[s.excl_start[i]:s.excl_start[i + 1]]}
    assert not (b & ex)


def test_G8_predicate_does_not_depend_on_the_roles_of_the_two_atoms(oracle):
    """G8: membership is a property of the unordered pair.  The two atoms below (found on config 4, bead 7, across the z
    face of the 10.5 x 10.5 x 13.5 box, r_c = 1.2) sit 2 ulp from r_c^2: a predicate that shifts 'atom i' first
    (xs_i = x_i - k L, d = xs_i - x_j) classifies them differently depending on which atom it calls i -- a kernel is
    free to choose -- while d = (x_i - x_j) - k L negates exactly under the swap.  Also on random pairs near r_c."""
    box = [10.5, 10.5, 13.5]
    A = np.float32([3.9472785, 5.670694, 13.426104])
    Bm = np.float32([4.2180476, 4.894643, 0.80042])

    def n_pairs(X):
        s = H.make_system("two", box, np.asarray(X, np.float64), [12.0, 12.0], [0.0, 0.0], [0, 0], [0.3], [0.5], r_cut=1.2)
        o = oracle.OracleSystem(s)
        a = len(oracle.pairs(o, np.asarray(X, np.float64), geom=1, brute=True))
        assert a == len(oracle.pairs(o, np.asarray(X, np.float64), geom=1, brute=False))
        return a

    assert n_pairs([A, Bm]) == n_pairs([Bm, A])
    # the value itself, by hand in numpy float32: d = (x_i - x_j) - k L with k = (0, 0, 1)
    d = (A - Bm).astype(np.float32) - np.float32([0.0, 0.0, 13.5])
    r2 = np.float32(np.float64(d[2]) * d[2] + np.float64(np.float32(np.float64(d[1]) * d[1] + np.float64(np.float32(d[0] * d[0])))))
    assert n_pairs([A, Bm]) == int(r2 < np.float32(1.2) * np.float32(1.2))
    rng = np.random.default_rng(8)
    for _ in range(200):
        P = rng.uniform(0, 1, 3) * box
        u = rng.normal(0, 1, 3)
        Qp = P + u / np.linalg.norm(u) * (1.2 + rng.uniform(-3e-7, 3e-7))
        X = np.float32([P, Qp])
        assert n_pairs(X) == n_pairs(X[::-1])


def test_G8_wrap_cells_and_stable_sort(oracle):
    s = W.config2()
    rng = np.random.default_rng(2)
    X = (s.R1 + rng.integers(-3, 4, (s.n_atoms, 3)) * np.asarray(s.box, float)).astype(np.float32)
    xw = oracle.wrap(X, s.box)
    L = s.box.astype(np.float32)
    assert (xw >= 0).all() and (xw < L).all()
    d = (xw.astype(float) - X.astype(float)) / L
    assert np.abs(d - np.round(d)).max() < 1e-6           # same point modulo the box
    dims = oracle.grid_dims(s.n_atoms, s.box, 8, 0.1)
    assert dims[0] >= 1 and dims[2] == int(np.floor(float(L[2]) / np.float32(0.1)))
    cell = oracle.cell_ids(xw, s.box, dims)
    assert cell.min() >= 0 and cell.max() < dims[0] * dims[1] * dims[2]
    cz = cell % dims[2]
    assert np.abs((cz + 0.5) * (L[2] / dims[2]) - xw[:, 2]).max() <= 0.5 * L[2] / dims[2] * 1.001
    perm = oracle.stable_sort_by_cell(cell, dims[0] * dims[1] * dims[2])
    assert sorted(perm.tolist()) == list(range(s.n_atoms))
    key = cell[perm].astype(np.int64) * s.n_atoms + perm
    assert (np.diff(key) > 0).all()                        # sorted by cell, ties by ascending index


def test_geom1_matches_geom0_physics(oracle):
    """The FP32-contract mode does its physics in FP64: same V_eff/grad as pure FP64 on float inputs."""
    s = H.tiny_chain()
    o, R = _tiny_path(oracle, s, 4)
    R32 = R.astype(np.float32).astype(np.float64)
    assert H.pairs_near_cutoff(s, R32[0], 1e-5) == 0
    v0, G0 = oracle.veff_grad(o, R32, geom=0, brute=True)
    v1, G1 = oracle.veff_grad(o, R32, geom=1, brute=False)
    assert v1 == pytest.approx(v0, rel=1e-12)
    assert H.rms_rel(G1, G0) < 1e-10


# ---------------------------------------------------------------- G8 edge branches (the cases bit-exact neighbour sets turn on)
def _wrap_by_hand(x, L):
    """The G8 wrap written out in numpy float32 scalars (every operation rounds to single precision).
    Returns (xw, took_negative_fixup, took_upper_fixup)."""
    x, L = np.float32(x), np.float32(L)
    invL = np.float32(1.0) / L
    t = x * invL
    f = np.floor(t)
    p = L * f
    xw = x - p
    lo = bool(xw < np.float32(0.0))
    if lo:
        xw = xw + L
    hi = bool(xw >= L)
    if hi:
        xw = xw - L
    return np.float32(xw), lo, hi


def test_G8_wrap_edge_inputs_stay_in_the_box(oracle):
    """What the mathematics fixes for a periodic box: the wrapped coordinate lies in [0, L) -- L itself
    excluded, or the cell index below would reach n -- and is the same point modulo L.  The inputs sit on and next to the
    box faces and their periodic copies, where x * (1/L) rounds onto an integer although x does not, so that
    x - L floor(x / L) comes out negative, or equal to L: both fix-ups of the G8 sequence are needed, and the test checks
    that it has inputs that take each of them (it cannot go vacuous)."""
    took_lo = took_hi = 0
    for L in (2.88, 3.10, 10.5, 13.5):
        Lf = np.float32(L)
        xs = [np.float32(-1e-9), np.float32(-0.0), Lf, np.nextafter(Lf, np.float32(0)), np.nextafter(Lf, np.float32(np.inf)),
              np.float32(1e6) * Lf, np.float32(-1e6) * Lf]
        for k in range(-3, 4):
            e = np.float32(k) * Lf
            x = e
            for _ in range(3):
                x = np.nextafter(x, np.float32(-np.inf))
                xs.append(x)
            x = e
            for _ in range(3):
                x = np.nextafter(x, np.float32(np.inf))
                xs.append(x)
            xs.append(e)
        X = np.zeros((len(xs), 3), np.float32)
        X[:, 0] = xs
        xw = oracle.wrap(X, [L, 5.0, 5.0])[:, 0]
        assert (xw >= 0).all() and (xw < Lf).all(), (L, X[~((xw >= 0) & (xw < Lf)), 0])
        for x, w in zip(xs, xw):
            hand, lo, hi = _wrap_by_hand(x, L)
            took_lo += lo
            took_hi += hi
            assert w.tobytes() == hand.tobytes() or (w == 0 and hand == 0), (L, x, w, hand)
            # the same point modulo L: distance to the nearest periodic copy of x, within the rounding of |x| / L turns
            d = (float(w) - float(x)) / float(Lf)
            assert abs(d - round(d)) * float(Lf) <= 4 * np.spacing(np.float32(max(abs(float(x)), float(Lf)))), (L, x, w)
    assert took_lo >= 1 and took_hi >= 1, (took_lo, took_hi)


def test_G8_cell_index_of_the_last_representable_coordinate(oracle):
    """xw = nextafter(L, 0) is inside the box, so its cell is the last one, n - 1; but xw * (n / L) can round up to n in
    FP32, and the index n would address the first bin of the next column.  The test looks for such (L, n) among the box
    lengths and bin counts of the configs, requires that it found some, and checks the oracle's cell ids there."""
    found = 0
    for L in (2.88, 3.10, 10.5, 13.5, 6.2):
        Lf = np.float32(L)
        xw = np.nextafter(Lf, np.float32(0))
        for n in list(range(1, 200)) + [256, 512, 1024, 2048, 4096]:
            sc = np.float32(n) * (np.float32(1.0) / Lf)
            if int(xw * sc) < n:
                continue
            found += 1
            X = np.array([[0.5, 0.5, xw], [xw, 0.5, 0.5]], np.float32)
            dims = [n if n <= 1024 else 1, 1, n]
            box = [L if n <= 1024 else 5.0, 5.0, L]
            cell = oracle.cell_ids(X, box, dims)
            cx0 = int(np.float32(0.5) * (np.float32(dims[0]) * (np.float32(1.0) / np.float32(box[0]))))
            assert cell[0] == (cx0 * 1 + 0) * n + (n - 1), (L, n, cell)
            if n <= 1024:
                cz1 = int(np.float32(0.5) * sc)
                assert cell[1] == ((n - 1) * 1 + 0) * n + cz1, (L, n, cell)
    assert found >= 3, found


@pytest.mark.parametrize("rc", [1.0, 1.5])
def test_G8_strict_inequality_at_exactly_r_cut(oracle, rc):
    """The cutoff test is r2 < r_c^2, strictly (reading G8).  With r_c = 1 or 1.5 and separations that are exact
    binary fractions, r2 == r_c^2 can be hit exactly in FP32: that pair is NOT listed, the pair one ulp closer is, the pair
    one ulp farther is not -- along each axis, in both atom orders, inside the box (k = 0) and across a face (k = +-1)."""
    L = 4.0                                     # exact in FP32, >= 2 r_c

    def n_pairs(xi, xj, axis):
        X = np.full((2, 3), 0.5, np.float32)
        X[0, axis], X[1, axis] = xi, xj
        s = H.make_system("two", [L] * 3, X.astype(np.float64), [12.0, 12.0], [0.0, 0.0], [0, 0], [0.3], [0.5], r_cut=rc)
        o = oracle.OracleSystem(s)
        out = []
        for Xo in (X, X[::-1].copy()):
            a = len(oracle.pairs(o, Xo.astype(np.float64), geom=1, brute=True))
            assert a == len(oracle.pairs(o, Xo.astype(np.float64), geom=1, brute=False))
            out.append(a)
        assert out[0] == out[1]
        return out[0]

    f = np.float32
    for axis in range(3):
        # inside the box: x_i = 1, x_j = 1 + r_c (exact)
        xi, xj = f(1.0), f(1.0 + rc)
        assert f(xj - xi) * f(xj - xi) == f(rc) * f(rc)               # the premise: r2 == r_c^2 exactly
        assert n_pairs(xi, xj, axis) == 0
        assert n_pairs(xi, np.nextafter(xj, f(0)), axis) == 1
        assert n_pairs(xi, np.nextafter(xj, f(9)), axis) == 0
        # across the face: x_i = 0.25, x_j = 0.25 + L - r_c; d0 = -(L - r_c), k = -1, d = d0 + L = r_c exactly
        xi, xj = f(0.25), f(0.25 + L - rc)
        assert f(f(xi - xj) + f(L)) == f(rc)
        assert n_pairs(xi, xj, axis) == 0
        assert n_pairs(xi, np.nextafter(xj, f(9)), axis) == 1         # farther from x_i directly = closer through the face
        assert n_pairs(xi, np.nextafter(xj, f(0)), axis) == 0


def test_G8_the_two_operand_orders_differ_only_within_ulps_of_r_cut(oracle):
    """Reading G8 forms d = (x_i - x_j) - k L; the list builder's superset test still shifts atom i first,
    d' = (x_i - k L) - x_j.  On the whole of config 2 (4.5 million atom pairs, by hand in numpy float32) the two
    memberships differ on at most a handful of pairs, all within a few ulp of r_c^2 -- far inside the 1e-4 relative
    margin the builder adds to r_list^2 -- and the oracle's FP32-contract pair list is the first of the two."""
    s = W.config2()
    o = oracle.OracleSystem(s)
    X = s.R1.astype(np.float32)
    xw = oracle.wrap(X, s.box)
    Lf = np.asarray(s.box, np.float32)
    iu, ju = np.triu_indices(s.n_atoms, 1)
    r2 = {}
    for order in ("pair", "shift_i"):
        acc = None
        for a in (2, 1, 0):                                            # fmaf(dz,dz, fmaf(dy,dy, dx*dx)) from the inside out
            xi, xj = xw[iu, a], xw[ju, a]
            d0 = xi - xj
            k = np.rint(d0 * (np.float32(1.0) / Lf[a]))
            kL = (k * Lf[a]).astype(np.float32)                        # k in {-1,0,1}: exact
            d = (d0 - kL) if order == "pair" else ((xi - kL) - xj)
            r2[(order, a)] = d
        dx, dy, dz = (r2[(order, a)].astype(np.float64) for a in (0, 1, 2))
        inner = (dx.astype(np.float32) * dx.astype(np.float32)).astype(np.float32)
        mid = (dy * dy + inner.astype(np.float64)).astype(np.float32)
        r2[order] = (dz * dz + mid.astype(np.float64)).astype(np.float32)
    rc2 = np.float32(s.r_cut) * np.float32(s.r_cut)
    inA, inB = r2["pair"] < rc2, r2["shift_i"] < rc2
    diff = np.nonzero(inA != inB)[0]
    assert len(diff) <= 8, len(diff)
    for t in diff:
        assert abs(float(r2["pair"][t]) - float(rc2)) <= 4 * np.spacing(rc2)
        assert abs(float(r2["shift_i"][t]) - float(rc2)) <= 4 * np.spacing(rc2)
    assert np.abs(r2["pair"].astype(np.float64) - r2["shift_i"]).max() <= 4 * np.spacing(np.float32(Lf.max() ** 2 / 2))
    # the oracle's list = order "pair" minus the exclusions
    ex = {(i, int(j)) for i in range(s.n_atoms) for j in s.excl_list[s.excl_start[i]:s.excl_start[i + 1]]}
    mine = {(int(i), int(j)) for i, j in zip(iu[inA], ju[inA])} - ex
    ref = {(int(i), int(j)) for i, j in oracle.pairs(o, X.astype(np.float64), geom=1, brute=False)}
    assert mine == ref, (len(mine), len(ref), len(mine ^ ref))
