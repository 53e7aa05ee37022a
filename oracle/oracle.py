"""ctypes loader for the FP64 CPU oracle (oracle/mop_oracle.c).

TEST INFRASTRUCTURE, NOT THE PRODUCT: only tests/, __graft_entry__.smoke() and
bench.py's cpu_baseline / --impl reference legs may import this module.  It
shares no code with the CUDA path (paper_2501_11962_b200/csrc) and never
imports the binding.

Every function takes a `system` object with the plain attributes the input
generators produce (n_atoms, box, r_cut, eps_rf, lj_shift, dt_path, nu, mass,
charge, type, n_types, c6, c12, bond_ij, bond_b0_kb, angle_ijk, angle_t0_kt,
excl_start, excl_list) and numpy arrays; see mop_oracle.c for the passage of
PAPER.md each step follows.
"""
import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "mop_oracle.c")
_LIB = os.path.join(_HERE, "liboracle.so")
_lib = None


def build(force=False):
    """Compile oracle/mop_oracle.c with gcc (FP contraction off, OpenMP on)."""
    if force or (not os.path.exists(_LIB)) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        cmd = ["gcc", "-O2", "-fopenmp", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC",
               "-o", _LIB, _SRC, "-lm"]
        subprocess.run(cmd, check=True)
    return _LIB


class _Sys(C.Structure):
    _fields_ = [
        ("n_atoms", C.c_int), ("box", C.c_float * 3), ("r_cut", C.c_float), ("eps_rf", C.c_float),
        ("lj_shift", C.c_int), ("dt_path", C.c_double), ("nu", C.c_double),
        ("mass", C.c_void_p), ("charge", C.c_void_p), ("type", C.c_void_p), ("n_types", C.c_int),
        ("c6", C.c_void_p), ("c12", C.c_void_p),
        ("n_bonds", C.c_int), ("bond_ij", C.c_void_p), ("bond_b0_kb", C.c_void_p),
        ("n_angles", C.c_int), ("angle_ijk", C.c_void_p), ("angle_t0_kt", C.c_void_p),
        ("excl_start", C.c_void_p), ("excl_list", C.c_void_p),
    ]


def _load():
    global _lib
    if _lib is None:
        build()
        L = C.CDLL(_LIB)
        L.orc_pairs.restype = C.c_long
        L.orc_bead.restype = C.c_long
        L.orc_veff_grad.restype = C.c_double
        L.orc_veff_grad_fd.restype = C.c_double
        L.orc_noise_normal.restype = C.c_double
        L.orc_bias.restype = C.c_double
        L.orc_cv_com_distance.restype = C.c_double
        L.orc_noise_bits.restype = C.c_uint64
        L.orc_num_threads.restype = C.c_int
        _lib = L
    return _lib


def _p(a):
    return None if a is None else a.ctypes.data_as(C.c_void_p)


class OracleSystem:
    """Holds contiguous copies of a system's arrays and the C struct pointing at them."""

    def __init__(self, system):
        s = system
        self.Q = int(s.n_atoms)
        self._keep = {}

        def arr(name, dtype, shape=None):
            a = np.ascontiguousarray(np.asarray(getattr(s, name), dtype=dtype))
            if shape is not None:
                a = a.reshape(shape)
            self._keep[name] = a
            return a

        st = _Sys()
        st.n_atoms = self.Q
        for d in range(3):
            st.box[d] = float(np.float32(s.box[d]))
        st.r_cut = float(np.float32(s.r_cut))
        st.eps_rf = float(np.float32(s.eps_rf))
        st.lj_shift = int(s.lj_shift)
        st.dt_path = float(s.dt_path)
        st.nu = float(s.nu)
        st.mass = _p(arr("mass", np.float32))
        st.charge = _p(arr("charge", np.float32))
        st.type = _p(arr("type", np.int32))
        st.n_types = int(s.n_types)
        st.c6 = _p(arr("c6", np.float32))
        st.c12 = _p(arr("c12", np.float32))
        b = arr("bond_ij", np.int32, (-1, 2))
        st.n_bonds = b.shape[0]
        st.bond_ij = _p(b)
        st.bond_b0_kb = _p(arr("bond_b0_kb", np.float32, (-1, 2)))
        a = arr("angle_ijk", np.int32, (-1, 3))
        st.n_angles = a.shape[0]
        st.angle_ijk = _p(a)
        st.angle_t0_kt = _p(arr("angle_t0_kt", np.float32, (-1, 2)))
        st.excl_start = _p(arr("excl_start", np.int32))
        st.excl_list = _p(arr("excl_list", np.int32))
        self.box = np.array([st.box[0], st.box[1], st.box[2]], dtype=np.float32)
        self.struct = st

    @property
    def ref(self):
        return C.byref(self.struct)


def num_threads():
    return int(_load().orc_num_threads())


def wrap(R32, box):
    """G8 FP32 wrap of one bead: R32 [Q][3] float32 -> xw [Q][3] float32."""
    L = _load()
    R32 = np.ascontiguousarray(R32, dtype=np.float32)
    out = np.empty_like(R32)
    b = (C.c_float * 3)(*[float(np.float32(x)) for x in box])
    L.orc_wrap(_p(R32), C.c_int(R32.shape[0]), b, _p(out))
    return out


def grid_dims(Q, box, cluster, bin_z):
    L = _load()
    b = (C.c_float * 3)(*[float(np.float32(x)) for x in box])
    d = (C.c_int * 3)()
    L.orc_grid_dims(C.c_int(Q), b, C.c_int(cluster), C.c_float(bin_z), d)
    return [d[0], d[1], d[2]]


def cell_ids(xw, box, dims):
    L = _load()
    xw = np.ascontiguousarray(xw, dtype=np.float32)
    b = (C.c_float * 3)(*[float(np.float32(x)) for x in box])
    d = (C.c_int * 3)(*dims)
    out = np.empty(xw.shape[0], dtype=np.int32)
    L.orc_cell_ids(_p(xw), C.c_int(xw.shape[0]), b, d, _p(out))
    return out


def stable_sort_by_cell(cell, ncell):
    L = _load()
    cell = np.ascontiguousarray(cell, dtype=np.int32)
    perm = np.empty(cell.shape[0], dtype=np.int32)
    L.orc_stable_sort_by_cell(_p(cell), C.c_int(cell.shape[0]), C.c_int(ncell), _p(perm))
    return perm


def pairs(osys, R, geom=1, brute=False):
    """In-range, non-excluded pairs (i<j) of one bead, sorted lexicographically."""
    L = _load()
    R = np.ascontiguousarray(R, dtype=np.float64).reshape(osys.Q, 3)
    n = L.orc_pairs(osys.ref, _p(R), C.c_int(geom), C.c_int(int(brute)), None, C.c_long(0))
    out = np.empty((n, 2), dtype=np.int32)
    n2 = L.orc_pairs(osys.ref, _p(R), C.c_int(geom), C.c_int(int(brute)), _p(out), C.c_long(n))
    assert n2 == n
    order = np.lexsort((out[:, 1], out[:, 0]))
    return out[order]


def bead(osys, R, geom=0, brute=False, s=None, want_force=True):
    """Force, energy terms and optional H s of one bead.

    Returns dict(F, Hs, U=(lj, coul, bond, angle), npairs)."""
    L = _load()
    R = np.ascontiguousarray(R, dtype=np.float64).reshape(osys.Q, 3)
    F = np.zeros((osys.Q, 3)) if want_force else None
    Hs = None
    if s is not None:
        s = np.ascontiguousarray(s, dtype=np.float64).reshape(osys.Q, 3)
        Hs = np.zeros((osys.Q, 3))
    u = np.zeros(4)
    n = L.orc_bead(osys.ref, _p(R), C.c_int(geom), C.c_int(int(brute)), _p(F), _p(s), _p(Hs), _p(u))
    return dict(F=F, Hs=Hs, U=u, npairs=int(n))


def veff_grad(osys, R, geom=0, brute=False, want_parts=False):
    """V_eff (eq. 3) and dV_eff/dR for a path R [N][Q][3].

    Returns (veff, grad) or, with want_parts, (veff, grad, dict(F, eta, Heta, U1, E_spring, npairs))."""
    L = _load()
    R = np.ascontiguousarray(R, dtype=np.float64)
    N = R.shape[0]
    assert R.shape[1:] == (osys.Q, 3)
    grad = np.zeros_like(R)
    nf = max(N - 1, 1)
    F = np.zeros((nf, osys.Q, 3))
    eta = np.zeros((nf, osys.Q, 3))
    Heta = np.zeros((nf, osys.Q, 3))
    parts = np.zeros(4)
    v = L.orc_veff_grad(osys.ref, C.c_int(N), _p(R), C.c_int(geom), C.c_int(int(brute)), _p(grad),
                        _p(F), _p(eta), _p(Heta), _p(parts))
    if want_parts:
        return float(v), grad, dict(F=F, eta=eta, Heta=Heta, U1=parts[0], E_spring=parts[1],
                                    npairs=int(parts[2]))
    return float(v), grad


def veff_grad_fd(osys, R, eps, geom=0, brute=False):
    """V_eff and -F_eff of eqs (5),(6),(7) as printed: Hessian term by the paper's finite difference
    [F(R + eps eta) - F(R - eps eta)]/(4 eps).  Returns (veff, grad)."""
    L = _load()
    R = np.ascontiguousarray(R, dtype=np.float64)
    N = R.shape[0]
    assert R.shape[1:] == (osys.Q, 3)
    grad = np.zeros_like(R)
    v = L.orc_veff_grad_fd(osys.ref, C.c_int(N), _p(R), C.c_double(eps), C.c_int(geom), C.c_int(int(brute)), _p(grad))
    return float(v), grad


def step(osys, R, V, dt, n_steps, geom=0, brute=False):
    """Velocity Verlet (eq. 4). Returns (R, V, energies[n_steps+1][3] = V_eff, E_kin, total)."""
    L = _load()
    R = np.array(R, dtype=np.float64, order="C")
    V = np.array(V, dtype=np.float64, order="C")
    N = R.shape[0]
    en = np.zeros((n_steps + 1, 3))
    L.orc_step(osys.ref, C.c_int(N), _p(R), _p(V), C.c_double(dt), C.c_int(n_steps), C.c_int(geom),
               C.c_int(int(brute)), _p(en))
    return R, V, en


KB = 0.0083144626   # kJ mol^-1 K^-1


def noise_bits(seed, step, idx):
    """The 64 random bits of the counter (seed, step, idx) of the thermostat's generator."""
    return int(_load().orc_noise_bits(C.c_uint64(seed), C.c_uint64(step), C.c_uint64(idx)))


def noise_normal(seed, step, idx):
    return float(_load().orc_noise_normal(C.c_uint64(seed), C.c_uint64(step), C.c_uint64(idx)))


def step_langevin(osys, R, V, dt, n_steps, gamma, temperature, seed=0, step0=0, geom=0, brute=False):
    """Velocity Verlet + exact Ornstein-Uhlenbeck velocity update (reading G19).  Returns (R, V, energies)."""
    L = _load()
    R = np.array(R, dtype=np.float64, order="C", copy=True)
    V = np.array(V, dtype=np.float64, order="C", copy=True)
    N = R.shape[0]
    en = np.zeros((n_steps + 1, 3))
    L.orc_step_langevin(osys.ref, C.c_int(N), _p(R), _p(V), C.c_double(dt), C.c_int(n_steps), C.c_double(gamma),
                        C.c_double(KB * temperature), C.c_uint64(seed), C.c_uint64(step0), C.c_int(geom),
                        C.c_int(int(brute)), _p(en))
    return R, V, en


def bias(osys, R, group_a, group_b, hills, sigma, height):
    """MoP bias V(S_e2e) of a path R [N][Q][3].  Returns (V, dV/dR [N][Q][3], (S, s1, sN))."""
    L = _load()
    R = np.ascontiguousarray(R, dtype=np.float64)
    ga = np.ascontiguousarray(group_a, dtype=np.int32)
    gb = np.ascontiguousarray(group_b, dtype=np.int32)
    h = np.ascontiguousarray(hills, dtype=np.float64).reshape(-1)
    g = np.zeros_like(R)
    out = np.zeros(3)
    v = L.orc_bias(osys.ref, C.c_int(R.shape[0]), _p(R), _p(ga), C.c_int(len(ga)), _p(gb), C.c_int(len(gb)),
                   _p(h) if len(h) else None, C.c_int(len(h)), C.c_double(sigma), C.c_double(height), _p(g), _p(out))
    return float(v), g, tuple(out)
