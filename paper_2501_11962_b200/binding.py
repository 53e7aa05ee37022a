"""Thin ctypes binding of libmop_b200.so (include/mop.h): argument marshalling only.

Every step of the hot path runs in the CUDA kernels behind the C-ABI; torch is used for device
memory and the stream handle.  There is no CPU fallback: if the library is missing or cannot be
loaded this module raises, and a context cannot be created without a CUDA device.
Names follow the C-ABI: mop_create / mop_set_topology / mop_eval_veff_grad / mop_step / mop_destroy.
"""
import ctypes as C
import os

import numpy as np

from . import build as _build

MOP_OK = 0
STATUS = {0: "MOP_OK", 1: "MOP_ERR_INVALID_ARG", 2: "MOP_ERR_NO_TOPOLOGY", 3: "MOP_ERR_BOX_TOO_SMALL",
          4: "MOP_ERR_OOM", 5: "MOP_ERR_CUDA", 6: "MOP_ERR_NONFINITE"}
EXPORTS = ["mop_create", "mop_set_topology", "mop_eval_veff_grad", "mop_step", "mop_destroy", "mop_last_error",
           "mop_get_stats", "mop_debug_get", "mop_debug_pairs", "mop_force_hvp", "mop_eval_veff_grad_host",
           "mop_set_timing", "mop_get_timing", "mop_eval_veff_grad_fd", "mop_step_continue",
           "mop_step_langevin_continue", "mop_debug_count_inrange", "mop_create_block", "mop_block_pass1",
           "mop_block_pass2", "mop_block_assemble", "mop_block_integrate", "mop_debug_set_list_capacity",
           "mop_step_langevin", "mop_debug_noise_bits", "mop_set_bias", "mop_add_hill", "mop_get_bias",
           "mop_eta_spring_noalloc", "mop_block_thermostat"]
MOP_NOALLOC_MAX_ATOM_BEADS = 33554432   # include/mop.h


class MopError(RuntimeError):
    def __init__(self, status, msg):
        super().__init__("%s: %s" % (STATUS.get(status, status), msg))
        self.status = status


class mop_params(C.Structure):
    _fields_ = [("n_atoms", C.c_int), ("n_beads", C.c_int), ("box", C.c_float * 3), ("r_cut", C.c_float),
                ("r_buf", C.c_float), ("eps_rf", C.c_float), ("lj_shift", C.c_int), ("dt_path", C.c_double),
                ("nu", C.c_double), ("device", C.c_int), ("stream", C.c_void_p)]


class mop_topology(C.Structure):
    _fields_ = [("mass", C.c_void_p), ("charge", C.c_void_p), ("type", C.c_void_p), ("n_types", C.c_int),
                ("c6", C.c_void_p), ("c12", C.c_void_p), ("n_bonds", C.c_int), ("bond_ij", C.c_void_p),
                ("bond_b0_kb", C.c_void_p), ("n_angles", C.c_int), ("angle_ijk", C.c_void_p),
                ("angle_t0_kt", C.c_void_p), ("excl_start", C.c_void_p), ("excl_list", C.c_void_p)]


_lib = None


def lib_path():
    return _build.LIB


def load(build_if_missing=True, path=None):
    """Loads the C-ABI library (building it with nvcc when it is missing or stale).  Raises if unavailable.
    path: load that build of the library instead (first call of the process only; the -DMOP_CHECK build of
    tests/sanitizer_target.py --checked)."""
    global _lib
    if _lib is not None:
        if path is not None:
            raise RuntimeError("the library is already loaded")
        return _lib
    if path is None:
        if build_if_missing:
            _build.build()
        path = _build.LIB
    if not os.path.exists(path):
        raise RuntimeError("%s is not built (run python -m paper_2501_11962_b200.build); there is no CPU fallback"
                           % os.path.basename(path))
    L = C.CDLL(path)
    L.mop_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(mop_params)]
    L.mop_set_topology.argtypes = [C.c_void_p, C.POINTER(mop_topology)]
    L.mop_eval_veff_grad.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]
    L.mop_step.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_int]
    L.mop_destroy.argtypes = [C.c_void_p]
    L.mop_destroy.restype = None
    L.mop_last_error.argtypes = [C.c_void_p]
    L.mop_last_error.restype = C.c_char_p
    L.mop_get_stats.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
    L.mop_debug_get.argtypes = [C.c_void_p, C.c_char_p, C.c_void_p, C.c_size_t]
    L.mop_debug_pairs.argtypes = [C.c_void_p, C.c_int, C.c_void_p, C.c_longlong, C.POINTER(C.c_longlong)]
    L.mop_force_hvp.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.mop_eval_veff_grad_host.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]
    L.mop_set_timing.argtypes = [C.c_void_p, C.c_int]
    L.mop_get_timing.argtypes = [C.c_void_p, C.POINTER(C.c_double)]
    L.mop_step_continue.argtypes = L.mop_step.argtypes
    L.mop_step_continue.restype = C.c_int
    L.mop_debug_count_inrange.argtypes = [C.c_void_p, C.c_int, C.POINTER(C.c_longlong), C.POINTER(C.c_ulonglong)]
    L.mop_debug_count_inrange.restype = C.c_int
    L.mop_debug_set_list_capacity.argtypes = [C.c_void_p, C.c_uint, C.c_uint, C.c_uint]
    L.mop_debug_set_list_capacity.restype = C.c_int
    L.mop_create_block.argtypes = [C.POINTER(C.c_void_p), C.POINTER(mop_params), C.c_int, C.c_int]
    L.mop_create_block.restype = C.c_int
    L.mop_block_pass1.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p]
    L.mop_block_pass1.restype = C.c_int
    L.mop_block_pass2.argtypes = [C.c_void_p, C.c_void_p]
    L.mop_block_pass2.restype = C.c_int
    L.mop_block_assemble.argtypes = [C.c_void_p, C.c_void_p, C.POINTER(C.c_double), C.c_void_p]
    L.mop_block_assemble.restype = C.c_int
    L.mop_block_integrate.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_int]
    L.mop_block_integrate.restype = C.c_int
    L.mop_block_thermostat.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.c_double, C.c_double, C.c_uint64, C.c_uint64]
    L.mop_block_thermostat.restype = C.c_int
    L.mop_eval_veff_grad_fd.argtypes = [C.c_void_p, C.c_void_p, C.c_double, C.POINTER(C.c_double), C.c_void_p]
    L.mop_eval_veff_grad_fd.restype = C.c_int
    L.mop_step_langevin.argtypes = [C.c_void_p, C.c_void_p, C.c_void_p, C.c_double, C.c_int, C.c_double, C.c_double,
                                    C.c_uint64, C.c_uint64]
    L.mop_step_langevin.restype = C.c_int
    L.mop_step_langevin_continue.argtypes = L.mop_step_langevin.argtypes
    L.mop_step_langevin_continue.restype = C.c_int
    L.mop_debug_noise_bits.argtypes = [C.c_void_p, C.c_uint64, C.c_uint64, C.c_int, C.c_void_p]
    L.mop_debug_noise_bits.restype = C.c_int
    L.mop_set_bias.argtypes = [C.c_void_p, C.c_void_p, C.c_int, C.c_void_p, C.c_int, C.c_double, C.c_double, C.c_int]
    L.mop_set_bias.restype = C.c_int
    L.mop_add_hill.argtypes = [C.c_void_p, C.c_double]
    L.mop_add_hill.restype = C.c_int
    L.mop_get_bias.argtypes = [C.c_void_p, C.POINTER(C.c_double), C.c_void_p, C.c_int, C.POINTER(C.c_int)]
    L.mop_get_bias.restype = C.c_int
    L.mop_eta_spring_noalloc.argtypes = [C.c_int, C.c_void_p, C.c_int, C.c_int, C.c_double, C.c_double, C.c_void_p,
                                         C.c_void_p, C.c_void_p, C.c_void_p, C.c_void_p, C.c_char_p, C.c_size_t]
    L.mop_eta_spring_noalloc.restype = C.c_int
    for n in ("mop_create", "mop_set_topology", "mop_eval_veff_grad", "mop_step", "mop_get_stats", "mop_debug_get",
              "mop_debug_pairs", "mop_force_hvp", "mop_eval_veff_grad_host", "mop_set_timing", "mop_get_timing"):
        getattr(L, n).restype = C.c_int
    _lib = L
    return L


def _ptr(t):
    return None if t is None else C.c_void_p(t.data_ptr())


def mop_eta_spring_noalloc(R, F, mass, dt_path, nu, eta_out, e_spring_out, stream=None):
    """eta^n and the spring energy (stage S4) for callers that must not allocate device memory: no context, and the
    library allocates nothing -- its working memory is a fixed array inside the library image (see include/mop.h for
    who needs this, the size limit MOP_NOALLOC_MAX_ATOM_BEADS and the rule against concurrent calls on one GPU).
    Every tensor is the caller's, already on the GPU: R [N][Q][3], F [N-1][Q][3], mass [Q] float32; eta_out
    [N-1][Q][3] float32 and e_spring_out (one float64) are written.  Nothing is allocated here either: the arguments
    are passed through as they are, so they must be contiguous.  Asynchronous on `stream` (default: torch's current)."""
    import torch
    L = load()
    N, Q = int(R.shape[0]), int(R.shape[1])
    for t, shape, dt in ((R, (N, Q, 3), torch.float32), (F, (N - 1, Q, 3), torch.float32), (mass, (Q,), torch.float32),
                         (eta_out, (N - 1, Q, 3), torch.float32), (e_spring_out, None, torch.float64)):
        if not (t.is_cuda and t.is_contiguous() and t.dtype == dt and t.device == R.device):
            raise ValueError("mop_eta_spring_noalloc takes contiguous CUDA tensors on one device (float32; energy float64)")
        if shape is not None and tuple(t.shape) != shape:
            raise ValueError("shape %s, expected %s" % (tuple(t.shape), shape))
    if e_spring_out.numel() != 1:
        raise ValueError("e_spring_out holds one float64")
    st = stream if stream is not None else torch.cuda.current_stream(R.device)
    err = C.create_string_buffer(512)
    s = L.mop_eta_spring_noalloc(R.device.index or 0, C.c_void_p(st.cuda_stream), Q, N, float(dt_path), float(nu), _ptr(R),
                                 _ptr(F), _ptr(mass), _ptr(eta_out), _ptr(e_spring_out), err, len(err))
    if s != MOP_OK:
        raise MopError(s, err.value.decode())


def _np(a, dtype, shape=None):
    a = np.ascontiguousarray(np.asarray(a, dtype=dtype))
    return a if shape is None else a.reshape(shape)


class Mop:
    """One context (device, system).  `system` carries the attributes of workloads.System."""

    def __init__(self, system, n_beads, device=0, r_buf=0.0, stream=None, block=None):
        """block = (first_bead, n_beads_path): mop_create_block -- the context owns beads [first_bead, first_bead +
        n_beads) of a longer path (bead-block mode, see MopBlockMethods below)."""
        import torch
        self.torch = torch
        self.L = load()
        if not torch.cuda.is_available():
            raise RuntimeError("no CUDA device: the MoP hot path has no CPU fallback")
        self.device = torch.device("cuda", device)
        self.Q, self.N = int(system.n_atoms), int(n_beads)
        self.nf = max(self.N - 1, 1)
        self.block = None
        if block is not None:
            n0, ntot = int(block[0]), int(block[1])
            self.block = (n0, ntot)
            self.nf = max(1 if ntot == 1 else min(self.N, ntot - 1 - n0), 1)
        p = mop_params()
        p.n_atoms, p.n_beads = self.Q, self.N
        for d in range(3):
            p.box[d] = float(np.float32(system.box[d]))
        p.r_cut, p.r_buf = float(system.r_cut), float(r_buf)
        p.eps_rf, p.lj_shift = float(system.eps_rf), int(system.lj_shift)
        p.dt_path, p.nu = float(system.dt_path), float(system.nu)
        p.device = device
        st = stream if stream is not None else torch.cuda.current_stream(self.device)
        self.stream = st
        p.stream = C.c_void_p(st.cuda_stream)
        self.ctx = C.c_void_p()
        if self.block is None:
            s = self.L.mop_create(C.byref(self.ctx), C.byref(p))
        else:
            s = self.L.mop_create_block(C.byref(self.ctx), C.byref(p), self.block[0], self.block[1])
        if s != MOP_OK:
            raise MopError(s, (self.L.mop_last_error(None) or b"").decode())
        self.set_topology(system)

    def _check(self, s):
        if s != MOP_OK:
            raise MopError(s, (self.L.mop_last_error(self.ctx) or b"").decode())

    def mop_set_topology(self, system):
        t = mop_topology()
        keep = []

        def arr(x, dtype, shape=None):
            a = _np(x, dtype, shape)
            keep.append(a)
            return a.ctypes.data_as(C.c_void_p) if a.size else None

        t.mass, t.charge, t.type = arr(system.mass, np.float32), arr(system.charge, np.float32), arr(system.type, np.int32)
        t.n_types = int(system.n_types)
        t.c6, t.c12 = arr(system.c6, np.float32), arr(system.c12, np.float32)
        b = _np(system.bond_ij, np.int32, (-1, 2))
        t.n_bonds = b.shape[0]
        t.bond_ij, t.bond_b0_kb = arr(b, np.int32), arr(system.bond_b0_kb, np.float32)
        a = _np(system.angle_ijk, np.int32, (-1, 3))
        t.n_angles = a.shape[0]
        t.angle_ijk, t.angle_t0_kt = arr(a, np.int32), arr(system.angle_t0_kt, np.float32)
        es = _np(system.excl_start, np.int32)
        keep.append(es)
        t.excl_start = es.ctypes.data_as(C.c_void_p)
        t.excl_list = arr(system.excl_list, np.int32)
        self._check(self.L.mop_set_topology(self.ctx, C.byref(t)))

    set_topology = mop_set_topology

    def _dev(self, R, shape):
        torch = self.torch
        if not isinstance(R, torch.Tensor):
            R = torch.as_tensor(np.ascontiguousarray(R, dtype=np.float32))
        R = R.to(device=self.device, dtype=torch.float32).contiguous()
        assert tuple(R.shape) == tuple(shape), (R.shape, shape)
        return R

    def mop_eval_veff_grad(self, R, want_grad=True, sync=True, grad_out=None):
        """R: [N][Q][3] float32 (torch cuda tensor, or anything castable).  Returns (veff | None, grad | None)."""
        R = self._dev(R, (self.N, self.Q, 3))
        grad = grad_out
        if want_grad and grad is None:
            grad = self.torch.empty_like(R)
        v = C.c_double(0.0)
        self._check(self.L.mop_eval_veff_grad(self.ctx, _ptr(R), C.byref(v) if sync else None,
                                              _ptr(grad) if want_grad else None))
        return (v.value if sync else None), (grad if want_grad else None)

    def mop_eval_veff_grad_fd(self, R, eps, sync=True, grad_out=None):
        """The paper's finite-difference form of the Hessian term (three force passes).  Returns (veff | None, grad)."""
        R = self._dev(R, (self.N, self.Q, 3))
        grad = grad_out if grad_out is not None else self.torch.empty_like(R)
        v = C.c_double(0.0)
        self._check(self.L.mop_eval_veff_grad_fd(self.ctx, _ptr(R), float(eps), C.byref(v) if sync else None, _ptr(grad)))
        return (v.value if sync else None), grad

    def mop_eval_veff_grad_host(self, R_host, grad_host=None):
        """HOST buffers (torch CPU tensors, ideally pinned, float32 [N][Q][3]).  Returns V_eff; fills grad_host."""
        assert not R_host.is_cuda and R_host.is_contiguous() and tuple(R_host.shape) == (self.N, self.Q, 3)
        assert R_host.dtype == self.torch.float32
        if grad_host is not None:
            assert not grad_host.is_cuda and grad_host.is_contiguous() and grad_host.shape == R_host.shape
            assert grad_host.dtype == self.torch.float32
        v = C.c_double(0.0)
        self._check(self.L.mop_eval_veff_grad_host(self.ctx, _ptr(R_host), C.byref(v), _ptr(grad_host)))
        return v.value

    def mop_set_timing(self, on):
        self._check(self.L.mop_set_timing(self.ctx, int(bool(on))))

    def mop_get_timing(self):
        """Mean ms per evaluation of each stage since mop_set_timing, and the number of evaluations averaged."""
        out = (C.c_double * 16)()
        self._check(self.L.mop_get_timing(self.ctx, out))
        k = ["S0_grid", "S1_pairlist", "S2_nb_force", "S3_bonded_force", "S4_eta", "S5_nb_hvp", "S6_bonded_hvp",
             "S7_assemble"]
        d = dict(zip(k, list(out)[:8]))
        d["evals"] = int(out[8])
        return d

    def mop_step(self, R, V, dt_pmd, n_steps):
        """In-place velocity Verlet on torch cuda tensors R, V [N][Q][3] float32."""
        assert R.is_cuda and V.is_cuda and R.is_contiguous() and V.is_contiguous()
        assert tuple(R.shape) == (self.N, self.Q, 3) and tuple(V.shape) == (self.N, self.Q, 3)
        self._check(self.L.mop_step(self.ctx, _ptr(R), _ptr(V), float(dt_pmd), int(n_steps)))

    def mop_step_continue(self, R, V, dt_pmd, n_steps):
        """mop_step without the initial evaluation: R must be what the previous mop_step* call left behind."""
        assert R.is_cuda and V.is_cuda and R.is_contiguous() and V.is_contiguous()
        assert tuple(R.shape) == (self.N, self.Q, 3) and tuple(V.shape) == (self.N, self.Q, 3)
        self._check(self.L.mop_step_continue(self.ctx, _ptr(R), _ptr(V), float(dt_pmd), int(n_steps)))

    def mop_step_langevin(self, R, V, dt_pmd, n_steps, gamma, temperature, seed=0, step0=0, cont=False):
        """In-place velocity Verlet + exact OU thermostat update on torch cuda tensors R, V [N][Q][3] float32.
        cont=True calls mop_step_langevin_continue (no initial evaluation)."""
        assert R.is_cuda and V.is_cuda and R.is_contiguous() and V.is_contiguous()
        assert tuple(R.shape) == (self.N, self.Q, 3) and tuple(V.shape) == (self.N, self.Q, 3)
        f = self.L.mop_step_langevin_continue if cont else self.L.mop_step_langevin
        self._check(f(self.ctx, _ptr(R), _ptr(V), float(dt_pmd), int(n_steps), float(gamma), float(temperature), int(seed),
                      int(step0)))

    # ---- bead-block mode (mop.h "bead-block mode"): pass 1, [halo exchange by the caller], pass 2, assembly
    def mop_block_pass1(self, R, R_right=None, keta_right_out=None):
        """R [n_beads][Q][3] cuda; R_right [Q][3] cuda = the bead after the block; keta_right_out [Q][3] cuda receives
        K eta of the block's last bead (both None for the path's last block)."""
        assert R.is_cuda and R.is_contiguous() and tuple(R.shape) == (self.N, self.Q, 3)
        for t in (R_right, keta_right_out):
            assert t is None or (t.is_cuda and t.is_contiguous() and tuple(t.shape) == (self.Q, 3) and t.dtype == R.dtype)
        self._check(self.L.mop_block_pass1(self.ctx, _ptr(R), _ptr(R_right), _ptr(keta_right_out)))

    def mop_block_pass2(self, R):
        self._check(self.L.mop_block_pass2(self.ctx, _ptr(R)))

    def mop_block_assemble(self, keta_left=None, grad_out=None, sync=True):
        """keta_left [Q][3] cuda from the left neighbour (None for the path's first block).  Returns (veff_local | None, grad)."""
        assert keta_left is None or (keta_left.is_cuda and keta_left.is_contiguous() and tuple(keta_left.shape) == (self.Q, 3))
        grad = grad_out if grad_out is not None else self.torch.empty((self.N, self.Q, 3), dtype=self.torch.float32,
                                                                      device=self.device)
        v = C.c_double(0.0)
        self._check(self.L.mop_block_assemble(self.ctx, _ptr(keta_left), C.byref(v) if sync else None, _ptr(grad)))
        return (v.value if sync else None), grad

    def mop_block_integrate(self, R, V, grad, dt_pmd, stage):
        assert R.is_cuda and V.is_cuda and grad.is_cuda and R.shape == V.shape == grad.shape
        self._check(self.L.mop_block_integrate(self.ctx, _ptr(R), _ptr(V), _ptr(grad), float(dt_pmd), int(stage)))

    def mop_block_thermostat(self, V, dt_pmd, gamma, temperature, seed=0, step=0):
        """The OU velocity update of mop_step_langevin on this context's beads, noise keyed by the whole-path index."""
        assert V.is_cuda and V.is_contiguous() and tuple(V.shape) == (self.N, self.Q, 3)
        self._check(self.L.mop_block_thermostat(self.ctx, _ptr(V), float(dt_pmd), float(gamma), float(temperature), int(seed),
                                                int(step)))

    def mop_set_bias(self, group_a, group_b, sigma, height, pace=0):
        """MoP bias on S_e2e = s(R^N) - s(R^1), s = COM distance of the two groups.  Empty groups switch it off."""
        ga, gb = _np(group_a, np.int32), _np(group_b, np.int32)
        self._check(self.L.mop_set_bias(self.ctx, ga.ctypes.data_as(C.c_void_p), len(ga), gb.ctypes.data_as(C.c_void_p),
                                        len(gb), float(sigma), float(height), int(pace)))

    def mop_add_hill(self, s_center):
        self._check(self.L.mop_add_hill(self.ctx, float(s_center)))

    def mop_get_bias(self):
        out = (C.c_double * 8)()
        n = C.c_int(0)
        hills = np.zeros(65536)
        self._check(self.L.mop_get_bias(self.ctx, out, hills.ctypes.data_as(C.c_void_p), len(hills), C.byref(n)))
        return dict(S=out[0], s1=out[1], sN=out[2], V=out[3], dVdS=out[4], n_hills=int(out[5]), hills=hills[:n.value].copy())

    def mop_debug_noise_bits(self, seed, step, n):
        out = np.empty(n, np.uint64)
        self._check(self.L.mop_debug_noise_bits(self.ctx, int(seed), int(step), int(n), out.ctypes.data_as(C.c_void_p)))
        return out

    def mop_force_hvp(self, R1, s=None):
        """Physical force (and H.s for a direction s) of one configuration [Q][3].  Returns (F, Hs) tensors."""
        R1 = self._dev(R1, (self.Q, 3))
        F = self.torch.empty_like(R1)
        Hs = None
        sd = None
        if s is not None:
            sd = self._dev(s, (self.Q, 3))
            Hs = self.torch.empty_like(R1)
        self._check(self.L.mop_force_hvp(self.ctx, _ptr(R1), _ptr(sd), _ptr(F), _ptr(Hs)))
        return F, Hs

    def mop_get_stats(self):
        out = (C.c_double * 16)()
        self._check(self.L.mop_get_stats(self.ctx, out))
        k = ["veff", "U1", "E_spring", "U_lj", "U_coul", "U_bond", "U_angle", "E_kin", "rebuilds", "entries", "units",
             "masks", "pair_slots", "launches", "reuses", "pair_slots_evaluated"]
        return dict(zip(k, list(out)[:16]))

    def dims(self):
        d = np.zeros(8, np.int32)
        self._check(self.L.mop_debug_get(self.ctx, b"dims", d.ctypes.data_as(C.c_void_p), d.nbytes))
        return dict(nx=int(d[0]), ny=int(d[1]), nz=int(d[2]), S=int(d[3]), nf=int(d[4]), cluster=int(d[5]),
                    groups=int(d[6]), bin_z=float(d[7:8].view(np.float32)[0]))

    def mop_debug_get(self, what):
        S = self.dims()["S"]
        shape, dt = {"cell": ((self.nf, self.Q), np.int32), "perm": ((self.nf, S), np.int32),
                     "xq": ((self.nf, S, 4), np.float32), "F": ((self.nf, self.Q, 3), np.float32),
                     "eta": ((self.nf, self.Q, 3), np.float32), "Heta": ((self.nf, self.Q, 3), np.float32)}[what]
        out = np.empty(shape, dt)
        self._check(self.L.mop_debug_get(self.ctx, what.encode(), out.ctypes.data_as(C.c_void_p), out.nbytes))
        return out

    def mop_debug_pairs(self, bead, cap=None):
        """Sorted (i<j) array of the in-range, non-excluded pairs of one force bead of the last evaluation."""
        n = C.c_longlong(0)
        if cap is None:
            self._check(self.L.mop_debug_pairs(self.ctx, bead, None, 0, C.byref(n)))
            cap = n.value
        out = np.empty((max(cap, 1), 2), np.int32)
        self._check(self.L.mop_debug_pairs(self.ctx, bead, out.ctypes.data_as(C.c_void_p), cap, C.byref(n)))
        out = out[:min(cap, n.value)]
        out = np.sort(out, axis=1)
        order = np.lexsort((out[:, 1], out[:, 0]))
        return out[order], int(n.value)

    def mop_debug_count_inrange(self, which=2):
        """In-range, non-excluded pair decisions of the PRODUCTION force kernel (counting instance) over the list of
        the last evaluation.  which: 0 bead 1, 1 the other force beads, 2 all force beads."""
        n, h = C.c_longlong(0), C.c_ulonglong(0)
        self._check(self.L.mop_debug_count_inrange(self.ctx, int(which), C.byref(n), C.byref(h)))
        self.last_pair_hash = int(h.value)
        return int(n.value)

    def mop_debug_pair_hash(self, which=2):
        """(count, fingerprint) of the production kernel's decided pair set (see mop.h)."""
        n = self.mop_debug_count_inrange(which)
        return n, self.last_pair_hash

    def mop_debug_set_list_capacity(self, units=0, entries=0, masks=0):
        self._check(self.L.mop_debug_set_list_capacity(self.ctx, int(units), int(entries), int(masks)))

    def mop_destroy(self):
        if getattr(self, "ctx", None) is not None and self.ctx.value:
            self.L.mop_destroy(self.ctx)
            self.ctx = C.c_void_p()

    close = mop_destroy

    def __del__(self):
        try:
            self.mop_destroy()
        except Exception:
            pass
