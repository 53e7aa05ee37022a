"""Small-system builders shared by the test modules (no method arithmetic here)."""
import numpy as np

from paper_2501_11962_b200 import workloads as W


def make_system(name, box, X, mass, charge, typ, sig, eps, bonds=(), bpar=(), angles=(), apar=(), r_cut=1.0,
                eps_rf=78.0, lj_shift=0, T=300.0, n_beads=1, excl=None):
    s = W._finish(name, box, r_cut, eps_rf, lj_shift, T, np.asarray(X, float), mass, charge, typ, sig, eps,
                  np.asarray(bonds, int).reshape(-1, 2), np.asarray(bpar, float).reshape(-1, 2),
                  np.asarray(angles, int).reshape(-1, 3), np.asarray(apar, float).reshape(-1, 2), n_beads)
    if excl is not None:
        s.excl_start, s.excl_list = excl
    return s


def two_atoms(r, eps=0.996, sig=0.34, q=(0.0, 0.0), box=4.0, r_cut=1.0, eps_rf=78.0, lj_shift=0, axis=0):
    X = np.full((2, 3), 1.0)
    X[1, axis] += r
    return make_system("pair", [box] * 3, X, [39.948, 39.948], list(q), [0, 0], [sig], [eps], r_cut=r_cut,
                       eps_rf=eps_rf, lj_shift=lj_shift)


def lj_cluster(n=32, L=2.4, seed=1, r_cut=1.0, lj_shift=1, masses=None):
    """n LJ atoms on a jittered lattice in a small periodic box (L >= 2 r_cut)."""
    rng = np.random.default_rng(seed)
    k = int(np.ceil(n ** (1 / 3)))
    g = np.stack(np.meshgrid(*[np.arange(k)] * 3, indexing="ij"), -1).reshape(-1, 3)[:n]
    X = (g + 0.5) * (L / k) + rng.normal(0, 0.03, (n, 3))
    m = np.full(n, 39.948) if masses is None else masses
    return make_system("ljc", [L] * 3, X, m, np.zeros(n), np.zeros(n, int), [0.34], [0.996], r_cut=r_cut,
                       eps_rf=0.0, lj_shift=lj_shift, T=120.0)


def tiny_water(n_side=2, L=2.2, seed=2, r_cut=1.0):
    s = W.water_box(n_side, L, seed, n_beads=1, r_cut=r_cut, name="tiny_water")
    return s


def tiny_chain(n=10, L=2.6, seed=3, r_cut=1.0, charged=True):
    """A bent bonded chain (bonds, angles, 1-2/1-3 exclusions, charges, LJ) plus 3 waters."""
    rng = np.random.default_rng(seed)
    X, bonds, angles, _ = W.serpentine_chain(n, 4, [(0.9, 0.9), (0.9, 1.33), (1.33, 1.33)], 0.8)
    X = X + rng.normal(0, 0.01, X.shape)
    cw = np.array([[1.9, 1.9, 1.9], [0.4, 1.9, 0.5], [1.9, 0.4, 1.2]])
    Xw = W.water_molecules(cw, rng)
    wb, wa = W.water_topology(3, n)
    Xall = np.concatenate([X, Xw], 0)
    q = rng.normal(0, 0.3, n) if charged else np.zeros(n)
    q = q - q.mean()
    charge = np.concatenate([q, np.tile([W.Q_O, W.Q_H, W.Q_H], 3)])
    mass = np.concatenate([np.full(n, W.M_CHAIN), np.tile([W.M_O, W.M_H, W.M_H], 3)])
    typ = np.concatenate([np.full(n, 2), np.tile([0, 1, 1], 3)])
    b = np.concatenate([bonds, wb], 0)
    a = np.concatenate([angles, wa], 0)
    bp = np.concatenate([np.tile([W.B_CHAIN, W.KB_BOND], (len(bonds), 1)), np.tile([W.B_OH, W.KB_BOND], (len(wb), 1))])
    ap = np.concatenate([np.tile([W.TH_CHAIN, W.KT_CHAIN], (len(angles), 1)),
                         np.tile([W.TH_HOH, W.KT_WATER], (len(wa), 1))])
    return make_system("tiny_chain", [L] * 3, Xall, mass, charge, typ, [0.3166, 0.0, 0.34], [0.65, 0.0, 0.4], b, bp,
                       a, ap, r_cut=r_cut)


def rms_rel(a, b):
    """G14: sqrt(sum |a-b|^2 / sum |b|^2)."""
    a = np.asarray(a, float)
    b = np.asarray(b, float)
    den = np.sqrt((b * b).sum())
    return float(np.sqrt(((a - b) ** 2).sum()) / (den if den > 0 else 1.0))


def pairs_near_cutoff(system, X, tol=1e-4):
    """Count atom pairs whose minimum-image distance is within tol of r_cut (G9 guard for FD pins)."""
    box = np.asarray(system.box, float)
    X = np.asarray(X, float)
    d = X[:, None, :] - X[None, :, :]
    d -= box * np.round(d / box)
    r = np.sqrt((d * d).sum(-1))
    iu = np.triu_indices(X.shape[0], 1)
    return int((np.abs(r[iu] - system.r_cut) < tol).sum())


TOL_MAX = 1e-3


def assert_close(a, b, tol_rms, tol_max=TOL_MAX):
    """The parity bar for a force-like array: G14's RMS relative error <= tol_rms (north_star: 1e-4) AND no single
    component farther from the reference than tol_max times the RMS magnitude of the reference components (an RMS over
    millions of components alone would let one component be off by a large multiple of the typical magnitude)."""
    a = np.asarray(a, float)
    b = np.asarray(b, float)
    assert a.shape == b.shape, (a.shape, b.shape)
    r = rms_rel(a, b)
    assert r <= tol_rms, "RMS relative error %.3e > %.1e" % (r, tol_rms)
    if b.size == 0:
        return
    scale = float(np.sqrt((b * b).mean()))
    err = np.abs(a - b)
    k = np.unravel_index(err.argmax(), err.shape)
    assert err[k] <= tol_max * max(scale, 1e-30), "max |delta| %.3e > %.1e x rms(ref) %.3e at component %s" % (
        err[k], tol_max, scale, k)


def pair_set_fingerprint(pairs_by_bead, Q):
    """The fingerprint mop_debug_count_inrange documents (include/mop.h), from a list of (bead index, pairs [n][2]):
    sum mod 2^64 of splitmix64(((bead * Q + min(i,j)) * Q + max(i,j)) + 0x9E3779B97F4A7C15)."""
    total = np.uint64(0)
    with np.errstate(over="ignore"):
        for bead, P in pairs_by_bead:
            P = np.asarray(P, np.int64)
            lo, hi = np.minimum(P[:, 0], P[:, 1]).astype(np.uint64), np.maximum(P[:, 0], P[:, 1]).astype(np.uint64)
            z = (np.uint64(bead) * np.uint64(Q) + lo) * np.uint64(Q) + hi + np.uint64(0x9E3779B97F4A7C15)
            z = (z ^ (z >> np.uint64(30))) * np.uint64(0xBF58476D1CE4E5B9)
            z = (z ^ (z >> np.uint64(27))) * np.uint64(0x94D049BB133111EB)
            z = z ^ (z >> np.uint64(31))
            total = total + z.sum(dtype=np.uint64)
    return int(total)
