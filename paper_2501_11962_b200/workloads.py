"""Seeded synthetic inputs for the MoP hot path (BASELINE.json configs 1-5).

This module serves both the tests/oracle and bench.py; it contains none of the
method's arithmetic (no potential, no force, no V_eff).  The only physics-shaped
step is the Brownian recursion that BASELINE.json prescribes for generating a
path, and it takes the force as a CALLBACK (`force_fn`) so that tests drive it
with the oracle and bench.py with the library.

The systems stand in for the paper's LJ cluster, water boxes, solvated protein
and the 151,850-atom hA2AR membrane system, whose structures
and force fields are not available here; sizes, densities, charge and topology
structure follow BASELINE.json `configs`, open choices (masses, force constants,
LJ of chain sites, packing) follow DESIGN.md "Input recipe".
Units: nm, ps, u, kJ/mol, e, K.
"""
from dataclasses import dataclass, field

import numpy as np

KB = 0.0083144626  # kJ mol^-1 K^-1

# water-like three-site molecule (config 2; W1/W2 in DESIGN.md)
M_O, M_H = 9.951, 4.032
Q_O, Q_H = -0.82, 0.41
B_OH, TH_HOH = 0.1, np.deg2rad(109.47)
KB_BOND = 1.0e5       # kJ mol^-1 nm^-2, all bonds
KT_WATER = 383.0      # kJ mol^-1 rad^-2
KT_CHAIN = 400.0
M_CHAIN, M_LIPID = 12.011, 14.027
B_CHAIN, TH_CHAIN = 0.15, np.deg2rad(110.0)


@dataclass
class System:
    name: str
    n_atoms: int
    box: np.ndarray            # [3] float32
    r_cut: float
    eps_rf: float
    lj_shift: int
    dt_path: float
    nu: float
    temperature: float
    mass: np.ndarray           # [Q] float32
    charge: np.ndarray         # [Q] float32
    type: np.ndarray           # [Q] int32
    n_types: int
    c6: np.ndarray             # [n_types*n_types] float32
    c12: np.ndarray
    bond_ij: np.ndarray        # [nb][2] int32
    bond_b0_kb: np.ndarray     # [nb][2] float32
    angle_ijk: np.ndarray      # [na][3] int32 (j central)
    angle_t0_kt: np.ndarray    # [na][2] float32
    excl_start: np.ndarray     # [Q+1] int32 CSR
    excl_list: np.ndarray      # int32
    R1: np.ndarray             # [Q][3] float64 start configuration (bead 1)
    n_beads: int = 1
    meta: dict = field(default_factory=dict)


# ----------------------------------------------------------------------------
# topology helpers
# ----------------------------------------------------------------------------
def exclusions_from_bonds(Q, bonds):
    """All pairs within 2 bonds (1-2 and 1-3), symmetric sorted CSR (reading G11)."""
    bonds = np.asarray(bonds, dtype=np.int64).reshape(-1, 2)
    if bonds.shape[0] == 0:
        return np.zeros(Q + 1, np.int32), np.zeros(0, np.int32)
    a = np.concatenate([bonds[:, 0], bonds[:, 1]])
    b = np.concatenate([bonds[:, 1], bonds[:, 0]])
    order = np.lexsort((b, a))
    a, b = a[order], b[order]
    start = np.zeros(Q + 1, np.int64)
    np.add.at(start, a + 1, 1)
    start = np.cumsum(start)
    pairs = [np.stack([a, b], 1)]
    # 1-3: for every centre j, all ordered pairs of its bonded neighbours
    deg = np.diff(start)
    for d in np.unique(deg):
        if d < 2:
            continue
        centres = np.flatnonzero(deg == d)
        nb = b[(start[centres][:, None] + np.arange(d)[None, :])]  # [nc][d]
        ii = np.repeat(nb, d, axis=1).reshape(-1)
        jj = np.tile(nb, (1, d)).reshape(-1)
        keep = ii != jj
        pairs.append(np.stack([ii[keep], jj[keep]], 1))
    p = np.concatenate(pairs, 0)
    key = np.unique(p[:, 0] * Q + p[:, 1])
    i, j = key // Q, key % Q
    es = np.zeros(Q + 1, np.int64)
    np.add.at(es, i + 1, 1)
    es = np.cumsum(es)
    return es.astype(np.int32), j.astype(np.int32)


def lj_table(sigma, eps):
    """Lorentz-Berthelot C6/C12 table for per-type sigma, eps (eps = 0: no LJ)."""
    sigma = np.asarray(sigma, float)
    eps = np.asarray(eps, float)
    s = 0.5 * (sigma[:, None] + sigma[None, :])
    e = np.sqrt(eps[:, None] * eps[None, :])
    c6 = 4.0 * e * s ** 6
    c12 = 4.0 * e * s ** 12
    return c6.astype(np.float32).reshape(-1), c12.astype(np.float32).reshape(-1)


_TET = np.array([[1, 1, 1], [1, -1, -1], [-1, 1, -1], [-1, -1, 1]], float) / np.sqrt(3.0)


def water_molecules(centres, rng):
    """Three-site molecules at O positions `centres`; the two H sit along two of the four
    tetrahedral body diagonals (angle exactly 109.47 deg, bond exactly 0.1 nm), chosen at
    random per molecule, so lattice neighbours never clash."""
    n = centres.shape[0]
    sign = rng.integers(0, 2, n) * 2 - 1
    pair = rng.integers(0, 6, n)
    combos = np.array([(0, 1), (0, 2), (0, 3), (1, 2), (1, 3), (2, 3)])
    u1 = _TET[combos[pair, 0]] * sign[:, None]
    u2 = _TET[combos[pair, 1]] * sign[:, None]
    X = np.empty((n, 3, 3))
    X[:, 0] = centres
    X[:, 1] = centres + B_OH * u1
    X[:, 2] = centres + B_OH * u2
    return X.reshape(-1, 3)


def water_topology(n_mol, first_atom):
    o = first_atom + 3 * np.arange(n_mol)
    bonds = np.concatenate([np.stack([o, o + 1], 1), np.stack([o, o + 2], 1)], 0)
    angles = np.stack([o + 1, o, o + 2], 1)
    return bonds, angles


def serpentine_chain(n_sites, n_strand, lattice_xy, z0, pitch_check=0.45):
    """Self-avoiding bonded chain: all-trans zig-zag strands along z (bond 0.15 nm, angle
    110 deg) standing on the 2-D points `lattice_xy` (visited in order), joined at the
    strand ends by two bridge sites so that every bond is exactly 0.15 nm (W4)."""
    h = B_CHAIN * np.sin(TH_CHAIN / 2.0)          # rise per site along z
    dlt = 0.5 * B_CHAIN * np.cos(TH_CHAIN / 2.0)  # zig-zag half amplitude (in x)
    pts = []
    k = 0
    up = True
    while len(pts) < n_sites:
        if k >= len(lattice_xy):
            raise ValueError("serpentine_chain: lattice too small for %d sites" % n_sites)
        x0, y0 = lattice_xy[k]
        levels = range(n_strand) if up else range(n_strand - 1, -1, -1)
        strand = [np.array([x0 + (dlt if (lv % 2 == 0) else -dlt), y0, z0 + lv * h]) for lv in levels]
        if pts:
            # two bridge sites between the previous strand end and this strand start
            pe, ps = pts[-1], strand[0]
            u = ps - pe
            D = np.linalg.norm(u)
            assert B_CHAIN < D <= 3 * B_CHAIN + 1e-9, D
            u = u / D
            c = 0.5 * (D - B_CHAIN)
            hh = np.sqrt(max(B_CHAIN ** 2 - c ** 2, 0.0))
            w = np.array([0.0, 0.0, 1.0 if not up else -1.0])  # outward from the turn
            for b in (pe + u * c + w * hh, ps - u * c + w * hh):
                if len(pts) < n_sites:
                    pts.append(b)
        for s in strand:
            if len(pts) < n_sites:
                pts.append(s)
        up = not up
        k += 1
    X = np.array(pts[:n_sites])
    idx = np.arange(n_sites)
    bonds = np.stack([idx[:-1], idx[1:]], 1)
    angles = np.stack([idx[:-2], idx[1:-1], idx[2:]], 1)
    return X, bonds, angles, k


def _snake(nx, ny, pitch, x0, y0):
    """Boustrophedon ordering of an nx x ny lattice."""
    out = []
    for ix in range(nx):
        ys = range(ny) if ix % 2 == 0 else range(ny - 1, -1, -1)
        for iy in ys:
            out.append((x0 + ix * pitch, y0 + iy * pitch))
    return out


def _carve(centres, sites, box, rmin):
    """Drop lattice centres closer than rmin (periodic) to any of `sites` (cell-binned)."""
    if sites.shape[0] == 0:
        return centres
    box = np.asarray(box, float)
    nc = np.maximum((box / max(rmin, 0.3)).astype(int), 1)
    cs = box / nc

    def cid(x):
        c = np.floor((x % box) / cs).astype(int) % nc
        return c

    sc = cid(sites)
    key = (sc[:, 0] * nc[1] + sc[:, 1]) * nc[2] + sc[:, 2]
    order = np.argsort(key, kind="stable")
    key_s = key[order]
    sites_s = sites[order]
    start = np.searchsorted(key_s, np.arange(nc.prod() + 1))
    keep = np.ones(centres.shape[0], bool)
    cc = cid(centres)
    for ox in (-1, 0, 1):
        for oy in (-1, 0, 1):
            for oz in (-1, 0, 1):
                c = (cc + np.array([ox, oy, oz])) % nc
                k = (c[:, 0] * nc[1] + c[:, 1]) * nc[2] + c[:, 2]
                lo, hi = start[k], start[k + 1]
                m = (hi - lo).max() if len(lo) else 0
                for t in range(int(m)):
                    sel = (lo + t) < hi
                    if not sel.any():
                        break
                    idx = np.where(sel, lo + t, 0)
                    d = centres - sites_s[idx]
                    d -= box * np.round(d / box)
                    close = (d * d).sum(1) < rmin * rmin
                    keep &= ~(close & sel)
    return centres[keep]


def _water_lattice(box, n_target, rng, avoid=None, rmin=0.3, jitter=0.012):
    """Face-centred-cubic lattice of molecule centres filling `box` (cube axes along the box, so
    the tetrahedral H directions of water_molecules point into voids), carved around `avoid`,
    thinned at random to exactly n_target; bounded rigid-body jitter per molecule."""
    box = np.asarray(box, float)
    vol = box.prod()
    a = (4.0 * vol / max(n_target, 1)) ** (1.0 / 3.0)   # conventional cell edge, 4 sites per cell
    basis = np.array([[0, 0, 0], [0.5, 0.5, 0], [0.5, 0, 0.5], [0, 0.5, 0.5]], float)
    for _ in range(400):
        n = np.maximum(np.floor(box / a).astype(int), 1)
        g = np.stack(np.meshgrid(*[np.arange(k) for k in n], indexing="ij"), -1).reshape(-1, 1, 3)
        c = ((g + basis[None, :, :] + 0.25) * (box / n)).reshape(-1, 3)
        if avoid is not None and len(avoid):
            c = _carve(c, avoid, box, rmin)
        if c.shape[0] >= n_target:
            break
        a *= 0.997
    else:
        raise RuntimeError("could not place %d molecules" % n_target)
    if c.shape[0] > n_target:
        keep = np.sort(rng.choice(c.shape[0], n_target, replace=False))
        c = c[keep]
    c = c + rng.uniform(-jitter, jitter, c.shape)
    return c, float((box / n).min() / np.sqrt(2.0))


def _finish(name, box, r_cut, eps_rf, lj_shift, T, X, mass, charge, typ, sig, eps, bonds, bpar, angles, apar,
            n_beads, meta=None):
    Q = X.shape[0]
    c6, c12 = lj_table(sig, eps)
    es, el = exclusions_from_bonds(Q, bonds)
    return System(
        name=name, n_atoms=Q, box=np.asarray(box, np.float32), r_cut=float(r_cut), eps_rf=float(eps_rf),
        lj_shift=int(lj_shift), dt_path=0.002, nu=50.0, temperature=float(T),
        mass=np.asarray(mass, np.float32), charge=np.asarray(charge, np.float32),
        type=np.asarray(typ, np.int32), n_types=len(sig), c6=c6, c12=c12,
        bond_ij=np.asarray(bonds, np.int32).reshape(-1, 2), bond_b0_kb=np.asarray(bpar, np.float32).reshape(-1, 2),
        angle_ijk=np.asarray(angles, np.int32).reshape(-1, 3),
        angle_t0_kt=np.asarray(apar, np.float32).reshape(-1, 2),
        excl_start=es, excl_list=el, R1=np.asarray(X, np.float64), n_beads=n_beads, meta=meta or {})


# ----------------------------------------------------------------------------
# the BASELINE.json configs
# ----------------------------------------------------------------------------
def config1(seed=0, n_side=8, n_beads=16):
    """512 LJ argon-like atoms, jittered simple-cubic lattice, 2.88 nm cube, no charges."""
    rng = np.random.default_rng(seed)
    a = 0.36
    g = np.stack(np.meshgrid(*[np.arange(n_side)] * 3, indexing="ij"), -1).reshape(-1, 3)
    X = (g + 0.5) * a + rng.normal(0.0, 0.02, (n_side ** 3, 3))
    Q = X.shape[0]
    L = n_side * a
    return _finish("c1_lj512" if n_side == 8 else "lj%d" % Q, [L, L, L], 1.0, 0.0, 1, 120.0, X,
                   np.full(Q, 39.948), np.zeros(Q), np.zeros(Q, int), [0.34], [0.996],
                   np.zeros((0, 2), int), np.zeros((0, 2)), np.zeros((0, 3), int), np.zeros((0, 2)), n_beads)


def water_box(n_side=10, L=3.10, seed=0, n_beads=64, T=300.0, r_cut=1.0, name=None):
    """n_side^3 three-site molecules on a lattice with random orientations (config 2)."""
    rng = np.random.default_rng(seed)
    g = np.stack(np.meshgrid(*[np.arange(n_side)] * 3, indexing="ij"), -1).reshape(-1, 3)
    c = (g + 0.5) * (L / n_side) + rng.uniform(-0.012, 0.012, (n_side ** 3, 3))
    n_mol = c.shape[0]
    X = water_molecules(c, rng)
    bonds, angles = water_topology(n_mol, 0)
    bpar = np.tile([B_OH, KB_BOND], (bonds.shape[0], 1))
    apar = np.tile([TH_HOH, KT_WATER], (angles.shape[0], 1))
    mass = np.tile([M_O, M_H, M_H], n_mol)
    q = np.tile([Q_O, Q_H, Q_H], n_mol)
    typ = np.tile([0, 1, 1], n_mol)
    return _finish(name or "c2_water3000", [L, L, L], r_cut, 78.0, 0, T, X, mass, q, typ,
                   [0.3166, 0.0], [0.650, 0.0], bonds, bpar, angles, apar, n_beads)


def config2(seed=0, n_beads=64):
    return water_box(10, 3.10, seed, n_beads)


def _assemble_solvated(name, box, r_cut, T, seed, n_total, chains, n_beads):
    """chains: list of dict(X, bonds, angles, type, mass, charge); water fills to n_total."""
    rng = np.random.default_rng(seed + 1000)
    n_chain = sum(c["X"].shape[0] for c in chains)
    assert (n_total - n_chain) % 3 == 0, "water count must be integral"
    n_w = (n_total - n_chain) // 3
    sites = np.concatenate([c["X"] for c in chains], 0)
    centres, a_w = _water_lattice(box, n_w, rng, avoid=sites, rmin=0.3)
    Xw = water_molecules(centres, rng)
    Xs, bonds, angles, bpar, apar, mass, q, typ = [], [], [], [], [], [], [], []
    off = 0
    for c in chains:
        n = c["X"].shape[0]
        Xs.append(c["X"])
        bonds.append(c["bonds"] + off)
        angles.append(c["angles"] + off)
        bpar.append(np.tile([B_CHAIN, KB_BOND], (c["bonds"].shape[0], 1)))
        apar.append(np.tile([TH_CHAIN, KT_CHAIN], (c["angles"].shape[0], 1)))
        mass.append(np.full(n, c["mass"]))
        q.append(c["charge"])
        typ.append(np.full(n, c["type"]))
        off += n
    wb, wa = water_topology(n_w, off)
    Xs.append(Xw)
    bonds.append(wb)
    angles.append(wa)
    bpar.append(np.tile([B_OH, KB_BOND], (wb.shape[0], 1)))
    apar.append(np.tile([TH_HOH, KT_WATER], (wa.shape[0], 1)))
    mass.append(np.tile([M_O, M_H, M_H], n_w))
    q.append(np.tile([Q_O, Q_H, Q_H], n_w))
    typ.append(np.tile([0, 1, 1], n_w))
    X = np.concatenate(Xs, 0)
    meta = dict(n_water=int(n_w), n_chain_sites=int(n_chain), water_nn_distance_nm=a_w)
    # types: 0 water O, 1 water H, 2 chain ("protein") site, 3 lipid-like site (W3)
    return _finish(name, box, r_cut, 78.0, 0, T, X, np.concatenate(mass), np.concatenate(q),
                   np.concatenate(typ), [0.3166, 0.0, 0.34, 0.375], [0.650, 0.0, 0.4, 0.4],
                   np.concatenate(bonds, 0), np.concatenate(bpar, 0), np.concatenate(angles, 0),
                   np.concatenate(apar, 0), n_beads, meta)


def _random_neutral_charges(n, rng, sd=0.3):
    q = rng.normal(0.0, sd, n)
    return q - q.mean()


def config3(seed=0, n_beads=32, n_total=23000, n_chain=2300, L=6.2):
    """Solvated globule: a bonded chain folded compactly at the box centre + water."""
    rng = np.random.default_rng(seed)
    pitch, n_strand = 0.43, 21
    n_lat = int(np.ceil(np.sqrt(n_chain / (n_strand + 2.0)))) + 1
    h = B_CHAIN * np.sin(TH_CHAIN / 2.0)
    x0 = 0.5 * L - 0.5 * (n_lat - 1) * pitch
    z0 = 0.5 * L - 0.5 * (n_strand - 1) * h
    X, bonds, angles, _ = serpentine_chain(n_chain, n_strand, _snake(n_lat, n_lat, pitch, x0, x0), z0)
    chain = dict(X=X, bonds=bonds, angles=angles, type=2, mass=M_CHAIN,
                 charge=_random_neutral_charges(n_chain, rng))
    return _assemble_solvated("c3_globule%d" % n_total, [L, L, L], 1.0, 300.0, seed, n_total, [chain], n_beads)


def config4(seed=0, n_beads=8, n_total=150000, box=(10.5, 10.5, 13.5), n_protein=4000, slab=4.0, r_cut=1.2,
            name=None):
    """Membrane-protein-shaped system: central slab of neutral 50-site lipid-like chains, one
    charged bonded chain crossing the slab, water above and below (and in the slab's voids)."""
    rng = np.random.default_rng(seed)
    box = np.asarray(box, float)
    h = B_CHAIN * np.sin(TH_CHAIN / 2.0)
    zc = 0.5 * box[2]
    # protein: strands a little taller than the slab, on a square lattice at the box centre
    pitch = 0.43
    n_strand_p = int(round((slab + 0.9) / h)) + 1
    n_lat = int(np.ceil(np.sqrt(n_protein / (n_strand_p + 2.0)))) + 1
    px0 = 0.5 * box[0] - 0.5 * (n_lat - 1) * pitch
    py0 = 0.5 * box[1] - 0.5 * (n_lat - 1) * pitch
    Xp, bp, ap, used = serpentine_chain(n_protein, n_strand_p, _snake(n_lat, n_lat, pitch, px0, py0),
                                        zc - 0.5 * (n_strand_p - 1) * h)
    chains = [dict(X=Xp, bonds=bp, angles=ap, type=2, mass=M_CHAIN,
                   charge=_random_neutral_charges(n_protein, rng))]
    foot_lo = Xp[:, :2].min(0) - 0.45
    foot_hi = Xp[:, :2].max(0) + 0.45
    # lipid-like hairpins: 24 + 2 + 24 = 50 sites, two strands 0.43 nm apart in y
    n_strand_l = 24
    gx = 0.46
    gy = 2 * pitch + 0.04
    nx = int(np.floor(box[0] / gx))
    ny = int(np.floor(box[1] / gy))
    gx, gy = box[0] / nx, box[1] / ny
    z0l = zc - 0.5 * (n_strand_l - 1) * h
    lipids = []
    for ix in range(nx):
        for iy in range(ny):
            x = (ix + 0.5) * gx
            y = (iy + 0.5) * gy - 0.5 * pitch
            if foot_lo[0] < x < foot_hi[0] and (foot_lo[1] < y + pitch) and (y < foot_hi[1]):
                continue
            lipids.append((x, y))
    # the atom count binds (W5): 3 must divide n_total - n_protein - 50 n_L
    while (n_total - n_protein - 50 * len(lipids)) % 3 != 0:
        lipids.pop(int(rng.integers(0, len(lipids))))
    for (x, y) in lipids:
        X, b, a, _ = serpentine_chain(50, n_strand_l, [(x, y), (x, y + pitch)], z0l)
        chains.append(dict(X=X, bonds=b, angles=a, type=3, mass=M_LIPID, charge=np.zeros(50)))
    s = _assemble_solvated(name or "c4_membrane%d" % n_total, box, r_cut, 310.0, seed, n_total, chains, n_beads)
    s.meta.update(n_lipid_chains=len(lipids), n_protein=n_protein)
    return s


def small_membrane(seed=0, n_beads=4):
    """A reduced copy of config 4 (same recipe and number density, 6.3 x 6.3 x 7.2 nm, r_c 1.2) that
    the oracle finishes in seconds; used for parity of the mixed topology (chain + lipids + water)."""
    vol_ratio = (6.3 * 6.3 * 7.2) / (10.5 * 10.5 * 13.5)
    n_total = int(round(150000 * vol_ratio))
    return config4(seed, n_beads, n_total, (6.3, 6.3, 7.2), 600, 3.0, 1.2, name="c4s_membrane_small")


# ----------------------------------------------------------------------------
# the path generator (BASELINE.json): R^{n+1} = R^n + a F(R^n) + N(0, 2 kT a),
# a_i = dt/(m_i nu); the force comes from the caller.
# ----------------------------------------------------------------------------
def brownian_path(system, n_beads, force_fn, seed=0, noise=True, dtype=np.float32):
    """Returns R [n_beads][Q][3].  force_fn(R_bead [Q][3] float64) -> F [Q][3].

    Generated in FP64 and cast once at the end; beads are never wrapped (image-consistent)."""
    rng = np.random.default_rng(seed + 7919)
    Q = system.n_atoms
    a = system.dt_path / (system.mass.astype(np.float64) * system.nu)
    sd = np.sqrt(2.0 * KB * system.temperature * a)
    R = np.empty((n_beads, Q, 3))
    R[0] = system.R1
    for n in range(n_beads - 1):
        F = np.asarray(force_fn(R[n]), dtype=np.float64).reshape(Q, 3)
        if not np.isfinite(F).all():
            raise FloatingPointError("non-finite force on bead %d" % n)
        R[n + 1] = R[n] + a[:, None] * F
        if noise:
            R[n + 1] += rng.normal(0.0, 1.0, (Q, 3)) * sd[:, None]
    return R.astype(dtype)


MAX_RECURSION_BEADS = 32


def folded_path(system, n_beads, force_fn, seed=0, noise=True, dtype=np.float32, first=0):
    """Beads [first, n_beads) of a path of any length from at most MAX_RECURSION_BEADS steps of the Brownian recursion.

    The explicit Euler recursion of the stiff three-site water is only stable for a few dozen steps,
    so a longer path walks the stable stretch back and forth: bead j is recursion bead j mod 2(L-1), reflected at L-1.
    Neighbouring beads stay one recursion step apart, which is all eqs (3),(5)-(7) look at.  For n_beads <= 32 this is
    brownian_path itself."""
    L = min(n_beads, MAX_RECURSION_BEADS)
    R = brownian_path(system, L, force_fn, seed=seed, noise=noise, dtype=dtype)
    if n_beads <= L and first == 0:
        return R
    idx = [j % (2 * (L - 1)) if L > 1 else 0 for j in range(first, n_beads)]
    idx = [j if j < L else 2 * (L - 1) - j for j in idx]
    return np.ascontiguousarray(R[idx])


def min_nonexcluded_distance(system, X, r_probe=0.25):
    """Smallest periodic distance between non-excluded atoms (generator sanity gate)."""
    box = np.asarray(system.box, float)
    Q = X.shape[0]
    nc = np.maximum((box / r_probe).astype(int), 1)
    c = np.floor((X % box) / (box / nc)).astype(int) % nc
    key = (c[:, 0] * nc[1] + c[:, 1]) * nc[2] + c[:, 2]
    order = np.argsort(key, kind="stable")
    ks = key[order]
    start = np.searchsorted(ks, np.arange(nc.prod() + 1))
    es, el = system.excl_start, system.excl_list
    best = np.inf
    excl = set()
    for i in range(Q):
        for e in range(es[i], es[i + 1]):
            excl.add((i, int(el[e])))
    for ox in (-1, 0, 1):
        for oy in (-1, 0, 1):
            for oz in (-1, 0, 1):
                cn = (c + np.array([ox, oy, oz])) % nc
                kn = (cn[:, 0] * nc[1] + cn[:, 1]) * nc[2] + cn[:, 2]
                lo, hi = start[kn], start[kn + 1]
                for t in range(int((hi - lo).max())):
                    sel = (lo + t) < hi
                    j = order[np.where(sel, lo + t, 0)]
                    d = X - X[j]
                    d -= box * np.round(d / box)
                    r = np.sqrt((d * d).sum(1))
                    r[~sel] = np.inf
                    r[j == np.arange(Q)] = np.inf
                    cand = np.flatnonzero(r < min(best, r_probe))
                    for i in cand:
                        if (int(i), int(j[i])) not in excl:
                            best = min(best, r[i])
    return best


CONFIGS = {1: config1, 2: config2, 3: config3, 4: config4}
