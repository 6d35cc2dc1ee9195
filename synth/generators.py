"""Seeded generators for the synthetic C-PCM workloads.

The paper measures on PDB proteins with 6-31G / 6-31G* and Lebedev grids
(PAPER.md:106, 114, 222); none of those data are available offline, so the
BASELINE.json configs replace them with the seeded recipe below (SURVEY.md
section 8(d), restated in DESIGN.md).  Everything returned is in atomic units
(bohr); the recipe's Angstrom figures are converted with ANGSTROM.

Nothing here evaluates the method (no integrals, no Boys function, no A
entries).  The only closed forms used are same-centre Gaussian self-overlaps,
needed to fold the normalisation into ``prim_coef`` as the C ABI expects
("prim_coef multiplies the raw primitive x^i y^j z^k exp(-a r^2)").
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field

import numpy as np

ANGSTROM = 1.8897261246  # bohr per Angstrom

# van der Waals (Bondi) radii in Angstrom, as listed in BASELINE.json configs[0]
_VDW = {"H": 1.20, "C": 1.70, "N": 1.55, "O": 1.52}
_Z = {"H": 1.0, "C": 6.0, "N": 7.0, "O": 8.0}


def cavity_radii(elements) -> np.ndarray:
    """Cavity radius of every atom in bohr: 1.2 x the van der Waals radius, as make_surface uses."""
    return np.array([_CAVITY_SCALE * _VDW[e] * ANGSTROM for e in elements], dtype=np.float64)


def nuclear_charges(elements) -> np.ndarray:
    """The vector z of Eq. 1 (nuclear charges of the solute's atoms)."""
    return np.array([_Z[e] for e in elements], dtype=np.float64)
_CAVITY_SCALE = 1.2          # PAPER.md:106 "20% larger than the Bondi radii"
_ZETA_TABLE_STANDIN = 4.9    # stands in for the tabulated zeta of Eq. 7

# atoms, surface points per atom, d shells?  per BASELINE.json configs[0..3]
CONFIG_ATOMS = {
    0: dict(n_atoms=12, n_pts=50, with_d=False),
    1: dict(n_atoms=300, n_pts=110, with_d=False),
    2: dict(n_atoms=1000, n_pts=110, with_d=False),
    3: dict(n_atoms=2000, n_pts=194, with_d=True),
}


@dataclass
class Basis:
    """Shell list in the layout ``pcm_setup`` takes (include/pcm.h)."""
    shell_l: np.ndarray       # int32 [nshell]  0,1,2
    shell_xyz: np.ndarray     # float64 [nshell,3] bohr
    shell_nprim: np.ndarray   # int32 [nshell]
    prim_exp: np.ndarray      # float64 [nprim_total]
    prim_coef: np.ndarray     # float64 [nprim_total], multiplies RAW primitives
    shell_atom: np.ndarray    # int32 [nshell] (bookkeeping only)
    d_pure: bool = True

    @property
    def nshell(self) -> int:
        return int(self.shell_l.shape[0])

    @property
    def ncomp(self) -> np.ndarray:
        nd = 5 if self.d_pure else 6
        return np.where(self.shell_l == 0, 1, np.where(self.shell_l == 1, 3, nd)).astype(np.int32)

    @property
    def bf_offset(self) -> np.ndarray:
        off = np.zeros(self.nshell + 1, dtype=np.int64)
        np.cumsum(self.ncomp, out=off[1:])
        return off

    @property
    def nbf(self) -> int:
        return int(self.ncomp.sum())

    @property
    def prim_offset(self) -> np.ndarray:
        off = np.zeros(self.nshell + 1, dtype=np.int64)
        np.cumsum(self.shell_nprim, out=off[1:])
        return off

    def subset(self, shells) -> "Basis":
        """Basis restricted to the listed shells (keeps order)."""
        shells = np.asarray(shells, dtype=np.int64)
        po = self.prim_offset
        idx = np.concatenate([np.arange(po[s], po[s + 1]) for s in shells]) if len(shells) else np.zeros(0, np.int64)
        return Basis(self.shell_l[shells].copy(), self.shell_xyz[shells].copy(), self.shell_nprim[shells].copy(),
                     self.prim_exp[idx].copy(), self.prim_coef[idx].copy(), self.shell_atom[shells].copy(), self.d_pure)


@dataclass
class Surface:
    """Molecular-surface (MS) points: positions, Gaussian exponents, switching values."""
    xyz: np.ndarray      # float64 [M,3] bohr
    zeta: np.ndarray     # float64 [M] bohr^-1   (Eq. 7)
    switch: np.ndarray   # float64 [M] S_k in (0,1]  (enters A_kk only, Eq. 3)
    atom: np.ndarray     # int32 [M] owning atom (bookkeeping only)

    @property
    def M(self) -> int:
        return int(self.xyz.shape[0])

    def subset(self, idx) -> "Surface":
        idx = np.asarray(idx, dtype=np.int64)
        return Surface(self.xyz[idx].copy(), self.zeta[idx].copy(), self.switch[idx].copy(), self.atom[idx].copy())


@dataclass
class Workload:
    name: str
    config: int
    seed: int
    elements: list
    atom_xyz: np.ndarray
    basis: Basis
    surface: Surface
    q: np.ndarray
    P: np.ndarray | None = None
    meta: dict = field(default_factory=dict)


# --------------------------------------------------------------------------- geometry
def make_chain(rng: np.random.Generator, n_atoms: int) -> np.ndarray:
    """Random chain, Angstrom recipe -> bohr.

    Atom 0 at the origin; bond length U[1.0,1.5] A, bond angle U[100,120] deg,
    dihedral U[0,2pi).  A draw is rejected (<=200 retries, then the draw with
    the largest clearance is kept) if the new atom is closer than 2.0 A to any
    atom other than its two predecessors.
    """
    xyz = np.zeros((n_atoms, 3))
    if n_atoms > 1:
        xyz[1] = [rng.uniform(1.0, 1.5), 0.0, 0.0]
    for i in range(2, n_atoms):
        best, best_clear = None, -1.0
        for _ in range(200):
            b = rng.uniform(1.0, 1.5)
            theta = math.radians(rng.uniform(100.0, 120.0))
            phi = rng.uniform(0.0, 2.0 * math.pi)
            p1, p2 = xyz[i - 1], xyz[i - 2]
            e1 = p1 - p2
            e1 /= np.linalg.norm(e1)
            if i >= 3:
                ref = xyz[i - 2] - xyz[i - 3]
            else:
                ref = np.array([0.0, 1.0, 0.0])
            n = np.cross(e1, ref)
            if np.linalg.norm(n) < 1e-8:
                n = np.cross(e1, np.array([0.0, 0.0, 1.0]))
                if np.linalg.norm(n) < 1e-8:
                    n = np.cross(e1, np.array([0.0, 1.0, 0.0]))
            n /= np.linalg.norm(n)
            m = np.cross(n, e1)
            # bond angle theta is the angle (i-2, i-1, i)
            d = -math.cos(theta) * e1 + math.sin(theta) * (math.cos(phi) * m + math.sin(phi) * n)
            cand = p1 + b * d
            if i > 2:
                clear = float(np.min(np.linalg.norm(xyz[: i - 2] - cand, axis=1)))
            else:
                clear = np.inf
            if clear >= 2.0:
                best = cand
                break
            if clear > best_clear:
                best, best_clear = cand, clear
        xyz[i] = best
    return xyz * ANGSTROM


def _elements(rng: np.random.Generator, config: int, n_atoms: int) -> list:
    if config == 0:
        n_heavy = 4
    else:
        n_heavy = n_atoms // 2
    heavy = list(rng.choice(["C", "N", "O"], size=n_heavy, p=[0.6, 0.2, 0.2]))
    el = heavy + ["H"] * (n_atoms - n_heavy)
    order = rng.permutation(n_atoms)
    return [el[j] for j in order]


# --------------------------------------------------------------------------- basis
def _dfact(n: int) -> int:
    return 1 if n <= 0 else n * _dfact(n - 2)


def _first_component_overlap(l: int, p: float) -> float:
    """Self-overlap integral of the first component of an l shell for a product
    exponent p (same centre): s: 1; p: x; d: sqrt(3) xy (pure) -- and xx for
    Cartesian d, which has the same value 3/(4 p^2) (pi/p)^1.5."""
    base = (math.pi / p) ** 1.5
    if l == 0:
        return base
    if l == 1:
        return base / (2.0 * p)
    return 3.0 * base / (4.0 * p * p)


def _contract(rng: np.random.Generator, l: int, exps: np.ndarray) -> np.ndarray:
    """raw U[0.1,1] coefficients x primitive normalisation, contracted function
    scaled to unit self-overlap of its first component."""
    raw = rng.uniform(0.1, 1.0, size=len(exps))
    # primitive normalisation of x^l exp(-a r^2): 1/sqrt( (2l-1)!!/(4a)^l (pi/2a)^1.5 )
    norm = np.array([1.0 / math.sqrt(_dfact(2 * l - 1) / (4.0 * a) ** l * (math.pi / (2.0 * a)) ** 1.5) for a in exps])
    c = raw * norm
    s = 0.0
    for i, ai in enumerate(exps):
        for j, aj in enumerate(exps):
            s += c[i] * c[j] * _first_component_overlap(l, ai + aj)
    return c / math.sqrt(s)


def make_basis(rng: np.random.Generator, elements: list, atom_xyz: np.ndarray, with_d: bool,
               d_pure: bool = True) -> Basis:
    """6-31G-shaped shells with seeded exponents: heavy = s(6) + sp(3) + sp(1)
    [+ d(1), exponent 0.8]; H = s(3) + s(1).  Exponents iid log-uniform on
    [0.1, 5000] bohr^-2, sorted descending within a shell; an sp shell is
    emitted as an s shell and a p shell with equal exponents."""
    L, X, NP, E, C, AT = [], [], [], [], [], []

    def draw(n):
        e = np.exp(rng.uniform(math.log(0.1), math.log(5000.0), size=n))
        return np.sort(e)[::-1].copy()

    def emit(l, exps, atom):
        L.append(l)
        X.append(atom_xyz[atom])
        NP.append(len(exps))
        E.extend(exps.tolist())
        C.extend(_contract(rng, l, exps).tolist())
        AT.append(atom)

    for a, el in enumerate(elements):
        if el == "H":
            emit(0, draw(3), a)
            emit(0, draw(1), a)
        else:
            emit(0, draw(6), a)
            for n in (3, 1):
                e = draw(n)
                emit(0, e, a)
                emit(1, e, a)
            if with_d:
                emit(2, np.array([0.8]), a)
    return Basis(np.array(L, np.int32), np.array(X, np.float64).reshape(-1, 3), np.array(NP, np.int32),
                 np.array(E, np.float64), np.array(C, np.float64), np.array(AT, np.int32), d_pure)


# --------------------------------------------------------------------------- surface
def make_surface(rng: np.random.Generator, elements: list, atom_xyz: np.ndarray, n_pts: int) -> Surface:
    """n_pts Fibonacci-lattice points per atom on spheres of 1.2 x vdW radius;
    points strictly inside another atom's sphere are dropped; equal weights
    w = 4 pi / n_pts; zeta_k = 4.9 / (R_I sqrt(w)) (Eq. 7);
    S_k iid U[0.1, 1] (configs[4]; used only by A_kk)."""
    from scipy.spatial import cKDTree

    radii = np.array([_CAVITY_SCALE * _VDW[e] * ANGSTROM for e in elements])
    n = np.arange(n_pts)
    z = 1.0 - (2.0 * n + 1.0) / n_pts
    phi = n * math.pi * (3.0 - math.sqrt(5.0))
    s = np.sqrt(np.maximum(0.0, 1.0 - z * z))
    unit = np.stack([s * np.cos(phi), s * np.sin(phi), z], axis=1)
    tree = cKDTree(atom_xyz)
    rmax = float(radii.max())
    w = 4.0 * math.pi / n_pts
    pts, zet, own = [], [], []
    for a in range(len(elements)):
        p = atom_xyz[a] + radii[a] * unit
        keep = np.ones(n_pts, dtype=bool)
        for b in tree.query_ball_point(atom_xyz[a], radii[a] + rmax):
            if b == a:
                continue
            keep &= ~(np.linalg.norm(p - atom_xyz[b], axis=1) < radii[b])
        p = p[keep]
        pts.append(p)
        zet.append(np.full(len(p), _ZETA_TABLE_STANDIN / (radii[a] * math.sqrt(w))))
        own.append(np.full(len(p), a, np.int32))
    xyz = np.concatenate(pts)
    sw = rng.uniform(0.1, 1.0, size=len(xyz))
    return Surface(xyz, np.concatenate(zet), sw, np.concatenate(own))


# --------------------------------------------------------------------------- P, q
def make_density(rng: np.random.Generator, nbf: int, max_cols: int = 256) -> np.ndarray:
    """P = C C^T, C iid N(0, 0.1^2) with min(max(1, nbf/4), max_cols) columns
    (BASELINE.json: "C.C^T, C random normal scaled 0.1"; the column count is a
    reading)."""
    ncol = max(1, min(nbf // 4, max_cols))
    Cm = rng.normal(0.0, 0.1, size=(nbf, ncol))
    P = Cm @ Cm.T
    return 0.5 * (P + P.T)


def make_charges(rng: np.random.Generator, M: int) -> np.ndarray:
    return rng.uniform(-0.05, 0.05, size=M)


# --------------------------------------------------------------------------- workloads
def make_workload(config: int, with_density: bool = True, d_pure: bool = True, n_atoms: int | None = None,
                  n_pts: int | None = None, with_d: bool | None = None, seed: int | None = None) -> Workload:
    """BASELINE.json configs[0..3].  ``n_atoms`` / ``n_pts`` / ``with_d`` override the
    config's values (used by tests for reduced-size cases of the same recipe)."""
    spec = dict(CONFIG_ATOMS[config])
    if n_atoms is not None:
        spec["n_atoms"] = n_atoms
    if n_pts is not None:
        spec["n_pts"] = n_pts
    if with_d is not None:
        spec["with_d"] = with_d
    seed = 1000 + config if seed is None else seed
    rng = np.random.Generator(np.random.PCG64(seed))
    xyz = make_chain(rng, spec["n_atoms"])
    el = _elements(rng, config, spec["n_atoms"])
    basis = make_basis(rng, el, xyz, spec["with_d"], d_pure)
    surf = make_surface(rng, el, xyz, spec["n_pts"])
    q = make_charges(rng, surf.M)
    P = make_density(rng, basis.nbf) if with_density else None
    return Workload(name=f"config{config}", config=config, seed=seed, elements=el, atom_xyz=xyz, basis=basis,
                    surface=surf, q=q, P=P, meta=dict(spec))


def make_solver_points(M: int, seed: int = 1004):
    """configs[4]: M points drawn from the configs[3] surface generator on a
    chain long enough to yield >= M points (n_atoms = smallest multiple of 500
    that does), seeded shuffle, first M kept.  Returns (Surface, q, q_true)."""
    n_atoms = 500
    while True:
        rng = np.random.Generator(np.random.PCG64(seed))
        xyz = make_chain(rng, n_atoms)
        el = _elements(rng, 3, n_atoms)
        surf = make_surface(rng, el, xyz, CONFIG_ATOMS[3]["n_pts"])
        if surf.M >= M:
            break
        n_atoms += 500
    order = rng.permutation(surf.M)[:M]
    surf = surf.subset(order)
    q = make_charges(rng, M)
    q_true = make_charges(rng, M)
    return surf, q, q_true
