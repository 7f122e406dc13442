"""Seeded input generators: crystals, spring-model phonons (omega, e, v_g) and random anharmonic IFC lists.

Recipe = SURVEY.md §8(d) table + §8(c) items 13-18 (restated in DESIGN.md §4).  Everything here is input preparation
on the host; none of the scattering-rate arithmetic lives in this file.

Conventions (SURVEY.md §8 header):
  * mesh N1 x N2 x N3, Gamma-centred, q-point index iq = i1 + N1*(i2 + N2*i3), q = sum_mu (i_mu/N_mu) b_mu
  * branch count nb = 3*natoms, mode index lam = iq*nb + j
  * eigenvector array eig[iq, j, 3*atom+alpha] (complex128), eigenvector of mode j contiguous
  * dynamical matrix in the CELL-OFFSET phase convention D_{ia,jb}(q) = sum_R Phi2(0i,Rj) e^{iq.R}/sqrt(m_i m_j),
    R = integer lattice translation of the cell holding atom j  (item 1: makes e(q+G) = e(q))
  * units: omega rad/ps, v_g Angstrom/ps, lengths Angstrom, masses u, Phi3 eV/A^3, Phi4 eV/A^4
"""
from __future__ import annotations

import itertools
from dataclasses import dataclass, field
from functools import lru_cache

import numpy as np

# CODATA 2018 (exact / recommended)
_E_CHARGE = 1.602176634e-19      # C  -> 1 eV in J
_AMU = 1.66053906660e-27         # kg
#: omega[rad/ps] = RADPS_PER_SQRT_EVA2U * sqrt(eigenvalue[eV / (A^2 u)])
RADPS_PER_SQRT_EVA2U = float(np.sqrt(_E_CHARGE / (1e-20 * _AMU)) * 1e-12)

BASE_SEED = 251000518            # item 18: default_rng(BASE_SEED + config_index)

CONFIG_NAMES = {
    0: "diamond 4x4x4 3ph all modes",
    1: "diamond 16x16x16 3ph all modes",
    2: "diamond 8x8x8 4ph, 32 target q x 6 branches",
    3: "diamond 16x16x16 4ph 16 target q x 6 branches + 3ph all modes + kappa",
    4: "sc8 (8 atoms, 24 branches): 3ph 12x12x12 all modes; 4ph 6x6x6 8 target q x 24 branches",
    # the paper's own mesh sizes on the diamond crystal of configs 0-3 -- not BASELINE.json configs:
    5: "paper mesh: diamond 32x32x32 3ph all 196,608 modes",
    6: "paper mesh: diamond 10x10x10 3ph all modes + kappa + 4ph 32 target q x 6 branches",
    7: "paper mesh: diamond 14x14x14 3ph all modes + kappa + 4ph 16 target q x 6 branches",
}
PAPER_MESHES = {5: (32, 32, 32), 6: (10, 10, 10), 7: (14, 14, 14)}


# ------------------------------------------------------------------------------------------------------------------
# crystals
# ------------------------------------------------------------------------------------------------------------------
@dataclass
class Crystal:
    lattvec: np.ndarray          # (3,3) rows a1,a2,a3, Cartesian, Angstrom
    positions: np.ndarray        # (natoms,3) Cartesian, Angstrom
    masses: np.ndarray           # (natoms,) u
    name: str = ""

    @property
    def natoms(self) -> int:
        return int(self.positions.shape[0])

    @property
    def volume(self) -> float:
        return float(abs(np.dot(self.lattvec[0], np.cross(self.lattvec[1], self.lattvec[2]))))


def diamond_crystal(a: float = 5.43, mass: float = 28.0855) -> Crystal:
    """Si-like diamond fcc, 2-atom cell (BASELINE.json config 0)."""
    lat = 0.5 * a * np.array([[0.0, 1.0, 1.0], [1.0, 0.0, 1.0], [1.0, 1.0, 0.0]])
    pos = np.array([[0.0, 0.0, 0.0], [0.25 * a, 0.25 * a, 0.25 * a]])
    return Crystal(lat, pos, np.array([mass, mass]), "diamond")


def sc8_crystal(rng: np.random.Generator, a: float = 6.0) -> Crystal:
    """Config 4: 8-atom simple-cubic cell, atoms on the 2x2x2 sub-grid + jitter U(-0.1,0.1) A (item 16).

    Draw order (item 18): jitter (8x3, row-major), then masses (8)."""
    grid = np.array([[x, y, z] for z in (0, 1) for y in (0, 1) for x in (0, 1)], dtype=float) * (a / 2.0)
    jitter = rng.uniform(-0.1, 0.1, size=(8, 3))
    masses = rng.uniform(20.0, 140.0, size=8)
    return Crystal(a * np.eye(3), grid + jitter, masses, "sc8")


def sc1_crystal(a: float = 3.0, mass: float = 30.0) -> Crystal:
    """1-atom simple-cubic test cell (closed-form |V|^2 pin)."""
    return Crystal(a * np.eye(3), np.zeros((1, 3)), np.array([mass]), "sc1")


# ------------------------------------------------------------------------------------------------------------------
# neighbours, harmonic spring model, phonons
# ------------------------------------------------------------------------------------------------------------------
def _sites_within(cr: Crystal, cutoff: float, nmax: int = 4):
    """For each basis atom i (cell 0): sorted list of sites (j, (n1,n2,n3)) with |tau_j + R - tau_i| <= cutoff,
    including the atom itself.  Returns (sites[i] list, vec dict)."""
    out = []
    for i in range(cr.natoms):
        lst = []
        for n in itertools.product(range(-nmax, nmax + 1), repeat=3):
            R = n[0] * cr.lattvec[0] + n[1] * cr.lattvec[1] + n[2] * cr.lattvec[2]
            for j in range(cr.natoms):
                d = np.linalg.norm(cr.positions[j] + R - cr.positions[i])
                if d <= cutoff + 1e-9:
                    lst.append((j, tuple(int(x) for x in n)))
        out.append(sorted(lst))
    return out


def _site_pos(cr: Crystal, site):
    j, n = site
    return cr.positions[j] + n[0] * cr.lattvec[0] + n[1] * cr.lattvec[1] + n[2] * cr.lattvec[2]


def spring_fc2(cr: Crystal, cutoff: float, kfun, trans_ratio: float = 0.0):
    """Second-order force constants of a bond-spring model.

    Every pair (i in cell 0, site (j,R)) with 0 < d <= cutoff is a bond with longitudinal stiffness k = kfun(key, d)
    (key = canonical undirected-bond key) and transverse stiffness trans_ratio*k (Born form, item 16):
        K = k rr^T + trans_ratio*k (1 - rr^T),  Phi2(0i,Rj) = -K,  Phi2(0i,0i) += +K   (translation invariance).
    Returns list of (i, j, cell(3), 3x3).  Bond keys are visited in sorted order so that seeded draws are reproducible.
    """
    sites = _sites_within(cr, cutoff)
    bonds = {}
    for i in range(cr.natoms):
        for (j, n) in sites[i]:
            if j == i and n == (0, 0, 0):
                continue
            key = min((i, j, n), (j, i, tuple(-x for x in n)))
            bonds.setdefault(key, None)
    kval = {}
    for key in sorted(bonds):
        i, j, n = key
        d = float(np.linalg.norm(_site_pos(cr, (j, n)) - cr.positions[i]))
        kval[key] = float(kfun(key, d))
    fc = {}
    for i in range(cr.natoms):
        for (j, n) in sites[i]:
            if j == i and n == (0, 0, 0):
                continue
            key = min((i, j, n), (j, i, tuple(-x for x in n)))
            k = kval[key]
            r = _site_pos(cr, (j, n)) - cr.positions[i]
            rh = r / np.linalg.norm(r)
            K = k * np.outer(rh, rh) + trans_ratio * k * (np.eye(3) - np.outer(rh, rh))
            fc[(i, j, n)] = fc.get((i, j, n), np.zeros((3, 3))) - K
            fc[(i, i, (0, 0, 0))] = fc.get((i, i, (0, 0, 0)), np.zeros((3, 3))) + K
    return [(i, j, n, m) for (i, j, n), m in sorted(fc.items(), key=lambda kv: kv[0])]


def qpoint_coords(mesh):
    """(N,3) integer mesh coordinates (i1,i2,i3) of q-point iq = i1 + N1*(i2 + N2*i3)."""
    N1, N2, N3 = (int(x) for x in mesh)
    iq = np.arange(N1 * N2 * N3)
    return np.stack([iq % N1, (iq // N1) % N2, iq // (N1 * N2)], axis=1)


def qpoint_index(coords, mesh):
    N1, N2, N3 = (int(x) for x in mesh)
    c = np.asarray(coords)
    return (c[..., 0] % N1) + N1 * ((c[..., 1] % N2) + N2 * (c[..., 2] % N3))


def phonons(cr: Crystal, fc2, mesh):
    """Diagonalise the spring-model dynamical matrix on the mesh -> omega (N,nb), eig (N,nb,nb), vg (N,nb,3).

    Item 17: one of each +-q pair is diagonalised and e(-q) = conj(e(q)), v(-q) = -v(q); real eigenvectors where
    q == -q; v_g is the Hellmann-Feynman diagonal e^H (dD/dq) e / (2 omega) in the stored basis.
    Item 8: the three acoustic omegas at Gamma are set to exactly 0.0.
    """
    mesh = np.asarray(mesh, dtype=np.int64)
    N = int(np.prod(mesh))
    nat = cr.natoms
    nb = 3 * nat
    coords = qpoint_coords(mesh)
    frac = coords / mesh[None, :]
    cells = np.array([n for (_, _, n, _) in fc2], dtype=float)            # (P,3)
    Rcart = cells @ cr.lattvec                                            # (P,3)
    blocks = np.zeros((len(fc2), nb, nb))
    for p, (i, j, n, m) in enumerate(fc2):
        blocks[p, 3 * i:3 * i + 3, 3 * j:3 * j + 3] = m / np.sqrt(cr.masses[i] * cr.masses[j])
    omega = np.zeros((N, nb))
    eig = np.zeros((N, nb, nb), dtype=np.complex128)
    vg = np.zeros((N, nb, 3))
    minus = qpoint_index(-coords, mesh)
    for iq in range(N):
        im = int(minus[iq])
        if im < iq:
            omega[iq] = omega[im]
            eig[iq] = np.conj(eig[im])
            vg[iq] = -vg[im]
            continue
        ph = np.exp(2j * np.pi * (cells @ frac[iq]))                      # (P,)
        D = np.tensordot(ph, blocks, axes=(0, 0))
        D = 0.5 * (D + D.conj().T)
        if im == iq:
            w2, vec = np.linalg.eigh(D.real)
            vec = vec.astype(np.complex128)
        else:
            w2, vec = np.linalg.eigh(D)
        w = RADPS_PER_SQRT_EVA2U * np.sqrt(np.maximum(w2, 0.0))
        if iq == 0:
            w[:3] = 0.0
        omega[iq] = w
        eig[iq] = vec.T                                                   # eig[iq, j, comp]
        for a in range(3):
            dD = np.tensordot(1j * Rcart[:, a] * ph, blocks, axes=(0, 0))
            dD = 0.5 * (dD + dD.conj().T)
            hf = np.real(np.einsum("cj,cd,dj->j", vec.conj(), dD, vec))
            with np.errstate(divide="ignore", invalid="ignore"):
                vg[iq, :, a] = np.where(w > 0, RADPS_PER_SQRT_EVA2U ** 2 * hf / (2.0 * np.where(w > 0, w, 1.0)), 0.0)
        if im == iq:
            vg[iq] = 0.0          # exact: dD/dq is i*antisymmetric there, real eigenvectors give 0 (item 20)
    return omega, eig, vg


# ------------------------------------------------------------------------------------------------------------------
# anharmonic cluster lists and random, symmetrised, sum-rule-compliant entries
# ------------------------------------------------------------------------------------------------------------------
def clusters(cr: Crystal, cutoff: float, order: int):
    """All clusters (i in cell 0; order-1 further sites) whose pairwise distances are all <= cutoff (item 13).

    Returns atoms (n,order) int32 and cells (n,order-1,3) int32 in sorted-cluster order."""
    sites = _sites_within(cr, cutoff)
    out = []
    for i in range(cr.natoms):
        S = sites[i]
        P = [_site_pos(cr, s) for s in S]
        ok = np.array([[np.linalg.norm(P[a] - P[b]) <= cutoff + 1e-9 for b in range(len(S))] for a in range(len(S))])
        for combo in itertools.product(range(len(S)), repeat=order - 1):
            if all(ok[a, b] for a, b in itertools.combinations(combo, 2)):
                out.append((i,) + tuple(S[c] for c in combo))
    out.sort()
    atoms = np.array([[c[0]] + [s[0] for s in c[1:]] for c in out], dtype=np.int32)
    cells = np.array([[s[1] for s in c[1:]] for c in out], dtype=np.int32).reshape(len(out), order - 1, 3)
    return atoms, cells


def _cluster_keys(atoms, cells):
    order = atoms.shape[1]
    return [tuple([(int(atoms[c, 0]), (0, 0, 0))] +
                  [(int(atoms[c, m]), tuple(int(x) for x in cells[c, m - 1])) for m in range(1, order)])
            for c in range(atoms.shape[0])]


def symmetry_maps(atoms, cells):
    """Index maps of the leg-permutation action (with re-anchoring to cell 0) and the sum-rule groups.

    Returns (img, gid): img[p] is an int array over flat entries (cluster*ncomp + comp) giving the entry that
    permutation p maps each entry to; gid[cluster] = id of the group {all clusters equal except for the last leg}."""
    order = atoms.shape[1]
    ncomp = 3 ** order
    keys = _cluster_keys(atoms, cells)
    index = {k: c for c, k in enumerate(keys)}
    n = len(keys)
    comp_tuples = list(itertools.product(range(3), repeat=order))
    comp_index = {t: a for a, t in enumerate(comp_tuples)}
    img = []
    for perm in itertools.permutations(range(order)):
        cmap = np.empty(n, dtype=np.int64)
        for c, k in enumerate(keys):
            legs = [k[m] for m in perm]
            s = legs[0][1]
            newk = tuple((a, (R[0] - s[0], R[1] - s[1], R[2] - s[2])) for (a, R) in legs)
            cmap[c] = index[newk]          # KeyError here would mean the cluster set is not closed (item 13)
        cperm = np.array([comp_index[tuple(t[m] for m in perm)] for t in comp_tuples], dtype=np.int64)
        img.append((cmap[:, None] * ncomp + cperm[None, :]).reshape(-1))
    gids = {}
    gid = np.empty(n, dtype=np.int64)
    for c, k in enumerate(keys):
        gid[c] = gids.setdefault(k[:-1], len(gids))
    return img, gid


def random_ifc(atoms, cells, sigma: float, rng: np.random.Generator, tol: float = 1e-12, maxit: int = 20000):
    """Raw N(0,sigma) entries (sorted-cluster x row-major component order), then alternate the two linear projections
    (acoustic sum rule over the last leg; average over leg permutations) until both residuals < tol, finishing on the
    permutation step (item 15).  Returns phi (n, 3**order) float64."""
    order = atoms.shape[1]
    ncomp = 3 ** order
    n = atoms.shape[0]
    phi = rng.normal(0.0, sigma, size=(n, ncomp))
    img, gid = symmetry_maps(atoms, cells)
    ng = int(gid.max()) + 1
    cnt = np.bincount(gid, minlength=ng).astype(float)

    def group_sums(p):
        s = np.zeros((ng, ncomp))
        np.add.at(s, gid, p)
        return s

    for _ in range(maxit):
        s = group_sums(phi)
        phi = phi - (s / cnt[:, None])[gid]
        flat = phi.reshape(-1)
        acc = np.zeros_like(flat)
        for m in img:
            acc += flat[m]
        phi = (acc / len(img)).reshape(n, ncomp)
        if np.abs(group_sums(phi)).max() < tol:
            break
    else:
        raise RuntimeError("IFC projection did not converge")
    return phi


# ------------------------------------------------------------------------------------------------------------------
# configs
# ------------------------------------------------------------------------------------------------------------------
@dataclass
class Inputs:
    """One fp_setup worth of inputs (one crystal, one mesh)."""
    name: str
    crystal: Crystal
    mesh: np.ndarray                      # (3,) int32
    omega: np.ndarray                     # (N,nb)
    eig: np.ndarray                       # (N,nb,nb) complex128
    vg: np.ndarray                        # (N,nb,3)
    ifc3: tuple | None = None             # (atoms (n,3) i32, cells (n,2,3) i32, phi (n,27) f64)
    ifc4: tuple | None = None             # (atoms (n,4), cells (n,3,3), phi (n,81))
    targets3: np.ndarray | None = None    # mode indices (int32) for the 3ph job, or None
    targets4: np.ndarray | None = None    # mode indices (int32) for the 4ph job, or None
    T: float = 300.0
    scale: float = 1.0
    extra: dict = field(default_factory=dict)

    @property
    def nq(self) -> int:
        return int(np.prod(self.mesh))

    @property
    def nb(self) -> int:
        return 3 * self.crystal.natoms


def _diamond_fc2(cr):
    def kfun(key, d):
        return 10.0 if d < 3.0 else 1.0        # k1 (2.351 A shell), k2 (3.840 A shell), eV/A^2
    return spring_fc2(cr, 4.0, kfun, trans_ratio=0.0)


@lru_cache(maxsize=None)
def _diamond_ifc3():
    cr = diamond_crystal()
    atoms, cells = clusters(cr, 4.0, 3)
    rng = np.random.default_rng(BASE_SEED + 0)           # "IFC3 as config 0" for configs 1 and 3
    return atoms, cells, random_ifc(atoms, cells, 5.0, rng)


@lru_cache(maxsize=None)
def _diamond_ifc4():
    cr = diamond_crystal()
    atoms, cells = clusters(cr, 2.5, 4)
    rng = np.random.default_rng(BASE_SEED + 2)           # config 2's stream: IFC4 entries, then config 2's targets
    phi = random_ifc(atoms, cells, 20.0, rng)
    targets2 = _target_modes(rng, 512, 32, 6)
    return atoms, cells, phi, targets2


@lru_cache(maxsize=None)
def _diamond_phonons(mesh):
    cr = diamond_crystal()
    return phonons(cr, _diamond_fc2(cr), mesh)


def _target_modes(rng, N, nq_targets, nb):
    """targets = sorted rng.choice(N, n, replace=False) q-points, all branches (item 18)."""
    qs = np.sort(rng.choice(N, nq_targets, replace=False))
    return (qs[:, None] * nb + np.arange(nb)[None, :]).reshape(-1).astype(np.int32)


@lru_cache(maxsize=None)
def _sc8_parts():
    rng = np.random.default_rng(BASE_SEED + 4)
    cr = sc8_crystal(rng)                                              # jitter, masses

    def kfun(key, d):
        return rng.uniform(2.0, 12.0)                                  # spring constants in sorted-bond order
    fc2 = spring_fc2(cr, 3.5, kfun, trans_ratio=0.2)
    a3, c3 = clusters(cr, 4.5, 3)
    p3 = random_ifc(a3, c3, 4.0, rng)                                  # IFC3
    a4, c4 = clusters(cr, 3.5, 4)
    p4 = random_ifc(a4, c4, 15.0, rng)                                 # IFC4
    t4 = _target_modes(rng, 216, 8, 24)                                # targets on the 6x6x6 mesh
    return cr, fc2, (a3, c3, p3), (a4, c4, p4), t4


def make_config(idx: int):
    """BASELINE.json config idx -> dict job-name -> Inputs  (jobs: '3ph', '4ph'; one mesh per Inputs)."""
    if idx in (0, 1, 2, 3):
        cr = diamond_crystal()
        mesh = {0: (4, 4, 4), 1: (16, 16, 16), 2: (8, 8, 8), 3: (16, 16, 16)}[idx]
        om, eg, vg = _diamond_phonons(mesh)
        N = int(np.prod(mesh))
        inp = Inputs(CONFIG_NAMES[idx], cr, np.array(mesh, dtype=np.int32), om, eg, vg)
        all_modes = np.arange(N * 6, dtype=np.int32)
        if idx in (0, 1, 3):
            inp.ifc3 = _diamond_ifc3()
            inp.targets3 = all_modes
        if idx in (2, 3):
            a4, c4, p4, t2 = _diamond_ifc4()
            inp.ifc4 = (a4, c4, p4)
            if idx == 2:
                inp.targets4 = t2
            else:                                  # config 3 reuses IFC3 (seed+0) and IFC4 (seed+2); its own stream
                rng = np.random.default_rng(BASE_SEED + 3)        # draws only its 16 target q-points
                inp.targets4 = _target_modes(rng, N, 16, 6)
        return {"main": inp}
    if idx in PAPER_MESHES:                        # same crystal, IFC3 (seed+0) and IFC4 (seed+2) as configs 0-3
        cr = diamond_crystal()
        mesh = PAPER_MESHES[idx]
        om, eg, vg = _diamond_phonons(mesh)
        N = int(np.prod(mesh))
        inp = Inputs(CONFIG_NAMES[idx], cr, np.array(mesh, dtype=np.int32), om, eg, vg)
        inp.ifc3 = _diamond_ifc3()
        inp.targets3 = np.arange(N * 6, dtype=np.int32)
        if idx != 5:
            a4, c4, p4, _ = _diamond_ifc4()
            inp.ifc4 = (a4, c4, p4)
            rng = np.random.default_rng(BASE_SEED + idx)          # draws only the target q-points
            inp.targets4 = _target_modes(rng, N, 32 if idx == 6 else 16, 6)
        return {"main": inp}
    if idx == 4:
        cr, fc2, i3, i4, t4 = _sc8_parts()
        om3, eg3, vg3 = phonons(cr, fc2, (12, 12, 12))
        om4, eg4, vg4 = phonons(cr, fc2, (6, 6, 6))
        j3 = Inputs(CONFIG_NAMES[4] + " [3ph]", cr, np.array((12, 12, 12), dtype=np.int32), om3, eg3, vg3, ifc3=i3,
                    targets3=np.arange(1728 * 24, dtype=np.int32))
        j4 = Inputs(CONFIG_NAMES[4] + " [4ph]", cr, np.array((6, 6, 6), dtype=np.int32), om4, eg4, vg4, ifc4=i4,
                    targets4=t4)
        return {"3ph": j3, "4ph": j4}
    raise ValueError(f"unknown config {idx}")


def make_tiny(kind: str, mesh=(3, 3, 3), seed: int = 7, with4: bool = True):
    """Small cases for oracle pins and parity tests.

    kind: 'diamond' (config-0 crystal and IFC lists on a small mesh), 'sc1' (1-atom cell, random IFCs within the
    first shell), 'sc8' (config-4 crystal on a small mesh)."""
    mesh = tuple(int(x) for x in mesh)
    N = int(np.prod(mesh))
    if kind == "diamond":
        cr = diamond_crystal()
        om, eg, vg = _diamond_phonons(mesh)
        inp = Inputs(f"tiny diamond {mesh}", cr, np.array(mesh, dtype=np.int32), om, eg, vg,
                     ifc3=_diamond_ifc3(), ifc4=_diamond_ifc4()[:3] if with4 else None)
    elif kind == "sc1":
        cr = sc1_crystal()
        rng = np.random.default_rng(seed)
        fc2 = spring_fc2(cr, 3.1, lambda key, d: 6.0, trans_ratio=0.3)
        om, eg, vg = phonons(cr, fc2, mesh)
        a3, c3 = clusters(cr, 3.1, 3)
        a4, c4 = clusters(cr, 3.1, 4)
        inp = Inputs(f"tiny sc1 {mesh}", cr, np.array(mesh, dtype=np.int32), om, eg, vg,
                     ifc3=(a3, c3, random_ifc(a3, c3, 5.0, rng)),
                     ifc4=(a4, c4, random_ifc(a4, c4, 20.0, rng)) if with4 else None)
    elif kind == "sc8":
        cr, fc2, i3, i4, _ = _sc8_parts()
        om, eg, vg = phonons(cr, fc2, mesh)
        inp = Inputs(f"tiny sc8 {mesh}", cr, np.array(mesh, dtype=np.int32), om, eg, vg, ifc3=i3,
                     ifc4=i4 if with4 else None)
    else:
        raise ValueError(kind)
    inp.targets3 = np.arange(N * inp.nb, dtype=np.int32)
    inp.targets4 = np.arange(N * inp.nb, dtype=np.int32)
    return inp
