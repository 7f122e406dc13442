"""Independent brute-force evaluation used ONLY to pin the oracle on tiny inputs (SURVEY.md §8(c) "What pins each part").

Different route from oracle/fp_oracle.c on purpose:
  * momentum conservation is decided by looping over ALL mode tuples and testing q +- q' (+- q'') - q_last == integer
    vector with exact rational arithmetic on the fractional coordinates (no modulo-combine of mesh indices);
  * the matrix element is the textbook "Fourier-transformed force-constant tensor contracted with eigenvectors":
    a dense (nb x nb x nb [x nb]) tensor is assembled with Cartesian phases exp(i q.R) (q = frac @ b, R = n @ a) and
    contracted by numpy.einsum, instead of per-cluster nested loops with integer phases;
  * unit constants are obtained by an explicit SI conversion chain.
Imports nothing from oracle/ or from the CUDA package.
"""
from __future__ import annotations

from fractions import Fraction

import numpy as np

HBAR = 1.054571817e-34
KB = 1.380649e-23
QE = 1.602176634e-19
AMU = 1.66053906660e-27


def si_chain_constants():
    """C3, C4 [1/ps], Ckappa [W/mK per unit], hbar/kB [ps K] by converting each factor to SI and back."""
    ev = QE
    ang = 1e-10
    radps = 1e12
    # Gamma3 [1/s] = (pi hbar / 4) * |V|^2 [ (J/m^3)^2 / kg^3 ] / omega^3 [s^-3] * delta(omega) [s]
    v3_unit = (ev / ang ** 3) ** 2 / AMU ** 3
    c3 = np.pi * HBAR / 4 * v3_unit / radps ** 3 / radps            # 1/s
    v4_unit = (ev / ang ** 4) ** 2 / AMU ** 4
    c4 = np.pi * HBAR ** 2 / 8 * v4_unit / radps ** 4 / radps        # 1/s
    # kappa = 1/(kB T^2 V N) sum f(f+1) (hbar w)^2 v^2 tau
    ck = HBAR ** 2 / KB * radps ** 2 * (ang * radps) ** 2 / radps / ang ** 3
    return c3 * 1e-12, c4 * 1e-12, ck, HBAR / KB * 1e12


def recip_cart(lattvec):
    return 2.0 * np.pi * np.linalg.inv(np.asarray(lattvec)).T        # rows b_mu, b_mu . a_nu = 2 pi delta


def frac_coords(inp):
    from fp_inputs import qpoint_coords
    c = qpoint_coords(inp.mesh)
    return [[Fraction(int(c[i, m]), int(inp.mesh[m])) for m in range(3)] for i in range(c.shape[0])]


def conserves(fr, qs, signs):
    """sum_k signs[k]*q_k is a reciprocal-lattice vector (integer fractional coordinates)."""
    for m in range(3):
        tot = sum(s * fr[q][m] for q, s in zip(qs, signs))
        if tot.denominator != 1:
            return False
    return True


def be(omega, T):
    return 1.0 / np.expm1(HBAR / KB * 1e12 * omega / T)


def _qcart(inp, iq):
    from fp_inputs import qpoint_coords
    c = qpoint_coords(inp.mesh)[iq] / np.asarray(inp.mesh, dtype=float)
    return c @ recip_cart(inp.crystal.lattvec)


def dense3(inp, q1, s1, q2):
    """T[a,b,c] = sum_t Phi_t / sqrt(m m m) exp(i s1 q1.Rj) exp(-i q2.Rk) scattered at (3i+al, 3j+be, 3k+ga)."""
    atoms, cells, phi = inp.ifc3
    nb = inp.nb
    T = np.zeros((nb, nb, nb), dtype=complex)
    k1, k2 = _qcart(inp, q1), _qcart(inp, q2)
    m = inp.crystal.masses
    A = inp.crystal.lattvec
    for t in range(atoms.shape[0]):
        i, j, k = atoms[t]
        Rj, Rk = cells[t, 0] @ A, cells[t, 1] @ A
        ph = np.exp(1j * s1 * (k1 @ Rj)) * np.exp(-1j * (k2 @ Rk)) / np.sqrt(m[i] * m[j] * m[k])
        T[3 * i:3 * i + 3, 3 * j:3 * j + 3, 3 * k:3 * k + 3] += phi[t].reshape(3, 3, 3) * ph
    return T


def dense4(inp, q1, s1, q2, s2, q3):
    atoms, cells, phi = inp.ifc4
    nb = inp.nb
    T = np.zeros((nb, nb, nb, nb), dtype=complex)
    k1, k2, k3 = _qcart(inp, q1), _qcart(inp, q2), _qcart(inp, q3)
    m = inp.crystal.masses
    A = inp.crystal.lattvec
    for t in range(atoms.shape[0]):
        i, j, k, l = atoms[t]
        Rj, Rk, Rl = cells[t, 0] @ A, cells[t, 1] @ A, cells[t, 2] @ A
        ph = (np.exp(1j * s1 * (k1 @ Rj)) * np.exp(1j * s2 * (k2 @ Rk)) * np.exp(-1j * (k3 @ Rl))
              / np.sqrt(m[i] * m[j] * m[k] * m[l]))
        T[3 * i:3 * i + 3, 3 * j:3 * j + 3, 3 * k:3 * k + 3, 3 * l:3 * l + 3] += phi[t].reshape(3, 3, 3, 3) * ph
    return T


def v3_dense(inp, lam, lam1, lam2, s):
    nb = inp.nb
    e0 = inp.eig[lam // nb, lam % nb]
    e1 = inp.eig[lam1 // nb, lam1 % nb]
    e2 = inp.eig[lam2 // nb, lam2 % nb]
    T = dense3(inp, lam1 // nb, s, lam2 // nb)
    return np.einsum("abc,a,b,c->", T, e0, e1 if s > 0 else e1.conj(), e2.conj())


def v4_dense(inp, lam, lam1, lam2, lam3, s1, s2):
    nb = inp.nb
    e = [inp.eig[x // nb, x % nb] for x in (lam, lam1, lam2, lam3)]
    T = dense4(inp, lam1 // nb, s1, lam2 // nb, s2, lam3 // nb)
    return np.einsum("abcd,a,b,c,d->", T, e[0], e[1] if s1 > 0 else e[1].conj(), e[2] if s2 > 0 else e[2].conj(),
                     e[3].conj())


def rates3_bruteforce(inp, lam, sigma, T=300.0):
    """Gamma+, Gamma-, counts for one target with constant sigma and NO energy filter (item 20), all tuples looped."""
    c3 = si_chain_constants()[0]
    fr = frac_coords(inp)
    nb, N = inp.nb, inp.nq
    q = lam // nb
    w = inp.omega.reshape(-1)
    out_g, out_c = [0.0, 0.0], [0, 0]
    if w[lam] == 0:
        return out_g, out_c
    for ch, s in enumerate((+1, -1)):
        for q1 in range(N):
            for q2 in range(N):
                if not conserves(fr, (q, q1, q2), (1, s, -1)):
                    continue
                T3 = dense3(inp, q1, s, q2)
                e0 = inp.eig[q, lam % nb]
                E1 = inp.eig[q1] if s > 0 else inp.eig[q1].conj()           # (j, comp)
                E2 = inp.eig[q2].conj()
                V = np.einsum("abc,a,jb,kc->jk", T3, e0, E1, E2)
                for j1 in range(nb):
                    for j2 in range(nb):
                        w1, w2 = w[q1 * nb + j1], w[q2 * nb + j2]
                        if w1 == 0 or w2 == 0:
                            continue
                        d = w[lam] + s * w1 - w2
                        g = np.exp(-(d / sigma) ** 2) / (sigma * np.sqrt(np.pi))
                        f1, f2 = be(w1, T), be(w2, T)
                        occ = (f1 - f2) if s > 0 else (f1 + f2 + 1.0)
                        out_g[ch] += occ * g / (w[lam] * w1 * w2) * abs(V[j1, j2]) ** 2
                        out_c[ch] += 1
        out_g[ch] *= c3 / N * (1.0 if s > 0 else 0.5)
    return out_g, out_c


def rates4_bruteforce(inp, lam, sigma, T=300.0):
    c4 = si_chain_constants()[1]
    fr = frac_coords(inp)
    nb, N = inp.nb, inp.nq
    q = lam // nb
    w = inp.omega.reshape(-1)
    out_g, out_c = [0.0, 0.0, 0.0], [0, 0, 0]
    if w[lam] == 0:
        return out_g, out_c
    f0 = be(w[lam], T)
    for ch, (s1, s2) in enumerate(((1, 1), (1, -1), (-1, -1))):
        for q1 in range(N):
            for q2 in range(N):
                for q3 in range(N):
                    if not conserves(fr, (q, q1, q2, q3), (1, s1, s2, -1)):
                        continue
                    T4 = dense4(inp, q1, s1, q2, s2, q3)
                    e0 = inp.eig[q, lam % nb]
                    E1 = inp.eig[q1] if s1 > 0 else inp.eig[q1].conj()
                    E2 = inp.eig[q2] if s2 > 0 else inp.eig[q2].conj()
                    E3 = inp.eig[q3].conj()
                    V = np.einsum("abcd,a,jb,kc,ld->jkl", T4, e0, E1, E2, E3)
                    for j1 in range(nb):
                        for j2 in range(nb):
                            for j3 in range(nb):
                                w1, w2, w3 = w[q1 * nb + j1], w[q2 * nb + j2], w[q3 * nb + j3]
                                if w1 == 0 or w2 == 0 or w3 == 0:
                                    continue
                                d = w[lam] + s1 * w1 + s2 * w2 - w3
                                g = np.exp(-(d / sigma) ** 2) / (sigma * np.sqrt(np.pi))
                                f1, f2, f3 = be(w1, T), be(w2, T), be(w3, T)
                                occ = ((1 + f1) if s1 > 0 else f1) * ((1 + f2) if s2 > 0 else f2) * f3 / f0
                                out_g[ch] += occ * g / (w[lam] * w1 * w2 * w3) * abs(V[j1, j2, j3]) ** 2
                                out_c[ch] += 1
        out_g[ch] *= c4 / N ** 2 * (1.0 / 6.0 if ch == 2 else 0.5)
    return out_g, out_c


def list4_bruteforce(inp, lam, ch, scale=1.0, ncut=2.0, T=300.0):
    """Adaptive-sigma 4ph process list of one target and channel by brute force over ALL (q', q'', q''') triples (rational
    momentum test), the window |Delta| <= ncut sigma with sigma = scale sqrt(sum_mu (B_mu . (v'' - v'''))^2 / 6) -- the
    reading of SURVEY.md §8(c) item 2 / DESIGN.md §3-2: the LAST TWO legs -- in plain numpy, and the weighted phase space
    of PAPER.md:163's Gaussian with the "/f" occupation forms (item 5).
    -> (set of (lam1, lam2, lam3), {triple: |Delta| - ncut sigma} for edge checks, WP sum incl. the symmetry weight / N^2)"""
    fr = frac_coords(inp)
    nb, N = inp.nb, inp.nq
    q = lam // nb
    w = inp.omega.reshape(N, nb)
    v = inp.vg.reshape(N, nb, 3)
    Bm = recip_cart(inp.crystal.lattvec) / np.asarray(inp.mesh, float)[:, None]      # rows B_mu = b_mu / N_mu
    s1, s2 = ((1, 1), (1, -1), (-1, -1))[ch]
    w0 = w[q, lam % nb]
    out, margin, wp = set(), {}, 0.0
    if w0 == 0:
        return out, margin, 0.0
    f0 = be(w0, T)
    for q1 in range(N):
        for q2 in range(N):
            for q3 in range(N):
                if not conserves(fr, (q, q1, q2, q3), (1, s1, s2, -1)):
                    continue
                dv = v[q2][:, None, :] - v[q3][None, :, :]                        # (j2, j3, 3): v'' - v'''
                sig = scale * np.sqrt(((dv @ Bm.T) ** 2).sum(axis=-1) / 6.0)       # (j2, j3)
                for j1 in range(nb):
                    w1 = w[q1, j1]
                    if w1 == 0:
                        continue
                    d = w0 + s1 * w1 + s2 * w[q2][:, None] - w[q3][None, :]
                    ok = (sig > 0) & (np.abs(d) <= ncut * sig) & (w[q2][:, None] != 0) & (w[q3][None, :] != 0)
                    f1 = be(w1, T)
                    for j2, j3 in zip(*np.nonzero(ok)):
                        t = (q1 * nb + j1, q2 * nb + int(j2), q3 * nb + int(j3))
                        out.add(t)
                        margin[t] = abs(d[j2, j3]) - ncut * sig[j2, j3]
                        w2, w3 = w[q2, j2], w[q3, j3]
                        f2, f3 = be(w2, T), be(w3, T)
                        occ = ((1 + f1) if s1 > 0 else f1) * ((1 + f2) if s2 > 0 else f2) * f3 / f0
                        g = np.exp(-(d[j2, j3] / sig[j2, j3]) ** 2) / (sig[j2, j3] * np.sqrt(np.pi))
                        wp += occ * g / (w0 * w1 * w2 * w3)
                    # near misses, for the edge rule of the set comparison
                    near = (sig > 0) & ~ok & (np.abs(np.abs(d) - ncut * sig) < 1e-9) & (w[q2][:, None] != 0) & (w[q3][None, :] != 0)
                    for j2, j3 in zip(*np.nonzero(near)):
                        margin[(q1 * nb + j1, q2 * nb + int(j2), q3 * nb + int(j3))] = abs(d[j2, j3]) - ncut * sig[j2, j3]
    return out, margin, wp * (1.0 / 6.0 if ch == 2 else 0.5) / N ** 2


def term4_dense(inp, lam, ch, triple, scale=1.0, T=300.0):
    """Contribution of ONE 4ph process (lam; lam1, lam2, lam3) of channel ch to Gamma(lam), in plain numpy: the dense-Fourier
    matrix element (v4_dense), PAPER.md:163's Gaussian with the adaptive sigma of the last two legs (item 2), the "/f"
    occupation form (item 5), C4/N^2 and the symmetry weight (items 6)."""
    c4 = si_chain_constants()[1]
    nb, N = inp.nb, inp.nq
    lam1, lam2, lam3 = (int(x) for x in triple)
    s1, s2 = ((1, 1), (1, -1), (-1, -1))[ch]
    w = inp.omega.reshape(-1)
    v = inp.vg.reshape(-1, 3)
    Bm = recip_cart(inp.crystal.lattvec) / np.asarray(inp.mesh, float)[:, None]
    sig = scale * np.sqrt((((v[lam2] - v[lam3]) @ Bm.T) ** 2).sum() / 6.0)
    d = w[lam] + s1 * w[lam1] + s2 * w[lam2] - w[lam3]
    g = np.exp(-(d / sig) ** 2) / (sig * np.sqrt(np.pi))
    f0, f1, f2, f3 = (be(w[x], T) for x in (lam, lam1, lam2, lam3))
    occ = ((1 + f1) if s1 > 0 else f1) * ((1 + f2) if s2 > 0 else f2) * f3 / f0
    V = v4_dense(inp, lam, lam1, lam2, lam3, s1, s2)
    return c4 / N ** 2 * (1.0 / 6.0 if ch == 2 else 0.5) * occ * g / (w[lam] * w[lam1] * w[lam2] * w[lam3]) * abs(V) ** 2


def term3_dense(inp, lam, ch, pair, scale=1.0, T=300.0):
    """The same for one 3ph process (lam; lam1, lam2): sigma from v' - v'', occupation f' - f'' (+) or f' + f'' + 1 (-)."""
    c3 = si_chain_constants()[0]
    N = inp.nq
    lam1, lam2 = (int(x) for x in pair)
    s = 1 if ch == 0 else -1
    w = inp.omega.reshape(-1)
    v = inp.vg.reshape(-1, 3)
    Bm = recip_cart(inp.crystal.lattvec) / np.asarray(inp.mesh, float)[:, None]
    sig = scale * np.sqrt((((v[lam1] - v[lam2]) @ Bm.T) ** 2).sum() / 6.0)
    d = w[lam] + s * w[lam1] - w[lam2]
    g = np.exp(-(d / sig) ** 2) / (sig * np.sqrt(np.pi))
    f1, f2 = be(w[lam1], T), be(w[lam2], T)
    occ = (f1 - f2) if s > 0 else (f1 + f2 + 1.0)
    V = v3_dense(inp, lam, lam1, lam2, s)
    return c3 / N * (1.0 if ch == 0 else 0.5) * occ * g / (w[lam] * w[lam1] * w[lam2]) * abs(V) ** 2
