"""Pins of the CPU oracle against what the paper and the mathematics fix (SURVEY.md §8(c) "What pins each part").

None of these tests touches the CUDA path.  Each is chosen so that a plausible oracle mistake (dropped term, wrong
sign or index, transposed operand, wrong conjugation, wrong prefactor) fails at least one of them.
"""
import math
from pathlib import Path

import numpy as np
import pytest

import fp_inputs as fi
from fp_inputs import Inputs
from oracle.oracle import Oracle
from tests import bruteforce as bf

GOLDEN = Path(__file__).parent / "golden"


# ---------------------------------------------------------------------------------------------------------------------
# constants and scalar pieces
# ---------------------------------------------------------------------------------------------------------------------
def test_constants_two_derivations():
    """C3, C4, C_kappa, hbar/kB: oracle's in-code derivation vs an explicit SI conversion chain vs the values printed
    in SURVEY.md §8(c) 'Constants' (stored in tests/golden/constants.txt)."""
    c = Oracle.constants()
    c3, c4, ck, hk = bf.si_chain_constants()
    assert c["C3"] == pytest.approx(c3, rel=1e-13)
    assert c["C4"] == pytest.approx(c4, rel=1e-13)
    assert c["Ckappa"] == pytest.approx(ck, rel=1e-13)
    assert c["hbar_over_kb"] == pytest.approx(hk, rel=1e-13)
    gold = dict(line.split()[:2] for line in (GOLDEN / "constants.txt").read_text().splitlines()
                if line and not line.startswith("#"))
    for key in ("C3", "C4", "Ckappa", "hbar_over_kb"):
        assert c[key] == pytest.approx(float(gold[key]), rel=2e-10)


def test_paper_gaussian_weight_formula():
    """PAPER.md:163 printed formula, evaluated by hand for one dyadic case: omega=4, omega'=2, omega''=5.5, sigma=0.5
    -> Delta = 0.5, exp(-1)/(0.5 sqrt(pi)) * (f'-f'')/(4*2*5.5).  Uses rates3 on a 1-q 'mesh' is not possible, so the
    same number is reached through a hand-built 2-q-point chain in test_window_edge; here BE and the Gaussian only."""
    T = 300.0
    x = 7.638232577577646 * 2.0 / T
    assert Oracle.be(2.0, T) == pytest.approx(1.0 / math.expm1(x), rel=1e-15)
    # small-x limit f -> 1/x - 1/2, large-x limit f -> exp(-x)
    assert Oracle.be(1e-6, T) == pytest.approx(T / (7.638232577577646 * 1e-6) - 0.5, rel=1e-9)
    assert Oracle.be(4000.0, T) == pytest.approx(math.exp(-7.638232577577646 * 4000.0 / T), rel=1e-12)


def test_sigma_closed_form_cubic():
    """Cubic cell: b_mu = (2 pi/a) e_mu, so sigma = scale (2 pi/(a N)) |dv| / sqrt(6)."""
    inp = fi.make_tiny("sc1", (5, 5, 5), with4=False)
    for scale in (1.0, 0.1):
        o = Oracle(inp, scale=scale)
        rng = np.random.default_rng(3)
        for _ in range(10):
            va, vb = rng.normal(size=3) * 40, rng.normal(size=3) * 40
            want = scale * (2 * np.pi / (3.0 * 5)) * np.linalg.norm(va - vb) / np.sqrt(6.0)
            assert o.sigma(va, vb) == pytest.approx(want, rel=1e-14)
    # non-cubic mesh: anisotropic N_mu enter per component
    inp2 = fi.make_tiny("sc1", (4, 2, 1), with4=False)
    o2 = Oracle(inp2)
    va, vb = np.array([3.0, -2.0, 5.0]), np.array([1.0, 1.0, 1.0])
    dv = va - vb
    want = np.sqrt(sum((2 * np.pi / (3.0 * n) * dv[m]) ** 2 for m, n in enumerate((4, 2, 1))) / 6.0)
    assert o2.sigma(va, vb) == pytest.approx(want, rel=1e-14)


def test_recip_vectors():
    inp = fi.make_tiny("diamond", (3, 2, 1), with4=False)
    B = Oracle.recip(inp.crystal.lattvec, inp.mesh)
    want = bf.recip_cart(inp.crystal.lattvec) / np.asarray(inp.mesh, dtype=float)[:, None]
    assert np.allclose(B, want, rtol=1e-14, atol=0)


def test_window_edge_inclusive_and_sigma_zero():
    """PAPER.md:163 '<= 2 sigma' is inclusive; sigma = 0 rejects (item 3).  Dyadic values: no rounding anywhere."""
    inp = fi.make_tiny("sc1", (2, 2, 2), with4=False)
    o = Oracle(inp, ncut=2.0)
    assert o.allowed(0.5, 0.25)            # |Delta| == 2 sigma exactly
    assert o.allowed(-0.5, 0.25)
    assert not o.allowed(0.5 + 2 ** -40, 0.25)
    assert not o.allowed(-(0.5 + 2 ** -40), 0.25)
    assert not o.allowed(0.0, 0.0)         # sigma == 0 rejects even Delta == 0
    assert Oracle(inp, ncut=math.inf).allowed(1e300, 1e-300)


# ---------------------------------------------------------------------------------------------------------------------
# matrix elements
# ---------------------------------------------------------------------------------------------------------------------
def _single_entry_sc1(order, comp, cells, mesh=(3, 3, 3), phi0=2.5):
    inp = fi.make_tiny("sc1", mesh, with4=False)
    atoms = np.zeros((1, order), dtype=np.int32)
    cl = np.array(cells, dtype=np.int32).reshape(1, order - 1, 3)
    phi = np.zeros((1, 3 ** order))
    idx = 0
    for c in comp:
        idx = idx * 3 + c
    phi[0, idx] = phi0
    if order == 3:
        inp.ifc3 = (atoms, cl, phi)
    else:
        inp.ifc4 = (atoms, cl, phi)
    return inp


def test_v3_closed_form_single_entry():
    """1-atom cell, single nonzero Phi^{a0 b0 c0} at one (Rj,Rk): |V3|^2 = Phi^2 |e^a0|^2 |e'^b0|^2 |e''^c0|^2 / m^3."""
    comp = (2, 0, 1)
    inp = _single_entry_sc1(3, comp, [[1, 0, -1], [0, 2, 1]])
    o = Oracle(inp)
    m = inp.crystal.masses[0]
    e = inp.eig.reshape(-1, 3)
    rng = np.random.default_rng(0)
    for _ in range(20):
        lam, lam1, lam2 = rng.integers(0, inp.nq * 3, size=3)
        for s in (+1, -1):
            want = 2.5 ** 2 * abs(e[lam, comp[0]]) ** 2 * abs(e[lam1, comp[1]]) ** 2 * abs(e[lam2, comp[2]]) ** 2 / m ** 3
            assert abs(o.v3(lam, lam1, lam2, s)) ** 2 == pytest.approx(want, rel=1e-12, abs=1e-30)


def test_v4_closed_form_single_entry():
    comp = (1, 2, 0, 2)
    inp = _single_entry_sc1(4, comp, [[1, 0, 0], [0, -1, 1], [2, 0, 1]])
    o = Oracle(inp)
    m = inp.crystal.masses[0]
    e = inp.eig.reshape(-1, 3)
    rng = np.random.default_rng(1)
    for _ in range(20):
        l0, l1, l2, l3 = rng.integers(0, inp.nq * 3, size=4)
        for s1, s2 in ((1, 1), (1, -1), (-1, -1)):
            want = 2.5 ** 2 * np.prod([abs(e[l, c]) ** 2 for l, c in zip((l0, l1, l2, l3), comp)]) / m ** 4
            assert abs(o.v4(l0, l1, l2, l3, s1, s2)) ** 2 == pytest.approx(want, rel=1e-12, abs=1e-30)


def _conserving_triplets(inp, rng, s, n):
    nb, N = inp.nb, inp.nq
    co = fi.qpoint_coords(inp.mesh)
    out = []
    while len(out) < n:
        q, q1 = rng.integers(0, N, size=2)
        q2 = int(fi.qpoint_index(co[q] + s * co[q1], inp.mesh))
        out.append((q * nb + rng.integers(nb), q1 * nb + rng.integers(nb), q2 * nb + rng.integers(nb)))
    return out


def _conserving_quartets(inp, rng, s1, s2, n):
    nb, N = inp.nb, inp.nq
    co = fi.qpoint_coords(inp.mesh)
    out = []
    while len(out) < n:
        q, q1, q2 = rng.integers(0, N, size=3)
        q3 = int(fi.qpoint_index(co[q] + s1 * co[q1] + s2 * co[q2], inp.mesh))
        out.append(tuple(int(x * nb + rng.integers(nb)) for x in (q, q1, q2, q3)))
    return out


@pytest.mark.parametrize("kind,mesh", [("diamond", (3, 3, 3)), ("diamond", (3, 2, 1)), ("sc8", (2, 3, 2))])
def test_v3_against_dense_fourier_einsum(kind, mesh):
    """Complex V3 (not only |V|) equals the dense Fourier-tensor einsum with Cartesian phases: pins the Phi index
    order (alpha slowest), the atom->component mapping, the mass scaling, both phases and both conjugation patterns."""
    inp = fi.make_tiny(kind, mesh, with4=False)
    o = Oracle(inp)
    rng = np.random.default_rng(5)
    for s in (+1, -1):
        for lam, lam1, lam2 in _conserving_triplets(inp, rng, s, 6):
            a = o.v3(lam, lam1, lam2, s)
            b = bf.v3_dense(inp, lam, lam1, lam2, s)
            assert a == pytest.approx(b, rel=1e-10, abs=1e-12)


@pytest.mark.parametrize("kind,mesh", [("diamond", (3, 3, 3)), ("diamond", (1, 2, 3)), ("sc8", (2, 2, 3))])
def test_v4_against_dense_fourier_einsum(kind, mesh):
    inp = fi.make_tiny(kind, mesh)
    o = Oracle(inp)
    rng = np.random.default_rng(6)
    for s1, s2 in ((1, 1), (1, -1), (-1, -1)):
        for l in _conserving_quartets(inp, rng, s1, s2, 4):
            a = o.v4(*l, s1, s2)
            b = bf.v4_dense(inp, *l, s1, s2)
            assert a == pytest.approx(b, rel=1e-10, abs=1e-12)


def test_v_permutation_symmetry():
    """With permutation-symmetrised IFCs, on momentum-conserving tuples:
    |V3-(l;l1,l2)| = |V3-(l;l2,l1)|, |V3+(l;l1,l2)| = |V3-(l2;l,l1)|, |V4++(l;l1,l2,l3)| = |V4--(l3;l,l1,l2)|,
    |V4+-(l;l1,l2,l3)| = |V4+-(l;l1,l3,l2)|, |V4++(l;l1,l2,l3)| = |V4++(l;l2,l1,l3)|."""
    inp = fi.make_tiny("diamond", (3, 3, 3))
    o = Oracle(inp)
    rng = np.random.default_rng(8)
    for l, l1, l2 in _conserving_triplets(inp, rng, -1, 6):
        assert abs(o.v3(l, l1, l2, -1)) == pytest.approx(abs(o.v3(l, l2, l1, -1)), rel=1e-10, abs=1e-13)
    for l, l1, l2 in _conserving_triplets(inp, rng, +1, 6):
        assert abs(o.v3(l, l1, l2, +1)) == pytest.approx(abs(o.v3(l2, l, l1, -1)), rel=1e-10, abs=1e-13)
    for l, l1, l2, l3 in _conserving_quartets(inp, rng, 1, 1, 4):
        a = abs(o.v4(l, l1, l2, l3, 1, 1))
        assert a == pytest.approx(abs(o.v4(l3, l, l1, l2, -1, -1)), rel=1e-10, abs=1e-13)
        assert a == pytest.approx(abs(o.v4(l, l2, l1, l3, 1, 1)), rel=1e-10, abs=1e-13)
    for l, l1, l2, l3 in _conserving_quartets(inp, rng, 1, -1, 4):
        assert abs(o.v4(l, l1, l2, l3, 1, -1)) == pytest.approx(abs(o.v4(l, l1, l3, l2, 1, -1)), rel=1e-10, abs=1e-13)


def test_v_sum_rule_gamma_acoustic():
    """Sum-rule-enforced IFCs: |V| vanishes when any leg is a Gamma acoustic mode (uniform translation)."""
    for kind, mesh in (("diamond", (3, 3, 3)), ("sc8", (2, 2, 2))):
        inp = fi.make_tiny(kind, mesh)
        o = Oracle(inp)
        nb = inp.nb
        rng = np.random.default_rng(9)
        scale3 = max(abs(o.v3(*t, 1)) for t in _conserving_triplets(inp, rng, 1, 8))
        scale4 = max(abs(o.v4(*t, 1, -1)) for t in _conserving_quartets(inp, rng, 1, -1, 4))
        co = fi.qpoint_coords(inp.mesh)
        for ac in range(3):                                   # Gamma acoustic mode index = 0*nb + ac
            q1 = int(rng.integers(1, inp.nq))
            j1, j2 = rng.integers(nb, size=2)
            # target leg acoustic: q=0 so q2 = q1 (+) ; middle leg acoustic: q1=0 so q2 = q ; last leg: q2=0 so q1=-q
            assert abs(o.v3(ac, q1 * nb + j1, q1 * nb + j2, +1)) < 1e-9 * scale3
            assert abs(o.v3(q1 * nb + j1, ac, q1 * nb + j2, +1)) < 1e-9 * scale3
            qm = int(fi.qpoint_index(-co[q1], inp.mesh))
            assert abs(o.v3(q1 * nb + j1, qm * nb + j2, ac, +1)) < 1e-9 * scale3
            q2 = int(rng.integers(0, inp.nq))
            q3 = int(fi.qpoint_index(co[q1] - co[q2], inp.mesh))      # q=0: q3 = q1 - q2
            assert abs(o.v4(ac, q1 * nb + j1, q2 * nb + j2, q3 * nb + j1, 1, -1)) < 1e-9 * scale4
            q3b = int(fi.qpoint_index(co[q1] + co[q2], inp.mesh))     # last... third leg acoustic (q2'=0): q3 = q+q1
            assert abs(o.v4(q1 * nb + j1, q2 * nb + j2, ac, q3b * nb + j2, 1, 1)) < 1e-9 * scale4


def test_gauge_and_cell_offset_invariance():
    """Rates are unchanged by e_lam -> e_lam exp(i theta_lam) and by adding N_mu a_mu to any cluster offset."""
    inp = fi.make_tiny("diamond", (3, 3, 3))
    tg = np.array([13, 40, 77, 160], dtype=np.int32)
    g3, _, c3 = Oracle(inp).rates3(tg)
    g4, _, c4 = Oracle(inp).rates4(tg[:2], 0, 4)
    rng = np.random.default_rng(11)
    ph = np.exp(2j * np.pi * rng.random((inp.nq, inp.nb)))
    inp2 = Inputs(inp.name, inp.crystal, inp.mesh, inp.omega, inp.eig * ph[:, :, None], inp.vg, inp.ifc3, inp.ifc4)
    a3, c3c, p3 = inp.ifc3
    a4, c4c, p4 = inp.ifc4
    c3s = c3c.copy(); c3s[::3, 0, :] += np.array([3, 0, -6]); c3s[1::4, 1, :] += np.array([0, 3, 3])
    c4s = c4c.copy(); c4s[::2, 2, :] += np.array([-3, 3, 0]); c4s[::5, 0, :] += np.array([6, 0, 0])
    inp2.ifc3 = (a3, c3s, p3)
    inp2.ifc4 = (a4, c4s, p4)
    h3, _, d3 = Oracle(inp2).rates3(tg)
    h4, _, d4 = Oracle(inp2).rates4(tg[:2], 0, 4)
    assert np.array_equal(c3, d3) and np.array_equal(c4, d4)
    assert np.allclose(g3, h3, rtol=1e-10, atol=0)
    assert np.allclose(g4, h4, rtol=1e-10, atol=0)


def test_quadratic_and_mass_scaling():
    """Gamma3 ~ s^2 under Phi -> s Phi; Gamma4 likewise.  (mass scaling is covered by the closed-form pins.)"""
    inp = fi.make_tiny("diamond", (3, 3, 3))
    tg = np.array([20, 100], dtype=np.int32)
    g3, _, _ = Oracle(inp).rates3(tg)
    g4, _, _ = Oracle(inp).rates4(tg[:1], 0, 3)
    inp2 = Inputs(inp.name, inp.crystal, inp.mesh, inp.omega, inp.eig, inp.vg,
                  (inp.ifc3[0], inp.ifc3[1], -3.0 * inp.ifc3[2]), (inp.ifc4[0], inp.ifc4[1], 0.5 * inp.ifc4[2]))
    h3, _, _ = Oracle(inp2).rates3(tg)
    h4, _, _ = Oracle(inp2).rates4(tg[:1], 0, 3)
    assert np.allclose(h3, 9.0 * g3, rtol=1e-12)
    assert np.allclose(h4, 0.25 * g4, rtol=1e-12)


# ---------------------------------------------------------------------------------------------------------------------
# enumeration, counts, brute force
# ---------------------------------------------------------------------------------------------------------------------
@pytest.mark.parametrize("kind,mesh", [("diamond", (2, 2, 2)), ("diamond", (3, 2, 1)), ("sc1", (2, 2, 2))])
def test_counts_closed_form_filter_disabled(kind, mesh):
    """ncut = inf, sigma_const > 0 (item 20): 3ph per channel N nb^2 - 6 nb + 9 [q = Gamma]; 4ph per channel by
    inclusion-exclusion over the three legs being one of the 3 zero modes at Gamma."""
    inp = fi.make_tiny(kind, mesh)
    o = Oracle(inp, ncut=math.inf, sigma_const=5.0)
    nb, N = inp.nb, inp.nq
    tg = inp.targets3
    _, _, c3 = o.rates3(tg, weights_only=True)
    _, _, c4 = o.rates4(tg, weights_only=True)
    for it, lam in enumerate(tg):
        q, j = divmod(int(lam), nb)
        if q == 0 and j < 3:
            assert (c3[it] == 0).all() and (c4[it] == 0).all()
            continue
        want3 = N * nb * nb - 6 * nb + (9 if q == 0 else 0)
        assert (c3[it] == want3).all()
        # 4ph: tuples (q1,j1,q2,j2,j3): N^2 nb^3 total. A_k = leg k is a zero mode.
        # |A1| = 3 * N * nb^2 (q1=0,j1<3; q2 free), same |A2|; |A3|: q3=0 fixes q2 given q1: N * nb^2 * 3.
        # |A1A2| = 9 * nb (q1=q2=0); |A1A3|: q1=0 and q3=0 -> q2 fixed: 9 nb; |A2A3| likewise 9 nb;
        # |A1A2A3|: q1=q2=0 -> q3 = q: 27 if q==0 else 0; and the pair terms need q3 reachable (always, one q2).
        a = 3 * N * nb * nb
        pair = 9 * nb
        # A1A2 forces q3 = q: no further constraint.  A1A3 forces q2 = +-q; A2A3 forces q1 = -+q.  Always one solution.
        triple = 27 if q == 0 else 0
        want4 = N * N * nb ** 3 - 3 * a + 3 * pair - triple
        assert (c4[it] == want4).all()


def test_list3_is_momentum_conserving_and_matches_bruteforce_set():
    """Filter on (adaptive sigma, 3x3x3): the oracle's process list equals, as a set, a brute-force scan over ALL
    (lam', lam'') pairs with rational momentum test and an independent numpy evaluation of the predicate."""
    inp = fi.make_tiny("diamond", (3, 3, 3), with4=False)
    o = Oracle(inp)
    fr = bf.frac_coords(inp)
    nb, N = inp.nb, inp.nq
    w = inp.omega.reshape(-1)
    v = inp.vg.reshape(-1, 3)
    B = bf.recip_cart(inp.crystal.lattvec) / np.asarray(inp.mesh, float)[:, None]
    total = 0
    for lam in (9, 50, 101):
        for ch, s in enumerate((1, -1)):
            got = set(map(tuple, o.list3(lam, ch)))
            total += len(got)
            want = set()
            for l1 in range(N * nb):
                for l2 in range(N * nb):
                    if w[l1] == 0 or w[l2] == 0:
                        continue
                    if not bf.conserves(fr, (lam // nb, l1 // nb, l2 // nb), (1, s, -1)):
                        continue
                    sig = np.sqrt(((B @ (v[l1] - v[l2])) ** 2).sum() / 6.0)
                    d = w[lam] + s * w[l1] - w[l2]
                    if sig > 0 and abs(d) <= 2 * sig:
                        want.add((l1, l2))
            # candidates within 1e-12 of the window edge may legitimately differ between two arithmetics
            diff = got ^ want
            for l1, l2 in diff:
                sig = np.sqrt(((B @ (v[l1] - v[l2])) ** 2).sum() / 6.0)
                d = w[lam] + s * w[l1] - w[l2]
                assert abs(abs(d) - 2 * sig) < 1e-10 * max(1.0, abs(d))
    assert total > 50


@pytest.mark.parametrize("kind,mesh,lams", [("diamond", (3, 3, 3), (31, 100)), ("diamond", (3, 2, 1), (8, 21)),
                                            ("sc1", (3, 3, 2), (20,))])
def test_list4_adaptive_sigma_matches_bruteforce_set_and_weights(kind, mesh, lams):
    """The 4ph ADAPTIVE-sigma path (SURVEY.md §8(c) item 2 / DESIGN.md §3-2: sigma from the last two legs, v2 - v3; the
    paper shows only compute_sigma(v1 - v2) for 3ph).  For each channel: (i) orc_list4 equals, as a set, a
    brute-force scan over ALL (lam1, lam2, lam3) with rational momentum test and an independent numpy evaluation of
    sigma and the window; (ii) orc_rates4's counts equal the list length; (iii) orc_rates4(weights_only) equals the
    direct sum of PAPER.md:163's Gaussian with the "/f" occupation forms over the brute-force list.  A sigma built from
    (v1, v2) instead, or a wrong sign of omega2 in Delta, fails (i), (ii) and (iii)."""
    inp = fi.make_tiny(kind, mesh)
    o = Oracle(inp)
    total = 0
    for lam in lams:
        t = np.array([lam], dtype=np.int32)
        _, wp, cnt = o.rates4(t, weights_only=True)
        for ch in range(3):
            want, margin, wsum = bf.list4_bruteforce(inp, lam, ch, scale=inp.scale, T=inp.T)
            got = set(map(tuple, o.list4(lam, ch).tolist()))
            assert len(got) == cnt[0, ch]                               # the list and the rate loop decide alike
            # candidates within rounding of the window edge may legitimately differ between two arithmetics
            for tr in got ^ want:
                assert tr in margin and abs(margin[tr]) < 1e-10
            if got == want:
                assert wp[0, ch] == pytest.approx(wsum, rel=1e-11)
            total += len(want)
    assert total > 200                                                  # the adaptive window really admits processes


def test_list4_partial_q_range_and_bounds():
    inp = fi.make_tiny("diamond", (3, 3, 3))
    o = Oracle(inp)
    full = o.list4(50, 1)
    part = np.concatenate([o.list4(50, 1, 0, 10), o.list4(50, 1, 10, 27)])
    assert np.array_equal(full, part)                                   # loop order: q' outermost
    assert len(np.unique(full, axis=0)) == len(full)
    with pytest.raises(ValueError):
        o.list4(50, 1, 0, 28)
    with pytest.raises(ValueError):
        o.rates4(np.array([50], dtype=np.int32), 5, 28)


@pytest.mark.parametrize("kind,lams", [("diamond", (4, 29)), ("sc1", (5, 13, 22))])
def test_rates3_bruteforce_2x2x2(kind, lams):
    """Full rates vs the brute-force/dense-Fourier route on 2x2x2 (constant sigma, filter off), both channels."""
    inp = fi.make_tiny(kind, (2, 2, 2), with4=False)
    o = Oracle(inp, ncut=math.inf, sigma_const=5.0)
    g, _, c = o.rates3(np.array(lams, dtype=np.int32))
    for it, lam in enumerate(lams):
        bg, bc = bf.rates3_bruteforce(inp, lam, 5.0)
        assert list(c[it]) == bc
        assert g[it] == pytest.approx(bg, rel=1e-10)


def test_rates3_bruteforce_unequal_mesh():
    inp = fi.make_tiny("diamond", (3, 2, 1), with4=False)
    o = Oracle(inp, ncut=math.inf, sigma_const=4.0)
    lams = (7, 20)
    g, _, c = o.rates3(np.array(lams, dtype=np.int32))
    for it, lam in enumerate(lams):
        bg, bc = bf.rates3_bruteforce(inp, lam, 4.0)
        assert list(c[it]) == bc
        assert g[it] == pytest.approx(bg, rel=1e-10)


def test_rates4_bruteforce_2x2x2():
    inp = fi.make_tiny("sc1", (2, 2, 2))
    o = Oracle(inp, ncut=math.inf, sigma_const=5.0)
    lams = (4, 17)
    g, _, c = o.rates4(np.array(lams, dtype=np.int32))
    for it, lam in enumerate(lams):
        bg, bc = bf.rates4_bruteforce(inp, lam, 5.0)
        assert list(c[it]) == bc
        assert g[it] == pytest.approx(bg, rel=1e-10)


def test_rates4_bruteforce_diamond_unequal_mesh():
    inp = fi.make_tiny("diamond", (2, 1, 3))
    o = Oracle(inp, ncut=math.inf, sigma_const=6.0)
    lam = 16
    g, _, c = o.rates4(np.array([lam], dtype=np.int32))
    bg, bc = bf.rates4_bruteforce(inp, lam, 6.0)
    assert list(c[0]) == bc
    assert g[0] == pytest.approx(bg, rel=1e-10)


def test_rates4_partial_ranges_add_up():
    inp = fi.make_tiny("diamond", (3, 3, 3))
    o = Oracle(inp)
    tg = np.array([30, 95], dtype=np.int32)
    g, w, c = o.rates4(tg, 0, 6)
    ga, wa, ca = o.rates4(tg, 0, 2)
    gb, wb, cb = o.rates4(tg, 2, 6)
    assert np.array_equal(c, ca + cb)
    assert np.allclose(g, ga + gb, rtol=1e-13) and np.allclose(w, wa + wb, rtol=1e-13)


def test_time_reversal():
    """Gamma^{ch}(q,j) = Gamma^{ch}(-q,j) and equal counts, inputs prepared per item 17."""
    inp = fi.make_tiny("diamond", (3, 3, 3))
    o = Oracle(inp)
    co = fi.qpoint_coords(inp.mesh)
    qs = np.array([1, 5, 14, 22])
    qm = fi.qpoint_index(-co[qs], inp.mesh)
    nb = inp.nb
    ta = (qs[:, None] * nb + np.arange(nb)).reshape(-1).astype(np.int32)
    tb = (qm[:, None] * nb + np.arange(nb)).reshape(-1).astype(np.int32)
    ga, wa, ca = o.rates3(ta)
    gb, wb, cb = o.rates3(tb)
    assert np.array_equal(ca, cb)
    assert np.allclose(ga, gb, rtol=1e-10) and np.allclose(wa, wb, rtol=1e-12)
    g4a, _, c4a = o.rates4(ta[6:9], 0, 27)
    # -q target: the q' range must be mirrored too, so use the full range for both
    g4b, _, c4b = o.rates4(tb[6:9], 0, 27)
    assert np.array_equal(c4a, c4b)
    assert np.allclose(g4a, g4b, rtol=1e-10)


# ---------------------------------------------------------------------------------------------------------------------
# weights
# ---------------------------------------------------------------------------------------------------------------------
def test_onshell_occupation_identities():
    """Delta = 0 exactly: (1+f1)(1+f2)f3/f = f1 f2 (1+f3) - ... forms of the 4ph factors and the 3ph analogue.
    Checks BE via detailed balance: for w = w3 - w1 - w2 (++): (1+f1)(1+f2) f3 / f == f1 f2 (1+f3)/(1+f) etc."""
    T = 300.0
    be = lambda w: Oracle.be(w, T)
    w1, w2, w = 21.0, 33.5, 12.25
    w3 = w + w1 + w2
    f, f1, f2, f3 = be(w), be(w1), be(w2), be(w3)
    # ++ : absorb lam,lam1,lam2 -> emit lam3.  detailed balance: f f1 f2 (1+f3) = (1+f)(1+f1)(1+f2) f3
    assert f * f1 * f2 * (1 + f3) == pytest.approx((1 + f) * (1 + f1) * (1 + f2) * f3, rel=1e-12)
    # so (1+f1)(1+f2) f3 / f == f1 f2 (1+f3) / (1+f)
    assert (1 + f1) * (1 + f2) * f3 / f == pytest.approx(f1 * f2 * (1 + f3) / (1 + f), rel=1e-12)
    # 3ph+: w2' = w + w1: detailed balance f f1 (1+f2') = (1+f)(1+f1) f2'  =>  f1 - f2' = (1+f1) f2' / f
    w2p = w + w1
    f2p = be(w2p)
    assert f * f1 * (1 + f2p) == pytest.approx((1 + f) * (1 + f1) * f2p, rel=1e-12)
    assert (f1 - f2p) == pytest.approx((1 + f1) * f2p / f, rel=1e-12)        # ShengBTE form == detailed-balance form
    # 3ph-: w = w1 + w2m
    w2m = 5.0
    w1m = w - w2m
    a, b = be(w1m), be(w2m)
    assert (a + b + 1) == pytest.approx((1 + a) * (1 + b) / (1 + f), rel=1e-12)


def test_weights_only_matches_direct_sum_and_high_T_scaling():
    """WP-only runs: (i) equal a direct numpy evaluation of PAPER.md:163 over the oracle's own process list,
    (ii) Gamma3 ~ T and Gamma4 ~ T^2 as T -> infinity (f -> kT/hbar w)."""
    inp = fi.make_tiny("diamond", (3, 3, 3))
    o = Oracle(inp)
    lam = 50
    _, wp, c = o.rates3(np.array([lam], dtype=np.int32), weights_only=True)
    w = inp.omega.reshape(-1)
    v = inp.vg.reshape(-1, 3)
    B = bf.recip_cart(inp.crystal.lattvec) / np.asarray(inp.mesh, float)[:, None]
    for ch, s in enumerate((1, -1)):
        tot = 0.0
        pairs = o.list3(lam, ch)
        assert len(pairs) == c[0, ch]
        for l1, l2 in pairs:
            sig = np.sqrt(((B @ (v[l1] - v[l2])) ** 2).sum() / 6.0)
            d = w[lam] + s * w[l1] - w[l2]
            f1, f2 = bf.be(w[l1], 300.0), bf.be(w[l2], 300.0)
            occ = f1 - f2 if s > 0 else f1 + f2 + 1
            tot += occ * np.exp(-d * d / sig ** 2) / (sig * np.sqrt(np.pi)) / (w[lam] * w[l1] * w[l2])
        tot *= (1.0 if s > 0 else 0.5) / inp.nq
        assert wp[0, ch] == pytest.approx(tot, rel=1e-11)
    tg = np.array([50, 120], dtype=np.int32)
    T1, T2 = 3.0e6, 6.0e6
    g1, _, _ = Oracle(inp, T=T1).rates3(tg)
    g2, _, _ = Oracle(inp, T=T2).rates3(tg)
    assert np.allclose(g2, 2.0 * g1, rtol=1e-4)
    h1, _, _ = Oracle(inp, T=T1).rates4(tg[:1], 0, 4)
    h2, _, _ = Oracle(inp, T=T2).rates4(tg[:1], 0, 4)
    assert np.allclose(h2, 4.0 * h1, rtol=1e-4)


def test_compensated_sum_vs_reordered_naive():
    """Oracle's compensated per-mode sum vs a naive float sum of the same terms in reversed order (< 1e-12)."""
    inp = fi.make_config(0)["main"]
    o = Oracle(inp)
    lam = 200
    g, wp, c = o.rates3(np.array([lam], dtype=np.int32))
    C3 = Oracle.constants()["C3"]
    w = inp.omega.reshape(-1)
    v = inp.vg.reshape(-1, 3)
    for ch, s in enumerate((1, -1)):
        terms = []
        for l1, l2 in o.list3(lam, ch):
            sig = o.sigma(v[l1], v[l2])
            d = w[lam] + s * w[l1] - w[l2]
            f1, f2 = Oracle.be(w[l1], 300.0), Oracle.be(w[l2], 300.0)
            occ = f1 - f2 if s > 0 else f1 + f2 + 1
            WP = occ * np.exp(-(d / sig) ** 2) / (sig * np.sqrt(np.pi)) / (w[lam] * w[l1] * w[l2])
            terms.append(WP * abs(o.v3(lam, l1, l2, s)) ** 2)
        naive = 0.0
        for t in reversed(terms):
            naive += t
        naive *= C3 / inp.nq * (1.0 if s > 0 else 0.5)
        assert g[0, ch] == pytest.approx(naive, rel=1e-12)


# ---------------------------------------------------------------------------------------------------------------------
# kappa
# ---------------------------------------------------------------------------------------------------------------------
def test_kappa_limits():
    """Constant Gamma: kappa = (1/Gamma) sum_lam C_lam v v / (V N); as T -> inf, C_lam -> kB, so
    kappa -> kB/(V N Gamma) sum v v."""
    inp = fi.make_tiny("diamond", (4, 4, 4), with4=False)
    T = 1.0e7
    o = Oracle(inp, T=T)
    gam = np.full(inp.nq * inp.nb, 0.25)
    k = o.kappa(gam)
    v = inp.vg.reshape(-1, 3)
    nz = inp.omega.reshape(-1) > 0
    vv = np.einsum("la,lb->ab", v[nz], v[nz])
    # kB [J/K] * (A/ps)^2 * ps / A^3 -> W/mK : 1e4 m^2/s^2 * 1e-12 s / 1e-30 m^3
    want = bf.KB * vv * 1e4 * 1e-12 / 1e-30 / (inp.crystal.volume * inp.nq * 0.25)
    assert np.allclose(k, want, rtol=1e-6, atol=1e-9 * abs(want).max())
    # (isotropy of a cubic crystal is NOT asserted: the Hellmann-Feynman diagonal velocities of item 17 depend on the
    #  basis chosen inside degenerate subspaces, which is a property of the inputs, not of the kappa formula)
    assert np.allclose(k, k.T, rtol=1e-14)
    # modes with Gamma <= 0 are skipped
    gam2 = gam.copy(); gam2[10] = 0.0; gam2[11] = -1.0
    k2 = o.kappa(gam2)
    assert k2[0, 0] < k[0, 0]
    # finite T: heat capacity form x^2 e^x/(e^x-1)^2 per mode
    o3 = Oracle(inp, T=300.0)
    k3 = o3.kappa(gam)
    w = inp.omega.reshape(-1)[nz]
    x = bf.HBAR * w * 1e12 / (bf.KB * 300.0)
    cl = bf.KB * x ** 2 * np.exp(x) / (np.exp(x) - 1) ** 2
    want3 = np.einsum("l,la,lb->ab", cl, v[nz], v[nz]) * 1e4 * 1e-12 / 1e-30 / (inp.crystal.volume * inp.nq * 0.25)
    assert np.allclose(k3, want3, rtol=1e-10, atol=1e-12 * abs(want3).max())
