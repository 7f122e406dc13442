"""-m gpu: the CUDA path (through the C ABI of include/fourphonon.h) against the CPU oracle, element by element.

Bars (BASELINE.json north_star): process counts bit-exact, rates / weighted phase space / kappa within 1e-9 relative.
See assert_rates_close for how "relative" is measured for modes whose rate is cancellation noise.
"""
import numpy as np
import pytest

import fp_inputs

pytestmark = pytest.mark.gpu

RTOL = 1e-9


@pytest.fixture(scope="module")
def fp():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("needs a CUDA device")
    import paper_2510_00518_b200 as fp
    fp.build_library(force=False)          # no-op when the in-tree .so is up to date
    fp.load_library()
    return fp


def PATHS(fp):
    """fused (lists in shared memory) and split (enumerator -> lists in the scratch -> evaluator, two streams)"""
    return (fp.FP_PATH_FUSED, fp.FP_PATH_SPLIT)


def _oracle(inp, **kw):
    from oracle.oracle import Oracle
    return Oracle(inp, **kw)


def assert_rates_close(got, ref, what):
    """|got - ref| <= 1e-9 * (largest |ref| of the channel) everywhere, and <= 1e-9 * |ref| itself wherever the mode's
    value is not cancellation noise (|ref| >= 1e-10 of the channel maximum: below that |V|^2 is the square of a sum
    that cancels to < 1e-5 of its terms, and no FP64 evaluation order reproduces another to 1e-9 of the result)."""
    got = np.asarray(got); ref = np.asarray(ref)
    assert got.shape == ref.shape
    scale = np.abs(ref).max(axis=0, keepdims=True)
    scale = np.where(scale > 0, scale, 1.0)
    err = np.abs(got - ref) / scale
    assert err.max() <= RTOL, f"{what}: max error relative to the channel maximum {err.max():.3e}"
    big = np.abs(ref) >= 1e-10 * scale
    if big.any():
        own = np.abs(got[big] - ref[big]) / np.abs(ref[big])
        assert own.max() <= RTOL, f"{what}: max error relative to own magnitude {own.max():.3e}"
    assert np.all(got[ref == 0] == 0.0), f"{what}: oracle zero where the GPU is nonzero"


def check3(fp, inp, targets, **kw):
    orc = _oracle(inp, **{k: v for k, v in kw.items() if k in ("ncut", "sigma_const", "T", "scale")})
    og, ow, oc = orc.rates3(targets)
    scratch = kw.pop("scratch_bytes", 64 << 20)
    for path in PATHS(fp):                                            # both execution paths meet the same bar
        with fp.Context.from_inputs(inp, scratch_bytes=scratch, **kw) as ctx:
            ctx.set_path(path)
            g, w, c = ctx.rates3(targets)
        assert np.array_equal(c, oc), f"3ph process counts are not bit-exact (path {path})"
        assert_rates_close(g, og, f"Gamma3 (path {path})")
        assert_rates_close(w, ow, f"WP3 (path {path})")
    return g, c


def check4(fp, inp, targets, qp=(0, None), **kw):
    orc = _oracle(inp, **{k: v for k, v in kw.items() if k in ("ncut", "sigma_const", "T", "scale")})
    og, ow, oc = orc.rates4(targets, qp[0], qp[1])
    scratch = kw.pop("scratch_bytes", 64 << 20)
    for path in PATHS(fp):
        with fp.Context.from_inputs(inp, scratch_bytes=scratch, **kw) as ctx:
            ctx.set_path(path)
            g, w, c = ctx.rates4(targets, qp[0], qp[1])
        assert np.array_equal(c, oc), f"4ph process counts are not bit-exact (path {path})"
        assert_rates_close(g, og, f"Gamma4 (path {path})")
        assert_rates_close(w, ow, f"WP4 (path {path})")
    return g, c


# ---- small cases: whole job element by element ----------------------------------------------------------------------------
def test_constants_match_oracle(fp):
    from oracle.oracle import Oracle
    a, b = fp.fp_constants(), Oracle.constants()
    for k in a:
        assert abs(a[k] - b[k]) <= 1e-14 * abs(b[k])


@pytest.mark.parametrize("kind,mesh", [("diamond", (3, 3, 3)), ("diamond", (4, 3, 2)), ("sc1", (5, 4, 3)),
                                       ("sc8", (2, 3, 2))])
def test_rates3_small(fp, kind, mesh):
    inp = fp_inputs.make_tiny(kind, mesh=mesh, with4=False)
    g, c = check3(fp, inp, inp.targets3)
    assert c.sum() > 0


def test_rates3_config0_all_modes(fp):
    inp = fp_inputs.make_config(0)["main"]
    g, c = check3(fp, inp, inp.targets3)
    assert c.sum() > 1e5


@pytest.mark.parametrize("kind,mesh,sl", [("diamond", (3, 3, 3), slice(5, 29)), ("diamond", (4, 2, 3), slice(40, 52)),
                                          ("sc1", (4, 3, 3), slice(0, None))])
def test_rates4_small(fp, kind, mesh, sl):
    inp = fp_inputs.make_tiny(kind, mesh=mesh)
    g, c = check4(fp, inp, inp.targets4[sl])
    assert c.sum() > 0


def test_rates4_many_branch_generic_path(fp):
    inp = fp_inputs.make_tiny("sc8", mesh=(2, 2, 3))
    check4(fp, inp, inp.targets4[30:36], qp=(3, 7))


def test_filter_disabled_constant_sigma_2x2x2(fp):
    """item 20: adaptive sigma vanishes on 2x2x2, so the brute-force configuration is ncut=inf with a fixed sigma."""
    inp = fp_inputs.make_tiny("diamond", mesh=(2, 2, 2))
    g3, c3 = check3(fp, inp, inp.targets3, ncut=float("inf"), sigma_const=5.0)
    nb, N = inp.nb, inp.nq
    for i, lam in enumerate(inp.targets3):
        expect = 0 if inp.omega.reshape(-1)[lam] == 0.0 else N * nb * nb - 6 * nb + (9 if lam // nb == 0 else 0)
        assert c3[i, 0] == expect and c3[i, 1] == expect
    check4(fp, inp, inp.targets4[3:15], ncut=float("inf"), sigma_const=5.0)


def test_adaptive_sigma_on_2x2x2_rejects_everything(fp):
    inp = fp_inputs.make_tiny("diamond", mesh=(2, 2, 2), with4=False)
    g, c = check3(fp, inp, inp.targets3)
    assert c.sum() == 0 and np.all(g == 0.0)


def test_list3_equals_oracle_list_as_sets(fp):
    inp = fp_inputs.make_tiny("diamond", mesh=(4, 4, 4), with4=False)
    orc = _oracle(inp)
    with fp.Context.from_inputs(inp, scratch_bytes=32 << 20) as ctx:
        for lam in (7, 100, 383):
            for ch in (0, 1):
                a = ctx.list3(lam, ch); b = orc.list3(lam, ch)
                assert len(a) == len(b)
                assert set(map(tuple, a.tolist())) == set(map(tuple, b.tolist()))


def test_list4_is_momentum_conserving_and_counts_match(fp):
    inp = fp_inputs.make_tiny("diamond", mesh=(3, 3, 3))
    orc = _oracle(inp)
    coords = fp_inputs.qpoint_coords(inp.mesh)
    nb = inp.nb
    lam = 31
    with fp.Context.from_inputs(inp, scratch_bytes=32 << 20) as ctx:
        for ch, (s1, s2) in enumerate(((1, 1), (1, -1), (-1, -1))):
            for qp in (0, 5, 26):
                tr = ctx.list4(lam, ch, qp)
                _, _, oc = orc.rates4(np.array([lam], dtype=np.int32), qp, qp + 1)
                assert len(tr) == oc[0, ch]
                assert len(set(map(tuple, tr.tolist()))) == len(tr)
                for l1, l2, l3 in tr:
                    assert l1 // nb == qp
                    q3 = (coords[lam // nb] + s1 * coords[l1 // nb] + s2 * coords[l2 // nb]) % inp.mesh
                    assert np.array_equal(q3, coords[l3 // nb])


# ---- boundary behaviour ------------------------------------------------------------------------------------------------------
def test_device_pointer_entry_points_match_host_entry_points(fp):
    import torch
    inp = fp_inputs.make_tiny("diamond", mesh=(3, 3, 3))
    dev = torch.device("cuda:0")
    om = torch.from_numpy(np.ascontiguousarray(inp.omega)).to(dev)
    eg = torch.from_numpy(np.ascontiguousarray(inp.eig)).to(dev)
    vg = torch.from_numpy(np.ascontiguousarray(inp.vg)).to(dev)
    with fp.Context.from_inputs(inp, scratch_bytes=32 << 20) as a, \
            fp.Context(inp.crystal.lattvec, inp.crystal.masses, om, eg, vg, inp.mesh, T=inp.T, ifc3=inp.ifc3,
                       ifc4=inp.ifc4, scratch_bytes=32 << 20) as b:
        t3 = inp.targets3
        g, w, c = a.rates3(t3)
        gd, wd, cd = b.rates3(torch.from_numpy(t3).to(dev))
        assert np.array_equal(g, gd.cpu().numpy()) and np.array_equal(w, wd.cpu().numpy())
        assert np.array_equal(c, cd.cpu().numpy())
        t4 = inp.targets4[10:16]
        g4, w4, c4 = a.rates4(t4)
        g4d, w4d, c4d = b.rates4(torch.from_numpy(t4).to(dev))
        assert np.array_equal(g4, g4d.cpu().numpy()) and np.array_equal(c4, c4d.cpu().numpy())
        k = a.kappa_rta(g.sum(axis=1))
        kd = b.kappa_rta(gd.sum(dim=1))
        assert np.array_equal(k, kd.cpu().numpy())


def test_rates4_partial_q_ranges_add_up(fp):
    inp = fp_inputs.make_tiny("diamond", mesh=(3, 3, 3))
    t = inp.targets4[20:26]
    with fp.Context.from_inputs(inp, scratch_bytes=32 << 20) as ctx:
        g, w, c = ctx.rates4(t)
        ga, wa, ca = ctx.rates4(t, 0, 11)
        gb, wb, cb = ctx.rates4(t, 11, 27)
        ge, we, ce = ctx.rates4(t, 5, 5)
    assert np.array_equal(c, ca + cb)
    assert np.allclose(g, ga + gb, rtol=1e-12, atol=0)
    assert np.all(ge == 0) and np.all(ce == 0)


def test_small_scratch_splits_targets_and_gives_identical_results(fp):
    """A scratch that holds a few targets at a time forces the bounded-memory loop (Algorithm 5)."""
    inp = fp_inputs.make_tiny("diamond", mesh=(3, 3, 3))
    t = inp.targets4[6:30]
    for path in PATHS(fp):                                            # chunking never changes a row's arithmetic
        with fp.Context.from_inputs(inp, scratch_bytes=256 << 20) as big:
            big.set_path(path)
            big.set_target_symmetry(False)
            big.profile_enable(True)
            g, w, c = big.rates4(t)
            n_big = big.profile_get().n_rates
            assert n_big == 1 or path != fp.FP_PATH_FUSED
        with fp.Context.from_inputs(inp, scratch_bytes=512 << 10) as small:
            small.set_path(path)
            small.set_target_symmetry(False)                          # (the candidate count below is that of all 24 targets)
            small.profile_enable(True)
            gs, ws, cs = small.rates4(t)
            p = small.profile_get()
            assert p.n_rates > n_big
            assert p.processes == int(cs.sum()) and p.prefiltered >= p.evaluated > 0
            assert p.candidates == len(t) * 3 * inp.nq ** 2 * inp.nb ** 3
        assert np.array_equal(c, cs) and np.array_equal(g, gs) and np.array_equal(w, ws)


def test_paths_agree(fp):
    """fused and split evaluate the same processes: identical counts, rates equal to rounding order."""
    inp = fp_inputs.make_tiny("diamond", mesh=(4, 4, 4))
    t = inp.targets4[24:48]
    res = []
    for path in PATHS(fp) + (fp.FP_PATH_SPLIT_SERIAL, fp.FP_PATH_AUTO):
        with fp.Context.from_inputs(inp, scratch_bytes=128 << 20) as ctx:
            ctx.set_path(path)
            res.append(ctx.rates4(t) + ctx.rates3(inp.targets3))
    for r in res[1:]:
        for a, b in zip(res[0], r):
            if a.dtype.kind == "i":
                assert np.array_equal(a, b)
            else:
                assert np.allclose(a, b, rtol=1e-12, atol=1e-13 * np.abs(a).max())
    assert all(np.array_equal(a, b) for a, b in zip(res[1], res[2]))   # overlap does not change the split path's bits


def test_run_to_run_determinism(fp):
    inp = fp_inputs.make_tiny("diamond", mesh=(3, 3, 3))
    with fp.Context.from_inputs(inp, scratch_bytes=32 << 20) as ctx:
        a = ctx.rates4(inp.targets4[6:12])
        b = ctx.rates4(inp.targets4[6:12])
    for x, y in zip(a, b):
        assert np.array_equal(x, y)


def test_empty_and_zero_mode_targets(fp):
    inp = fp_inputs.make_tiny("diamond", mesh=(3, 3, 3))
    with fp.Context.from_inputs(inp, scratch_bytes=32 << 20) as ctx:
        g, w, c = ctx.rates3(np.zeros(0, dtype=np.int32))
        assert g.shape == (0, 2)
        g, w, c = ctx.rates3(np.array([0, 1, 2], dtype=np.int32))          # the three Gamma acoustic modes
        assert np.all(g == 0) and np.all(w == 0) and np.all(c == 0)
        g, w, c = ctx.rates4(np.array([0, 1, 2], dtype=np.int32))
        assert np.all(g == 0) and np.all(w == 0) and np.all(c == 0)


def test_error_codes(fp):
    inp = fp_inputs.make_tiny("diamond", mesh=(3, 3, 3), with4=False)
    with fp.Context.from_inputs(inp, scratch_bytes=32 << 20) as ctx:
        with pytest.raises(fp.FourPhononError) as e:
            ctx.rates4(inp.targets4[:2])
        assert e.value.code == fp.FP_ESTATE
        with pytest.raises(fp.FourPhononError) as e:
            ctx.rates3(np.array([inp.nq * inp.nb], dtype=np.int32))
        assert e.value.code == fp.FP_EINVAL
        with pytest.raises(fp.FourPhononError) as e:
            ctx.rates3(np.array([-1], dtype=np.int32))
        assert e.value.code == fp.FP_EINVAL
    with pytest.raises(fp.FourPhononError) as e:
        fp.Context.from_inputs(inp, T=0.0)
    assert e.value.code == fp.FP_EINVAL
    with pytest.raises(fp.FourPhononError) as e:
        fp.Context.from_inputs(inp, scale=-1.0)
    assert e.value.code == fp.FP_EINVAL
    bad = np.array(inp.omega, copy=True); bad.reshape(-1)[10] = float("nan")
    with pytest.raises(fp.FourPhononError) as e:
        fp.Context(inp.crystal.lattvec, inp.crystal.masses, bad, inp.eig, inp.vg, inp.mesh, ifc3=inp.ifc3)
    assert e.value.code == fp.FP_EINVAL
    atoms = np.array(inp.ifc3[0], copy=True); atoms[0, 1] = 7
    with pytest.raises(fp.FourPhononError) as e:
        fp.Context(inp.crystal.lattvec, inp.crystal.masses, inp.omega, inp.eig, inp.vg, inp.mesh,
                   ifc3=(atoms, inp.ifc3[1], inp.ifc3[2]))
    assert e.value.code == fp.FP_EINVAL
    with pytest.raises(fp.FourPhononError) as e:                           # workspace below the resident tables
        fp.Context.from_inputs(inp, workspace_bytes=4096)
    assert e.value.code == fp.FP_ENOMEM
    with fp.Context.from_inputs(inp, scratch_bytes=1) as ctx:             # sized by fp_workspace_bytes: setup fits,
        need = ctx.workspace.numel()
    with pytest.raises(fp.FourPhononError) as e:                           # ... but not one target's row arrays
        with fp.Context.from_inputs(inp, workspace_bytes=need - 60000) as ctx:
            ctx.rates3(inp.targets3[:4])
    assert e.value.code == fp.FP_ENOMEM


def test_kappa_matches_oracle(fp):
    inp = fp_inputs.make_config(0)["main"]
    orc = _oracle(inp)
    with fp.Context.from_inputs(inp, scratch_bytes=64 << 20) as ctx:
        g, w, c = ctx.rates3(inp.targets3)
        gt = g.sum(axis=1)
        k = ctx.kappa_rta(gt)
    ok = orc.kappa(gt)
    assert np.abs(k - ok).max() <= RTOL * np.abs(ok).max()
    assert np.allclose(k, k.T, rtol=1e-12, atol=1e-12 * np.abs(k).max())    # symmetric by construction


# ---- BASELINE.json's full sizes, sampled: the oracle evaluates a seeded sample of targets (and a q' range for 4ph) -------
def _sample(targets, n, seed, always=()):
    rng = np.random.default_rng(seed)
    pick = set(int(x) for x in rng.choice(np.asarray(targets), n, replace=False)) | set(int(x) for x in always)
    return np.array(sorted(pick), dtype=np.int32)


FULL_SCRATCH = 4 << 30


def test_full_size_config1_3ph_sampled_modes(fp):
    """config 1 (= the 3ph leg of config 3): 16x16x16, 24 of the 24,576 target modes incl. a Gamma acoustic mode."""
    inp = fp_inputs.make_config(1)["main"]
    t = _sample(inp.targets3, 23, 11, always=(0, 5, 24575))
    g, c = check3(fp, inp, t, scratch_bytes=FULL_SCRATCH)
    assert np.all(c[t == 0] == 0) and c.sum() > 100000


def test_full_size_config2_4ph_sampled(fp):
    """config 2: 8x8x8, three of the 192 targets over a q' range of 8 of the 512 points, all three channels."""
    inp = fp_inputs.make_config(2)["main"]
    t = np.ascontiguousarray(inp.targets4[[0, 77, 191]])
    g, c = check4(fp, inp, t, qp=(37, 45), scratch_bytes=FULL_SCRATCH)
    assert c.sum() > 100000


def test_full_size_config3_4ph_sampled(fp):
    """config 3: 16x16x16, two of the 96 targets (one acoustic, one optical branch) over q' in [1000, 1003)."""
    inp = fp_inputs.make_config(3)["main"]
    t = np.ascontiguousarray(inp.targets4[[1, 53]])
    g, c = check4(fp, inp, t, qp=(1000, 1003), scratch_bytes=FULL_SCRATCH)
    assert c.sum() > 100000


def test_full_size_config4_sampled(fp):
    """config 4 (8 atoms, 24 branches, generic kernels): 3ph at 12x12x12 on four modes, 4ph at 6x6x6 on one target x one q'."""
    jobs = fp_inputs.make_config(4)
    j3, j4 = jobs["3ph"], jobs["4ph"]
    check3(fp, j3, _sample(j3.targets3, 3, 12, always=(7,)), scratch_bytes=FULL_SCRATCH)
    g, c = check4(fp, j4, np.ascontiguousarray(j4.targets4[[29]]), qp=(17, 18), scratch_bytes=FULL_SCRATCH)
    assert c.sum() > 10000


def test_list_overflow_falls_back_to_fused(fp):
    """With the filter disabled every candidate is allowed, so the list slots of the group path (a quarter of the
    candidates a unit can meet, at least 2048 entries) fill up on a 16x8x8 mesh (two 32-point tiles per unit: 2304
    candidates): k_enum_g marks the rows whose slot filled up and the driver redoes those rows through the fused kernel."""
    inp = fp_inputs.make_tiny("diamond", mesh=(16, 8, 8))
    t = np.ascontiguousarray(inp.targets4[[100, 205]])
    kw = dict(ncut=np.inf, sigma_const=5.0)
    og, ow, oc = _oracle(inp, **kw).rates4(t, 5, 6)
    with fp.Context.from_inputs(inp, scratch_bytes=256 << 20, **kw) as ctx:
        ctx.set_path(fp.FP_PATH_SPLIT_SERIAL)
        ctx.profile_enable(True)
        g, w, c = ctx.rates4(t, 5, 6)
        p = ctx.profile_get()
    assert p.list_overflows > 0 and p.n_enum > 0
    assert np.array_equal(c, oc)
    assert_rates_close(g, og, "Gamma4 (overflow fallback)")
    assert_rates_close(w, ow, "WP4 (overflow fallback)")
    # the ordinary filter never comes near the slot size
    with fp.Context.from_inputs(inp, scratch_bytes=256 << 20) as ctx:
        ctx.set_path(fp.FP_PATH_SPLIT_SERIAL)
        ctx.profile_enable(True)
        ctx.rates4(t, 5, 6)
        assert ctx.profile_get().list_overflows == 0


def test_pair_symmetry_of_the_4ph_channels(fp):
    """fp_setup detects that the (symmetrised) IFC4 list is invariant under the exchange of its last two legs; the split path
    then lists each unordered {lambda'', lambda'''} pair of the +- and -- channels once.  Counts must not change at all, rates
    only by summation order; about half of the matrix elements are evaluated."""
    inp = fp_inputs.make_tiny("diamond", mesh=(4, 4, 4))
    t = inp.targets4[30:54]
    res = {}
    for on in (True, False):
        with fp.Context.from_inputs(inp, scratch_bytes=256 << 20) as ctx:
            ctx.set_path(fp.FP_PATH_SPLIT_SERIAL)
            ctx.set_symmetry(on)
            ctx.set_target_symmetry(False)
            assert ctx.get_symmetry() == on
            ctx.profile_enable(True)
            res[on] = ctx.rates4(t)
            p = ctx.profile_get()
            res[on] += (p.evaluated, p.processes)
    (g1, w1, c1, e1, p1), (g0, w0, c0, e0, p0) = res[True], res[False]
    assert np.array_equal(c1, c0) and p1 == p0 == int(c0.sum())
    assert e0 == p0 and e1 < 0.62 * e0                               # ++ is not reduced, +- and -- are halved
    assert np.allclose(g1, g0, rtol=1e-12, atol=1e-13 * np.abs(g0).max())
    assert np.allclose(w1, w0, rtol=1e-12, atol=1e-13 * np.abs(w0).max())
    # the 3ph - channel (lambda' <-> lambda'') in the same way
    r3 = {}
    for on in (True, False):
        with fp.Context.from_inputs(inp, scratch_bytes=256 << 20) as ctx:
            ctx.set_path(fp.FP_PATH_SPLIT_SERIAL)
            ctx.set_symmetry(on)
            ctx.profile_enable(True)
            r3[on] = ctx.rates3(inp.targets3) + (ctx.profile_get().evaluated,)
    assert np.array_equal(r3[True][2], r3[False][2]) and r3[True][3] < 0.8 * r3[False][3]
    assert np.allclose(r3[True][0], r3[False][0], rtol=1e-12, atol=1e-13 * np.abs(r3[False][0]).max())
    assert np.allclose(r3[True][1], r3[False][1], rtol=1e-12, atol=1e-13 * np.abs(r3[False][1]).max())


def test_asymmetric_ifc_disables_the_pair_symmetry(fp):
    """An IFC4 list that is not symmetric in its last two legs (one entry perturbed) must be evaluated over the full
    domain -- and still match the oracle, which never uses any symmetry."""
    inp = fp_inputs.make_tiny("diamond", mesh=(3, 3, 3))
    a4, c4, p4 = inp.ifc4
    p4 = p4.copy()
    p4[3, 1 * 27 + 0 * 9 + 1 * 3 + 2] += 0.37                        # component (y,x,y,z) of one quartet
    inp.ifc4 = (a4, c4, p4)
    t = inp.targets4[7:19]
    with fp.Context.from_inputs(inp, scratch_bytes=64 << 20) as ctx:
        assert ctx.get_symmetry_mask() & 2 == 0 and ctx.get_symmetry_mask() & 1 == 1   # IFC3 is still symmetric
    check4(fp, inp, t)
    a3, c3, p3 = inp.ifc3
    p3 = p3.copy()
    p3[5, 0 * 9 + 1 * 3 + 2] -= 0.21                                 # component (x,y,z) of one triplet
    inp.ifc3 = (a3, c3, p3)
    with fp.Context.from_inputs(inp, scratch_bytes=64 << 20) as ctx:
        assert ctx.get_symmetry_mask() == 0
    check3(fp, inp, inp.targets3[::5])


def test_time_reversal_reuse_over_targets(fp):
    """fp_setup finds the generated mode arrays time-reversal symmetric bit for bit (fp_inputs sets e(-q) = conj(e(q)),
    v(-q) = -v(q), reading 17); fp_rates3 / full-range fp_rates4 then evaluate one target of each {(q,j), (-q,j)} pair.
    Counts must not change at all, rates only by rounding order; about half of the 3ph work is done; a partial q' range
    does not use it; a mode array that breaks the symmetry turns it off -- and every variant still matches the oracle."""
    inp = fp_inputs.make_tiny("diamond", mesh=(4, 3, 3))
    orc = _oracle(inp)
    og3, ow3, oc3 = orc.rates3(inp.targets3)
    res = {}
    for on in (True, False):
        with fp.Context.from_inputs(inp, scratch_bytes=256 << 20) as ctx:
            ctx.set_target_symmetry(on)
            assert ctx.get_target_symmetry() == on
            ctx.profile_enable(True)
            res[on] = ctx.rates3(inp.targets3) + (ctx.profile_get().evaluated,)
    (g1, w1, c1, e1), (g0, w0, c0, e0) = res[True], res[False]
    assert np.array_equal(c1, c0) and np.array_equal(c1, oc3)
    assert e1 < 0.62 * e0
    assert np.allclose(g1, g0, rtol=1e-12, atol=1e-13 * np.abs(g0).max())
    assert_rates_close(g1, og3, "Gamma3 (time reversal)")
    assert_rates_close(w1, ow3, "WP3 (time reversal)")
    # 4ph: all branches of a q-point and of its partner -q, whole q' range (reuse) and a partial range (none)
    N1, N2, N3 = (int(x) for x in inp.mesh)
    q = 1 + N1 * (2 + N2 * 1)
    qm = (N1 - 1) % N1 + N1 * ((N2 - 2) % N2 + N2 * ((N3 - 1) % N3))
    t4 = np.array([q * inp.nb + j for j in range(inp.nb)] + [qm * inp.nb + j for j in range(inp.nb)], dtype=np.int32)
    og4, ow4, oc4 = orc.rates4(t4)
    ogp, owp, ocp = orc.rates4(t4, 3, 9)
    with fp.Context.from_inputs(inp, scratch_bytes=256 << 20) as ctx:
        ctx.profile_enable(True)
        g, w, c = ctx.rates4(t4)
        ev_full = ctx.profile_get().evaluated
        gp, wp_, cp = ctx.rates4(t4, 3, 9)
        ctx.set_target_symmetry(False)
        ctx.profile_reset()
        g_, w_, c_ = ctx.rates4(t4)
        assert ctx.profile_get().evaluated == 2 * ev_full
    assert np.array_equal(c, oc4) and np.array_equal(c_, oc4) and np.array_equal(cp, ocp)
    assert np.array_equal(c[:inp.nb], c[inp.nb:])
    assert_rates_close(g, og4, "Gamma4 (time reversal)")
    assert_rates_close(gp, ogp, "Gamma4 (partial q' range)")
    assert np.allclose(g, g_, rtol=1e-12, atol=1e-13 * np.abs(g_).max())
    # broken symmetry: one eigenvector component of one mode changed by an ulp-scale amount
    import copy
    bad = copy.copy(inp)
    bad.eig = inp.eig.copy()
    bad.eig.reshape(-1)[5 * inp.nb * inp.nb * 2 + 3] *= (1.0 + 1e-12)
    with fp.Context.from_inputs(bad, scratch_bytes=256 << 20) as ctx:
        assert not ctx.get_target_symmetry()
        gb, wb, cb = ctx.rates3(inp.targets3)
    assert np.array_equal(cb, oc3)
    assert np.allclose(gb, og3, rtol=1e-9, atol=1e-9 * np.abs(og3).max())


def test_per_process_terms(fp):
    """fp_terms3 / fp_terms4: the process lists of fp_list3/4 with each process's
    contribution to Gamma.  The terms sum to the oracle's Gamma of that target, channel (and q'), their number is the
    oracle's count, and sampled terms equal an independent numpy evaluation (dense-Fourier matrix element x weights; a
    matrix element that vanishes by symmetry is rounding noise on both sides, hence the floor of 1e-14 of the largest term)."""
    from . import bruteforce as bf
    inp = fp_inputs.make_tiny("diamond", mesh=(3, 3, 3))
    orc = _oracle(inp)
    rng = np.random.default_rng(5)
    with fp.Context.from_inputs(inp, scratch_bytes=256 << 20) as ctx:
        for lam in (7, 40, 101):
            og, ow, oc = orc.rates3(np.array([lam], dtype=np.int32))
            for ch in (0, 1):
                pairs, g = ctx.terms3(lam, ch)
                assert len(g) == int(oc[0, ch]) and np.array_equal(pairs, ctx.list3(lam, ch))
                assert abs(g.sum() - og[0, ch]) <= 1e-9 * abs(og[0, ch])
                for i in rng.choice(len(g), size=min(4, len(g)), replace=False):
                    ref = bf.term3_dense(inp, lam, ch, pairs[i])
                    assert abs(g[i] - ref) <= 1e-8 * abs(ref) + 1e-14 * g.max(), (lam, ch, pairs[i], g[i], ref)
        for lam, qp in ((8, 5), (61, 20), (20, 3)):
            og, ow, oc = orc.rates4(np.array([lam], dtype=np.int32), qp, qp + 1)
            for ch in (0, 1, 2):
                triples, g = ctx.terms4(lam, ch, qp)
                assert len(g) == int(oc[0, ch]) and np.array_equal(triples, ctx.list4(lam, ch, qp))
                assert abs(g.sum() - og[0, ch]) <= 1e-9 * max(abs(og[0, ch]), 1e-10 * np.abs(og).max())   # (floor: DESIGN.md §5.2)
                for i in rng.choice(len(g), size=min(3, len(g)), replace=False):
                    ref = bf.term4_dense(inp, lam, ch, triples[i])
                    assert abs(g[i] - ref) <= 1e-8 * abs(ref) + 1e-14 * np.abs(og).max(), (lam, ch, triples[i], g[i], ref)


def test_mixed_precision_mode(fp):
    """fp_set_precision(FP_PREC_MIXED): the level-2 contraction in FP32.  Counts and
    the weighted phase space must not change at all (the decision and the weights stay FP64); Gamma carries the FP32
    rounding of |V|^2 -- checked against the oracle at 2e-5 relative to the channel's largest rate, and it must really
    differ from the FP64 result (the switch does something).  Off by default."""
    inp = fp_inputs.make_tiny("diamond", mesh=(4, 4, 4))
    t = np.ascontiguousarray(inp.targets4[12:36])
    og, ow, oc = _oracle(inp).rates4(t, 3, 12)
    og3, ow3, oc3 = _oracle(inp).rates3(inp.targets3)
    with fp.Context.from_inputs(inp, scratch_bytes=256 << 20) as ctx:
        assert ctx.get_precision() == fp.FP_PREC_FP64
        g64, w64, c64 = ctx.rates4(t, 3, 12)
        ctx.set_precision(fp.FP_PREC_MIXED)
        assert ctx.get_precision() == fp.FP_PREC_MIXED
        g, w, c = ctx.rates4(t, 3, 12)
        g3, w3, c3 = ctx.rates3(inp.targets3)
    assert np.array_equal(c, oc) and np.array_equal(w, w64) and np.array_equal(c3, oc3)
    assert_rates_close(w3, ow3, "WP3 (mixed)")
    for a, ref, what in ((g, og, "Gamma4"), (g3, og3, "Gamma3")):
        scale = np.abs(ref).max(axis=0, keepdims=True)
        err = np.abs(a - ref) / scale
        assert err.max() < 2e-5, (what, err.max())
    assert np.abs(g - g64).max() > 0.0
    assert_rates_close(g64, og, "Gamma4 (FP64)")


def test_long_ifc3_list_reads_the_block_table_from_global_memory(fp):
    """ADVICE.md / include/fourphonon.h "Limits": an IFC3 list with more contraction blocks (atomA, atomB, R_A - R_B mod mesh)
    than the shared memory of one SM can hold as a per-row table (about 1,400) is still served -- the 3ph kernels then read
    Mhat from the level-0 table in global memory.  A synthetic list of 1,700 triplets, one block each, on an 8x8x8 mesh: rates,
    weighted phase space and counts of a few targets against the oracle on the group path and the fused path, and the
    per-process terms."""
    import copy
    base = fp_inputs.make_tiny("diamond", mesh=(8, 8, 8), with4=False)
    rng = np.random.default_rng(11)
    n = 1700
    combos = rng.permutation(4 * 512)[:n]                            # distinct (atom j, atom k, R_j - R_k mod 8)
    aj, ak, dr = combos // 1024, (combos // 512) % 2, combos % 512
    d3 = np.stack([dr % 8, (dr // 8) % 8, dr // 64], axis=1)
    Rk = rng.integers(-1, 2, size=(n, 3))
    atoms = np.stack([rng.integers(0, 2, size=n), aj, ak], axis=1).astype(np.int32)
    cells = np.concatenate([Rk + d3, Rk], axis=1).reshape(n, 2, 3).astype(np.int32)
    phi = rng.normal(0.0, 0.5, size=(n, 27))
    inp = copy.copy(base)
    inp.ifc3 = (np.ascontiguousarray(atoms), np.ascontiguousarray(cells), np.ascontiguousarray(phi))
    t = np.array([5, 700, 1501, 3070], dtype=np.int32)
    og, ow, oc = _oracle(inp).rates3(t)
    assert oc.sum() > 1000
    for path in (fp.FP_PATH_AUTO, fp.FP_PATH_FUSED):
        with fp.Context.from_inputs(inp, scratch_bytes=1 << 30) as ctx:
            ctx.set_path(path)
            g, w, c = ctx.rates3(t)
            assert np.array_equal(c, oc)
            assert_rates_close(g, og, f"Gamma3 (long IFC3 list, path {path})")
            assert_rates_close(w, ow, f"WP3 (long IFC3 list, path {path})")
            if path == fp.FP_PATH_FUSED:
                pairs, gp = ctx.terms3(int(t[1]), 1)
                assert len(gp) == int(oc[1, 1]) and abs(gp.sum() - og[1, 1]) <= 1e-9 * abs(og[1, 1])
