"""-m gpu: parity at BASELINE.json's full sizes (north_star: "bit-exact counts and 1e-9 rates on all five configs").

The oracle cannot evaluate V for 10^10 processes, but in its weights-only mode (orc_rates3/4 with weights_only = 1: the
same loops, the same pinned window decision, the same weights, |V|^2 replaced by 1) it walks ~5x10^8 candidates/s on
16 cores.  So over FULL q' ranges these tests compare what the enumerator and the weight code decide -- process counts
bit-exact, weighted phase space WP to 1e-9 -- and over narrow q' ranges (tests/test_gpu_parity.py and below) the rates
Gamma themselves.  Every comparison runs on the configuration bench.py times (FP_PATH_AUTO with a 48 GB scratch, which
picks the group path) as well as on the fused and two-stream split paths with a small scratch.

Also here: kappa at 16x16x16 (config 1) and the self-check of the FP32 pre-filter's superset claim:
counts with every FP32 test disabled (fp_set_prefilter(ctx, 0)) equal the counts with the filter on, bit for bit.
"""
import numpy as np
import pytest

import fp_inputs

from .test_gpu_parity import RTOL, _oracle, assert_rates_close, fp  # noqa: F401  (fp is the module fixture)

pytestmark = pytest.mark.gpu

BENCH_SCRATCH = 48 << 30          # bench.py's default (--scratch-gb 48)
SMALL_SCRATCH = 4 << 30


def _configs(fp):
    """(label, scratch, path): the bench configuration first"""
    return (("auto/48GB", BENCH_SCRATCH, fp.FP_PATH_AUTO), ("fused/4GB", SMALL_SCRATCH, fp.FP_PATH_FUSED),
            ("split/4GB", SMALL_SCRATCH, fp.FP_PATH_SPLIT))


def _counts_and_wp4(fp, inp, targets, qp=(0, None), configs=None):
    """GPU rates4 on every configuration vs the oracle's weights-only pass: counts bit-exact, WP to 1e-9."""
    _, ow, oc = _oracle(inp).rates4(targets, qp[0], qp[1], weights_only=True)
    out = None
    for label, scratch, path in (configs or _configs(fp)):
        with fp.Context.from_inputs(inp, scratch_bytes=scratch) as ctx:
            ctx.set_path(path)
            g, w, c = ctx.rates4(targets, qp[0], qp[1])
        assert np.array_equal(c, oc), f"4ph process counts are not bit-exact ({label})"
        assert_rates_close(w, ow, f"WP4 ({label})")
        if out is not None:                                           # the paths agree on Gamma to summation order
            assert_rates_close(g, out[0], f"Gamma4 ({label} vs {_configs(fp)[0][0]})")
        else:
            out = (g, w, c)
    return out


def test_config3_six_branches_full_q_range_counts_and_wp(fp):
    """config 3 (16x16x16): the six branches of one target q-point over ALL 4096 q' -- 6.5x10^10 of the step's 1.05x10^12
    candidates (6 %), 1.4x10^9 processes -- counts bit-exact and WP to 1e-9 against the oracle."""
    inp = fp_inputs.make_config(3)["main"]
    t = np.ascontiguousarray(inp.targets4[30:36])
    assert len(set(int(x) // inp.nb for x in t)) == 1 and sorted(int(x) % inp.nb for x in t) == list(range(6))
    g, w, c = _counts_and_wp4(fp, inp, t)
    assert c.sum() > 10 ** 9


def test_config2_all_targets_full_q_range_counts_and_wp(fp):
    """config 2 (8x8x8): all 192 targets over all 512 q': the whole job's counts (1.3x10^9 processes) and WP."""
    inp = fp_inputs.make_config(2)["main"]
    g, w, c = _counts_and_wp4(fp, inp, inp.targets4)
    assert c.sum() > 10 ** 9


def test_config4_4ph_eight_targets_full_q_range_and_gamma_samples(fp):
    """config 4 (8 atoms, 24 branches, 6x6x6, generic kernels): eight targets spread over branches and q-points over all
    216 q' (counts + WP), and Gamma itself on three (target, q') pairs."""
    j4 = fp_inputs.make_config(4)["4ph"]
    idx = [0, 23, 29, 50, 77, 100, 150, 191]
    t = np.ascontiguousarray(j4.targets4[idx])
    g, w, c = _counts_and_wp4(fp, j4, t)
    assert c.sum() > 10 ** 8
    orc = _oracle(j4)
    for ti, qp in ((3, 5), (77, 100), (170, 211)):
        tt = np.ascontiguousarray(j4.targets4[[ti]])
        og, ow, oc = orc.rates4(tt, qp, qp + 1)
        for label, scratch, path in _configs(fp):
            with fp.Context.from_inputs(j4, scratch_bytes=scratch) as ctx:
                ctx.set_path(path)
                gg, ww, cc = ctx.rates4(tt, qp, qp + 1)
            assert np.array_equal(cc, oc)
            assert_rates_close(gg, og, f"Gamma4 config 4 target {ti} q' {qp} ({label})")
            assert_rates_close(ww, ow, f"WP4 config 4 target {ti} q' {qp} ({label})")


def test_config3_gamma_on_the_bench_configuration(fp):
    """Gamma (with V) over a narrow q' range on FP_PATH_AUTO with the bench's 48 GB scratch: six branches of one q-point."""
    inp = fp_inputs.make_config(3)["main"]
    t = np.ascontiguousarray(inp.targets4[60:66])
    og, ow, oc = _oracle(inp).rates4(t, 2222, 2224)
    with fp.Context.from_inputs(inp, scratch_bytes=BENCH_SCRATCH) as ctx:
        g, w, c = ctx.rates4(t, 2222, 2224)
    assert np.array_equal(c, oc)
    assert_rates_close(g, og, "Gamma4 (auto/48GB)")
    assert_rates_close(w, ow, "WP4 (auto/48GB)")


def test_config1_all_modes_counts_wp_and_kappa_at_16cubed(fp):
    """config 1 (3ph, 16x16x16): ALL 24,576 target modes -- counts bit-exact and WP to 1e-9 against the oracle's
    weights-only pass (1.5x10^8 processes), Gamma on a sample (tests/test_gpu_parity.py), and kappa_RTA of the GPU's
    own Gamma_3 against orc_kappa of the same array."""
    inp = fp_inputs.make_config(1)["main"]
    orc = _oracle(inp)
    _, ow, oc = orc.rates3(inp.targets3, weights_only=True)
    first = None
    for label, scratch, path in _configs(fp):
        with fp.Context.from_inputs(inp, scratch_bytes=scratch) as ctx:
            ctx.set_path(path)
            g, w, c = ctx.rates3(inp.targets3)
            gt = g.sum(axis=1)
            k = ctx.kappa_rta(gt)
        assert np.array_equal(c, oc), f"3ph process counts are not bit-exact ({label})"
        assert_rates_close(w, ow, f"WP3 ({label})")
        ok = orc.kappa(gt)
        assert np.abs(k - ok).max() <= RTOL * np.abs(ok).max(), f"kappa ({label})"
        if first is None:
            first = g
        else:
            assert_rates_close(g, first, f"Gamma3 ({label} vs auto)")
    assert oc.sum() > 10 ** 8


def _counts_filter_on_off(fp, inp, targets, qp, order=4):
    res = []
    with fp.Context.from_inputs(inp, scratch_bytes=SMALL_SCRATCH) as ctx:
        for on in (True, False):
            ctx.set_prefilter(on)
            ctx.profile_reset(); ctx.profile_enable(True)
            g, w, c = ctx.rates4(targets, qp[0], qp[1]) if order == 4 else ctx.rates3(targets)
            res.append((g, w, c, ctx.profile_get()))
    (g1, w1, c1, p1), (g0, w0, c0, p0) = res
    assert p0.prefiltered > 5 * p1.prefiltered                        # the switch really removed the filter
    assert np.array_equal(c1, c0), "counts depend on the FP32 pre-filter"
    assert np.array_equal(w1, w0) and np.array_equal(g1, g0)          # the same processes in the same order
    return c1


def test_prefilter_is_a_superset_config2_whole_job(fp):
    """the FP32 tests admit every candidate the pinned FP64 decision allows.  Checked on the GPU itself
    at full size: all 3.3x10^10 candidates of config 2 decided with and without the filter, per-(target, channel) counts
    (and rates: same lists, same order) bit-identical."""
    inp = fp_inputs.make_config(2)["main"]
    c = _counts_filter_on_off(fp, inp, inp.targets4, (0, None))
    assert c.sum() > 10 ** 9


def test_prefilter_is_a_superset_config3_one_percent(fp):
    """... and on two targets of config 3 over all q' (2.2x10^10 of 1.05x10^12 candidates, 2 %), plus the 3ph leg in full."""
    inp = fp_inputs.make_config(3)["main"]
    c = _counts_filter_on_off(fp, inp, np.ascontiguousarray(inp.targets4[[13, 88]]), (0, None))
    assert c.sum() > 10 ** 8
    c3 = _counts_filter_on_off(fp, inp, inp.targets3[::7], None, order=3)
    assert c3.sum() > 10 ** 7


# ---- the paper's own mesh sizes: fp_inputs configs 5-7 ---------------------------
def test_paper_mesh_32cubed_3ph_sampled(fp):
    """3ph at 32x32x32 (196,608 modes): counts + WP of 768 targets spread over the mesh against the oracle's
    weights-only pass, Gamma (with V) of 24 of them; the whole job runs on the bench configuration."""
    inp = fp_inputs.make_config(5)["main"]
    orc = _oracle(inp)
    t = np.ascontiguousarray(inp.targets3[5::256])
    assert len(t) == 768
    _, ow, oc = orc.rates3(t, weights_only=True)
    tg = np.ascontiguousarray(t[::32])
    og, ogw, ogc = orc.rates3(tg)
    with fp.Context.from_inputs(inp, scratch_bytes=BENCH_SCRATCH) as ctx:
        g, w, c = ctx.rates3(t)
        ga, wa, ca = ctx.rates3(inp.targets3)                         # all modes in one call: the same rows, bit for bit
    assert np.array_equal(c, oc), "3ph process counts are not bit-exact at 32^3"
    assert_rates_close(w, ow, "WP3 32^3")
    assert np.array_equal(c[::32], ogc)
    assert_rates_close(g[::32], og, "Gamma3 32^3")
    assert np.array_equal(ca[5::256], c) and np.array_equal(ga[5::256], g) and np.array_equal(wa[5::256], w)


@pytest.mark.parametrize("cfg", [6, 7])
def test_paper_mesh_4ph_sampled_and_3ph_kappa(fp, cfg):
    """3ph + 4ph at 10x10x10 and 14x14x14: lcm 10 / 14 is not a power of two (the `% L` phase index and
    the table look-up of q coordinates at size).  4ph: two targets over ALL q' (counts + WP), Gamma of six branches on
    two q'; 3ph: all modes counts + WP, kappa of the GPU's Gamma_3 against orc_kappa."""
    inp = fp_inputs.make_config(cfg)["main"]
    orc = _oracle(inp)
    t2 = np.ascontiguousarray(inp.targets4[[7, 52]])
    _counts_and_wp4(fp, inp, t2, configs=_configs(fp)[:2])
    t6 = np.ascontiguousarray(inp.targets4[18:24])
    q0 = inp.nq // 3
    og, ow, oc = orc.rates4(t6, q0, q0 + 2)
    _, ow3, oc3 = orc.rates3(inp.targets3, weights_only=True)
    with fp.Context.from_inputs(inp, scratch_bytes=BENCH_SCRATCH) as ctx:
        g, w, c = ctx.rates4(t6, q0, q0 + 2)
        g3, w3, c3 = ctx.rates3(inp.targets3)
        gt = g3.sum(axis=1)
        k = ctx.kappa_rta(gt)
    assert np.array_equal(c, oc)
    assert_rates_close(g, og, f"Gamma4 config {cfg}")
    assert_rates_close(w, ow, f"WP4 config {cfg}")
    assert np.array_equal(c3, oc3), "3ph process counts are not bit-exact"
    assert_rates_close(w3, ow3, f"WP3 config {cfg}")
    ok = orc.kappa(gt)
    assert np.abs(k - ok).max() <= RTOL * np.abs(ok).max()
