"""-m gpu, collected last: fp_kappa_rta_static -- the RTA kappa for callers that cannot allocate (static device scratch,
include/fourphonon.h) -- against the existing fp_kappa_rta on the same rates, within the 1e-9 the other tests use, on two
calls in a row (the calls share the static array, which keeps the last call's contents), with host and with device
buffers; and the rejection of a mesh beyond FP_NOALLOC_MAX_MODES.  Passes alone in a fresh process and after the others.
"""
import numpy as np
import pytest

import fp_inputs

from .test_gpu_parity import RTOL, fp  # noqa: F401  (fp is the module fixture)

pytestmark = pytest.mark.gpu


def _close(k, ref):
    return np.abs(np.asarray(k) - np.asarray(ref)).max() <= RTOL * np.abs(ref).max()


def test_kappa_rta_static_matches_kappa_rta_on_two_calls_in_a_row(fp):
    import torch
    inp = fp_inputs.make_tiny("diamond", mesh=(4, 4, 4), with4=False)
    with fp.Context.from_inputs(inp, scratch_bytes=64 << 20) as ctx:
        g3, _, _ = ctx.rates3(inp.targets3)
        gt1 = g3.sum(axis=1)
        gt2 = 0.5 * gt1 + 0.25 * gt1.max()                           # different rates: stale scratch would show
        ref1, ref2 = ctx.kappa_rta(gt1), ctx.kappa_rta(gt2)          # the existing path
        assert np.abs(ref1).max() > 0 and not _close(ref2, ref1)
        # host buffers: two calls in a row, then the first again
        k1 = ctx.kappa_rta_static(gt1)
        k2 = ctx.kappa_rta_static(gt2)
        k1b = ctx.kappa_rta_static(gt1)
        assert _close(k1, ref1), np.abs(k1 - ref1).max() / np.abs(ref1).max()
        assert _close(k2, ref2), np.abs(k2 - ref2).max() / np.abs(ref2).max()
        assert np.array_equal(k1, k1b)                               # fixed summation order: reproducible
        # device buffers (asynchronous): two calls back to back on the current stream, read afterwards
        d1, d2 = torch.from_numpy(gt1).cuda(), torch.from_numpy(gt2).cuda()
        kd1 = ctx.kappa_rta_static(d1)
        kd2 = ctx.kappa_rta_static(d2)
        torch.cuda.synchronize()
        assert np.array_equal(kd1.cpu().numpy(), k1) and np.array_equal(kd2.cpu().numpy(), k2)
        # zero and negative rates are skipped exactly as in fp_kappa_rta
        gt3 = gt1.copy(); gt3[::5] = 0.0; gt3[3::7] = -1.0
        assert _close(ctx.kappa_rta_static(gt3), ctx.kappa_rta(gt3))


def test_kappa_rta_static_rejects_meshes_beyond_its_scratch(fp):
    inp = fp_inputs.make_tiny("sc1", mesh=(28, 28, 28), with4=False)  # 21,952 q-points x 3 branches = 65,856 modes
    assert inp.nq * inp.nb > fp.FP_NOALLOC_MAX_MODES
    with fp.Context.from_inputs(inp, scratch_bytes=64 << 20) as ctx:
        gt = np.ones(inp.nq * inp.nb)
        with pytest.raises(fp.FourPhononError) as err:
            ctx.kappa_rta_static(gt)
        assert err.value.code == fp.FP_EINVAL and "FP_NOALLOC_MAX_MODES" in str(err.value)
        assert np.abs(ctx.kappa_rta(gt)).max() > 0                   # the existing path still serves this mesh
