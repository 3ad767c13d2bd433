"""nms_azimuthal_average_noalloc (csrc/k_noalloc.cu): the |q|-histogram average with its scratch in a static device array,
for callers that cannot call cudaMalloc.  Checked against the existing path (nms_azimuthal_average) on the same maps: counts
and bin abscissae bit-exact, averages within the tolerance the existing histogram test uses (rtol 2e-6: the two paths differ
in the order of the fp64 additions, then round once to fp32).  Two calls in a row with different shapes, so that the second
one would see the first one's leftovers if the scratch were not cleared.

Collected last on purpose (the suite runs with pytest -x); it must pass alone in a fresh process and after the other tests.
"""
import os
import sys

import numpy as np
import pytest

sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
import nms_inputs as ni  # noqa: E402

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def nms():
    import torch
    assert torch.cuda.is_available(), "GPU tests need a CUDA device"
    import paper_2601_18444_b200 as mod
    return mod


def _dev(a):
    import torch
    return None if a is None else torch.as_tensor(np.ascontiguousarray(a), device="cuda")


def _both_paths(nms, h, maps, n_maps, nb, q_lo, q_hi):
    import torch
    out = []
    for fn in (nms.nms_azimuthal_average, nms.nms_azimuthal_average_noalloc):
        I = torch.full((n_maps, nb), -7.0, dtype=torch.float32, device="cuda")
        qb = torch.full((nb,), -7.0, dtype=torch.float32, device="cuda")
        cnt = torch.full((nb,), -7, dtype=torch.int32, device="cuda")
        fn(h, maps, n_maps, nb, q_lo, q_hi, I, qb, cnt)
        nms.nms_synchronize(h)
        out.append((I.cpu().numpy(), qb.cpu().numpy(), cnt.cpu().numpy()))
    return out


def _compare(ref, got, what):
    I_ref, q_ref, c_ref = ref
    I_got, q_got, c_got = got
    assert np.array_equal(c_got, c_ref), what + ": counts"
    assert np.array_equal(q_got, q_ref), what + ": bin abscissae"
    assert c_ref.sum() > 0
    np.testing.assert_allclose(I_got, I_ref, rtol=2e-6, atol=0, err_msg=what)


def test_noalloc_histogram_matches_existing_path_twice(nms):
    import torch
    with nms.Context(0) as ctx:
        h = ctx.h
        # call 1: C2 (Cartesian 128 x 128 detector), its own 13 kinds and bin range
        w2 = ni.make_config("C2")
        nms.nms_set_sample(h, _dev(w2.pos), _dev(w2.N), _dev(w2.m), w2.R)
        k2 = list(w2.kinds)
        maps2 = torch.empty((len(k2), w2.grid.n_q), dtype=torch.float32, device="cuda")
        nms.nms_compute(h, w2.grid, k2, maps2)
        ref, got = _both_paths(nms, h, maps2, len(k2), w2.n_bins, w2.q_lo, w2.q_hi)
        _compare(ref, got, "C2 histogram, first call")

        # call 2, straight after it: C1 (polar detector) with a finer histogram than its rings (many empty bins, which must
        # read 0 with count 0 although call 1 left sums and counts in the shared scratch), 2 maps instead of 13
        w1 = ni.make_config("C1")
        nms.nms_set_sample(h, _dev(w1.pos), _dev(w1.N), _dev(w1.m), w1.R)
        k1 = [ni.KIND_INDEX["NUC"], ni.KIND_INDEX["NM"]]
        maps1 = torch.empty((2, w1.grid.n_q), dtype=torch.float32, device="cuda")
        nms.nms_compute(h, w1.grid, k1, maps1)
        ref, got = _both_paths(nms, h, maps1, 2, 200, 0.5, 2.0)
        _compare(ref, got, "C1 fine histogram, second call")
        assert (ref[2] == 0).sum() > 50
        assert np.all(got[0][:, ref[2] == 0] == 0.0)

        # the same call again: identical counts, averages within the tolerance again
        ref3, got3 = _both_paths(nms, h, maps1, 2, 200, 0.5, 2.0)
        _compare(ref3, got3, "C1 fine histogram, third call")

        # a second context on the same device shares the scratch (serialised here by the synchronize in _both_paths)
        with nms.Context(0) as ctx_b:
            hb = ctx_b.h
            nms.nms_set_sample(hb, _dev(w2.pos), _dev(w2.N), _dev(w2.m), w2.R)
            nms.nms_compute(hb, w2.grid, k2, maps2)
            ref, got = _both_paths(nms, hb, maps2, len(k2), w2.n_bins, w2.q_lo, w2.q_hi)
            _compare(ref, got, "C2 histogram, second context")


def test_noalloc_limits_and_errors(nms):
    import torch
    with nms.Context(0) as ctx:
        h = ctx.h
        w1 = ni.make_config("C1")
        out = torch.empty((5, 16385), dtype=torch.float32, device="cuda")
        maps = torch.zeros((5, w1.grid.n_q), dtype=torch.float32, device="cuda")
        with pytest.raises(nms.NmsError) as e:                          # no grid yet
            nms.nms_azimuthal_average_noalloc(h, maps, 1, 64, 0.0, 1.0, out)
        assert e.value.status == nms.NMS_E_STATE
        nms.nms_set_sample(h, _dev(w1.pos), _dev(w1.N), _dev(w1.m), w1.R)
        nms.nms_compute(h, w1.grid, [0, 1, 2, 3, 4], maps)
        with pytest.raises(nms.NmsError) as e:                          # more bins than the static scratch holds
            nms.nms_azimuthal_average_noalloc(h, maps, 1, 16385, 0.0, 3.0, out)
        assert e.value.status == nms.NMS_E_UNSUPPORTED and "16384" in str(e.value)
        with pytest.raises(nms.NmsError) as e:                          # n_maps * n_bins beyond it
            nms.nms_azimuthal_average_noalloc(h, maps, 5, 16384, 0.0, 3.0, out)
        assert e.value.status == nms.NMS_E_UNSUPPORTED and "65536" in str(e.value)
        with pytest.raises(nms.NmsError) as e:                          # ring mode: not this entry point
            nms.nms_azimuthal_average_noalloc(h, maps, 4, w1.grid.n0, 0.0, 0.0, out)
        assert e.value.status == nms.NMS_E_ARG
        # at the limit: 4 maps x 16384 bins = 65536 sums
        ref, got = _both_paths(nms, h, maps, 4, 16384, 0.0, 3.0)
        _compare(ref, got, "C1 histogram at the scratch limit")
