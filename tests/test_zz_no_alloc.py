"""teuk_get_folded_static (include/teuk.h): the allocation-free variant of teuk_get_folded -- the same kernel writing into
the library's file-scope `static __device__` scratch array instead of a cudaMalloc'ed buffer -- must return the planes of
the existing path BIT FOR BIT, on two calls in a row (the array is shared and keeps the previous call's contents), on
grids of different sizes, and must refuse grids beyond its fixed capacity.  Collected last on purpose (the suite runs
with `pytest -x`); it passes alone in a fresh process and after the other tests."""
import numpy as np
import pytest

from paper_1006_0663_b200 import inputs

pytestmark = pytest.mark.gpu


@pytest.fixture(scope="module")
def teuk():
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_1006_0663_b200 import teuk as t
    return t


def _handle(teuk, n_r, n_theta):
    w = inputs.config(2).scaled(n_r=n_r, n_theta=n_theta, rstar_min=-30.0, rstar_max=60.0, precision=1)
    w = w.scaled(dt_override=inputs.stable_dt(w))
    return teuk.Teuk.from_workload(w)


def test_static_scratch_matches_the_allocating_path_on_consecutive_calls(teuk):
    big = _handle(teuk, 1000, 40)            # 8 * 40 * 1008 = 322 560 doubles: inside the 524 288 limit
    small = _handle(teuk, 75, 6)             # a later, smaller call must not see the larger call's leftovers
    for g in (big, small, big):
        for variant in (1, 2):
            for half in (False, True):
                ref = g.folded(half, variant)                # existing path: cudaMalloc'ed scratch
                first = g.folded_static(half, variant)
                second = g.folded_static(half, variant)      # two calls in a row on the shared array
                assert np.array_equal(first, ref) and np.array_equal(second, ref)
                assert np.isfinite(ref).all() and np.abs(ref).max() > 0
    # the output buffer is written in full (pre-filled with a sentinel)
    out = np.full((8, 6, 75), np.nan)
    small.folded_static(False, 1, out)
    assert np.array_equal(out, small.folded(False, 1))


def test_static_scratch_rejects_what_does_not_fit(teuk):
    g = _handle(teuk, 4096, 32)              # 8 * 32 * 4096 = 1 048 576 doubles > TEUK_STATIC_SCRATCH_DOUBLES
    assert 8 * 32 * 4096 > teuk.STATIC_SCRATCH_DOUBLES
    with pytest.raises(teuk.TeukError) as e:
        g.folded_static(False, 1)
    assert e.value.code == teuk.ECAPACITY and "capacity" in str(e.value)
    ok = _handle(teuk, 64, 8)
    for bad_variant in (0, 3):
        with pytest.raises(teuk.TeukError) as e:
            ok.folded_static(False, bad_variant)
        assert e.value.code == teuk.EINVAL
    dd = teuk.Teuk.from_workload(inputs.config(3).scaled(n_r=64, n_theta=8))
    with pytest.raises(teuk.TeukError) as e:
        dd.folded_static(False, 1)                           # fp64 handles only, like teuk_get_folded
    assert e.value.code == teuk.EINVAL
