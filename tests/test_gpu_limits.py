"""-m gpu: the largest geometry the library takes (MKF_MAX_LAYERS = 64 layers, one 64-step plan) through the fit, the
backward fit, the hit index and the build, against the oracle. With 64 plan steps the build kernel reads
its trellis back from the workspace instead of staging it in shared memory (the other build tests stage it)."""
import numpy as np
import pytest

from workloads import datagen

pytestmark = pytest.mark.gpu


def _events():
    g = datagen.geometry_barrel(64, 3.0, 110.0, 140.0, 0.004)
    ev = datagen.make_events(g, 21, 2, 400, n_noise=6000, pt_range=(0.8, 10.0))
    return ev, datagen.default_params(max_cand=8)


def test_fit_and_backward_fit_on_64_layers():
    from test_gpu_fit import check_backward, check_fit
    ev, prm = _events()
    assert ev["seeds"]["track_hits"].shape[0] == 64
    r, h = check_fit(ev, prm)
    assert (r["nfit"] >= 60).mean() > 0.9
    check_backward(ev, prm)


def test_hit_index_and_build_on_64_layers():
    from test_gpu_build import check_index, compare_build, run_build
    ev, prm = _events()
    check_index(ev, prm)
    r, h = run_build(ev, prm)
    assert h["hit_ids"].shape[0] == 64
    compare_build(ev, prm, r, h)
    assert (r["nhits"] >= 50).mean() > 0.8


def test_more_than_64_layers_is_refused():
    from paper_2002_06295_b200 import binding as B
    g = datagen.geometry_barrel(65, 3.0, 110.0, 140.0, 0.004)
    with pytest.raises(B.MkfError):
        B.Context(g, datagen.default_params())
