"""-m gpu: mkf_build_hit_index_static, the hit index for callers that cannot allocate (its scratch is a fixed device
array inside the library), against the existing mkf_build_hit_index on two calls in a row. Integer / index work and
copied floats: the bar is bit-exact (the bar tests/test_gpu_build.py holds the existing path to against the oracle).
Collected last on purpose (file name): a failure here must not hide the other tests under `pytest -x`."""
import numpy as np
import pytest
import torch

from workloads import datagen

pytestmark = pytest.mark.gpu


def _both(ctx, B, ev, poison, steady=False):
    """(existing path, static path) outputs for one event set; the static path's outputs start from `poison`.
    steady: the static call must leave the device's free memory as it found it (no allocation by the library)."""
    hits = B.hits_to_device(ev["hits"])
    nev, nh = hits["n_events"], hits["x"].shape[0]
    ref, ws = B.alloc_hit_index(ctx, nev, nh)
    ctx.build_hit_index(hits, ref, ws)
    got, _ = B.alloc_hit_index(ctx, nev, nh)
    for k in ("bin_off", "sorted_id"):
        got[k].fill_(poison)
    got["vmax"].fill_(float(poison)); got["packed"].fill_(float(poison))
    torch.cuda.synchronize()
    free0 = torch.cuda.mem_get_info()[0]
    ctx.build_hit_index_static(hits, got)
    torch.cuda.synchronize()
    if steady:
        assert torch.cuda.mem_get_info()[0] == free0
    return ({k: v.cpu().numpy() for k, v in ref.items()}, {k: v.cpu().numpy() for k, v in got.items()}, nh)


def _same(ref, got, nh):
    assert np.array_equal(got["bin_off"], ref["bin_off"])
    assert np.array_equal(got["sorted_id"], ref["sorted_id"])
    assert np.array_equal(got["vmax"].view(np.uint32), ref["vmax"].view(np.uint32))
    c0 = 4 * (nh + (nh & 1))                                   # positions, then (from a whole sector on) covariances
    assert np.array_equal(got["packed"][:4 * nh].view(np.uint32), ref["packed"][:4 * nh].view(np.uint32))
    assert np.array_equal(got["packed"][c0:c0 + 8 * nh].view(np.uint32), ref["packed"][c0:c0 + 8 * nh].view(np.uint32))


def test_static_hit_index_matches_existing_path_on_two_calls_in_a_row():
    from paper_2002_06295_b200 import binding as B
    big, prm = datagen.config(3, scale=0.015, seed=3)          # 3 events x 38 layers, ~240 k hits
    small, _ = datagen.config(3, scale=0.005, seed=4)          # 1 event: fewer hits, so the shared scratch keeps
    assert small["hits"]["x"].shape[0] < big["hits"]["x"].shape[0] <= B.STATIC_MAX_HITS      # stale words of call 1
    ctx = B.Context(big["geom"], prm)
    n0 = ctx.launch_count()
    r1, g1, nh1 = _both(ctx, B, big, 7)
    r2, g2, nh2 = _both(ctx, B, small, -3, steady=True)                  # second call right after the first, same scratch
    _same(r1, g1, nh1)
    _same(r2, g2, nh2)
    assert ctx.launch_count() - n0 == 4                        # one kernel per call on either path
    # a third call on the first input again gives the first result (nothing left over from call 2 matters)
    r3, g3, nh3 = _both(ctx, B, big, 11, steady=True)
    _same(r1, g3, nh3)
    ctx.close()


def test_static_hit_index_limits_and_empty_input():
    from paper_2002_06295_b200 import binding as B
    ev, prm = datagen.config(2, scale=0.01)
    ctx = B.Context(ev["geom"], prm)
    nl = len(ev["geom"]["layers"])
    # beyond the fixed scratch: refused with a clear error, nothing launched, outputs untouched
    n = B.STATIC_MAX_HITS + 1
    hits = dict(n_events=1, layer_off=torch.zeros(nl + 1, dtype=torch.int32, device="cuda"),
                x=torch.zeros(n, device="cuda"), y=torch.zeros(n, device="cuda"), z=torch.zeros(n, device="cuda"),
                V=torch.zeros((6, n), device="cuda"))
    hits["layer_off"][1:] = n
    out, _ = B.alloc_hit_index(ctx, 1, n)
    out["sorted_id"].fill_(5)
    n0 = ctx.launch_count()
    with pytest.raises(B.MkfError, match="MKF_STATIC_MAX_HITS"):
        ctx.build_hit_index_static(hits, out)
    torch.cuda.synchronize()
    assert ctx.launch_count() == n0 and int(out["sorted_id"].min()) == 5
    # no hits at all: all offsets zero, as the existing path
    e = dict(n_events=2, layer_off=torch.zeros(2 * (nl + 1), dtype=torch.int32, device="cuda"), x=torch.zeros(0, device="cuda"),
             y=torch.zeros(0, device="cuda"), z=torch.zeros(0, device="cuda"), V=torch.zeros((6, 0), device="cuda"))
    o2, _ = B.alloc_hit_index(ctx, 2, 1)                       # (an empty tensor has a null data pointer)
    o2["bin_off"].fill_(9); o2["vmax"].fill_(9.0)
    ctx.build_hit_index_static(e, o2)
    torch.cuda.synchronize()
    assert int(o2["bin_off"].abs().max()) == 0 and float(o2["vmax"].abs().max()) == 0.0
    ctx.close()
