"""-m gpu: track building at the FULL size of configs[2] (100 events, 100 k seeds, 3.7 M hits), in the launch
configuration bench.py times: properties that hold for every track at any size, and the 25 events of one generator chunk
compared with the oracle element by element (the oracle builds a chunk in a few seconds, not the whole workload)."""
import numpy as np
import pytest

from oracle import mkfo
from workloads import assemble, datagen

pytestmark = pytest.mark.gpu


def test_build_config2_full_size_properties_and_one_chunk_against_the_oracle():
    from gpu_helpers import gpu_build
    from test_gpu_build import compare_build
    ev, prm = assemble.make_build_workload(2, 0, 1.0)
    geom, hits, s = ev["geom"], ev["hits"], ev["seeds"]
    nev, n, nl = hits["n_events"], s["par"].shape[1], len(geom["layers"])
    assert nev == assemble.BUILD_EVENTS[2] and n == 100000
    h = gpu_build(ev, prm)
    hid = h["hit_ids"]                                         # [mpl, n]
    has = hid >= 0
    # counts, scores (U13) and hit lists are consistent for every track
    assert np.array_equal(has.sum(0), h["nhits"])
    assert ((hid == -1).sum(0) == h["nmiss"]).all()
    sc = np.float32(prm["score_hit"]) * h["nhits"] - np.float32(prm["score_miss"]) * h["nmiss"] - h["chi2"]
    assert np.abs(sc - h["score"]).max() <= 1e-3 * np.maximum(np.abs(h["score"]), 1.0).max()
    assert (h["nhits"] >= 3).all() and (h["chi2"] >= 0).all()
    # every hit of a track lies in the track's event and on the layer of its plan step, and is taken once
    lo = hits["layer_off"].reshape(nev, nl + 1)
    plan_off, plan_layers = np.asarray(geom["plan_off"]), np.asarray(geom["plan_layers"])
    evs = s["event"].astype(np.int64)
    for st in range(hid.shape[0]):
        m = has[st]
        if not m.any():
            continue
        lay = plan_layers[plan_off[s["plan"][m].astype(int)] + st]
        assert (hid[st][m] >= lo[evs[m], lay]).all() and (hid[st][m] < lo[evs[m], lay + 1]).all()
    srt = np.sort(np.where(has, hid, -np.arange(1, hid.shape[0] + 1)[:, None]), axis=0)
    assert (np.diff(srt, axis=0) != 0).all()
    # the seed's own three hits are in its track
    for k in range(3):
        assert (hid == s["hits"][k][None]).any(0).all()
    # chunk 2 of the generator (events 50..74) against the oracle
    k = 2
    per = assemble.BUILD_CHUNK[2]
    cev, cprm = datagen.config(2, scale=per / assemble.BUILD_EVENTS[2], seed=64 * 0 + k)
    cs = cev["seeds"]
    o = mkfo.Oracle(cev["geom"], cprm)
    idx = o.build_hit_index(cev["hits"])
    r = o.build_tracks(cev["hits"], idx, cs["par"], cs["cov"], cs["q"], cs["event"], cs["hits"], cs["plan"])
    sel = np.nonzero((evs >= k * per) & (evs < (k + 1) * per))[0]
    assert sel.shape[0] == cs["par"].shape[1] and np.array_equal(s["par"][:, sel], cs["par"])
    nh0 = int(lo[k * per, 0])                                  # the chunk's hit ids were offset by this
    hs = {kk: (v[..., sel] if isinstance(v, np.ndarray) and v.ndim >= 1 and v.shape[-1] == n else v) for kk, v in h.items()}
    hs["hit_ids"] = np.where(hs["hit_ids"] >= 0, hs["hit_ids"] - nh0, hs["hit_ids"])
    compare_build(cev, cprm, r, hs)
