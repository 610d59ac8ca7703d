"""Pins for hit masking between iterations (reading R9 of DESIGN.md): the selection rules on
a hand-made case, and the defining property of a masked index: the next iteration behaves as if the masked hits had
been taken out of the event."""
import numpy as np

from oracle import mkfo
from workloads import datagen


def test_mask_rules_by_hand():
    # 4 tracks x 3 plan steps over 10 hits
    hit_ids = np.array([[0, 3, 6, 8], [1, -1, 7, 9], [2, 5, -2, 4]], np.int32)
    nhits = np.array([3, 2, 2, 3], np.int32)
    chi2 = np.array([1.0, 0.0, 0.0, 6.0], np.float32)          # ndf = 2 n - 5 = 1 for 3 hits
    m = mkfo.mask_hits(10, hit_ids, nhits, chi2, min_hits=3, max_chi2_ndf=5.0)
    assert m.tolist() == [1, 1, 1, 0, 0, 0, 0, 0, 0, 0]          # track 0 only: 1, 2 too short, 3 has chi2 / ndf = 6 > 5
    m = mkfo.mask_hits(10, hit_ids, nhits, chi2, min_hits=3, max_chi2_ndf=6.0)
    assert m.tolist() == [1, 1, 1, 0, 1, 0, 0, 0, 1, 1]          # the cut is inclusive
    m = mkfo.mask_hits(10, hit_ids, nhits, chi2, keep=np.array([0, 1, 1, 1], np.uint8), min_hits=3, max_chi2_ndf=6.0)
    assert m.tolist() == [0, 0, 0, 0, 1, 0, 0, 0, 1, 1]          # duplicates do not mask
    m = mkfo.mask_hits(10, hit_ids, nhits, chi2, min_hits=2, max_chi2_ndf=5.0, mask=m)
    assert m.tolist() == [1, 1, 1, 0, 1, 0, 0, 0, 1, 1]          # masks accumulate; 2-hit tracks have ndf < 0: never selected
    assert mkfo.mask_hits(10, hit_ids, nhits, np.full(4, np.nan, np.float32), min_hits=0).sum() == 0


def remove_hits(ev, mask):
    """The event without the masked hits, and old id -> new id."""
    h, nl = ev["hits"], len(ev["geom"]["layers"])
    keep = mask == 0
    new_id = np.where(keep, np.cumsum(keep) - 1, -1).astype(np.int32)
    lo = h["layer_off"].reshape(h["n_events"], nl + 1)
    cum = np.concatenate([[0], np.cumsum(keep)])
    h2 = dict(n_events=h["n_events"], layer_off=cum[lo].astype(np.int32).reshape(-1), x=h["x"][keep], y=h["y"][keep], z=h["z"][keep],
              V=np.ascontiguousarray(h["V"][:, keep]))
    return h2, new_id


def test_masked_index_equals_index_of_the_event_without_those_hits():
    ev, prm = datagen.config(2, scale=0.02)                    # 2 barrel events with noise
    o = mkfo.Oracle(ev["geom"], prm)
    rng = np.random.default_rng(5)
    nh = ev["hits"]["x"].shape[0]
    mask = (rng.random(nh) < 0.3).astype(np.uint8)
    im = o.build_hit_index(ev["hits"], mask=mask)
    h2, new_id = remove_hits(ev, mask)
    i2 = o.build_hit_index(h2)
    assert np.array_equal(im["bin_off"], i2["bin_off"]) and len(im["sorted_id"]) == int((mask == 0).sum())
    assert np.array_equal(new_id[im["sorted_id"]], i2["sorted_id"])
    assert np.array_equal(im["vmax"], i2["vmax"])
    # no mask = all-zero mask = the plain index
    i0 = o.build_hit_index(ev["hits"])
    iz = o.build_hit_index(ev["hits"], mask=np.zeros(nh, np.uint8))
    assert all(np.array_equal(i0[k], iz[k]) for k in i0)


def test_second_iteration_on_masked_hits():
    ev, prm = datagen.config(2, scale=0.03)
    o = mkfo.Oracle(ev["geom"], prm)
    s, h = ev["seeds"], ev["hits"]
    nh = h["x"].shape[0]
    idx = o.build_hit_index(h)
    r1 = o.build_tracks(h, idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    # mask the hits of the good tracks among the first half of the seeds, then build the second half again
    n = s["par"].shape[1]
    first = np.arange(n) < n // 2
    mask = mkfo.mask_hits(nh, r1["hit_ids"][:, first], r1["nhits"][first], r1["chi2"][first].astype(np.float32), min_hits=8, max_chi2_ndf=5.0)
    assert 0 < mask.sum() < nh
    sel = ~first
    args = (s["par"][:, sel], s["cov"][:, sel], s["q"][sel], s["event"][sel])
    rm = o.build_tracks(h, o.build_hit_index(h, mask=mask), *args, s["hits"][:, sel], s["plan"][sel])
    # (a) no masked hit is picked up beyond the seed's own three hits
    picked = rm["hit_ids"][3:][rm["hit_ids"][3:] >= 0]
    assert mask[picked].sum() == 0
    # (b) identical to building on the event with those hits taken out (seed hits are read by id: keep them in)
    keep_seed = np.zeros(nh, bool); keep_seed[s["hits"][:, sel].ravel()] = True
    mask2 = np.where(keep_seed, 0, mask).astype(np.uint8)
    rm2 = o.build_tracks(h, o.build_hit_index(h, mask=mask2), *args, s["hits"][:, sel], s["plan"][sel])
    h2, new_id = remove_hits(ev, mask2)
    r2 = o.build_tracks(h2, o.build_hit_index(h2), *args, new_id[s["hits"][:, sel]], s["plan"][sel])
    mapped = np.where(rm2["hit_ids"] >= 0, new_id[np.maximum(rm2["hit_ids"], 0)], rm2["hit_ids"])
    assert np.array_equal(mapped, r2["hit_ids"]) and np.array_equal(rm2["nhits"], r2["nhits"])
    assert np.allclose(rm2["chi2"], r2["chi2"], rtol=0, atol=0)
    # (c) the tracks of the second half that do not overlap the masked hits are unchanged
    r1s = {k: r1[k][..., sel] for k in ("hit_ids", "nhits")}
    untouched = np.array([not mask[c[c >= 0]].any() for c in r1s["hit_ids"].T])
    assert untouched.sum() > 10
