"""-m gpu: hit index (bit-exact), track building (hit lists identical up to small oracle margins) and duplicate
removal (exact) against the oracle."""
import numpy as np
import pytest

from oracle import mkfo
from workloads import datagen
from workloads import parity

pytestmark = pytest.mark.gpu


def check_index(ev, prm):
    from gpu_helpers import gpu_hit_index
    o = mkfo.Oracle(ev["geom"], prm)
    ref = o.build_hit_index(ev["hits"])
    got = gpu_hit_index(ev, prm)
    assert np.array_equal(got["bin_off"], ref["bin_off"])
    assert np.array_equal(got["sorted_id"], ref["sorted_id"])
    assert np.array_equal(got["vmax"].view(np.uint32), ref["vmax"].view(np.uint32))     # bit-exact floats
    # packed copy: the hits in sorted order, positions then covariances
    sid = ref["sorted_id"]
    h = ev["hits"]
    nh = len(sid)
    c0 = 4 * (nh + (nh & 1))                                  # the covariance block starts on a whole sector
    pos, cv = got["packed"][:4 * nh].reshape(nh, 4), got["packed"][c0:c0 + 8 * nh].reshape(nh, 8)
    assert np.array_equal(pos[:, 3].copy().view(np.int32), sid)
    assert np.array_equal(pos[:, 0], h["x"][sid]) and np.array_equal(pos[:, 1], h["y"][sid]) and np.array_equal(pos[:, 2], h["z"][sid])
    assert np.array_equal(cv[:, :6], h["V"][:, sid].T)
    return ref


def test_hit_index_barrel_bit_exact():
    ev, prm = datagen.config(2, scale=0.05)           # 5 events x 17 layers
    check_index(ev, prm)


def test_hit_index_endcap_bit_exact():
    ev, prm = datagen.config(3, scale=0.015)          # 3 events x 38 layers, ~80k hits each
    check_index(ev, prm)


def test_hit_index_empty_layers_and_crowded_bins():
    """Layers without hits, and all hits of a layer in one bin (exercises the heap-sort branch)."""
    g = datagen.geometry_barrel(3, 10.0, 30.0, 50.0, 0.02)
    n1 = 700
    rng = np.random.default_rng(3)
    # layer 0: empty; layer 1: n1 hits at (nearly) the same place; layer 2: 5 hits spread out
    ph2 = np.linspace(-3, 3, 5)
    x = np.concatenate([20 * np.cos(0.3 + 1e-6 * rng.random(n1)), 30 * np.cos(ph2)])
    y = np.concatenate([20 * np.sin(0.3 + 1e-6 * rng.random(n1)), 30 * np.sin(ph2)])
    z = np.concatenate([np.full(n1, 1.0), np.linspace(-40, 40, 5)])
    V = np.zeros((6, n1 + 5), np.float32); V[0] = V[2] = 1e-5; V[5] = 1e-4; V[1] = 3e-6
    hits = dict(n_events=1, layer_off=np.array([0, 0, n1, n1 + 5], np.int32), x=x.astype(np.float32), y=y.astype(np.float32),
                z=z.astype(np.float32), V=V)
    check_index(dict(geom=g, hits=hits), datagen.default_params())


@pytest.mark.parametrize("n_per_layer", [6001, 12000])
def test_hit_index_large_segments_odd_and_even_counts(n_per_layer):
    """Segments beyond 4096 hits on average take the 1024-thread instance of the index kernel; 12000 hits per segment
    exceed the id list it keeps in shared memory (the rest goes through the workspace). An odd total moves the
    covariance block of the packed copy by one record (whole-sector records)."""
    g = datagen.geometry_barrel(3, 10.0, 30.0, 50.0, 0.02)
    rng = np.random.default_rng(11 + n_per_layer)
    radii = np.array([l["pos"] for l in g["layers"]])
    n = 3 * n_per_layer
    ph = rng.uniform(-np.pi, np.pi, n); r = np.repeat(radii, n_per_layer)
    x, y, z = r * np.cos(ph), r * np.sin(ph), rng.uniform(-50, 50, n)
    V = np.zeros((6, n), np.float32); V[0] = rng.uniform(1e-6, 1e-4, n); V[2] = rng.uniform(1e-6, 1e-4, n); V[5] = rng.uniform(1e-5, 1e-3, n)
    V[1] = 0.3 * np.sqrt(V[0] * V[2])
    hits = dict(n_events=1, layer_off=(np.arange(4) * n_per_layer).astype(np.int32), x=x.astype(np.float32), y=y.astype(np.float32),
                z=z.astype(np.float32), V=V)
    assert (n % 2 == 1) == (n_per_layer % 2 == 1)
    check_index(dict(geom=g, hits=hits), datagen.default_params())


def compare_build(ev, prm, r, h, min_same=0.999):
    n = r["nhits"].shape[0]
    same = np.all(h["hit_ids"] == r["hit_ids"], axis=0)
    frac = same.mean()
    # mismatches only where the oracle itself was within 1e-3 of a decision boundary (U20)
    assert np.all(r["margin"][~same] < 1e-3), (np.sort(r["margin"][~same])[-5:], frac)
    assert frac >= min_same, frac
    assert np.array_equal(h["nhits"][same], r["nhits"][same])
    assert np.array_equal(h["nmiss"][same], r["nmiss"][same])
    assert np.array_equal(h["status"][same], r["status"][same])
    ok = same & ((r["status"] & 32) == 0)
    # the state sits on the layer of the last found hit
    geom = ev["geom"]
    plan_off, plan_layers = np.asarray(geom["plan_off"]), np.asarray(geom["plan_layers"])
    hid = r["hit_ids"]
    has = hid >= 0
    last = hid.shape[0] - 1 - np.argmax(has[::-1], axis=0)
    lay = plan_layers[plan_off[ev["seeds"]["plan"].astype(int)] + last]
    kinds = np.array([l["kind"] for l in geom["layers"]])[lay]
    pos = np.array([abs(l["pos"]) for l in geom["layers"]])[lay]
    # a candidate that ended on missed layers has been propagated beyond its last hit: find the surface it is on
    # from the state itself (barrel if its radius matches a barrel layer better than its z matches a disk)
    pe = parity.param_errors(h["par"], r["par"], np.maximum(pos, 1.0))[ok]
    xe = parity.chi2_errors(h["chi2"], r["chi2"])[ok]
    se = np.abs(h["score"] - r["score"])[ok] / np.maximum(np.abs(r["score"][ok]), 1.0)
    assert pe.max() <= parity.TOL_PAR, pe.max()
    assert xe.max() <= parity.TOL_CHI2, xe.max()
    assert se.max() <= parity.TOL_CHI2, se.max()
    # covariance: on the surface the state sits on (the last crossed layer, hit or miss)
    crossed = hid >= -1
    lastc = hid.shape[0] - 1 - np.argmax(crossed[::-1], axis=0)
    layc = plan_layers[plan_off[ev["seeds"]["plan"].astype(int)] + lastc]
    kindc = np.array([l["kind"] for l in geom["layers"]])[layc]
    ce = parity.cov_errors(h["cov"], r["cov"], r["par"], kindc)[ok]
    assert ce.max() <= parity.TOL_COV, ce.max()                              # north_star: 1e-3 on every element, every track
    return frac


def run_build(ev, prm, brute=False, packed=True):
    from gpu_helpers import gpu_build
    s = ev["seeds"]
    o = mkfo.Oracle(ev["geom"], prm)
    idx = o.build_hit_index(ev["hits"])
    r = o.build_tracks(ev["hits"], idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"], brute_force=brute)
    h = gpu_build(ev, prm, packed=packed)
    return r, h


def test_build_barrel_config2_sample():
    ev, prm = datagen.config(2, scale=0.05)           # 5 events x 1000 seeds, 20k noise hits each
    r, h = run_build(ev, prm)
    frac = compare_build(ev, prm, r, h)
    assert (r["nhits"] >= 10).mean() > 0.8


def test_build_barrel_unpacked_gather_path_and_brute_force_oracle():
    ev, prm = datagen.config(2, scale=0.01)
    r, h = run_build(ev, prm, brute=True, packed=False)       # oracle tries every hit of the layer
    compare_build(ev, prm, r, h)


def test_build_barrel_endcap_config3_sample():
    ev, prm = datagen.config(3, scale=0.015)          # 3 events x ~1500 seeds, 38 layers, propagateToZ, 5 % inefficiency
    r, h = run_build(ev, prm)
    compare_build(ev, prm, r, h)
    assert (r["nmiss"] > 0).mean() > 0.1 and ((r["status"] & 32) != 0).sum() >= 0


def test_build_config4_like_eight_candidates_and_duplicate_removal():
    from gpu_helpers import gpu_build
    ev, prm = datagen.config(4, scale=1 / 64.0)       # one high-occupancy event, 6000 seeds, max_cand 8
    s = ev["seeds"]
    o = mkfo.Oracle(ev["geom"], prm)
    idx = o.build_hit_index(ev["hits"])
    r = o.build_tracks(ev["hits"], idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    h = gpu_build(ev, prm, dedup=True)
    compare_build(ev, prm, r, h)
    # duplicate removal is integer-only: the oracle on the GPU's own built tracks must agree exactly
    d = o.remove_duplicates(h["track_off"], h["hit_ids"], h["nhits"], h["score"])
    assert np.array_equal(h["keep"], d["keep"]) and np.array_equal(h["n_kept"], d["n_kept"])


def test_remove_duplicates_exact_on_synthetic_overlaps():
    import torch
    from paper_2002_06295_b200 import binding as B
    rng = np.random.default_rng(11)
    g = datagen.geometry_barrel(12, 4.0, 48.0, 100.0, 0.02)
    prm = datagen.default_params()
    n_events, per_ev, mpl, hits_per_ev = 3, 400, 12, 3000
    n = n_events * per_ev
    hit_ids = np.full((mpl, n), -1, np.int32)
    for i in range(n):
        ev = i // per_ev
        if i % 3 and i > ev * per_ev:                                  # derive from the previous track: heavy overlap
            hit_ids[:, i] = hit_ids[:, i - 1]
            k = rng.integers(0, mpl, rng.integers(1, 9))
            hit_ids[k, i] = ev * hits_per_ev + rng.integers(0, hits_per_ev, k.size)
        else:
            hit_ids[:, i] = ev * hits_per_ev + rng.integers(0, hits_per_ev, mpl)
        hit_ids[rng.random(mpl) < 0.2, i] = -1
    nhits = (hit_ids >= 0).sum(0).astype(np.int32)
    score = np.round(rng.normal(200, 30, n)).astype(np.float32)         # rounded: many exact ties
    toff = (np.arange(n_events + 1) * per_ev).astype(np.int32)
    ref = mkfo.Oracle(g, prm).remove_duplicates(toff, hit_ids, nhits, score)
    ctx = B.Context(g, prm)
    nh = n_events * hits_per_ev
    keep = torch.empty(n, dtype=torch.uint8, device="cuda"); nk = torch.empty(n_events, dtype=torch.int32, device="cuda")
    ws = torch.empty(ctx.workspace_bytes(B.CALL_REMOVE_DUPLICATES, n_events, nh, n), dtype=torch.uint8, device="cuda")
    ctx.remove_duplicates(nh, torch.from_numpy(toff).cuda(), torch.from_numpy(hit_ids).cuda(), torch.from_numpy(nhits).cuda(),
                          torch.from_numpy(score).cuda(), keep, nk, ws)
    torch.cuda.synchronize()
    assert np.array_equal(keep.cpu().numpy(), ref["keep"]) and np.array_equal(nk.cpu().numpy(), ref["n_kept"])
    assert 0.2 < ref["keep"].mean() < 0.95
    ctx.close()


def test_build_host_entry_point_matches_device_path():
    from gpu_helpers import gpu_build
    from paper_2002_06295_b200 import binding as B
    ev, prm = datagen.config(2, scale=0.02)
    h = gpu_build(ev, prm, dedup=True)
    ctx = B.Context(ev["geom"], prm)
    s = ev["seeds"]
    r = ctx.build_host(ev["hits"], s, np.ascontiguousarray(s["event"]), np.ascontiguousarray(s["hits"]),
                       np.ascontiguousarray(s["plan"]), dedup=True)
    for k in ("hit_ids", "nhits", "nmiss", "chi2", "score", "par", "cov", "keep"):
        assert np.array_equal(r[k], h[k]), k
    ctx.close()


def test_fit_of_built_tracks_chained_from_build_output():
    """PAPER.md:25 'Fitting simply applies the KF procedure to all hits identified during building': the hit_ids
    array written by mkf_build_tracks is the track_hits input of mkf_fit as it is (-1 / -2 entries are skipped)."""
    import torch
    from paper_2002_06295_b200 import binding as B
    from gpu_helpers import gpu_build
    ev, prm = datagen.config(3, scale=0.01)
    s = ev["seeds"]
    hb = gpu_build(ev, prm)
    ctx = B.Context(ev["geom"], prm)
    hits = B.hits_to_device(ev["hits"])
    sd = B.to_device(dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"]), ["par", "cov", "q", "plan"])
    th = torch.from_numpy(hb["hit_ids"]).cuda()
    n = s["par"].shape[1]
    out = B.alloc_fit_out(n)
    ctx.fit(hits, sd, sd["plan"], th, out, out["chi2"], out["nfit"], out["status"])
    torch.cuda.synchronize()
    g = {k: v.cpu().numpy() for k, v in out.items()}
    r = mkfo.Oracle(ev["geom"], prm).fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], hb["hit_ids"])
    assert np.array_equal(g["nfit"], r["nfit"]) and np.array_equal(g["status"].view(np.uint32), r["status"])
    ok = (r["nfit"] > 0)
    # a built track without missed layers is fitted through exactly the same sequence of steps, so the total chi2
    # agrees with the build's (with a miss the build also applied the material of the missed layer; the fit,
    # which goes from hit to hit, does not)
    full = ok & (g["nfit"] == hb["nhits"]) & ((hb["status"] & 32) == 0) & (hb["nmiss"] == 0)
    assert full.mean() > 0.3
    lay, kinds, pos = parity.last_layer_of_fit(ev["geom"], s["plan"], hb["hit_ids"], r["nfit"])
    assert parity.param_errors(g["par"], r["par"], pos)[ok].max() <= parity.TOL_PAR
    assert parity.cov_errors(g["cov"], r["cov"], r["par"], kinds)[ok].max() <= parity.TOL_COV
    assert parity.chi2_errors(g["chi2"], r["chi2"])[ok].max() <= parity.TOL_CHI2
    assert (np.abs(g["chi2"][full] - hb["chi2"][full]) <= 1e-3 * np.maximum(hb["chi2"][full], 1.0)).all()
    ctx.close()


def test_degenerate_inputs():
    """No seeds, events without hits, seeds whose hits are not on their plan, no tracks for duplicate removal."""
    import torch
    from paper_2002_06295_b200 import binding as B
    g = datagen.geometry_barrel(6, 4.0, 24.0, 50.0, 0.02)
    prm = datagen.default_params()
    ev = datagen.make_events(g, 5, 2, 40, n_noise=600)
    o = mkfo.Oracle(g, prm)
    # event 1 emptied: all its hits removed
    h = ev["hits"]
    lo = h["layer_off"].reshape(2, 7)
    n0 = int(lo[0, 6])
    sub = dict(n_events=2, layer_off=np.concatenate([lo[0], np.full(7, n0)]).astype(np.int32), x=h["x"][:n0].copy(), y=h["y"][:n0].copy(),
               z=h["z"][:n0].copy(), V=np.ascontiguousarray(h["V"][:, :n0]))
    from gpu_helpers import gpu_hit_index
    ref = o.build_hit_index(sub)
    got = gpu_hit_index(dict(geom=g, hits=sub), prm)
    assert np.array_equal(got["bin_off"], ref["bin_off"]) and np.array_equal(got["sorted_id"], ref["sorted_id"])
    assert np.array_equal(got["vmax"], ref["vmax"]) and np.all(got["vmax"][12:] == 0)
    # seeds of event 0 only; the last seed gets hits that are not in plan order -> TRUNCATED seed returned
    s = ev["seeds"]
    m = s["event"] == 0
    seeds = {k: np.ascontiguousarray(v[..., m]) for k, v in s.items() if k in ("par", "cov", "q", "plan", "event", "hits")}
    seeds["hits"][:, -1] = seeds["hits"][::-1, -1]
    r = o.build_tracks(sub, ref, seeds["par"], seeds["cov"], seeds["q"], seeds["event"], seeds["hits"], seeds["plan"])
    ctx = B.Context(g, prm)
    dh = B.hits_to_device(sub)
    idx, ws = B.alloc_hit_index(ctx, 2, n0)
    ctx.build_hit_index(dh, idx, ws)
    sd = B.to_device(seeds, ["par", "cov", "q", "plan", "event", "hits"])
    n = seeds["par"].shape[1]
    out = B.alloc_build_out(n, ctx.max_plan_len)
    ctx.build_tracks(dh, idx, sd, sd["event"], sd["hits"], sd["plan"], out, out["chi2"], out["score"], out["nhits"], out["nmiss"],
                     out["hit_ids"], out["status"])
    torch.cuda.synchronize()
    hid = out["hit_ids"].cpu().numpy()
    same = np.all(hid == r["hit_ids"], axis=0)
    assert same.mean() >= 0.97 and np.all(r["margin"][~same] < 1e-3)
    st = out["status"].cpu().numpy().view(np.uint32)
    assert np.array_equal(st[same], r["status"][same]) and (r["status"][-1] & 32) and same[-1]
    assert np.array_equal(out["nhits"].cpu().numpy()[same], r["nhits"][same])
    # zero seeds: nothing launched
    e = {k: v[..., :0].contiguous() for k, v in sd.items()}
    out0 = B.alloc_build_out(0, ctx.max_plan_len)
    before = ctx.launch_count()
    ctx.build_tracks(dh, idx, e, e["event"], e["hits"], e["plan"], out0, out0["chi2"], out0["score"], out0["nhits"], out0["nmiss"],
                     out0["hit_ids"], out0["status"])
    assert ctx.launch_count() == before
    # duplicate removal with an event that has no tracks
    toff = torch.tensor([0, n, n], dtype=torch.int32, device="cuda")
    keep = torch.empty(n, dtype=torch.uint8, device="cuda"); nk = torch.empty(2, dtype=torch.int32, device="cuda")
    ws2 = torch.empty(ctx.workspace_bytes(B.CALL_REMOVE_DUPLICATES, 2, n0, n), dtype=torch.uint8, device="cuda")
    ctx.remove_duplicates(n0, toff, out["hit_ids"], out["nhits"], out["score"], keep, nk, ws2)
    torch.cuda.synchronize()
    d = o.remove_duplicates(np.array([0, n, n], np.int32), hid, out["nhits"].cpu().numpy(), out["score"].cpu().numpy())
    assert np.array_equal(keep.cpu().numpy(), d["keep"]) and np.array_equal(nk.cpu().numpy(), d["n_kept"]) and nk[1].item() == 0
    # workspace too small is an error code, not a crash
    with pytest.raises(B.MkfError):
        ctx.remove_duplicates(n0, toff, out["hit_ids"], out["nhits"], out["score"], keep, nk, ws2[:64])
    ctx.close()


@pytest.mark.parametrize("cap", [1, 2])
def test_u14_ties_lower_hit_id_then_lower_parent_rank(cap):
    """Keys 3 and 4 of the total order U14 on the hand-placed twin-hit event (tests/hand_events.py): the expected lists
    are written by hand; the oracle is pinned to the same lists in tests/test_oracle_build.py."""
    from gpu_helpers import gpu_build
    from hand_events import tie_event, TIE_EXPECTED
    ev, prm = tie_event()
    prm = dict(prm, max_cand=cap)
    for packed in (True, False):
        h = gpu_build(ev, prm, packed=packed)
        assert list(h["hit_ids"][:, 0]) == TIE_EXPECTED[cap]
        assert h["nhits"][0] == 5 and h["nmiss"][0] == 0 and h["status"][0] == 0
    r, _ = run_build(ev, prm)
    assert np.array_equal(h["hit_ids"], r["hit_ids"]) and abs(h["chi2"][0] - r["chi2"][0]) <= 1e-3 * max(r["chi2"][0], 1.0)


def test_u14_tie_on_the_last_layer():
    from gpu_helpers import gpu_build
    from hand_events import tie_event
    ev, prm = tie_event()
    hh = ev["hits"]
    g4 = dict(ev["geom"], layers=ev["geom"]["layers"][:4], plan_off=np.array([0, 4], np.int32), plan_layers=np.arange(4, dtype=np.int32))
    sub = dict(n_events=1, x=hh["x"][:5].copy(), y=hh["y"][:5].copy(), z=hh["z"][:5].copy(), V=np.ascontiguousarray(hh["V"][:, :5]),
               layer_off=np.array([0, 1, 2, 3, 5], np.int32))
    h = gpu_build(dict(geom=g4, hits=sub, seeds=ev["seeds"]), dict(prm, max_cand=2))
    assert list(h["hit_ids"][:, 0]) == [0, 1, 2, 3]


def test_nan_child_is_dropped_and_its_parent_offered_to_best_short():
    """Reading R1: same hand-placed event and hand-written lists as the oracle pin of the same name."""
    from gpu_helpers import gpu_build
    from hand_events import nan_child_event
    ev, prm = nan_child_event(bad_layer=4)
    h = gpu_build(ev, dict(prm, max_cand=1))
    assert list(h["hit_ids"][:, 0]) == [0, 1, 2, 3, -2, -2]
    assert h["nhits"][0] == 4 and h["nmiss"][0] == 0 and (h["status"][0] & 32) == 0
    assert np.all(np.isfinite(h["par"][:, 0])) and np.all(np.isfinite(h["cov"][:, 0]))
    r, _ = run_build(ev, dict(prm, max_cand=1))
    lay = ev["geom"]["layers"][3]
    assert parity.param_errors(h["par"], r["par"], np.array([abs(lay["pos"])])).max() <= parity.TOL_PAR
    assert parity.cov_errors(h["cov"], r["cov"], r["par"], np.array([1])).max() <= parity.TOL_COV
    assert abs(h["chi2"][0] - r["chi2"][0]) <= 1e-3 * max(r["chi2"][0], 1.0)
    h3 = gpu_build(ev, dict(prm, max_cand=3))
    assert list(h3["hit_ids"][:, 0]) == [0, 1, 2, 3, -1, 5] and h3["nhits"][0] == 5 and h3["nmiss"][0] == 1
    ev3, _ = nan_child_event(bad_layer=3)
    h4 = gpu_build(ev3, dict(prm, max_cand=1))
    assert (h4["status"][0] & 32) and h4["nhits"][0] == 3 and list(h4["hit_ids"][:, 0]) == [0, 1, 2, -2, -2, -2]


def test_build_with_scores_where_a_miss_can_outrank_a_hit():
    """score_hit + score_miss < chi2_cut: a miss child (score - 1) outranks a hit child with chi2 > 6 (score + 5 - chi2),
    so a parent's children are no longer ordered hits-first; the selection must still follow the total order U14
    (on the oracle this changes 45 % of the hit lists of this sample)."""
    ev, prm = datagen.config(2, scale=0.03)
    prm = dict(prm, score_hit=5.0, score_miss=1.0)
    r, h = run_build(ev, prm)
    compare_build(ev, prm, r, h)
    base = run_build(ev, datagen.default_params(max_cand=6))[0]
    assert (np.any(base["hit_ids"] != r["hit_ids"], axis=0)).mean() > 0.3       # the parameters do change the answer
