"""Pins for the oracle hit index (C8), window (U11), combinatorial build (C9) and duplicate removal (C10).

None of these re-type the oracle's formula: bins are checked against hand-placed golden azimuths and against
edge *directions* (cross products), the window against brute force over every hit of the layer, the build's
binned search against its own brute-force mode and against simulation truth, and the duplicate removal against a
set-based O(n^2) Python loop."""
import os

import numpy as np
import pytest

from oracle import mkfo
from workloads import datagen
from hand_events import tie_event, nan_child_event, TIE_EXPECTED

GOLD = os.path.join(os.path.dirname(__file__), "golden")


@pytest.fixture(scope="module")
def small_build_event():
    """configs[2] at 2 events, 1000 particles + 20k noise hits each (17 barrel layers)."""
    ev, prm = datagen.config(2, scale=0.02, seed=3)
    return ev, prm


@pytest.fixture(scope="module")
def small_endcap_event():
    """configs[3] at 1 event (barrel + endcap, 38 layers, inefficiency, secondaries, noise)."""
    ev, prm = datagen.config(3, scale=0.005, seed=5)
    return ev, prm


def one_layer_hits(x, y, z, nl=1):
    n = len(x)
    V = np.zeros((6, n), np.float32)
    V[0] = V[2] = 9e-6
    V[5] = 1e-4
    return dict(n_events=1, layer_off=np.array([0, n], np.int32), x=np.asarray(x, np.float32),
                y=np.asarray(y, np.float32), z=np.asarray(z, np.float32), V=V)


def test_phi_bins_golden():
    """golden/phi_bins.txt: hand-placed azimuths → bin of 63 (C8)."""
    rows = np.loadtxt(os.path.join(GOLD, "phi_bins.txt"))
    g = datagen.geometry_barrel(1, 10.0, 10.0, 100.0, 0.02)
    o = mkfo.Oracle(g, datagen.default_params())
    phi = rows[:, 0]
    h = one_layer_hits(10 * np.cos(phi), 10 * np.sin(phi), np.zeros_like(phi))
    idx = o.build_hit_index(h)
    cnt = np.diff(idx["bin_off"].astype(np.int64)).reshape(40, 63)
    for k, (ph, b) in enumerate(rows):
        # z=0 → eta=0 → eta bin 20 (the bin whose lower edge is eta=0)
        pos = np.nonzero(idx["sorted_id"] == k)[0][0]
        binid = np.searchsorted(idx["bin_off"], pos, side="right") - 1
        assert binid % 63 == int(b), (ph, b, binid % 63)
        assert binid // 63 == 20
    assert cnt.sum() == len(phi)


def test_hit_index_invariants_and_edge_directions(small_build_event):
    ev, prm = small_build_event
    g, h = ev["geom"], ev["hits"]
    o = mkfo.Oracle(g, prm)
    idx = o.build_hit_index(h)
    nl, nb = len(g["layers"]), 63 * 40
    bo = idx["bin_off"].astype(np.int64)
    sid = idx["sorted_id"]
    nh = len(h["x"])
    assert bo[0] == 0 and bo[-1] == nh and np.all(np.diff(bo) >= 0)
    assert np.array_equal(np.sort(sid), np.arange(nh))                        # a permutation of all hits
    lo = h["layer_off"].reshape(-1, nl + 1)
    x, y, z = (h[k].astype(np.float64) for k in "xyz")
    edges = -np.pi + 2 * np.pi * np.arange(64) / 63
    ex, ey = np.cos(edges), np.sin(edges)
    for e in range(h["n_events"]):
        for l in range(nl):
            seg = e * nl + l
            b0, b1 = bo[seg * nb], bo[(seg + 1) * nb]
            assert b0 == lo[e, l] and b1 == lo[e, l + 1]                      # a segment holds exactly its layer
            ids = sid[b0:b1]
            assert np.array_equal(np.sort(ids), np.arange(lo[e, l], lo[e, l + 1]))
            binid = np.searchsorted(bo[seg * nb:(seg + 1) * nb + 1], np.arange(b0, b1), side="right") - 1
            ip, ie = binid % 63, binid // 63
            # within a bin ids ascend (stable)
            same = binid[1:] == binid[:-1]
            assert np.all(ids[1:][same] > ids[:-1][same])
            # phi: the hit direction lies between the bin's two edge directions (cross products; no atan2 floor)
            hx, hy = x[ids], y[ids]
            c_lo = ex[ip] * hy - ey[ip] * hx
            c_hi = ex[ip + 1] * hy - ey[ip + 1] * hx
            r = np.hypot(hx, hy)
            assert np.all(c_lo >= -1e-9 * r) and np.all(c_hi <= 1e-9 * r)
            # eta: sinh(edge) brackets z/r
            L = g["layers"][l]
            ee = L["eta_lo"] + (L["eta_hi"] - L["eta_lo"]) * np.arange(41) / 40
            t = z[ids] / r
            inside = (t >= np.sinh(ee[0])) & (t < np.sinh(ee[40]))
            okk = (np.sinh(ee[ie]) <= t * (1 + 1e-12) + 1e-12) & (t * (1 - 1e-12) - 1e-12 <= np.sinh(ee[ie + 1]))
            assert np.all(okk[inside])
            assert np.all((ie[~inside] == 0) | (ie[~inside] == 39))            # outside → clamped to edge bins
    # vmax: upper bound of hit variance along any in-plane direction and along z
    vm = idx["vmax"].reshape(-1, 2)
    V = h["V"].astype(np.float64)
    for e in range(h["n_events"]):
        for l in range(nl):
            sl = slice(lo[e, l], lo[e, l + 1])
            if lo[e, l + 1] == lo[e, l]:
                continue
            lam = 0.5 * (V[0, sl] + V[2, sl]) + np.sqrt(0.25 * (V[0, sl] - V[2, sl]) ** 2 + V[1, sl] ** 2)
            assert vm[e * nl + l, 0] >= lam.max() * (1 - 1e-6) and vm[e * nl + l, 0] <= lam.max() * (1 + 1e-5)
            assert vm[e * nl + l, 1] == V[5, sl].max().astype(np.float32)


def _window_superset(ev, prm, n_seeds):
    """U11: every hit with chi2 < cut lies inside the window (brute force over the whole layer)."""
    g, h, s = ev["geom"], ev["hits"], ev["seeds"]
    o = mkfo.Oracle(g, prm)
    idx = o.build_hit_index(h)
    nl, nb = len(g["layers"]), 63 * 40
    lo = h["layer_off"].reshape(-1, nl + 1)
    bo, sid = idx["bin_off"].astype(np.int64), idx["sorted_id"]
    vm = idx["vmax"].reshape(-1, 2)
    npass = nchecked = 0
    rng = np.random.default_rng(1)
    for i in rng.choice(s["par"].shape[1], n_seeds, replace=False):
        u = s["par"][:, i].astype(np.float64)
        Cm = np.zeros((6, 6))
        for a in range(6):
            for b in range(a + 1):
                Cm[a, b] = Cm[b, a] = s["cov"][a * (a + 1) // 2 + b, i]
        Cm /= 25.0                                                             # a moderately wide state
        e = s["event"][i]
        pl = g["plan_layers"][g["plan_off"][s["plan"][i]]:g["plan_off"][s["plan"][i] + 1]]
        for lay in pl[1:]:
            L = g["layers"][lay]
            rc, u1, F, C1, sp = mkfo.propagate(L["kind"], L["pos"], g["bz"], int(s["q"][i]), u, Cm)
            if rc:
                continue
            v = u1[2] if L["kind"] == 0 else np.hypot(u1[0], u1[1])
            if v < L["lo"] or v > L["hi"]:
                continue
            seg = e * nl + lay
            if lo[e, lay + 1] == lo[e, lay]:
                continue
            e0, e1, p0, npb = o.window(lay, u1, C1, vm[seg])
            inwin = set()
            for ie in range(e0, e1 + 1):
                for k in range(npb):
                    b = seg * nb + ie * 63 + (p0 + k) % 63
                    inwin.update(sid[bo[b]:bo[b + 1]].tolist())
            for hid in range(lo[e, lay], lo[e, lay + 1]):
                m = np.array([h["x"][hid], h["y"][hid], h["z"][hid]], np.float64)
                rc2, c2 = mkfo.chi2(u1, C1, m, h["V"][:, hid].astype(np.float64))
                nchecked += 1
                if rc2 == 0 and c2 < prm["chi2_cut"]:
                    npass += 1
                    assert hid in inwin, (i, lay, hid, c2)
            assert len(inwin) < lo[e, lay + 1] - lo[e, lay] or npb == 63      # the window actually prunes
            u, Cm = u1, C1
    return npass, nchecked


def test_window_is_superset_of_chi2_cut_barrel(small_build_event):
    ev, prm = small_build_event
    npass, nchecked = _window_superset(ev, prm, 12)
    assert npass > 50 and nchecked > 100000


def test_window_is_superset_of_chi2_cut_endcap(small_endcap_event):
    ev, prm = small_endcap_event
    npass, nchecked = _window_superset(ev, prm, 6)
    assert npass > 20


def _build(ev, prm, brute, sel=None):
    g, h, s = ev["geom"], ev["hits"], ev["seeds"]
    o = mkfo.Oracle(g, prm)
    idx = o.build_hit_index(h)
    sl = slice(None) if sel is None else sel
    return o.build_tracks(h, idx, s["par"][:, sl], s["cov"][:, sl], s["q"][sl], s["event"][sl], s["hits"][:, sl],
                          s["plan"][sl], brute_force=brute)


def test_binned_search_equals_brute_force_barrel(small_build_event):
    """north_star: 'brute-force all-hits search on tiny events agreeing with the binned search' — exact identity."""
    ev, prm = small_build_event
    sel = slice(0, 400)
    a = _build(ev, prm, True, sel)
    b = _build(ev, prm, False, sel)
    for k in ("hit_ids", "nhits", "nmiss", "status"):
        assert np.array_equal(a[k], b[k]), k
    for k in ("par", "cov", "chi2", "score"):
        assert np.array_equal(a[k], b[k]), k
    assert b["n_chi2_evals"] * 20 < a["n_chi2_evals"]                          # and the window prunes >95 %


def test_binned_search_equals_brute_force_endcap(small_endcap_event):
    ev, prm = small_endcap_event
    n = ev["seeds"]["par"].shape[1]
    sel = slice(0, min(n, 300))
    a = _build(ev, prm, True, sel)
    b = _build(ev, prm, False, sel)
    for k in ("hit_ids", "nhits", "nmiss", "status", "par", "cov", "chi2", "score"):
        assert np.array_equal(a[k], b[k]), k


def test_build_finds_truth_on_clean_event():
    """Sanity (C9): noise-free barrel event, every seed's winner = its truth hits for >= 99 % of seeds, and the
    fit over the found hits equals mkfo_fit over the same hits (building = propagate+update)."""
    g = datagen.geometry_barrel(17, 4.0, 110.0, 150.0, np.linspace(0.01, 0.04, 17))
    ev = datagen.make_events(g, 11, 1, 300)
    prm = datagen.default_params()
    r = _build(ev, prm, False)
    th = ev["seeds"]["track_hits"]
    found = r["hit_ids"]
    same = np.all((found == th) | ((th < 0) & (found < 0)), axis=0)
    assert same.mean() >= 0.99
    # chained fit equality on tracks without misses
    o = mkfo.Oracle(g, prm)
    s = ev["seeds"]
    f = o.fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], np.where(found >= 0, found, -1))
    okk = (r["status"] == 0) & (f["status"] == 0) & (r["nmiss"] == 0)
    assert okk.sum() > 200
    assert np.allclose(f["chi2"][okk], r["chi2"][okk], rtol=1e-9, atol=1e-9)
    assert np.allclose(f["par"][:, okk], r["par"][:, okk], rtol=1e-9, atol=1e-12)


def test_build_rules_on_hand_placed_event():
    """Hand-placed single straight-ish track: per-seed cap, miss counting, stop after 2 consecutive misses,
    short-track preservation (C9)."""
    g = datagen.geometry_barrel(10, 4.0, 40.0, 100.0, 0.0)
    ev = datagen.make_events(g, 2, 1, 1, material=False)
    prm = datagen.default_params(material_flags=0)
    h, s = ev["hits"], ev["seeds"]
    assert s["par"].shape[1] == 1
    o = mkfo.Oracle(g, prm)

    def run(keep_layers, **kw):
        lo = h["layer_off"]
        keep = np.array([l in keep_layers for l in range(10)])
        ids = np.nonzero(keep)[0]                                             # one hit per layer, hit id == layer
        hh = dict(n_events=1, x=h["x"][ids], y=h["y"][ids], z=h["z"][ids], V=h["V"][:, ids],
                  layer_off=np.concatenate([[0], np.cumsum(keep)]).astype(np.int32))
        remap = -np.ones(10, np.int32); remap[ids] = np.arange(len(ids))
        p2 = dict(prm); p2.update(kw)
        oo = mkfo.Oracle(g, p2)
        idx = oo.build_hit_index(hh)
        r = oo.build_tracks(hh, idx, s["par"], s["cov"], s["q"], s["event"], remap[s["hits"]], s["plan"])
        back = np.where(r["hit_ids"][:, 0] >= 0, ids[np.maximum(r["hit_ids"][:, 0], 0)], r["hit_ids"][:, 0])
        return r, back

    r, ids = run(range(10))
    assert list(ids) == list(range(10)) and r["nhits"][0] == 10 and r["nmiss"][0] == 0
    assert abs(r["score"][0] - (30 * 10 - r["chi2"][0])) < 1e-9               # U13
    r, ids = run([0, 1, 2, 3, 5, 6, 7, 8, 9])                                  # one hole: counted as one miss
    assert list(ids) == [0, 1, 2, 3, -1, 5, 6, 7, 8, 9] and r["nmiss"][0] == 1 and r["nhits"][0] == 9
    assert abs(r["score"][0] - (30 * 9 - 15 - r["chi2"][0])) < 1e-9
    r, ids = run([0, 1, 2, 3, 4, 7, 8, 9])                                     # two consecutive holes: stop, keep short
    assert list(ids[:7]) == [0, 1, 2, 3, 4, -1, -1] and r["nhits"][0] == 5 and r["nmiss"][0] == 2
    assert np.all(ids[7:] == -2)
    r, ids = run([0, 1, 2, 5, 6, 7, 8, 9])                                     # stops with 3 hits < min_hits_keep
    assert r["status"][0] & 32 and r["nhits"][0] == 3                          # TRUNCATED: the seed itself
    r, ids = run([0, 1, 2, 5, 6, 7, 8, 9], max_consec_miss=3)                  # a looser rule bridges the gap
    assert r["nhits"][0] == 8 and r["nmiss"][0] == 2


def test_top_n_cap_equals_full_sort_when_cap_is_loose(small_build_event):
    """With a cap no pool can reach, the answer equals the cap-8 answer wherever the margin says the cap never
    bit (score gap recorded), and a cap of 1 (greedy) still returns valid tracks with fewer or equal score."""
    ev, prm = small_build_event
    sel = slice(0, 200)
    r8 = _build(ev, dict(prm, max_cand=8), False, sel)
    r1 = _build(ev, dict(prm, max_cand=1), False, sel)
    r64 = _build(ev, dict(prm, max_cand=64), False, sel)
    assert np.all(r64["score"] >= r8["score"] - 1e-9)                          # a wider beam never loses
    assert np.all(r8["score"] >= r1["score"] - 1e-9)
    assert (r64["score"] == r8["score"]).mean() > 0.97


# ---- C10 ------------------------------------------------------------------------------------------------
def _dedup_brute(track_off, hit_ids, nhits, score, frac):
    n = hit_ids.shape[1]
    keep = np.ones(n, np.uint8)
    for e in range(len(track_off) - 1):
        rng_ = range(track_off[e], track_off[e + 1])
        sets = {i: set(int(v) for v in hit_ids[:, i] if v >= 0) for i in rng_}
        for i in rng_:
            for j in rng_:
                if i == j:
                    continue
                mn = min(nhits[i], nhits[j])
                if mn <= 0:
                    continue
                sh = len(sets[i] & sets[j])
                if sh > frac * mn and (score[j] > score[i] or (score[j] == score[i] and j < i)):
                    keep[i] = 0
    return keep


def test_remove_duplicates_matches_set_brute_force():
    rng = np.random.default_rng(7)
    nev, per, mpl = 3, 120, 12
    n = nev * per
    track_off = np.arange(nev + 1, dtype=np.int32) * per
    hit_ids = np.full((mpl, n), -1, np.int32)
    base = rng.integers(0, 400, size=(mpl, n))
    for i in range(n):
        ev = i // per
        if i % per >= 40 and rng.random() < 0.6:                               # a near-copy of an earlier track
            src = ev * per + rng.integers(0, 40)
            col = hit_ids[:, src].copy()
            chg = rng.random(mpl) < rng.choice([0.2, 0.45, 0.55])
            col[chg] = base[chg, i] + 1000 * ev + 400 * np.arange(mpl)[chg]
        else:
            col = base[:, i] + 1000 * ev + 400 * np.arange(mpl)
        drop = rng.random(mpl) < 0.2
        col[drop] = rng.choice([-1, -2])
        hit_ids[:, i] = col
    hit_ids += 0
    nhits = (hit_ids >= 0).sum(0).astype(np.int32)
    score = np.round(rng.normal(200, 50, n)).astype(np.float32)                # rounded → exact ties occur
    o = mkfo.Oracle(datagen.geometry_barrel(2, 4, 8, 10, 0.0), datagen.default_params())
    r = o.remove_duplicates(track_off, hit_ids, nhits, score)
    want = _dedup_brute(track_off, hit_ids, nhits, score, 0.5)
    assert np.array_equal(r["keep"], want)
    assert 0.1 < 1 - want.mean() < 0.8
    assert np.array_equal(r["n_kept"], want.reshape(nev, per).sum(1))
    # invariants: the best track of each event survives; identical twins: exactly the lower index survives
    for e in range(nev):
        sl = slice(e * per, (e + 1) * per)
        assert r["keep"][sl][np.argmax(score[sl])] == 1
    hit2 = np.concatenate([hit_ids[:, :5], hit_ids[:, :5]], 1)
    r2 = o.remove_duplicates(np.array([0, 10], np.int32), hit2, np.tile(nhits[:5], 2), np.tile(score[:5], 2))
    assert list(r2["keep"][5:]) == [0] * 5 and r2["n_kept"][0] <= 5


def test_remove_duplicates_on_built_tracks(small_build_event):
    """Seeding the same particle twice must leave one track (PAPER.md:5 'duplicate tracks ... explicitly removed')."""
    ev, prm = small_build_event
    s = ev["seeds"]
    first = np.nonzero(s["event"] == 0)[0][:100]
    sel = np.concatenate([first, first[:50]])
    g, h = ev["geom"], ev["hits"]
    o = mkfo.Oracle(g, prm)
    idx = o.build_hit_index(h)
    r = o.build_tracks(h, idx, s["par"][:, sel], s["cov"][:, sel], s["q"][sel], s["event"][sel], s["hits"][:, sel], s["plan"][sel])
    d = o.remove_duplicates(np.array([0, len(sel)], np.int32), r["hit_ids"], r["nhits"], r["score"].astype(np.float32))
    assert np.all(d["keep"][100:] == 0)                                        # the later twin goes
    assert d["keep"][:100].mean() > 0.95


# ---- U14 keys 3 and 4 (lower parent rank, lower hit id) ------------------------------------------------------
@pytest.mark.parametrize("cap", [1, 2])
def test_u14_ties_lower_hit_id_then_lower_parent_rank(cap):
    ev, prm = tie_event()
    s = ev["seeds"]
    o = mkfo.Oracle(ev["geom"], dict(prm, max_cand=cap))
    idx = o.build_hit_index(ev["hits"])
    for brute in (False, True):
        r = o.build_tracks(ev["hits"], idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"], brute_force=brute)
        assert list(r["hit_ids"][:, 0]) == TIE_EXPECTED[cap]
        assert r["nhits"][0] == 5 and r["nmiss"][0] == 0 and r["status"][0] == 0
    # the twins really tie: building with only one of them gives the same chi2 and score bit for bit
    for drop in (3, 4):
        keep = np.array([i for i in range(6) if i != drop])
        h = ev["hits"]
        sub = dict(n_events=1, x=h["x"][keep], y=h["y"][keep], z=h["z"][keep], V=np.ascontiguousarray(h["V"][:, keep]),
                   layer_off=np.array([0, 1, 2, 3, 4, 5], np.int32))
        r1 = o.build_tracks(sub, o.build_hit_index(sub), s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
        assert r1["chi2"][0] == r["chi2"][0] and r1["score"][0] == r["score"][0]


def test_u14_tie_on_the_last_layer_reaches_the_output_through_best_short():
    """The same twins on the LAST layer (no later layer to break the tie): the final choice among equal candidates is
    the first in rank order (stable), i.e. again the lower hit id."""
    ev, prm = tie_event()
    h, s = ev["hits"], ev["seeds"]
    g4 = datagen.geometry_barrel(5, 4.0, 20.0, 100.0, 0.0)
    g4 = dict(g4, layers=g4["layers"][:4], plan_off=np.array([0, 4], np.int32), plan_layers=np.arange(4, dtype=np.int32))
    sub = dict(n_events=1, x=h["x"][:5], y=h["y"][:5], z=h["z"][:5], V=np.ascontiguousarray(h["V"][:, :5]),
               layer_off=np.array([0, 1, 2, 3, 5], np.int32))
    o = mkfo.Oracle(g4, dict(prm, max_cand=2))
    r = o.build_tracks(sub, o.build_hit_index(sub), s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    assert list(r["hit_ids"][:, 0]) == [0, 1, 2, 3]


# ---- R1: a child whose update is not finite ------------------------------------------------------------------
def test_nan_child_is_dropped_and_its_parent_offered_to_best_short():
    """Reading R1 (C9.4 / C9.6): the non-finite child never becomes a candidate; its parent, as it stood before the
    layer, competes for the seed's best-short slot. Expected lists written by hand."""
    ev, prm = nan_child_event(bad_layer=4)
    s = ev["seeds"]
    # cap 1: on disk 4 the only ranked child is the accepted bad hit (chi2 < cut beats the miss child); it is not
    # finite -> dropped, the live set is empty and the parent (hits 0..3, 4 >= min_hits_keep) is the best short
    o = mkfo.Oracle(ev["geom"], dict(prm, max_cand=1))
    idx = o.build_hit_index(ev["hits"])
    r = o.build_tracks(ev["hits"], idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    assert list(r["hit_ids"][:, 0]) == [0, 1, 2, 3, -2, -2]
    assert r["nhits"][0] == 4 and r["nmiss"][0] == 0 and (r["status"][0] & 32) == 0
    assert np.all(np.isfinite(r["par"][:, 0])) and np.all(np.isfinite(r["cov"][:, 0]))
    # cap 3: after disk 3 the live set is [hits 0..3, hits 0..2 + one miss]. On disk 4 the ranked children are the bad
    # hit on the first (score 150 - chi2), then the first one's miss child and the bad hit on the second (both
    # 105 - chi2, in either order). Both bad-hit children are dropped (the second one's parent has 3 hits < 4: no
    # offer); the miss child lives on, finds hit 5 and wins with 5 hits and one miss (135 - chi2) over the offered
    # parent (120 - chi2')
    o3 = mkfo.Oracle(ev["geom"], dict(prm, max_cand=3))
    r2 = o3.build_tracks(ev["hits"], idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    assert list(r2["hit_ids"][:, 0]) == [0, 1, 2, 3, -1, 5]
    assert r2["nhits"][0] == 5 and r2["nmiss"][0] == 1
    # with a sane covariance on that hit the full track is found
    ev_ok = dict(ev, hits=dict(ev["hits"], V=ev["hits"]["V"].copy()))
    ev_ok["hits"]["V"][0, 4] = ev["hits"]["V"][0, 3]
    r3 = o.build_tracks(ev_ok["hits"], o.build_hit_index(ev_ok["hits"]), s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    assert list(r3["hit_ids"][:, 0]) == [0, 1, 2, 3, 4, 5]
    # bad hit on the layer right after the seed: the parent has 3 hits < min_hits_keep -> nothing qualifies, TRUNCATED seed
    ev3, _ = nan_child_event(bad_layer=3)
    r4 = o.build_tracks(ev3["hits"], o.build_hit_index(ev3["hits"]), s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    assert (r4["status"][0] & 32) and r4["nhits"][0] == 3 and list(r4["hit_ids"][:, 0]) == [0, 1, 2, -2, -2, -2]
