"""Pins for overlap-hit recovery (reading R15; PAPER.md:55 'more than one hit per layer can be assigned')."""
import numpy as np

from oracle import mkfo
from workloads import datagen


def _barrel():
    return datagen.geometry_barrel(10, 4.0, 40.0, 100.0, 0.0)


def _one_track_event(dup_layers, module_same=False):
    """One track through 10 barrel layers without material; on each layer in dup_layers the hit is present twice with
    independent smearing (ids: the copies come right after their first hit). Returns hits, seeds, module."""
    g = _barrel()
    ev = datagen.make_events(g, 2, 1, 1, material=False, overlap_frac=0.0)
    h, s = ev["hits"], ev["seeds"]
    rng = np.random.default_rng(1)
    ids, mod, lay_of = [], [], []
    for l in range(10):
        ids.append(l); mod.append(100 * l + 7); lay_of.append(l)
        if l in dup_layers:
            ids.append(l); mod.append(100 * l + (7 if module_same else 8)); lay_of.append(l)
    ids = np.array(ids)
    x, y, z = h["x"][ids].astype(np.float64), h["y"][ids].astype(np.float64), h["z"][ids].astype(np.float64)
    second = np.concatenate([[False], ids[1:] == ids[:-1]])
    # move the copies by a fraction of the resolution along the surface (rphi 0.003, z 0.01)
    r = np.hypot(x, y)
    dphi = rng.standard_normal(len(ids)) * 0.003 / r * second
    c, sn = np.cos(dphi), np.sin(dphi)
    x, y = x * c - y * sn, x * sn + y * c
    z = z + rng.standard_normal(len(ids)) * 0.01 * second
    lo = np.concatenate([[0], np.cumsum(np.bincount(lay_of, minlength=10))]).astype(np.int32)
    hits = dict(n_events=1, x=x.astype(np.float32), y=y.astype(np.float32), z=z.astype(np.float32), V=np.ascontiguousarray(h["V"][:, ids]),
                layer_off=lo)
    first_id = np.array([int(np.nonzero((np.array(lay_of) == l) & ~second)[0][0]) for l in range(10)])
    seeds = {k: np.ascontiguousarray(s[k]) for k in ("par", "cov", "q", "plan", "event")}
    seeds["hits"] = first_id[:3].reshape(3, 1).astype(np.int32)
    return g, hits, seeds, np.array(mod, np.int32), first_id


def _run(g, hits, seeds, module, **kw):
    prm = datagen.default_params(material_flags=0, **kw)
    o = mkfo.Oracle(g, prm)
    idx = o.build_hit_index(hits)
    return o.build_tracks(hits, idx, seeds["par"], seeds["cov"], seeds["q"], seeds["event"], seeds["hits"], seeds["plan"], module=module)


def test_second_hit_is_taken_once_per_layer_from_another_module_only():
    g, hits, seeds, module, first = _one_track_event({4, 7})
    base = _run(g, hits, seeds, None)                                  # without modules: today's build
    r = _run(g, hits, seeds, module)
    assert "hit_ids2" not in base
    # one of the two copies is the layer's hit, the other its second hit; elsewhere no second hit
    h1, h2 = r["hit_ids"][:, 0], r["hit_ids2"][:, 0]
    for l in range(10):
        if l in (4, 7):
            assert {int(h1[l]), int(h2[l])} == {int(first[l]), int(first[l]) + 1}, l
        else:
            assert h1[l] == first[l] and h2[l] == -2
    assert r["nhits"][0] == 12 and base["nhits"][0] == 10 and r["nmiss"][0] == 0
    assert abs(r["score"][0] - (30.0 * 12 - r["chi2"][0])) < 1e-9       # U13 with the overlap hits counted
    # the copies in the SAME module as the first hit: nothing is taken, the result is today's, bit for bit
    g2, hits2, seeds2, module2, _ = _one_track_event({4, 7}, module_same=True)
    r2 = _run(g2, hits2, seeds2, module2)
    b2 = _run(g2, hits2, seeds2, None)
    assert np.all(r2["hit_ids2"] == -2)
    for k in ("hit_ids", "nhits", "chi2", "score", "par", "cov"):
        assert np.array_equal(r2[k], b2[k]), k


def test_second_hit_improves_the_state_like_one_more_measurement():
    """The state after a layer with two hits equals the Kalman update with both (order: best first), so its position
    variance along rphi is below the single-hit one by the textbook factor when the prior is weak against the hits."""
    g, hits, seeds, module, first = _one_track_event({9})
    r = _run(g, hits, seeds, module)
    b = _run(g, hits, seeds, None)
    assert r["hit_ids2"][9, 0] >= 0
    # rphi variance at the last layer (x-y block projected on the tangent)
    def ctt(res):
        P, Cv = res["par"][:, 0], res["cov"][:, 0]
        R = np.hypot(P[0], P[1]); tx, ty = -P[1] / R, P[0] / R
        return tx * tx * Cv[0] + 2 * tx * ty * Cv[1] + ty * ty * Cv[2]
    v1, v2 = ctt(b), ctt(r)
    sig2 = 0.003 ** 2
    # single hit: 1/v1 = 1/prior + 1/sig2 ; two hits: 1/v2 = 1/prior + 2/sig2  =>  1/v2 - 1/v1 = 1/sig2
    assert abs((1 / v2 - 1 / v1) * sig2 - 1.0) < 0.02


def test_overlap_recovery_on_simulated_events():
    """30 % of the crossings seen twice: the build with modules picks up most second hits of the seeded particles, never
    two hits of one module on a layer, never the same hit twice; without modules it equals the plain build."""
    g = datagen.geometry_barrel(17, 4.0, 110.0, 150.0, np.linspace(0.01, 0.04, 17))
    ev = datagen.make_events(g, 5, 2, 400, n_noise=6000, overlap_frac=0.3)
    prm = datagen.default_params(max_cand=6)
    s, h = ev["seeds"], ev["hits"]
    o = mkfo.Oracle(g, prm)
    idx = o.build_hit_index(h)
    r = o.build_tracks(h, idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"], module=h["module"])
    b = o.build_tracks(h, idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    bf = o.build_tracks(h, idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"], module=h["module"], brute_force=True)
    for k in ("hit_ids", "hit_ids2", "nhits", "chi2"):
        assert np.array_equal(r[k], bf[k]), k                          # binned search == brute force with the feature on
    h1, h2 = r["hit_ids"], r["hit_ids2"]
    two = h2 >= 0
    assert np.all(h1[two] >= 0) and np.all(h1[two] != h2[two])
    assert np.all(h["module"][h1[two]] != h["module"][h2[two]])
    assert np.all(ev["hit_layer"][h1[two]] == ev["hit_layer"][h2[two]])
    assert np.array_equal(r["nhits"], (h1 >= 0).sum(0) + two.sum(0))
    # truth: second hits of the seeded particle that exist on layers where the track has its particle's first hit
    part = ev["hit_particle"]
    pid = s["particle"]
    right = two & (part[np.maximum(h2, 0)] == pid[None]) & (part[np.maximum(h1, 0)] == pid[None])
    n_truth_pairs = 0
    sig = part >= 0
    import collections
    pairs = collections.Counter(zip(part[sig].tolist(), ev["hit_layer"][sig].tolist()))
    seeded = set(pid.tolist())
    n_truth_pairs = sum(1 for (pp, ll), v in pairs.items() if v == 2 and pp in seeded and ll >= 3)
    assert right.sum() > 0.85 * n_truth_pairs
    assert (two & ~right).sum() < 0.05 * two.sum()                      # and few wrong ones
    assert r["score"].mean() > b["score"].mean() + 5.0
