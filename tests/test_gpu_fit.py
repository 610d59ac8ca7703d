"""-m gpu: mkf_fit (CUDA, fp32) against the fp64 oracle on the same seeded inputs (tolerances: BASELINE.json
north_star; U19 of DESIGN.md §3 says how 'relative' is read)."""
import numpy as np
import pytest

from oracle import mkfo
from workloads import datagen
from workloads import parity

pytestmark = pytest.mark.gpu


def check_fit(ev, prm, seeds=None, min_good=0.99):
    from gpu_helpers import gpu_fit
    s = seeds if seeds is not None else ev["seeds"]
    o = mkfo.Oracle(ev["geom"], prm)
    r = o.fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    h = gpu_fit(ev, prm, s)
    # integer outputs: identical
    assert np.array_equal(h["nfit"], r["nfit"])
    assert np.array_equal(h["status"], r["status"])
    ok = r["nfit"] > 0
    assert ok.mean() >= min_good
    lay, kinds, pos = parity.last_layer_of_fit(ev["geom"], s["plan"], s["track_hits"], r["nfit"])
    pe = parity.param_errors(h["par"], r["par"], pos)[ok]
    ce = parity.cov_errors(h["cov"], r["cov"], r["par"], kinds)[ok]
    xe = parity.chi2_errors(h["chi2"], r["chi2"])[ok]
    assert pe.max() <= parity.TOL_PAR, pe.max()
    assert xe.max() <= parity.TOL_CHI2, xe.max()
    assert ce.max() <= parity.TOL_COV, ce.max()
    return r, h


def test_fit_config0_full():
    ev, prm = datagen.config(0)                       # 10 000 helices, 10 layers: 79 CTAs, ragged last CTA
    r, h = check_fit(ev, prm)
    assert r["nfit"].sum() == 100000


def test_fit_config1_sample():
    ev, prm = datagen.config(1, scale=0.0125)          # 50 000 helices, 17 layers incl. low-pT tracks that stop early
    r, h = check_fit(ev, prm)
    assert (r["nfit"] < 17).mean() > 0.03              # the short (near-grazing) tracks are in the sample


def test_fit_barrel_endcap_truth_hits():
    ev, prm = datagen.config(3, scale=0.01)            # 2 events of the 38-layer geometry: propagateToZ on disks
    r, h = check_fit(ev, prm, min_good=0.9)
    kinds = np.array([l["kind"] for l in ev["geom"]["layers"]])
    lay, k, pos = parity.last_layer_of_fit(ev["geom"], ev["seeds"]["plan"], ev["seeds"]["track_hits"], r["nfit"])
    assert (k == 1).sum() > 100 and (k == 0).sum() > 100


def test_fit_material_flags_and_status_paths():
    ev, prm = datagen.config(0, scale=0.05)
    for flags in (0, 1, 2):
        check_fit(ev, dict(prm, material_flags=flags))
    # status paths, with the states frozen (covariance x1e-8, no scattering noise) so that the hits cannot pull
    # them back: 0.2 GeV cannot reach r = 36 cm (radius of curvature 17.5 cm) -> PROP_UNREACHABLE; 0.05 GeV loses
    # all its energy -> STOPPED_ELOSS; 0.226..0.24 GeV straddles the grazing threshold at r = 40 cm -> GRAZING
    from gpu_helpers import gpu_fit
    s = {k: np.array(v[..., :64]) for k, v in ev["seeds"].items() if k in ("par", "cov", "q", "plan", "track_hits")}
    s["cov"] *= 1e-8
    for flags, ipt, want in ((2, np.r_[np.full(32, 5.0), np.full(32, 20.0)], (1, 16)),
                             (0, 1.0 / np.linspace(0.226, 0.24, 64), (2,))):
        s["par"][3] = ipt
        p2 = dict(prm, material_flags=flags)
        r = mkfo.Oracle(ev["geom"], p2).fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
        h = gpu_fit(ev, p2, s)
        assert np.array_equal(h["nfit"], r["nfit"]) and np.array_equal(h["status"], r["status"])
        for bit in want:
            assert (r["status"] & bit).any(), bit
        assert (r["status"] == 0).any() or flags == 2
        ok = r["nfit"] > 0
        lay, kinds, pos = parity.last_layer_of_fit(ev["geom"], s["plan"], s["track_hits"], r["nfit"])
        assert parity.param_errors(h["par"], r["par"], pos)[ok].max() <= parity.TOL_PAR
        z = r["nfit"] == 0                           # tracks that never fitted a hit return their seed unchanged
        if z.any():
            assert np.array_equal(h["par"][:, z], s["par"][:, z]) and np.array_equal(h["cov"][:, z], s["cov"][:, z])


def test_fit_empty_and_no_hits():
    import torch
    from paper_2002_06295_b200 import binding as B
    ev, prm = datagen.config(0, scale=0.01)
    ctx = B.Context(ev["geom"], prm)
    hits = B.hits_to_device(ev["hits"])
    s = ev["seeds"]
    sd = B.to_device(s, ["par", "cov", "q", "plan", "track_hits"])
    # n = 0: nothing launched, OK
    e = {k: v[..., :0].contiguous() for k, v in sd.items()}
    out = B.alloc_fit_out(0)
    before = ctx.launch_count()
    ctx.fit(hits, e, e["plan"], e["track_hits"], out, out["chi2"], out["nfit"], out["status"])
    assert ctx.launch_count() == before
    # tracks without any hit: state returned unchanged, nfit 0, chi2 0
    sd["track_hits"].fill_(-1)
    n = s["par"].shape[1]
    out = B.alloc_fit_out(n)
    ctx.fit(hits, sd, sd["plan"], sd["track_hits"], out, out["chi2"], out["nfit"], out["status"])
    torch.cuda.synchronize()
    assert int(out["nfit"].sum()) == 0 and float(out["chi2"].abs().sum()) == 0.0
    assert torch.equal(out["par"][:4], sd["par"][:4]) and torch.equal(out["cov"], sd["cov"])
    ctx.close()


def test_fit_host_entry_point_matches_device_path():
    from gpu_helpers import gpu_fit
    from paper_2002_06295_b200 import binding as B
    ev, prm = datagen.config(0, scale=0.1)
    h = gpu_fit(ev, prm)
    ctx = B.Context(ev["geom"], prm)
    s = ev["seeds"]
    r = ctx.fit_host(ev["hits"], s, np.ascontiguousarray(s["plan"]), np.ascontiguousarray(s["track_hits"]))
    for k in ("par", "cov", "chi2", "nfit"):
        assert np.array_equal(r[k], h[k]), k
    n = s["par"].shape[1]
    assert r["d2h_bytes"] == n * (27 * 4 + 12) and r["h2d_bytes"] > n * 27 * 4
    ctx.close()


def test_fit_quarter_of_configs1_in_bench_launch_configuration_sampled():
    """1 M helices (a quarter of configs[1], generated exactly as bench.py does, same launch configuration: 7813 CTAs
    of 128 threads); the oracle checks a sample of 60 000 tracks taken across the whole range."""
    import sys, os
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    from gpu_helpers import gpu_fit
    geom, prm, hits, seeds, _ = bench.make_fit_workload(3, 0.25)
    n = seeds["par"].shape[1]
    assert n == 1000000
    h = gpu_fit(dict(geom=geom, hits=hits), prm, seeds)
    sel = np.sort(np.random.default_rng(0).choice(n, 60000, replace=False))
    sub = {k: np.ascontiguousarray(v[..., sel]) for k, v in seeds.items()}
    r = mkfo.Oracle(geom, prm).fit(hits, sub["par"], sub["cov"], sub["q"], sub["plan"], sub["track_hits"])
    assert np.array_equal(h["nfit"][sel], r["nfit"]) and np.array_equal(h["status"][sel], r["status"])
    ok = r["nfit"] > 0
    lay, kinds, pos = parity.last_layer_of_fit(geom, sub["plan"], sub["track_hits"], r["nfit"])
    assert parity.param_errors(h["par"][:, sel], r["par"], pos)[ok].max() <= parity.TOL_PAR
    assert parity.cov_errors(h["cov"][:, sel], r["cov"], r["par"], kinds)[ok].max() <= parity.TOL_COV
    assert parity.chi2_errors(h["chi2"][sel], r["chi2"])[ok].max() <= parity.TOL_CHI2
    # property that holds at any size: every track ends on the layer of its last fitted hit (the update moves the
    # point along the tangent plane, so the radius may exceed the layer's by shift^2 / 2R)
    R = np.hypot(h["par"][0], h["par"][1])
    radii = np.array([l["pos"] for l in geom["layers"]])
    fitted = h["nfit"] > 0
    dR = R[fitted] - radii[h["nfit"][fitted] - 1]
    assert dR.min() > -2e-5 * 110 and dR.max() < 0.1 and np.quantile(np.abs(dR), 0.99) < 1e-3
    assert np.isfinite(h["chi2"]).all() and np.isfinite(h["cov"]).all()


def check_backward(ev, prm):
    """mkf_fit_backward against the oracle (R7). Seeds: the ORACLE's forward fit (so that both sides start from the
    same float32 numbers) with the covariance x100, hit lists cut at the last fitted hit."""
    from gpu_helpers import gpu_fit
    s = ev["seeds"]
    o = mkfo.Oracle(ev["geom"], prm)
    f = o.fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    th = s["track_hits"].copy()
    th[np.cumsum(th >= 0, 0) > f["nfit"][None]] = -1
    sb = dict(par=f["par"].astype(np.float32), cov=(100.0 * f["cov"]).astype(np.float32), q=s["q"], plan=s["plan"],
              track_hits=np.ascontiguousarray(th))
    r = o.fit_backward(ev["hits"], sb["par"], sb["cov"], sb["q"], sb["plan"], sb["track_hits"])
    h = gpu_fit(ev, prm, sb, backward=True)
    assert np.array_equal(h["nfit"], r["nfit"]) and np.array_equal(h["status"], r["status"])
    has = th >= 0
    ok = (r["nfit"] > 0) & (r["nfit"] == has.sum(0))                   # went all the way in: state on the first hit's layer
    assert ok.mean() > 0.95
    geom = ev["geom"]
    lay = np.asarray(geom["plan_layers"])[np.asarray(geom["plan_off"])[s["plan"].astype(int)] + np.argmax(has, 0)]
    kinds = np.array([l["kind"] for l in geom["layers"]])[lay]
    pos = np.array([abs(l["pos"]) for l in geom["layers"]])[lay]
    assert parity.param_errors(h["par"], r["par"], pos)[ok].max() <= parity.TOL_PAR
    assert parity.cov_errors(h["cov"], r["cov"], r["par"], kinds)[ok].max() <= parity.TOL_COV
    assert parity.chi2_errors(h["chi2"], r["chi2"])[ok].max() <= parity.TOL_CHI2
    return r, h


def test_fit_backward_barrel():
    ev, prm = datagen.config(0, scale=0.5)
    check_backward(ev, prm)
    ev, prm = datagen.config(1, scale=0.005)          # 20 000 helices, 17 layers, tracks of unequal length
    check_backward(ev, prm)


def test_fit_backward_barrel_endcap_with_curling_tracks():
    ev, prm = datagen.config(3, scale=0.01)           # disks and cylinders, soft tracks that come back in radius
    r, h = check_backward(ev, prm)
    assert (r["status"] != 0).sum() >= 1


def test_fit_on_shuffled_hits_with_48_byte_records_is_bit_identical():
    """mkf_hits.rec (mkf_pack_hits): the same hits gathered from 48-byte records instead of the nine SoA planes, on hit
    ids in random order; the result must not change by a bit, forward and backward, and equals the id-ordered fit."""
    import torch
    from paper_2002_06295_b200 import binding as B
    from workloads import assemble
    ev, prm = datagen.config(1, scale=0.01)           # 40 000 helices, 17 layers
    s = {k: ev["seeds"][k] for k in ("par", "cov", "q", "plan", "track_hits")}
    h2, s2 = assemble.shuffle_hit_order(ev["hits"], s, 5)
    assert not np.array_equal(s2["track_hits"], s["track_hits"])
    from gpu_helpers import gpu_fit
    base = gpu_fit(ev, prm, s)
    ctx = B.Context(ev["geom"], prm)
    dh = B.hits_to_device(h2)
    sd = B.to_device(s2, ["par", "cov", "q", "plan", "track_hits"])
    n = s["par"].shape[1]
    for backward in (False, True):
        outs = []
        for use_rec in (False, True):
            if use_rec:
                dh["rec"] = torch.empty(12 * h2["x"].shape[0], dtype=torch.float32, device="cuda")
                ctx.pack_hits(dh, dh["rec"])
            else:
                dh.pop("rec", None)
            out = B.alloc_fit_out(n)
            ctx.fit(dh, sd, sd["plan"], sd["track_hits"], out, out["chi2"], out["nfit"], out["status"], backward=backward)
            torch.cuda.synchronize()
            outs.append({k: v.cpu().numpy() for k, v in out.items()})
        for k in ("par", "cov", "chi2", "nfit", "status"):
            assert np.array_equal(outs[0][k], outs[1][k]), (backward, k)
            if not backward:
                assert np.array_equal(outs[1][k].view(np.uint32) if k == "status" else outs[1][k], base[k]), k
    rec = dh["rec"].cpu().numpy().reshape(-1, 12)
    assert np.array_equal(rec[:, 0], h2["x"]) and np.array_equal(rec[:, 3:9], h2["V"].T) and not rec[:, 9:].any()
    ctx.close()


def test_fit_host_pipeline_over_several_track_ranges():
    """mkf_fit_host / mkf_fit_backward_host work on ranges of 256 k tracks on three streams: 600 k tracks (3 ranges, the
    last one ragged) must give exactly the device path's result; a second call reuses the context's arena."""
    import sys, os
    sys.path.insert(0, os.path.dirname(os.path.dirname(os.path.abspath(__file__))))
    import bench
    from gpu_helpers import gpu_fit
    from paper_2002_06295_b200 import binding as B
    geom, prm, hits, seeds, _ = bench.make_fit_workload(9, 0.15)
    n = seeds["par"].shape[1]
    assert n == 600000
    h = gpu_fit(dict(geom=geom, hits=hits), prm, seeds)
    ctx = B.Context(geom, prm)
    for rep in range(2):
        r = ctx.fit_host(hits, seeds, seeds["plan"], seeds["track_hits"])
        for k in ("par", "cov", "chi2", "nfit"):
            assert np.array_equal(r[k], h[k]), k
        assert np.array_equal(r["status"], h["status"])
        assert r["d2h_bytes"] == n * (27 * 4 + 12)
        assert r["h2d_bytes"] == hits["x"].shape[0] * 36 + 4 * len(hits["layer_off"]) + n * (27 * 4 + 2 + 4 * seeds["track_hits"].shape[0])
    hb = gpu_fit(dict(geom=geom, hits=hits), prm, seeds, backward=True)
    rb = ctx.fit_host(hits, seeds, seeds["plan"], seeds["track_hits"], backward=True)
    for k in ("par", "cov", "chi2", "nfit"):
        assert np.array_equal(rb[k], hb[k]), k
    ctx.close()


def test_fit_flags_indices_outside_the_call():
    """A plan id that is no plan of the geometry, or a hit id >= n_hits: the track is flagged (TRUNCATED) instead of
    reading out of bounds; its neighbours are not disturbed."""
    from gpu_helpers import gpu_fit
    ev, prm = datagen.config(0, scale=0.02)
    s = {k: ev["seeds"][k].copy() for k in ("par", "cov", "q", "plan", "track_hits")}
    base = gpu_fit(ev, prm, s)
    s["plan"][3] = 5
    s["plan"][4] = -1
    nh = ev["hits"]["x"].shape[0]
    s["track_hits"][6, 10] = nh + 7
    h = gpu_fit(ev, prm, s)
    for i in (3, 4):
        assert h["status"][i] == 32 and h["nfit"][i] == 0 and np.array_equal(h["par"][:, i], s["par"][:, i])
    assert (h["status"][10] & 32) and h["nfit"][10] == 6 and base["nfit"][10] == 10
    others = np.ones(len(h["nfit"]), bool); others[[3, 4, 10]] = False
    for k in ("par", "cov", "chi2", "nfit", "status"):
        assert np.array_equal(h[k][..., others], base[k][..., others]), k
    hb = gpu_fit(ev, prm, s, backward=True)                         # the backward kernel flags the plan ids the same way
    assert hb["status"][3] == 32 and hb["status"][4] == 32 and hb["nfit"][3] == 0
