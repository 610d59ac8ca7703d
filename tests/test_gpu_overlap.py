"""-m gpu: overlap-hit recovery (mkf_build_tracks_overlap, reading R15) against the oracle."""
import numpy as np
import pytest
import torch

from oracle import mkfo
from workloads import datagen, parity

pytestmark = pytest.mark.gpu


def gpu_build_overlap(ev, prm, packed=True):
    from paper_2002_06295_b200 import binding as B
    s = ev["seeds"]
    ctx = B.Context(ev["geom"], prm)
    hits = B.hits_to_device(ev["hits"], with_module=True)
    nh = hits["x"].shape[0]
    idx, ws = B.alloc_hit_index(ctx, hits["n_events"], nh, packed=packed)
    ctx.build_hit_index(hits, idx, ws)
    sd = B.to_device(dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"], event=s["event"], hits=s["hits"]),
                     ["par", "cov", "q", "plan", "event", "hits"])
    n = s["par"].shape[1]
    out = B.alloc_build_out(n, ctx.max_plan_len)
    h2 = torch.full((ctx.max_plan_len, n), 99, dtype=torch.int32, device="cuda")
    ctx.build_tracks(hits, idx, sd, sd["event"], sd["hits"], sd["plan"], out, out["chi2"], out["score"], out["nhits"],
                     out["nmiss"], out["hit_ids"], out["status"], hit_ids2=h2)
    torch.cuda.synchronize()
    r = {k: v.cpu().numpy() for k, v in out.items()}
    r["hit_ids2"] = h2.cpu().numpy()
    # without `module` the call is refused
    plain = B.hits_to_device(ev["hits"])
    with pytest.raises(B.MkfError):
        ctx.build_tracks(plain, idx, sd, sd["event"], sd["hits"], sd["plan"], out, out["chi2"], out["score"], out["nhits"],
                         out["nmiss"], out["hit_ids"], out["status"], hit_ids2=h2)
    ctx.close()
    return r


def check(ev, prm, packed=True, min_same=0.995):
    s, h = ev["seeds"], ev["hits"]
    o = mkfo.Oracle(ev["geom"], prm)
    idx = o.build_hit_index(h)
    r = o.build_tracks(h, idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"], module=h["module"])
    g = gpu_build_overlap(ev, prm, packed=packed)
    same = np.all(g["hit_ids"] == r["hit_ids"], axis=0) & np.all(g["hit_ids2"] == r["hit_ids2"], axis=0)
    assert np.all(r["margin"][~same] < 1e-3), np.sort(r["margin"][~same])[-5:]
    assert same.mean() >= min_same, same.mean()
    assert np.array_equal(g["nhits"][same], r["nhits"][same]) and np.array_equal(g["nmiss"][same], r["nmiss"][same])
    ok = same & ((r["status"] & 32) == 0)
    assert parity.chi2_errors(g["chi2"], r["chi2"])[ok].max() <= parity.TOL_CHI2
    assert (np.abs(g["score"] - r["score"])[ok] / np.maximum(np.abs(r["score"][ok]), 1.0)).max() <= parity.TOL_CHI2
    assert (r["hit_ids2"] >= 0).sum() > 0
    return r, g


def test_overlap_recovery_barrel():
    g = datagen.geometry_barrel(17, 4.0, 110.0, 150.0, np.linspace(0.01, 0.04, 17))
    ev = datagen.make_events(g, 5, 3, 600, n_noise=8000, overlap_frac=0.3)
    r, h = check(ev, datagen.default_params(max_cand=6))
    assert (r["hit_ids2"] >= 0).sum() > 2000
    check(ev, datagen.default_params(max_cand=6), packed=False)


def test_overlap_recovery_barrel_endcap():
    g = datagen.geometry_barrel_endcap()
    ev = datagen.make_events(g, 3, 2, 800, n_secondary=1500, n_noise=6000, spectrum="soft", pt_range=(0.3, 50.0), n_hard=20,
                             eta_max=2.5, eff=0.95, seed_on_pixel=True, overlap_frac=0.25)
    check(ev, datagen.default_params(max_cand=8))


def test_overlap_hand_placed_event():
    import sys, os
    sys.path.insert(0, os.path.dirname(os.path.abspath(__file__)))
    from test_oracle_overlap import _one_track_event
    g, hits, seeds, module, first = _one_track_event({4, 7})
    hits = dict(hits, module=module)
    ev = dict(geom=g, hits=hits, seeds=seeds)
    prm = datagen.default_params(material_flags=0)
    r = gpu_build_overlap(ev, prm)
    h1, h2 = r["hit_ids"][:, 0], r["hit_ids2"][:, 0]
    for l in range(10):
        if l in (4, 7):
            assert {int(h1[l]), int(h2[l])} == {int(first[l]), int(first[l]) + 1}, l
        else:
            assert h1[l] == first[l] and h2[l] == -2
    assert r["nhits"][0] == 12
