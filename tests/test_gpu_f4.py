"""-m gpu: SURVEY f4's remaining items against the oracle: energy-loss straggling (material flag 4, reading R12) and the
non-uniform field hook (bz_layer, reading R13), in the forward fit, the backward fit and the building."""
import numpy as np
import pytest

from oracle import mkfo
from workloads import datagen, parity

pytestmark = pytest.mark.gpu


def check_fit(ev, prm, min_full=0.9):
    from gpu_helpers import gpu_fit
    s = ev["seeds"]
    o = mkfo.Oracle(ev["geom"], prm)
    r = o.fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    h = gpu_fit(ev, prm)
    assert np.array_equal(h["nfit"], r["nfit"]) and np.array_equal(h["status"], r["status"])
    ok = r["nfit"] > 0
    lay, kinds, pos = parity.last_layer_of_fit(ev["geom"], s["plan"], s["track_hits"], r["nfit"])
    assert parity.param_errors(h["par"], r["par"], pos)[ok].max() <= parity.TOL_PAR
    assert parity.cov_errors(h["cov"], r["cov"], r["par"], kinds)[ok].max() <= parity.TOL_COV
    assert parity.chi2_errors(h["chi2"], r["chi2"])[ok].max() <= parity.TOL_CHI2
    # backward from the oracle's forward result
    th = s["track_hits"].copy()
    th[np.cumsum(th >= 0, 0) > r["nfit"][None]] = -1
    sb = dict(par=r["par"].astype(np.float32), cov=(100.0 * r["cov"]).astype(np.float32), q=s["q"], plan=s["plan"], track_hits=np.ascontiguousarray(th))
    rb = o.fit_backward(ev["hits"], sb["par"], sb["cov"], sb["q"], sb["plan"], sb["track_hits"])
    hb = gpu_fit(ev, prm, sb, backward=True)
    assert np.array_equal(hb["nfit"], rb["nfit"]) and np.array_equal(hb["status"], rb["status"])
    has = th >= 0
    okb = (rb["nfit"] > 0) & (rb["nfit"] == has.sum(0))
    assert okb.mean() > min_full
    geom = ev["geom"]
    layb = np.asarray(geom["plan_layers"])[np.asarray(geom["plan_off"])[s["plan"].astype(int)] + np.argmax(has, 0)]
    kb = np.array([l["kind"] for l in geom["layers"]])[layb]
    pb = np.array([abs(l["pos"]) for l in geom["layers"]])[layb]
    assert parity.param_errors(hb["par"], rb["par"], pb)[okb].max() <= parity.TOL_PAR
    assert parity.cov_errors(hb["cov"], rb["cov"], rb["par"], kb)[okb].max() <= parity.TOL_COV
    assert parity.chi2_errors(hb["chi2"], rb["chi2"])[okb].max() <= parity.TOL_CHI2
    return r, h


def test_fit_with_energy_loss_straggling():
    g = datagen.geometry_barrel(12, 4.0, 48.0, 150.0, 0.05)
    ev = datagen.make_events(g, 4, 1, 20000, pt_range=(0.25, 3.0), eta_max=0.8, straggle=True, shuffle=False)
    r7, h7 = check_fit(ev, datagen.default_params(material_flags=7))
    r3, h3 = check_fit(ev, datagen.default_params(material_flags=3))
    ok = (r7["nfit"] > 3) & (r3["nfit"] > 3)
    # the flag does something: sigma^2(ipt) grows, on the GPU as in the oracle
    assert np.median(h7["cov"][9][ok] / h3["cov"][9][ok]) > 1.02
    assert np.median(r7["cov"][9][ok] / r3["cov"][9][ok]) > 1.02
    # dE/dx and straggling without scattering: the term is the whole process noise
    check_fit(ev, datagen.default_params(material_flags=6))


def test_fit_and_build_in_a_layerwise_field():
    g = datagen.geometry_barrel(10, 4.0, 40.0, 100.0, 0.02)
    g["bz_layer"] = np.linspace(3.8, 2.6, 10).astype(np.float32)
    ev = datagen.make_events(g, 9, 1, 20000, shuffle=False)
    r, h = check_fit(ev, datagen.default_params())
    # the uniform hook is no hook, bit for bit
    from gpu_helpers import gpu_fit
    g0 = {k: v for k, v in g.items() if k != "bz_layer"}
    a = gpu_fit(dict(ev, geom=g0), datagen.default_params())
    b = gpu_fit(dict(ev, geom=dict(g0, bz_layer=np.full(10, g0["bz"], np.float32))), datagen.default_params())
    for k in ("par", "cov", "chi2", "nfit"):
        assert np.array_equal(a[k], b[k]), k
    assert not np.array_equal(a["par"], h["par"])
    # building, barrel + endcap with noise, in a field that falls off outwards
    from gpu_helpers import gpu_build
    gbe = datagen.geometry_barrel_endcap()
    gbe["bz_layer"] = np.array([3.8 - 0.012 * (abs(l["pos"]) if l["kind"] == 0 else 0.5 * abs(l["pos"])) for l in gbe["layers"]], np.float32)
    evb = datagen.make_events(gbe, 3, 2, 600, n_secondary=1000, n_noise=4000, spectrum="soft", pt_range=(0.3, 50.0), n_hard=20,
                              eta_max=2.5, eff=0.95, seed_on_pixel=True)
    prm = datagen.default_params(max_cand=6)
    s = evb["seeds"]
    o = mkfo.Oracle(gbe, prm)
    idx = o.build_hit_index(evb["hits"])
    rb = o.build_tracks(evb["hits"], idx, s["par"], s["cov"], s["q"], s["event"], s["hits"], s["plan"])
    hb = gpu_build(evb, prm)
    same = np.all(hb["hit_ids"] == rb["hit_ids"], axis=0)
    assert same.mean() >= 0.995 and np.all(rb["margin"][~same] < 1e-3)
    assert (rb["nhits"] >= 8).mean() > 0.5
    xe = parity.chi2_errors(hb["chi2"], rb["chi2"])[same & ((rb["status"] & 32) == 0)]
    assert xe.max() <= parity.TOL_CHI2
