"""-m gpu: the two-filter smoother (mkf_fit_smooth, reading R14) against the oracle at every fitted hit."""
import numpy as np
import pytest
import torch

from oracle import mkfo
from workloads import datagen, parity

pytestmark = pytest.mark.gpu


def gpu_smooth(ev, prm, seeds=None):
    from paper_2002_06295_b200 import binding as B
    s = seeds if seeds is not None else ev["seeds"]
    ctx = B.Context(ev["geom"], prm)
    hits = B.hits_to_device(ev["hits"])
    sd = B.to_device(s, ["par", "cov", "q", "plan", "track_hits"])
    n = s["par"].shape[1]
    mpl = s["track_hits"].shape[0]
    par_s = torch.full((mpl, 6, n), 7.0, dtype=torch.float32, device="cuda")
    cov_s = torch.full((mpl, 21, n), 7.0, dtype=torch.float32, device="cuda")
    o = B.alloc_fit_out(n)
    ws = torch.empty(max(ctx.workspace_bytes(B.CALL_FIT_SMOOTH, 0, 0, n), 256), dtype=torch.uint8, device="cuda")
    ctx.fit_smooth(hits, sd, sd["plan"], sd["track_hits"], par_s, cov_s, o["chi2"], o["nfit"], o["status"], ws)
    torch.cuda.synchronize()
    r = dict(par_s=par_s.cpu().numpy(), cov_s=cov_s.cpu().numpy(), chi2=o["chi2"].cpu().numpy(), nfit=o["nfit"].cpu().numpy(),
             status=o["status"].cpu().numpy().view(np.uint32))
    with pytest.raises(B.MkfError):
        ctx.fit_smooth(hits, sd, sd["plan"], sd["track_hits"], par_s, cov_s, o["chi2"], o["nfit"], o["status"], ws[:64])
    ctx.close()
    return r


def check_smooth(ev, prm, min_smoothed=0.9):
    s = ev["seeds"]
    geom = ev["geom"]
    r = mkfo.Oracle(geom, prm).fit_smooth(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    h = gpu_smooth(ev, prm)
    assert np.array_equal(h["nfit"], r["nfit"]) and np.array_equal(h["status"], r["status"])
    assert parity.chi2_errors(h["chi2"], r["chi2"])[r["nfit"] > 0].max() <= parity.TOL_CHI2
    mpl, _, n = r["par_s"].shape
    plan_off, plan_layers = np.asarray(geom["plan_off"]), np.asarray(geom["plan_layers"])
    smoothed_ref = np.any(r["cov_s"] != 0, axis=1)                     # (mpl, n)
    smoothed_gpu = np.any(h["cov_s"] != 0, axis=1)
    assert np.array_equal(smoothed_ref, smoothed_gpu)
    assert (smoothed_ref.sum(0) == r["nfit"])[r["status"] == 0].all()
    assert smoothed_ref.any(0).mean() > min_smoothed
    assert not np.any(h["par_s"][~np.repeat(smoothed_gpu[:, None, :], 6, 1)])          # zero where there is nothing
    worst = [0.0, 0.0]
    for st in range(mpl):
        m = smoothed_ref[st]
        if not m.any():
            continue
        lay = plan_layers[plan_off[s["plan"].astype(int)] + np.minimum(st, np.diff(plan_off)[s["plan"].astype(int)] - 1)]
        kinds = np.array([l["kind"] for l in geom["layers"]])[lay]
        pos = np.array([abs(l["pos"]) for l in geom["layers"]])[lay]
        pe = parity.param_errors(h["par_s"][st][:, m], r["par_s"][st][:, m], pos[m])
        ce = parity.cov_errors(h["cov_s"][st][:, m], r["cov_s"][st][:, m], r["par_s"][st][:, m], kinds[m])
        worst = [max(worst[0], pe.max()), max(worst[1], ce.max())]
    assert worst[0] <= parity.TOL_PAR and worst[1] <= parity.TOL_COV, worst
    return r, h


def test_smoother_barrel_config0_and_config1_samples():
    ev, prm = datagen.config(0, scale=0.3)
    check_smooth(ev, prm)
    ev, prm = datagen.config(1, scale=0.003)          # 12 000 helices, 17 layers, tracks of unequal length
    check_smooth(ev, prm)


def test_smoother_barrel_endcap_with_gaps_and_straggling():
    ev, prm = datagen.config(3, scale=0.01)           # disks and cylinders, 5 % missing hits, soft tracks
    r, h = check_smooth(ev, dict(prm, material_flags=7), min_smoothed=0.8)
    assert (r["status"] != 0).sum() >= 1
