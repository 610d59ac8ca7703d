"""Pins for the oracle's strip clustering (reading R8 of DESIGN.md): hand-worked cases for every rule
of the passage, and an independent brute-force formulation on random data."""
import numpy as np

from oracle import mkfo
from workloads import datagen


def run(adc, noise=4.0, bad=None, off=None, **kw):
    adc = np.asarray(adc)
    n = len(adc)
    return mkfo.cluster_strips([0, n] if off is None else off, adc, np.full(n, noise, np.float32) if np.isscalar(noise) else noise,
                               np.zeros(n, np.uint8) if bad is None else bad, **kw)


def test_hand_worked_rules():
    # noise 4: channel threshold 8 (strict), seed threshold 12 (strict)
    r = run([0, 30, 50, 30, 0, 0, 40, 0])
    assert r["first"].tolist() == [1, 6] and r["last"].tolist() == [3, 6] and r["charge"].tolist() == [110, 40]
    assert np.allclose(r["bary"], [(30 * 1.5 + 50 * 2.5 + 30 * 3.5) / 110, 6.5])
    # thresholds are strict: 8 = 2 sigma does not join, 12 = 3 sigma does not seed
    assert run([8, 30, 8])["first"].tolist() == [1] and run([8, 30, 8])["last"].tolist() == [1]
    assert len(run([9, 12, 9, 11])["first"]) == 0                       # no strip above 12 -> no seed -> no cluster
    assert run([9, 13, 9, 11, 0], clus_thr=0.0)["last"].tolist() == [3]
    # quadrature cut: 13^2 + 9^2 + 9^2 = 331 <= 25 * 3 * 16 = 1200 -> rejected; 30^2 = 900 > 400 -> kept
    assert len(run([9, 13, 9])["first"]) == 0 and len(run([0, 30, 0])["first"]) == 1
    # exactly at the cut: 20^2 = 400 is not > 25 * 16 = 400
    assert len(run([0, 20, 0])["first"]) == 0 and len(run([0, 21, 0])["first"]) == 1
    # minimum charge
    assert len(run([0, 30, 0], min_charge=31)["first"]) == 0 and len(run([0, 30, 0], min_charge=30)["first"]) == 1
    # a good strip below threshold splits (max_holes = 0); a bad strip is bridged (max_bad = 1); two bad strips split
    assert run([30, 0, 30])["first"].tolist() == [0, 2]
    bad = np.array([0, 1, 0], np.uint8)
    r = run([30, 0, 30], bad=bad)
    assert r["first"].tolist() == [0] and r["last"].tolist() == [2] and r["charge"].tolist() == [60] and np.allclose(r["bary"], [1.5])
    assert run([30, 0, 0, 30], bad=np.array([0, 1, 1, 0], np.uint8))["first"].tolist() == [0, 3]
    assert run([30, 0, 0, 30], bad=np.array([0, 1, 1, 0], np.uint8), max_bad=2)["first"].tolist() == [0]
    assert run([30, 0, 30], max_holes=1)["first"].tolist() == [0]
    # a bad strip never counts, whatever it reads; a trailing bad strip does not extend the cluster
    r = run([30, 500, 0], bad=np.array([0, 1, 0], np.uint8))
    assert r["first"].tolist() == [0] and r["last"].tolist() == [0] and r["charge"].tolist() == [30]
    # clusters never cross a module boundary; strip indices are local to the module
    r = run([0, 30, 30, 30, 30, 0], off=[0, 3, 6])
    assert r["module"].tolist() == [0, 1] and r["first"].tolist() == [1, 0] and r["last"].tolist() == [2, 1]


def brute_force(off, adc, noise, bad, seed_thr, chan_thr, clus_thr, min_charge, max_holes, max_bad):
    """Different formulation: label passing strips, link two of them iff the strips strictly between satisfy the gap
    rule (checked pair by pair, not by scanning), clusters = connected components."""
    out = []
    for m in range(len(off) - 1):
        b, e = off[m], off[m + 1]
        a = adc[b:e].astype(np.float32); nz = noise[b:e]; bd = bad[b:e] != 0
        ok = (~bd) & (a > np.float32(chan_thr) * nz)
        idx = np.nonzero(ok)[0]
        if idx.size == 0:
            continue
        groups = [[idx[0]]]
        for u, v in zip(idx[:-1], idx[1:]):
            between = np.arange(u + 1, v)
            linked = (bd[between].sum() <= max_bad) and ((~bd[between]).sum() <= max_holes)
            if linked:
                groups[-1].append(v)
            else:
                groups.append([v])
        for gidx in groups:
            gidx = np.array(gidx)
            if not (a[gidx] > np.float32(seed_thr) * nz[gidx]).any():
                continue
            q2 = int((adc[b:e][gidx].astype(np.int64) ** 2).sum()); n2 = float((nz[gidx].astype(np.float64) ** 2).sum())
            ch = int(adc[b:e][gidx].astype(np.int64).sum())
            if q2 > clus_thr * clus_thr * n2 and ch >= min_charge:
                out.append((m, int(gidx[0]), int(gidx[-1]), ch, float((adc[b:e][gidx].astype(np.float64) * (gidx + 0.5)).sum() / ch)))
    return out


def test_equals_brute_force_on_random_modules():
    for seed, kw in ((1, {}), (2, dict(max_holes=1, max_bad=0)), (3, dict(max_holes=2, max_bad=2, min_charge=0)), (4, dict(clus_thr=8.0))):
        d = datagen.make_strips(seed, 300, strips_per_module=128, occupancy=0.05, bad_frac=0.05)
        prm = datagen.default_strip_params(**kw)
        r = mkfo.cluster_strips(d["module_off"], d["adc"], d["noise"], d["bad"], **prm)
        ref = brute_force(d["module_off"], d["adc"], d["noise"], d["bad"], **prm)
        assert len(ref) > 200
        got = list(zip(r["module"].tolist(), r["first"].tolist(), r["last"].tolist(), r["charge"].tolist()))
        assert got == [t[:4] for t in ref]
        assert np.allclose(r["bary"], [t[4] for t in ref], rtol=1e-6)
        # invariants: ordered, disjoint, inside the module, no bad strip at either end
        key = r["module"].astype(np.int64) * 10000 + r["first"]
        assert np.all(np.diff(key) > 0) and np.all(r["last"] >= r["first"])
        assert np.all(r["bary"] > r["first"]) and np.all(r["bary"] < r["last"] + 1)
