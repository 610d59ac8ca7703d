"""Pins for SURVEY f4's two remaining items: energy-loss straggling (reading R12) and the non-uniform field hook
(reading R13). Hit masking (R9) has its own file."""
import os

import numpy as np

from oracle import mkfo
from workloads import datagen

GOLD = os.path.join(os.path.dirname(__file__), "golden")
M_PI = 0.13957039


def cidx(i, j):
    return i * (i + 1) // 2 + j if j <= i else j * (j + 1) // 2 + i


def test_straggling_variance_golden_and_scaling():
    for p, t, v in np.loadtxt(os.path.join(GOLD, "straggling.txt"), ndmin=2):
        assert abs(mkfo.straggling_var(p, t) - v) < 2e-4 * v
    # linear in the thickness; ~ 1/beta^2 (1 - beta^2/2) Tmax: grows towards low momentum per unit of Tmax
    assert abs(mkfo.straggling_var(1.0, 0.04) / mkfo.straggling_var(1.0, 0.02) - 2.0) < 1e-12
    assert mkfo.straggling_var(0.3, 0.02) < mkfo.straggling_var(3.0, 0.02)       # Tmax ~ (beta gamma)^2 wins


def test_material_with_straggling_adds_exactly_the_ipt_term():
    """flags 7 against flags 3 on one state: the same state, the same covariance except C[ipt, ipt], which grows by
    (ipt1 E1 / p1^2)^2 sigma_E^2 (a shift dE of the energy at fixed direction moves ipt by ipt1 E1 / p1^2 dE)."""
    rng = np.random.default_rng(3)
    for kind, pos in ((0, 30.0), (1, 55.0)):
        for _ in range(20):
            th = rng.uniform(0.6, 1.2); phi = rng.uniform(-3, 3); ipt = rng.choice([-1, 1]) / rng.uniform(0.4, 5.0)
            if kind == 0:
                u = np.array([pos * np.cos(phi), pos * np.sin(phi), 3.0, ipt, phi + rng.uniform(-0.3, 0.3), th])
            else:
                u = np.array([10 * np.cos(phi), 10 * np.sin(phi), pos, ipt, phi, th])
            A = rng.standard_normal((6, 6)) * 1e-3
            Cm = A @ A.T
            rc3, u3, C3, th0, dE = mkfo.material(kind, 0.03, 3, u, Cm)
            rc7, u7, C7, _, _ = mkfo.material(kind, 0.03, 7, u, Cm)
            assert rc3 == 0 and rc7 == 0 and np.array_equal(u3, u7)
            D = C7 - C3
            st = np.sin(th)
            pn = abs(st * (u[0] * np.cos(u[4]) + u[1] * np.sin(u[4])) / np.hypot(u[0], u[1])) if kind == 0 else abs(np.cos(th))
            t = 0.03 / pn
            p = 1 / (abs(ipt) * st)
            E1 = np.sqrt(p * p + M_PI ** 2) - dE
            p1 = np.sqrt(E1 * E1 - M_PI ** 2)
            want = (u3[3] * E1 / p1 ** 2) ** 2 * mkfo.straggling_var(p, t)
            assert abs(D[3, 3] - want) < 1e-9 * want
            D[3, 3] = 0
            assert np.abs(D).max() == 0
    # the same term on the way back (R7): flags 7 vs 3 with dir = -1 differ in C[ipt, ipt] only, and by a positive amount
    rc3, u3, C3, _, _ = mkfo.material_dir(0, 0.03, 3, -1, u * 0 + np.array([30.0, 0, 3, 0.8, 0.1, 1.0]), np.eye(6) * 1e-6)
    rc7, u7, C7, _, _ = mkfo.material_dir(0, 0.03, 7, -1, np.array([30.0, 0, 3, 0.8, 0.1, 1.0]), np.eye(6) * 1e-6)
    D = C7 - C3
    assert D[3, 3] > 0 and np.count_nonzero(D) == 1 and np.array_equal(u3, u7)


def _low_momentum_event(straggle, scatter, seed=4, n=6000):
    """Soft pions (0.25-0.6 GeV) through 12 thick layers (x/X0 = 0.05): the regime where straggling matters."""
    g = datagen.geometry_barrel(12, 4.0, 48.0, 150.0, 0.05)
    return datagen.make_events(g, seed, 1, n, pt_range=(0.25, 0.6), eta_max=0.5, straggle=straggle, scatter=scatter, shuffle=False)


def _ipt_pull(ev, flags):
    prm = datagen.default_params(material_flags=flags)
    s = ev["seeds"]
    r = mkfo.Oracle(ev["geom"], prm).fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    tr = ev["truth"]
    pid = s["particle"]
    nlay = (s["track_hits"] >= 0).sum(0)
    good = (r["status"] == 0) & (r["nfit"] == nlay) & (nlay >= 8) & (s["q"] == tr["q"][pid])
    fs = tr["final_state"][:, pid]
    pull = ((r["par"][3] - fs[3]) / np.sqrt(r["cov"][cidx(3, 3)]))[good]
    return pull, good.sum()


def test_straggling_pulls_on_a_straggling_truth():
    """Truth whose energy loss fluctuates as a Gaussian of the R12 width. Without scattering in the truth the curvature
    error is set by the measurement and by those fluctuations alone: the filter with flag 4 has unit ipt pulls, the
    filter without it is off by an order of magnitude; on a truth without fluctuations it is the other way round. With
    scattering on (the usual workload) the term is a small correction and the pulls stay unit."""
    ev = _low_momentum_event(True, False)
    pull6, n6 = _ipt_pull(ev, 2 | 4)
    pull2, _ = _ipt_pull(ev, 2)
    assert n6 > 5000
    assert abs(pull6.std() - 1.0) < 0.04 and abs(pull6.mean()) < 0.05
    assert pull2.std() > 5.0
    ev0 = _low_momentum_event(False, False)
    pull2b, _ = _ipt_pull(ev0, 2)
    pull6b, _ = _ipt_pull(ev0, 2 | 4)
    assert abs(pull2b.std() - 1.0) < 0.12 and pull6b.std() < 0.6
    ev_ms = _low_momentum_event(True, True)
    pull7, n7 = _ipt_pull(ev_ms, 7)
    assert n7 > 5000 and abs(pull7.std() - 1.0) < 0.05 and abs(pull7.mean()) < 0.06


def test_field_hook_uniform_is_identical_and_radius_follows_the_layer_field():
    ev, prm = datagen.config(0, scale=0.05)
    s = ev["seeds"]
    g = ev["geom"]
    r0 = mkfo.Oracle(g, prm).fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    g1 = dict(g, bz_layer=np.full(len(g["layers"]), g["bz"], np.float32))
    r1 = mkfo.Oracle(g1, prm).fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    for k in ("par", "cov", "chi2"):
        assert np.array_equal(r0[k], r1[k]), k
    # closed form: one propagation step from layer 3 to layer 4 turns the momentum by w s with w = -q kappa Bz_4 ipt
    bzl = np.linspace(3.8, 2.0, len(g["layers"])).astype(np.float32)
    o2 = mkfo.Oracle(dict(g, bz_layer=bzl), datagen.default_params(material_flags=0))
    par = np.array([[16.0], [0.0], [1.0], [0.5], [0.2], [1.3]], np.float32)
    cov = np.zeros((21, 1), np.float32); cov[[0, 2, 5, 9, 14, 20]] = 1e-4
    x4 = 20.0 * np.cos(0.05); y4 = 20.0 * np.sin(0.05)
    hits = dict(n_events=1, layer_off=np.array([0, 0, 0, 0, 0, 1] + [1] * 6, np.int32), x=np.array([x4], np.float32),
                y=np.array([y4], np.float32), z=np.array([2.0], np.float32), V=np.full((6, 1), 0, np.float32))
    hits["V"][[0, 2, 5]] = 1e6                                                   # a hit that pulls nothing
    th = np.full((10, 1), -1, np.int32); th[4, 0] = 0
    r = o2.fit(hits, par, cov, np.array([1], np.int8), np.zeros(1, np.int8), th)
    assert r["nfit"][0] == 1
    rc, u1, F, C1, sp = mkfo.propagate(0, 20.0, float(bzl[4]), 1, par[:, 0].astype(np.float64))
    assert rc == 0 and abs((r["par"][4, 0] - 0.2) - (-0.0029979246 * float(bzl[4]) * 0.5 * sp)) < 1e-7
    rc, u0, F, C1, sp0 = mkfo.propagate(0, 20.0, 3.8, 1, par[:, 0].astype(np.float64))
    assert abs(u0[4] - u1[4]) > 1e-3                                             # and the global field would have turned it differently


def test_field_hook_pulls_on_a_truth_in_the_same_field():
    """Truth stepped in the layer-wise field, filter in the same field: unit pulls; filter in the uniform field: biased."""
    g = datagen.geometry_barrel(10, 4.0, 40.0, 100.0, 0.02)
    g["bz_layer"] = np.linspace(3.8, 2.6, 10).astype(np.float32)
    ev = datagen.make_events(g, 9, 1, 4000, shuffle=False)
    s = ev["seeds"]
    prm = datagen.default_params()
    tr = ev["truth"]; pid = s["particle"]
    fs = tr["final_state"][:, pid]

    def pull(geom):
        r = mkfo.Oracle(geom, prm).fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
        good = (r["status"] == 0) & (r["nfit"] == 10) & (s["q"] == tr["q"][pid])
        return ((r["par"][3] - fs[3]) / np.sqrt(r["cov"][cidx(3, 3)]))[good]
    p_ok = pull(g)
    assert len(p_ok) > 3000 and abs(p_ok.std() - 1.0) < 0.05 and abs(p_ok.mean()) < 0.08
    g_uniform = {k: v for k, v in g.items() if k != "bz_layer"}
    p_bad = pull(g_uniform)
    assert abs(p_bad.mean()) > 0.5 or p_bad.std() > 1.3
