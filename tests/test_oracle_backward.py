"""Pins for the oracle's backward propagation, reverse material and backward fit (reading R7)."""
import numpy as np

from oracle import mkfo
from workloads import datagen, parity

BZ = 3.8


def test_backward_propagation_inverts_forward_propagation():
    rng = np.random.default_rng(2)
    for trial in range(200):
        kind = trial % 2
        pt = 0.6 + 5 * rng.random(); q = 1 if rng.random() < 0.5 else -1
        phi_pos = rng.uniform(-np.pi, np.pi)
        if kind == 0:
            r0, R = 20.0, 27.0
            u = np.array([r0 * np.cos(phi_pos), r0 * np.sin(phi_pos), rng.uniform(-10, 10), 1 / pt, phi_pos + rng.uniform(-0.4, 0.4),
                          rng.uniform(0.7, 2.4)])
            back = r0
        else:
            th = rng.uniform(0.3, 0.9)
            u = np.array([8 * np.cos(phi_pos), 8 * np.sin(phi_pos), 30.0, 1 / pt, phi_pos + rng.uniform(-0.4, 0.4), th])
            R, back = 38.0, 30.0
        rc, u1, F, _, s = mkfo.propagate_dir(kind, R, BZ, q, +1, u)
        assert rc == 0 and s > 0
        rc, u2, Fb, _, sb = mkfo.propagate_dir(kind, back, BZ, q, -1, u1)
        assert rc == 0 and sb < 0 and abs(sb + s) < 1e-9 * max(1, s)
        assert np.allclose(u2, u, atol=1e-9)
        # F_back F_fwd is the identity on directions tangent to the start surface
        n0 = np.array([u[0], u[1], 0, 0, 0, 0]) / np.hypot(u[0], u[1]) if kind == 0 else np.array([0, 0, 1.0, 0, 0, 0])
        Pt = np.eye(6) - np.outer(n0, n0)
        assert np.allclose(Fb @ F @ Pt, Pt, atol=1e-8)
        # a forward-only call refuses the backward target and vice versa
        assert mkfo.propagate_dir(kind, back - (3 if kind == 0 else 5), BZ, q, +1, u1)[0] != 0
        assert mkfo.propagate_dir(kind, R + 5, BZ, q, -1, u)[0] != 0


def test_reverse_material_gives_the_energy_back_and_adds_noise():
    u = np.array([30.0, 0.0, 5.0, 1 / 0.8, 0.2, 1.2])
    C0 = np.diag([1e-4, 1e-4, 1e-4, 1e-3, 1e-5, 1e-5])
    rc, u1, C1, th0, dE = mkfo.material_dir(0, 0.03, 3, +1, u, C0)
    assert rc == 0 and u1[3] > u[3] and dE > 0
    rc, u2, C2, th0b, dEb = mkfo.material_dir(0, 0.03, 3, -1, u1, C1)
    assert rc == 0 and u2[3] < u1[3]
    assert abs(u2[3] / u[3] - 1) < 2e-6                     # dE is evaluated at slightly different momenta: second order
    assert abs(dEb / dE - 1) < 2e-3 and abs(th0b / th0 - 1) < 2e-3
    # scattering noise is added both ways (variances grow monotonically); dir = +1 equals the plain call
    assert C2[4, 4] > C1[4, 4] > C0[4, 4] and C2[5, 5] > C1[5, 5] > C0[5, 5]
    rc, u1p, C1p, _, _ = mkfo.material(0, 0.03, 3, u, C0)
    assert np.array_equal(u1p, u1) and np.array_equal(C1p, C1)


def test_backward_fit_pulls_at_the_innermost_hit(small_fit_event):
    """Seeds = forward-fit states at the last hit with covariance x100; the backward fit must give unbiased
    parameters with unit pulls at the innermost layer, against the truth there BEFORE that layer's material."""
    ev, prm = small_fit_event
    s = ev["seeds"]
    g = ev["geom"]
    o = mkfo.Oracle(g, prm)
    f = o.fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    good = (f["status"] == 0) & (f["nfit"] == 10)
    b = o.fit_backward(ev["hits"], f["par"].astype(np.float32), (100.0 * f["cov"]).astype(np.float32), s["q"], s["plan"], s["track_hits"])
    tr = ev["truth"]
    pid = s["particle"]
    good &= (b["status"] == 0) & (b["nfit"] == 10) & (s["q"] == tr["q"][pid])
    assert good.mean() > 0.99
    N = good.sum()
    # truth at the first layer, before its material: the generated particle propagated from its vertex
    R0 = g["layers"][0]["pos"]
    truth = np.zeros((6, len(pid)))
    for k, i in enumerate(pid):
        u0 = np.array([tr["vx"][i], tr["vy"][i], tr["vz"][i], 1 / tr["pt"][i], tr["phi"][i], tr["theta"][i]])
        rc, u1, _, _, _ = mkfo.propagate(0, R0, g["bz"], int(tr["q"][i]), u0)
        truth[:, k] = u1 if rc == 0 else np.nan
    P, Cv = b["par"], b["cov"]
    R = np.hypot(P[0], P[1])
    assert np.nanmax(np.abs(R[good] - R0)) < 0.02
    tx, ty = -P[1] / R, P[0] / R
    dt = (P[0] - truth[0]) * tx + (P[1] - truth[1]) * ty
    ctt = tx * tx * Cv[parity.cidx(0, 0)] + 2 * tx * ty * Cv[parity.cidx(1, 0)] + ty * ty * Cv[parity.cidx(1, 1)]
    dphi = np.angle(np.exp(1j * (P[4] - truth[4])))
    for name, d, v in [("rphi", dt, ctt), ("z", P[2] - truth[2], Cv[parity.cidx(2, 2)]), ("ipt", P[3] - truth[3], Cv[parity.cidx(3, 3)]),
                       ("phi", dphi, Cv[parity.cidx(4, 4)]), ("theta", P[5] - truth[5], Cv[parity.cidx(5, 5)])]:
        pull = (d / np.sqrt(v))[good]
        assert abs(pull.mean()) < 4 / np.sqrt(N), (name, pull.mean())
        assert abs(pull.std() - 1.0) < 4 / np.sqrt(2 * N) + 0.02, (name, pull.std())
    # total chi2 ~ chi2(2n - 5) as for the forward fit (weak prior)
    c2 = b["chi2"][good]
    assert abs(c2.mean() - 15.0) < 4 * np.sqrt(30.0 / N) + 0.3
    # the backward estimate of the curvature is as precise as the forward one (same hits, same lever arm)
    rel = np.sqrt(b["cov"][parity.cidx(3, 3)][good] / f["cov"][parity.cidx(3, 3)][good])
    assert 0.8 < np.median(rel) < 1.25
