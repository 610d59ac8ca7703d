"""Pins for the two-filter smoother (reading R14): the combination step against the information-form mean,
straight tracks against the global least-squares line at every layer, unit pulls at every layer against the truth
after that layer, covariance never above either filter's."""
import numpy as np

from oracle import mkfo
from workloads import datagen


def cidx(i, j):
    return i * (i + 1) // 2 + j if j <= i else j * (j + 1) // 2 + i


def unpack(cov21):
    C = np.zeros((6, 6))
    for i in range(6):
        for j in range(6):
            C[i, j] = cov21[cidx(i, j)]
    return C


def test_combine_equals_information_form_mean():
    rng = np.random.default_rng(2)
    for kind in (0, 1):
        for _ in range(20):
            phi = rng.uniform(-3, 3)
            uf = np.array([30 * np.cos(phi), 30 * np.sin(phi), 5.0, 0.7, phi + 0.2, 1.1]) if kind == 0 else \
                np.array([9.0 * np.cos(phi), 9.0 * np.sin(phi), 40.0, 0.7, phi, 0.5])
            r = np.hypot(uf[0], uf[1])
            T = np.zeros((5, 6))
            if kind == 0:
                T[0, 0], T[0, 1], T[1, 2] = -uf[1] / r, uf[0] / r, 1.0
            else:
                T[0, 0] = T[1, 1] = 1.0
            T[2, 3] = T[3, 4] = T[4, 5] = 1.0
            A, B = rng.standard_normal((5, 5)) * 1e-2, rng.standard_normal((5, 5)) * 1e-2
            Pf, Pb = A @ A.T + 1e-6 * np.eye(5), B @ B.T + 1e-6 * np.eye(5)
            ab = rng.standard_normal(5) * 1e-2
            ub = uf + T.T @ ab
            rc, us, Cs = mkfo.smooth_combine(kind, uf, T.T @ Pf @ T, ub, T.T @ Pb @ T)
            assert rc == 0
            Wf, Wb = np.linalg.inv(Pf), np.linalg.inv(Pb)
            Ps = np.linalg.inv(Wf + Wb)
            a_s = Ps @ (Wb @ ab)                                      # forward estimate at the origin
            assert np.allclose(T @ (us - uf), a_s, rtol=1e-8, atol=1e-14)
            assert np.allclose(T @ Cs @ T.T, Ps, rtol=1e-8, atol=1e-18)
            # nothing along the normal, and never above either input
            nrm = np.array([uf[0] / r, uf[1] / r, 0, 0, 0, 0]) if kind == 0 else np.array([0, 0, 1.0, 0, 0, 0])
            assert np.abs(Cs @ nrm).max() < 1e-15
            assert np.linalg.eigvalsh(Pf - T @ Cs @ T.T).min() > -1e-12 and np.linalg.eigvalsh(Pb - T @ Cs @ T.T).min() > -1e-12
    # phi differences are taken modulo 2 pi
    uf = np.array([30.0, 0, 0, 0.5, 3.1, 1.0]); ub = uf.copy(); ub[4] = -3.1
    P = np.eye(6) * 1e-4; P[0, 0] = 0
    rc, us, Cs = mkfo.smooth_combine(0, uf, P, ub, P)
    assert abs(us[4] - (3.1 + 0.5 * (2 * np.pi - 6.2))) < 1e-12


def test_straight_tracks_smoothed_state_is_the_least_squares_line_everywhere():
    """Bz -> 0, no material, weak prior: at EVERY layer the smoothed z and its variance are those of the global weighted
    least-squares line through all hits (the forward filter alone only reaches that at the last layer)."""
    rng = np.random.default_rng(5)
    g = datagen.geometry_barrel(8, 5.0, 40.0, 200.0, 0.0, bz=1e-9)
    prm = datagen.default_params(material_flags=0)
    radii = np.array([l["pos"] for l in g["layers"]])
    n = 40
    phi0 = rng.uniform(-np.pi, np.pi, n); cot = rng.uniform(-1, 1, n); z0 = rng.uniform(-5, 5, n)
    sz = 0.002
    zs = z0[None] + cot[None] * radii[:, None] + rng.standard_normal((8, n)) * sz
    hx = (radii[:, None] * np.cos(phi0)[None]).astype(np.float32)
    hy = (radii[:, None] * np.sin(phi0)[None]).astype(np.float32)
    hz = zs.astype(np.float32)
    V = np.zeros((6, 8 * n), np.float32); V[0] = V[2] = 0.003 ** 2; V[5] = sz ** 2
    hits = dict(n_events=1, layer_off=np.arange(9, dtype=np.int32) * n, x=hx.reshape(-1), y=hy.reshape(-1), z=hz.reshape(-1), V=V)
    th = (np.arange(8)[:, None] * n + np.arange(n)[None]).astype(np.int32)
    par = np.stack([hx[0], hy[0], hz[0], np.full(n, 1.0), phi0, np.arctan2(1.0, cot)]).astype(np.float32)   # near the truth: linear regime
    cov = np.zeros((21, n), np.float32)
    for k, v in zip([0, 2, 5, 9, 14, 20], [1.0, 1.0, 1e4, 1.0, 1.0, 1e2]):
        cov[k] = v
    o = mkfo.Oracle(g, prm)
    par2 = par.copy()
    for _ in range(3):                                                # iterate the linearisation point of theta
        r = o.fit_smooth(hits, par2, cov, np.ones(n, np.int8), np.zeros(n, np.int8), th)
        par2[5] = r["par_s"][0, 5]
    assert np.all(r["status"] == 0) and np.all(r["nfit"] == 8)
    A = np.stack([np.ones(8), radii], 1)
    AtA_inv = np.linalg.inv(A.T @ A)
    for i in range(n):
        coef = AtA_inv @ A.T @ hz[:, i].astype(float)
        for l in range(8):
            zfit = coef[0] + coef[1] * radii[l]
            var = sz ** 2 * (A[l] @ AtA_inv @ A[l])
            assert abs(r["par_s"][l, 2, i] - zfit) < 0.03 * np.sqrt(var), (i, l)
            assert abs(r["cov_s"][l, cidx(2, 2), i] - var) < 0.02 * var, (i, l)


def test_smoothed_pulls_are_unit_at_every_layer_and_covariance_shrinks():
    g = datagen.geometry_barrel(10, 4.0, 40.0, 100.0, 0.02)
    ev = datagen.make_events(g, 21, 1, 5000, shuffle=False, keep_truth=True)
    prm = datagen.default_params()
    s = ev["seeds"]
    o = mkfo.Oracle(g, prm)
    r = o.fit_smooth(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    f = o.fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    assert np.array_equal(r["nfit"], f["nfit"]) and np.allclose(r["chi2"], f["chi2"])
    tr = ev["truth"]; pid = s["particle"]
    good = (r["status"] == 0) & (r["nfit"] == 10) & (s["q"] == tr["q"][pid])
    assert good.mean() > 0.99
    N = good.sum()
    ts = tr["states"][:, :, pid]                                       # (10, 6, n)
    for l in range(10):
        P, Cv = r["par_s"][l], r["cov_s"][l]
        R = np.hypot(P[0], P[1])
        assert np.abs(R[good] - g["layers"][l]["pos"]).max() < 1e-3    # stays on its layer up to the tangent-plane shift^2 / 2R
        tx, ty = -P[1] / R, P[0] / R
        dt = (P[0] - ts[l, 0]) * tx + (P[1] - ts[l, 1]) * ty
        ctt = tx * tx * Cv[cidx(0, 0)] + 2 * tx * ty * Cv[cidx(1, 0)] + ty * ty * Cv[cidx(1, 1)]
        dphi = np.angle(np.exp(1j * (P[4] - ts[l, 4])))
        for name, d, v in [("rphi", dt, ctt), ("z", P[2] - ts[l, 2], Cv[cidx(2, 2)]), ("ipt", P[3] - ts[l, 3], Cv[cidx(3, 3)]),
                           ("phi", dphi, Cv[cidx(4, 4)]), ("theta", P[5] - ts[l, 5], Cv[cidx(5, 5)])]:
            pull = (d / np.sqrt(v))[good]
            assert abs(pull.mean()) < 4.5 / np.sqrt(N), (l, name, pull.mean())
            assert abs(pull.std() - 1.0) < 4.5 / np.sqrt(2 * N) + 0.015, (l, name, pull.std())
    # at the last layer the smoothed state is the forward filter's (the backward prior carries 1e-4 of the information)
    assert np.allclose(r["par_s"][9][:, good], f["par"][:, good], rtol=0, atol=2e-3 * np.sqrt(f["cov"][[0, 2, 5, 9, 14, 20]][:, good]).max())
    assert np.allclose(r["cov_s"][9][9, good], f["cov"][9, good], rtol=2e-3)
    # sigma(ipt) of the smoothed state: the same at every layer up to the material between them, and below the forward
    # filter's at the inner layers by a large factor
    fwd_first = o.fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], np.where(np.arange(10)[:, None] < 4, s["track_hits"], -1))
    assert np.median(r["cov_s"][3][9, good] / fwd_first["cov"][9, good]) < 0.2
