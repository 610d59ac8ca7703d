"""Pins for the oracle fit (C7): pulls ~ N(0,1), chi2 ~ chi2(2n-5), PSD covariance (U2), straight-line least squares."""
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


def test_pulls_and_chi2_on_config0(small_fit_event):
    ev, prm = small_fit_event
    s = ev["seeds"]
    o = mkfo.Oracle(ev["geom"], prm)
    r = o.fit(ev["hits"], s["par"], s["cov"], s["q"], s["plan"], s["track_hits"])
    n = s["par"].shape[1]
    assert n >= 1900
    tr = ev["truth"]
    pid = s["particle"]
    good = (r["status"] == 0) & (r["nfit"] == 10) & (s["q"] == tr["q"][pid])
    assert good.mean() > 0.995
    N = good.sum()
    # total chi2 ~ chi2(2n-5) (U3): mean 15, variance 30
    c2 = r["chi2"][good]
    assert abs(c2.mean() - 15.0) < 4 * np.sqrt(30.0 / N)
    assert abs(c2.var() - 30.0) < 6.0
    fs = tr["final_state"][:, pid]
    P, Cv = r["par"], r["cov"]
    R = np.hypot(P[0], P[1])
    assert np.allclose(R[good], 40.0, atol=1e-6)                                # state sits on the last layer
    tx, ty = -P[1] / R, P[0] / R
    dt = (P[0] - fs[0]) * tx + (P[1] - fs[1]) * ty
    ctt = tx * tx * Cv[cidx(0, 0)] + 2 * tx * ty * Cv[cidx(1, 0)] + ty * ty * Cv[cidx(1, 1)]
    dphi = np.angle(np.exp(1j * (P[4] - fs[4])))
    for name, d, v in [("rphi", dt, ctt), ("z", P[2] - fs[2], Cv[cidx(2, 2)]), ("ipt", P[3] - fs[3], Cv[cidx(3, 3)]),
                       ("phi", dphi, Cv[cidx(4, 4)]), ("theta", P[5] - fs[5], Cv[cidx(5, 5)])]:
        pull = (d / np.sqrt(v))[good]
        assert abs(pull.mean()) < 4 / np.sqrt(N), name
        assert abs(pull.std() - 1.0) < 4 / np.sqrt(2 * N) + 0.01, name


def test_covariance_psd_and_singular_along_normal(small_fit_event):
    """U2: symmetric, eigenvalues >= -1e-10 lmax, rank 5 (null along the surface normal), local 5x5 block PD."""
    ev, prm = small_fit_event
    s = ev["seeds"]
    o = mkfo.Oracle(ev["geom"], prm)
    sel = slice(0, 200)
    r = o.fit(ev["hits"], s["par"][:, sel], s["cov"][:, sel], s["q"][sel], s["plan"][sel], s["track_hits"][:, sel])
    for i in range(200):
        if r["status"][i]:
            continue
        C = unpack(r["cov"][:, i])
        w = np.linalg.eigvalsh(C)
        assert w[0] >= -1e-10 * w[-1]
        x, y = r["par"][0, i], r["par"][1, i]
        rr = np.hypot(x, y)
        T = np.zeros((5, 6))
        T[0, 0], T[0, 1] = -y / rr, x / rr
        T[1, 2] = T[2, 3] = T[3, 4] = T[4, 5] = 1
        np.linalg.cholesky(T @ C @ T.T)                                          # raises if not PD


def test_straight_track_fit_equals_weighted_least_squares():
    """Bz -> 0, no material: the filter over all hits with a very weak prior must reproduce the linear weighted
    least-squares straight-line fit (r-z plane: z = z0 + cot(theta) * r, exact for a track from the axis)."""
    rng = np.random.default_rng(5)
    g = datagen.geometry_barrel(8, 5.0, 40.0, 200.0, 0.0, bz=1e-9)
    prm = datagen.default_params(material_flags=0)
    radii = np.array([l["pos"] for l in g["layers"]])
    n = 50
    phi0 = rng.uniform(-np.pi, np.pi, n); cot = rng.uniform(-1, 1, n); z0 = rng.uniform(-5, 5, n)
    sz = 0.002
    zs = z0[None] + cot[None] * radii[:, None] + rng.standard_normal((8, n)) * sz
    hx = (radii[:, None] * np.cos(phi0)[None]).astype(np.float32)
    hy = (radii[:, None] * np.sin(phi0)[None]).astype(np.float32)
    hz = zs.astype(np.float32)
    V = np.zeros((6, 8 * n), np.float32); V[0] = V[2] = 0.003 ** 2; V[5] = sz ** 2
    hits = dict(n_events=1, layer_off=np.arange(9, dtype=np.int32) * n, x=hx.reshape(-1), y=hy.reshape(-1),
                z=hz.reshape(-1), V=V)
    th = (np.arange(8)[:, None] * n + np.arange(n)[None]).astype(np.int32)
    par = np.stack([hx[0], hy[0], hz[0], np.full(n, 1.0), phi0, np.full(n, np.pi / 2)]).astype(np.float32)
    cov = np.zeros((21, n), np.float32)
    for k, v in zip([0, 2, 5, 9, 14, 20], [1.0, 1.0, 1e4, 1.0, 1.0, 1e2]):
        cov[k] = v
    o = mkfo.Oracle(g, prm)
    # the filter linearises z1 = z0 + s cot(theta) about its current theta, which starts far off (pi/2): iterate
    # the linearisation point (error squares each pass) before comparing with the *linear* least squares
    par2 = par.copy()
    for _ in range(5):
        r = o.fit(hits, par2, cov, np.ones(n, np.int8), np.zeros(n, np.int8), th)
        par2[5] = r["par"][5]
    assert np.all(r["status"] == 0) and np.all(r["nfit"] == 8)
    A = np.stack([np.ones(8), radii], 1)
    for i in range(n):
        coef, *_ = np.linalg.lstsq(A, hz[:, i].astype(float), rcond=None)
        cot_fit = 1 / np.tan(r["par"][5, i])
        assert abs(cot_fit - coef[1]) < 3e-6                                    # 0.05 sigma of the slope
        assert abs(r["par"][2, i] - (coef[0] + coef[1] * 40.0)) < 4e-5          # z at the last layer
        # variance of the slope: sigma^2 / sum (r - rbar)^2, mapped to theta
        var_cot = sz ** 2 / np.sum((radii - radii.mean()) ** 2)
        var_th = var_cot * np.sin(r["par"][5, i]) ** 4
        assert abs(r["cov"][20, i] - var_th) < 0.02 * var_th
