"""Pins for the oracle's material terms (C5) and chi2 / Kalman update (C6). CPU only."""
import math
import os

import numpy as np

from oracle import mkfo

GOLD = os.path.join(os.path.dirname(__file__), "golden")
M_PI = 0.13957039


def test_highland_golden():
    for p, t, th0 in np.loadtxt(os.path.join(GOLD, "highland.txt"), ndmin=2):
        assert abs(mkfo.highland(p, t) - th0) < 1e-4 * th0 + 5e-8


def test_bethe_bloch_minimum_golden():
    vmin, bg_at, pdg = np.loadtxt(os.path.join(GOLD, "bethe_minimum.txt"))
    bgs = np.linspace(1.5, 6.0, 451)
    vals = np.array([mkfo.dedx(bg * M_PI) for bg in bgs]) / 2.329 * 1e3      # MeV cm^2/g
    i = int(np.argmin(vals))
    assert abs(vals[i] - vmin) < 2e-3
    assert abs(bgs[i] - bg_at) < 0.15
    assert abs(vals[i] - pdg) / pdg < 0.03                                       # sanity vs tabulated (with delta)
    # 1/beta^2 rise at low momentum and logarithmic rise at high momentum
    assert mkfo.dedx(0.1) > 2 * mkfo.dedx(0.45) and mkfo.dedx(100.0) > 1.2 * mkfo.dedx(0.45)


def state_on_barrel(rng, R=20.0):
    a0 = rng.uniform(-np.pi, np.pi)
    return np.array([R * np.cos(a0), R * np.sin(a0), rng.uniform(-10, 10), 1.0 / rng.uniform(0.4, 5), a0 + rng.uniform(-0.8, 0.8),
                     rng.uniform(0.7, 2.4)])


def test_material_energy_loss_and_jacobian():
    rng = np.random.default_rng(0)
    for kind in (0, 1):
        for _ in range(50):
            u = state_on_barrel(rng)
            C = np.diag([1e-4, 1e-4, 1e-4, 1e-2, 1e-4, 1e-4])
            C[3, 4] = C[4, 3] = 3e-4
            rc, u1, C1, th0, dE = mkfo.material(kind, 0.03, 2, u, C)              # dE/dx only
            assert rc == 0 and th0 == 0.0
            st = np.sin(u[5])
            p = 1 / (u[3] * st); E = math.hypot(p, M_PI)
            if kind == 0:
                pn = abs(st * (u[0] * np.cos(u[4]) + u[1] * np.sin(u[4])) / 20.0)
            else:
                pn = abs(np.cos(u[5]))
            assert abs(dE - mkfo.dedx(p) * (0.03 / pn) * 9.37) < 1e-15
            p1 = 1 / (u1[3] * st)
            assert abs(math.hypot(p1, M_PI) - (E - dE)) < 1e-12                     # energy bookkeeping
            assert u1[3] > u[3] and np.all(u1[[0, 1, 2, 4, 5]] == u[[0, 1, 2, 4, 5]])
            # J33 against the finite-difference derivative of ipt' wrt ipt (dropped term is O(dE/E))
            h = 1e-6 * u[3]
            up, um = u.copy(), u.copy(); up[3] += h; um[3] -= h
            Jfd = (mkfo.material(kind, 0.03, 2, up, C)[1][3] - mkfo.material(kind, 0.03, 2, um, C)[1][3]) / (2 * h)
            J = C1[3, 3] / C[3, 3]
            assert abs(math.sqrt(J) - Jfd) < 3 * dE / E * Jfd + 1e-9
            assert np.isclose(C1[3, 4], C[3, 4] * math.sqrt(J)) and C1[4, 4] == C[4, 4]
            assert np.allclose(C1, C1.T)


def test_multiple_scattering_Q_matches_monte_carlo():
    """Q (incl. the ipt-theta correlation) equals the sample covariance of a direction kick by two independent
    N(0,theta0) angles at fixed |p| (C5)."""
    rng = np.random.default_rng(1)
    u = np.array([20.0, 0.0, 3.0, 1.25, 0.2, 0.9])
    C = np.zeros((6, 6))
    rc, u1, C1, th0, dE = mkfo.material(0, 0.02, 1, u, C)                         # MS only
    assert rc == 0 and dE == 0 and np.all(u1 == u)
    p = 1 / (u[3] * np.sin(u[5]))
    pn = abs(np.sin(u[5]) * np.cos(u[4]))
    assert abs(th0 - mkfo.highland(p, 0.02 / pn)) < 1e-15
    n = 400000
    al, be = rng.standard_normal(n) * th0, rng.standard_normal(n) * th0
    th = u[5] + al; ph = u[4] + be / np.sin(u[5]); ipt = 1 / (p * np.sin(th))
    S = np.cov(np.stack([ipt, ph, th]))
    Q = C1[3:, 3:]
    assert np.allclose(np.diag(S), np.diag(Q), rtol=0.01)
    assert abs(S[0, 2] - Q[0, 2]) < 0.01 * abs(Q[0, 2]) and Q[0, 2] < 0        # cot(theta)>0: anti-correlated
    assert abs(Q[0, 1]) == 0 and abs(Q[1, 2]) == 0
    assert np.all(C1[:3, :] == 0)                                                # no position noise


def test_material_stops_when_energy_exhausted():
    u = np.array([20.0, 0.0, 0.0, 1 / 0.02, 0.0, np.pi / 2])                      # p = 20 MeV
    rc = mkfo.material(0, 0.5, 3, u, np.eye(6) * 1e-4)[0]
    assert rc == 16


def rand_spd(rng, n, scale):
    M = rng.standard_normal((n, n))
    return (M @ M.T + n * np.eye(n)) * scale


def V6_to_mat(V6):
    return np.array([[V6[0], V6[1], V6[3]], [V6[1], V6[2], V6[4]], [V6[3], V6[4], V6[5]]])


def test_update_equals_information_form_and_gain_form():
    rng = np.random.default_rng(2)
    H = np.hstack([np.eye(3), np.zeros((3, 3))])
    for _ in range(100):
        C = rand_spd(rng, 6, 1e-3)
        Vm = rand_spd(rng, 3, 1e-4)
        V6 = np.array([Vm[0, 0], Vm[1, 0], Vm[1, 1], Vm[2, 0], Vm[2, 1], Vm[2, 2]])
        u = rng.standard_normal(6)
        m = u[:3] + rng.standard_normal(3) * 0.05
        rc, u1, C1, c2 = mkfo.update(u, C, m, V6)
        assert rc == 0
        Ci = np.linalg.inv(C); Vi = np.linalg.inv(Vm)
        C_info = np.linalg.inv(Ci + H.T @ Vi @ H)
        u_info = C_info @ (Ci @ u + H.T @ Vi @ m)
        assert np.allclose(C1, C_info, rtol=1e-9, atol=1e-15)
        assert np.allclose(u1, u_info, rtol=1e-9, atol=1e-12)
        S = C[:3, :3] + Vm
        K = C[:, :3] @ np.linalg.inv(S)
        assert np.allclose(C1, C - K @ H @ C, rtol=1e-9, atol=1e-15)           # gain form == Joseph form in fp64
        r = m - u[:3]
        assert np.isclose(c2, r @ np.linalg.solve(S, r), rtol=1e-11)
        assert np.isclose(mkfo.chi2(u, C, m, V6)[1], c2, rtol=1e-14)
        # filtered residual chi2 identity: chi2 = r'^T V^-1 r' + (u1-u)^T C^-1 (u1-u)
        rp = m - u1[:3]
        assert np.isclose(c2, rp @ Vi @ rp + (u1 - u) @ Ci @ (u1 - u), rtol=1e-8)
        assert np.allclose(C1, C1.T) and np.all(np.linalg.eigvalsh(C1) > 0)


def test_update_rejects_non_positive_definite_S():
    C = -np.eye(6)
    rc, *_ = mkfo.update(np.zeros(6), C, np.zeros(3), np.array([0.5, 0, 0.5, 0, 0, 0.5]))
    assert rc == 4
