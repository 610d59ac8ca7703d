"""Pins for the oracle's helix propagation and Jacobian (C1-C4, U5, U6). CPU only."""
import math
import os

import numpy as np
import pytest

from oracle import mkfo

KAPPA = 0.0029979246
BZ = 3.8
GOLD = os.path.join(os.path.dirname(__file__), "golden")


def rand_state(rng, r0max=60.0, ptmin=0.3, ptmax=20.0):
    r0 = rng.uniform(0.0, r0max)
    a0 = rng.uniform(-np.pi, np.pi)
    pt = ptmin * (ptmax / ptmin) ** rng.random()
    # mostly outward-going
    phi = a0 + rng.uniform(-1.0, 1.0)
    eta = rng.uniform(-1.5, 1.5)
    return np.array([r0 * np.cos(a0), r0 * np.sin(a0), rng.uniform(-20, 20), 1.0 / pt, phi,
                     2 * np.arctan(np.exp(-eta))]), int(rng.choice([-1, 1]))


def rk4_path(u, q, s, n=2000):
    """Brute force: integrate dx/ds=cos phi, dy/ds=sin phi, dz/ds=cot theta, dphi/ds=omega (Lorentz force)."""
    w = -q * KAPPA * BZ * u[3]
    y = np.array([u[0], u[1], u[2], u[4]])
    f = lambda v: np.array([np.cos(v[3]), np.sin(v[3]), 1.0 / np.tan(u[5]), w])
    h = s / n
    for _ in range(n):
        k1 = f(y); k2 = f(y + 0.5 * h * k1); k3 = f(y + 0.5 * h * k2); k4 = f(y + h * k3)
        y = y + h / 6 * (k1 + 2 * k2 + 2 * k3 + k4)
    return y


def test_lorentz_sign_and_radius():
    """q=+1 in +Bz turns clockwise (F = q v x B); radius = pT/(kappa Bz) — golden/radius.txt."""
    pt, bz, rho = np.loadtxt(os.path.join(GOLD, "radius.txt"))
    u = np.array([0, 0, 0, 1.0 / pt, 0.0, np.pi / 2])
    u1 = mkfo.helix_step(bz, +1, u, 0.5 * np.pi * rho)        # quarter turn
    assert abs(u1[0] - rho) < 2e-4 and abs(u1[1] + rho) < 2e-4  # ends at (rho, -rho): clockwise
    assert abs(u1[4] + np.pi / 2) < 2e-6                             # rho in the file has 4 decimals
    u1 = mkfo.helix_step(bz, -1, u, 0.5 * np.pi * rho)
    assert abs(u1[0] - rho) < 2e-4 and abs(u1[1] - rho) < 2e-4  # negative charge: counter-clockwise


def test_helix_step_matches_numerical_integration():
    rng = np.random.default_rng(1)
    for _ in range(20):
        u, q = rand_state(rng)
        s = rng.uniform(1, 40)
        u1 = mkfo.helix_step(BZ, q, u, s)
        y = rk4_path(u, q, s)
        assert np.allclose([u1[0], u1[1], u1[2], u1[4]], y, atol=1e-8)
        assert u1[3] == u[3] and u1[5] == u[5]


def test_propagate_to_r_lands_on_cylinder_first_outward_crossing():
    rng = np.random.default_rng(2)
    n_ok = 0
    for _ in range(3000):
        u, q = rand_state(rng)
        r0 = math.hypot(u[0], u[1])
        R = r0 + rng.uniform(0.5, 40)
        rc, u1, F, C1, s = mkfo.propagate(0, R, BZ, q, u)
        if rc:
            continue
        n_ok += 1
        assert abs(math.hypot(u1[0], u1[1]) - R) < 1e-9 * R
        assert s > 0 and abs(-q * KAPPA * BZ * u[3] * s) < np.pi
        assert u1[0] * np.cos(u1[4]) + u1[1] * np.sin(u1[4]) >= 0          # outward
        # the point is ON the helix through u (C1) ...
        assert np.allclose(u1, mkfo.helix_step(BZ, q, u, s), atol=1e-10)
        # ... and it is the FIRST crossing: radius stays below R on the way (sampled)
        for f in (0.1, 0.3, 0.5, 0.7, 0.9, 0.99):
            um = mkfo.helix_step(BZ, q, u, f * s)
            assert math.hypot(um[0], um[1]) < R
    assert n_ok > 2000


def test_propagate_to_r_second_algebraic_form():
    """Independent derivation (chord/tan-half-angle quadratic): G lam^2 + 2 A lam - D = 0, s = lam atan(tau)/tau."""
    rng = np.random.default_rng(3)
    worst = 0.0
    for _ in range(5000):
        u, q = rand_state(rng, ptmin=0.2, ptmax=50)
        r0 = math.hypot(u[0], u[1])
        R = r0 + rng.uniform(0.1, 40)
        rc, u1, F, C1, s = mkfo.propagate(0, R, BZ, q, u)
        w = -q * KAPPA * BZ * u[3]
        cp, sp = np.cos(u[4]), np.sin(u[4])
        A = u[0] * cp + u[1] * sp; B = u[1] * cp - u[0] * sp; D = R * R - r0 * r0
        G = 1 + w * B - D * w * w / 4
        disc = A * A + D * G
        reach = disc >= 0 and A + math.sqrt(max(disc, 0)) > 0
        if reach:
            lam = D / (A + math.sqrt(disc)); tau = w * lam / 2
            s2 = lam * math.atan(tau) / tau
        assert (rc == 0) == bool(reach), (u, q, R)
        if rc == 0:
            worst = max(worst, abs(s - s2) / s)
    assert worst < 1e-9


def test_straight_line_limit():
    rng = np.random.default_rng(4)
    for _ in range(200):
        u, q = rand_state(rng)
        u[3] = 1e-7                                                   # pT = 1e7 GeV
        r0 = math.hypot(u[0], u[1]); R = r0 + rng.uniform(1, 40)
        rc, u1, *_ , s = mkfo.propagate(0, R, BZ, q, u)
        assert rc == 0
        A = u[0] * np.cos(u[4]) + u[1] * np.sin(u[4]); D = R * R - r0 * r0
        s_line = -A + math.sqrt(A * A + D)
        assert abs(s - s_line) < 1e-6 * s_line                      # sagitta at pT=1e7 GeV is O(1e-8) relative
        assert np.allclose(u1[:2], u[:2] + s_line * np.array([np.cos(u[4]), np.sin(u[4])]), atol=1e-6)
        assert abs(u1[2] - (u[2] + s_line / np.tan(u[5]))) < 1e-6 * max(1, abs(u1[2]))


def test_composition():
    rng = np.random.default_rng(5)
    for _ in range(300):
        u, q = rand_state(rng, r0max=20)
        r0 = math.hypot(u[0], u[1])
        rc1, ua, *_ = mkfo.propagate(0, r0 + 10, BZ, q, u)
        rc2, ub, *_ = mkfo.propagate(0, r0 + 25, BZ, q, u)
        if rc1 or rc2:
            continue
        rc3, uc, *_ = mkfo.propagate(0, r0 + 25, BZ, q, ua)
        assert rc3 == 0 and np.allclose(ub, uc, atol=1e-9)
        # barrel then disk then the same disk directly
        Z = ub[2] + (5 if ub[5] < np.pi / 2 else -5)
        rc4, ud, *_ = mkfo.propagate(1, Z, BZ, q, ub)
        rc5, ue, *_ = mkfo.propagate(1, Z, BZ, q, u)
        if rc4 == 0 and rc5 == 0:
            assert np.allclose(ud, ue, atol=1e-9)


def test_propagate_to_z_exact_plane():
    rng = np.random.default_rng(6)
    for k in range(400):
        u, q = rand_state(rng)
        fwd = u[5] < np.pi / 2
        Z = u[2] + (1 if fwd else -1) * rng.uniform(1, 60)
        rc, u1, F, C1, s = mkfo.propagate(1, Z, BZ, q, u)
        if rc:
            assert abs(KAPPA * BZ * u[3] * (Z - u[2]) * np.tan(u[5])) >= np.pi
            continue
        assert u1[2] == pytest.approx(Z, abs=1e-12)
        assert s == pytest.approx((Z - u[2]) * np.tan(u[5]), rel=1e-14)
        if k < 40:
            y = rk4_path(u, q, s)
            assert np.allclose([u1[0], u1[1], u1[2], u1[4]], y, atol=1e-8)
    # backward is unreachable
    u = np.array([1.0, 0, 10.0, 1.0, 0.0, 1.0])
    assert mkfo.propagate(1, 5.0, BZ, 1, u)[0] == 1


def test_loopers_and_unreachable():
    # pT = 0.1 GeV: rho = 8.78 cm, from the origin the helix never reaches r = 20
    u = np.array([0, 0, 0, 10.0, 0.3, 1.2])
    assert mkfo.propagate(0, 20.0, BZ, 1, u)[0] == 1
    # reaches r = 17.5 only after more than half a turn? from origin max r = 2 rho = 17.56 at exactly half turn
    rc, u1, *_ , s = mkfo.propagate(0, 17.0, BZ, 1, u)
    assert rc == 0 and abs(KAPPA * BZ * 10.0 * s) < np.pi
    # inward-pointing start at (15,0): circle centre (15, 8.78), exit through r = 15.5 after ~120 deg (reachable),
    # exit through r = 26 (max reach 26.16) only after ~230 deg of turning -> unreachable (U6)
    u = np.array([15.0, 0, 0, 10.0, np.pi, 1.2])
    rc, u1, *_, s = mkfo.propagate(0, 15.5, BZ, 1, u)
    assert rc == 0 and np.pi / 2 < abs(KAPPA * BZ * 10.0 * s) < np.pi
    assert mkfo.propagate(0, 26.0, BZ, 1, u)[0] == 1


def test_start_on_surface_gives_zero_step_not_full_turn():
    """U5: propagating to the radius the state already sits on must give s ~ 0, not a spurious turn."""
    rng = np.random.default_rng(7)
    for _ in range(200):
        u, q = rand_state(rng)
        r0 = math.hypot(u[0], u[1])
        if u[0] * np.cos(u[4]) + u[1] * np.sin(u[4]) <= 0.1 * r0:
            continue
        for R in (r0, r0 * (1 - 1e-7), r0 * (1 + 1e-7), float(np.float32(r0))):
            rc, u1, F, C1, s = mkfo.propagate(0, R, BZ, q, u)
            assert rc == 0 and abs(s) < 1e-3
            assert np.allclose(u1, u, atol=1e-3)


@pytest.mark.parametrize("kind", [0, 1])
def test_jacobian_vs_central_differences_and_null_vector(kind):
    rng = np.random.default_rng(8 + kind)
    worst = 0.0
    n = 0
    while n < 200:
        u, q = rand_state(rng)
        if kind == 0:
            pos = math.hypot(u[0], u[1]) + rng.uniform(1, 30)
        else:
            if abs(np.pi / 2 - u[5]) < 0.3:
                continue
            pos = u[2] + (1 if u[5] < np.pi / 2 else -1) * rng.uniform(2, 40)
        rc, u1, F, C1, s = mkfo.propagate(kind, pos, BZ, q, u, np.eye(6))
        if rc:
            continue
        if kind == 0 and (u1[0] * np.cos(u1[4]) + u1[1] * np.sin(u1[4])) / pos < 0.3:
            continue
        n += 1
        Ffd = np.zeros((6, 6))
        for j in range(6):
            h = 1e-6 * max(1.0, abs(u[j]))
            up, um = u.copy(), u.copy()
            up[j] += h; um[j] -= h
            Ffd[:, j] = (mkfo.propagate(kind, pos, BZ, q, up)[1] - mkfo.propagate(kind, pos, BZ, q, um)[1]) / (2 * h)
        worst = max(worst, np.max(np.abs(F - Ffd) / (1 + np.abs(Ffd))))
        nvec = np.array([u1[0], u1[1], 0, 0, 0, 0]) if kind == 0 else np.array([0, 0, 1.0, 0, 0, 0])
        assert np.max(np.abs(nvec @ F)) < 1e-9 * max(1.0, np.max(np.abs(F))) * np.linalg.norm(nvec)
        # C1 = F C F^T with C = I
        assert np.allclose(C1, F @ F.T, rtol=1e-12, atol=1e-12)
    assert worst < 5e-6


def test_covariance_transport_is_congruence():
    rng = np.random.default_rng(11)
    u, q = rand_state(rng)
    M = rng.standard_normal((6, 6)); C = M @ M.T * 1e-4
    rc, u1, F, C1, s = mkfo.propagate(0, math.hypot(u[0], u[1]) + 10, BZ, q, u, C)
    assert rc == 0
    assert np.allclose(C1, F @ C @ F.T, rtol=1e-12, atol=1e-18)
    assert np.allclose(C1, C1.T)
