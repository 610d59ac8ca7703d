"""Seeded synthetic detector events (the ONLY module shared by the CUDA path, the oracle's tests and bench.py).

It holds none of the method's arithmetic (no Kalman filter, no covariance transport, no chi2, no binning, no
selection): it is a toy detector *simulation* in numpy float64 that stands in for the paper's simulated ttbar
PU50/PU70 CMS-2017 events (PAPER.md:25,51,57 — not available here) with the shapes BASELINE.json `configs`
gives. It imports neither the CUDA binding nor oracle/.

Recipe: particles are charged pions in a uniform field Bz; truth is stepped exactly along the
helix from surface to surface in plan order; on each crossed surface a hit is made (Gaussian smearing within the
surface only), then the truth loses the mean Bethe-Bloch energy and is scattered by two independent N(0,theta0)
angles at fixed |p|. Seeds are 3-point helices through the first three hits with an inflated covariance.
All random numbers come from one numpy Generator(PCG64(seed)) in a fixed draw order.
"""
import numpy as np

KAPPA = 0.0029979246  # GeV/(T cm)
M_PION = 0.13957039
M_E = 0.51099895e-3


# ------------------------------------------------------------------------------------------------------
# geometry tables
# ------------------------------------------------------------------------------------------------------
def _barrel_layer(r, zmax, xx0, sig_t, sig_l):
    eta = float(np.arcsinh(zmax / r))
    return dict(kind=0, pos=float(r), lo=float(-zmax), hi=float(zmax), xx0=float(xx0), eta_lo=-eta, eta_hi=eta,
                sig_t=sig_t, sig_l=sig_l)


def _disk_layer(z, rlo, rhi, xx0, sig_t, sig_l):
    a, b = float(np.arcsinh(abs(z) / rhi)), float(np.arcsinh(abs(z) / rlo))
    lo, hi = (a, b) if z > 0 else (-b, -a)
    return dict(kind=1, pos=float(z), lo=float(rlo), hi=float(rhi), xx0=float(xx0), eta_lo=lo, eta_hi=hi,
                sig_t=sig_t, sig_l=sig_l)


def geometry_barrel(n_layers, r_first, r_last, zmax, xx0, bz=3.8, n_phi_bins=63, n_eta_bins=40):
    """Idealised barrel: n_layers concentric cylinders, one plan (all layers inner to outer)."""
    radii = np.linspace(r_first, r_last, n_layers)
    xx0 = np.broadcast_to(np.asarray(xx0, float), (n_layers,))
    layers = [_barrel_layer(r, zmax, x, 0.003, 0.01) for r, x in zip(radii, xx0)]
    return dict(layers=layers, bz=float(bz), n_phi_bins=n_phi_bins, n_eta_bins=n_eta_bins,
                plan_off=np.array([0, n_layers], np.int32), plan_layers=np.arange(n_layers, dtype=np.int32),
                pixel_layers=np.arange(n_layers), name="barrel%d" % n_layers)


def geometry_barrel_endcap(bz=3.8, n_phi_bins=63, n_eta_bins=40):
    """Own rounded numbers 'shaped like' a CMS-2017-type tracker: 14 barrel cylinders and
    12 disks per side = 38 layers; two nested-envelope plans (eta>=0, eta<0) of 26 layers each."""
    L = []
    idx = {}

    def add(name, lay):
        idx[name] = len(L)
        L.append(lay)

    for i, r in enumerate([3.0, 6.8, 10.9, 16.0]):
        add("PXB%d" % i, _barrel_layer(r, 27.0, 0.02, 0.003, 0.01))
    for i, r in enumerate([25.0, 34.0, 42.0, 50.0]):
        add("TIB%d" % i, _barrel_layer(r, 70.0, 0.03, 0.01, 0.5))
    for i, r in enumerate([61.0, 69.0, 78.0, 87.0, 97.0, 110.0]):
        add("TOB%d" % i, _barrel_layer(r, 110.0, 0.03, 0.01, 0.5))
    for sgn, tag in ((1, "P"), (-1, "N")):
        for i, z in enumerate([30.0, 38.0, 48.0]):
            add("PXF%s%d" % (tag, i), _disk_layer(sgn * z, 4.5, 16.5, 0.02, 0.003, 0.01))
        for i, z in enumerate([78.0, 91.0, 105.0]):
            add("TID%s%d" % (tag, i), _disk_layer(sgn * z, 22.0, 51.0, 0.03, 0.01, 0.5))
        for i, z in enumerate([130.0, 155.0, 185.0, 215.0, 245.0, 280.0]):
            add("TEC%s%d" % (tag, i), _disk_layer(sgn * z, 22.0, 110.0, 0.03, 0.01, 0.5))
    plans = []
    for tag in ("P", "N"):
        p = ["PXB%d" % i for i in range(4)] + ["PXF%s%d" % (tag, i) for i in range(3)]
        p += ["TIB%d" % i for i in range(4)] + ["TID%s%d" % (tag, i) for i in range(3)]
        p += ["TOB%d" % i for i in range(6)] + ["TEC%s%d" % (tag, i) for i in range(6)]
        plans.append([idx[n] for n in p])
    plan_off = np.cumsum([0] + [len(p) for p in plans]).astype(np.int32)
    pixel = [i for n, i in idx.items() if n.startswith("PX")]
    return dict(layers=L, bz=float(bz), n_phi_bins=n_phi_bins, n_eta_bins=n_eta_bins, plan_off=plan_off,
                plan_layers=np.concatenate(plans).astype(np.int32), pixel_layers=np.array(sorted(pixel)),
                name="barrel_endcap38")


def default_params(**kw):
    p = dict(chi2_cut=30.0, max_cand=6, max_consec_miss=2, min_hits_keep=4, score_hit=30.0, score_miss=15.0,
             graze_cos_min=0.25, material_flags=3, dup_frac=0.5)
    p.update(kw)
    return p


# ------------------------------------------------------------------------------------------------------
# truth physics (simulation side; not the filter)
# ------------------------------------------------------------------------------------------------------
def _dedx_si(p):
    """Mean -dE/dx [GeV/cm] of a pion in silicon (Bethe-Bloch, no density correction)."""
    E = np.sqrt(p * p + M_PION ** 2)
    bg2 = (p / M_PION) ** 2
    b2 = (p / E) ** 2
    g = E / M_PION
    tmax = 2 * M_E * bg2 / (1 + 2 * g * M_E / M_PION + (M_E / M_PION) ** 2)
    return 0.307075e-3 * (14.0 / 28.0855) * 2.329 / b2 * (0.5 * np.log(2 * M_E * bg2 * tmax / (173e-9) ** 2) - b2)


def _sigma_e(p, t):
    """Width [GeV] of the energy-loss fluctuation in thickness t (radiation lengths along the path): Bohr's variance
    with the relativistic factor, xi Tmax (1 - beta^2/2) (the truth straggles as a Gaussian of this width)."""
    E = np.sqrt(p * p + M_PION ** 2)
    b2 = (p / E) ** 2
    g = E / M_PION
    tmax = 2 * M_E * (p / M_PION) ** 2 / (1 + 2 * g * M_E / M_PION + (M_E / M_PION) ** 2)
    xi = 0.5 * 0.307075e-3 * (14.0 / 28.0855) * 2.329 * (t * 9.37) / b2
    return np.sqrt(xi * tmax * (1 - 0.5 * b2))


def _theta0(p, t):
    E = np.sqrt(p * p + M_PION ** 2)
    return 0.0136 / ((p / E) * p) * np.sqrt(t) * (1 + 0.038 * np.log(t))


def _path_to_layer(lay, a, st):
    """Transverse path s to the layer for every particle; ok=False where it cannot be reached going forward
    with less than half a turn."""
    x, y, z, ipt, phi, th = st
    w = a * ipt
    if lay["kind"] == 1:
        s = (lay["pos"] - z) * np.tan(th)
        ok = (s > -1e-9) & (np.abs(w * s) < np.pi)
        return s, ok
    R = lay["pos"]
    cp, sp = np.cos(phi), np.sin(phi)
    A = x * cp + y * sp
    B = y * cp - x * sp
    D = R * R - (x * x + y * y)
    G = 1 + w * B - 0.25 * D * w * w
    disc = A * A + D * G
    ok = disc >= 0
    sq = np.sqrt(np.where(ok, disc, 0.0))
    den = A + sq
    ok &= den > 0
    lam = D / np.where(ok, den, 1.0)
    tau = 0.5 * w * lam
    s = lam * np.where(np.abs(tau) > 1e-12, np.arctan(tau) / np.where(tau == 0, 1.0, tau), 1.0)
    ok &= s > -1e-9
    return s, ok


def _step(a, st, s):
    x, y, z, ipt, phi, th = st
    w = a * ipt
    h = 0.5 * w * s
    sc = np.where(np.abs(h) > 1e-9, np.sin(h) / np.where(h == 0, 1.0, h), 1.0)
    return [x + s * sc * np.cos(phi + h), y + s * sc * np.sin(phi + h), z + s / np.tan(th), ipt, phi + w * s, th]


def simulate(geom, rng, ev_of, plan_of, q, st0, eff=1.0, material=True, truth_graze=0.30, straggle=False, scatter=True, keep_truth=False, keep_cross=False):
    """Step every particle through its plan. Returns per plan step, per particle: hit position (3), the layer,
    and a validity mask; also the truth state after the last crossed layer (after its material).
    st0 = [x,y,z,ipt,phi,theta] arrays (float64)."""
    n = len(q)
    layers = geom["layers"]
    a0 = -q * KAPPA
    bz_layer = geom.get("bz_layer")                       # field hook: Bz of the step that ends on a layer
    st = [np.array(v, float) for v in st0]
    alive = np.ones(n, bool)
    plan_off, plan_layers = geom["plan_off"], geom["plan_layers"]
    mpl = int(np.max(np.diff(plan_off)))
    hx = np.zeros((mpl, n)); hy = np.zeros((mpl, n)); hz = np.zeros((mpl, n))
    hl = np.full((mpl, n), -1, np.int32)
    tstates = np.full((mpl, 6, n), np.nan) if keep_truth else None    # truth after each crossed layer (after its material)
    xing = np.zeros((3, mpl, n)) if keep_cross else None              # true crossing points (for a second, overlapping-module hit)
    for step in range(mpl):
        # fixed draw order per step: smear1, smear2, efficiency, scatter alpha, scatter beta
        g1, g2 = rng.standard_normal(n), rng.standard_normal(n)
        ue = rng.random(n)
        ga, gb = rng.standard_normal(n), rng.standard_normal(n)
        gs = rng.standard_normal(n) if straggle else None   # drawn only when asked for: the other workloads keep their draws
        for pl in range(len(plan_off) - 1):
            if step >= plan_off[pl + 1] - plan_off[pl]:
                continue
            li = int(plan_layers[plan_off[pl] + step])
            lay = layers[li]
            a = a0 * (geom["bz"] if bz_layer is None else float(bz_layer[li]))
            sel = alive & (plan_of == pl)
            if not sel.any():
                continue
            ii = np.nonzero(sel)[0]
            sub = [v[ii] for v in st]
            s, ok = _path_to_layer(lay, a[ii], sub)
            w = a[ii] * sub[3]
            loop = ok & (np.abs(w * s) >= np.pi)
            ok &= ~loop
            new = _step(a[ii], sub, np.where(ok, s, 0.0))
            r1 = np.hypot(new[0], new[1])
            if lay["kind"] == 0:
                acc = (new[2] >= lay["lo"]) & (new[2] <= lay["hi"])
                cosa = (new[0] * np.cos(new[4]) + new[1] * np.sin(new[4])) / np.maximum(r1, 1e-12)
                graze = ok & acc & (cosa < truth_graze)
                pn = np.abs(np.sin(new[5]) * cosa)
            else:
                acc = (r1 >= lay["lo"]) & (r1 <= lay["hi"])
                graze = ok & acc & (np.abs(np.cos(new[5])) < 0.06)
                pn = np.abs(np.cos(new[5]))
            cross = ok & acc & ~graze
            # particles that graze stop for good
            alive[ii[graze]] = False
            jj = ii[cross]
            if jj.size == 0:
                continue
            nx = [v[cross] for v in new]
            # hit (smearing within the surface only)
            made = ue[jj] < eff
            if lay["kind"] == 0:
                R = lay["pos"]
                ph = np.arctan2(nx[1], nx[0]) + g1[jj] * lay["sig_t"] / R
                px, py, pz = R * np.cos(ph), R * np.sin(ph), nx[2] + g2[jj] * lay["sig_l"]
            else:
                rr = np.hypot(nx[0], nx[1])
                ph = np.arctan2(nx[1], nx[0]) + g1[jj] * lay["sig_t"] / rr
                rr = rr + g2[jj] * lay["sig_l"]
                px, py, pz = rr * np.cos(ph), rr * np.sin(ph), np.full(jj.size, lay["pos"])
            hx[step, jj] = px; hy[step, jj] = py; hz[step, jj] = pz
            if keep_cross:
                xing[0, step, jj] = nx[0]; xing[1, step, jj] = nx[1]; xing[2, step, jj] = nx[2]
            hl[step, jj] = np.where(made, li, -1)
            # material on the truth
            if material and lay["xx0"] > 0:
                t = lay["xx0"] / np.maximum(pn[cross], 1e-6)
                sth = np.sin(nx[5])
                p = 1.0 / (np.abs(nx[3]) * np.abs(sth))
                th0 = _theta0(p, t)
                E = np.sqrt(p * p + M_PION ** 2) - _dedx_si(p) * t * 9.37
                if straggle:
                    E = E + gs[jj] * _sigma_e(p, t)
                stopped = E <= M_PION * 1.0001
                p1 = np.sqrt(np.maximum(E * E - M_PION ** 2, 1e-12))
                if not scatter:                              # energy loss only (isolates the straggling term in the pins)
                    th0 = 0.0 * th0
                th_new = nx[5] + ga[jj] * th0
                ph_new = nx[4] + gb[jj] * th0 / sth
                nx[5] = th_new
                nx[4] = ph_new
                nx[3] = 1.0 / (p1 * np.abs(np.sin(th_new)))
                alive[jj[stopped]] = False
            for k in range(6):
                st[k][jj] = nx[k]
                if keep_truth:
                    tstates[step, k, jj] = nx[k]
    if keep_truth or keep_cross:
        return hx, hy, hz, hl, np.stack(st), tstates, xing
    return hx, hy, hz, hl, np.stack(st)


def hit_cov(lay, x, y):
    """V (6: xx,xy,yy,xz,yz,zz) of a hit on `lay` at azimuth of (x,y): U4 — sigma_n = sig_t along the normal."""
    r = np.hypot(x, y)
    cx, cy = x / r, y / r
    n = len(x)
    V = np.zeros((6, n))
    if lay["kind"] == 0:
        V[0] = lay["sig_t"] ** 2; V[2] = lay["sig_t"] ** 2; V[5] = lay["sig_l"] ** 2
    else:
        sr2, st2 = lay["sig_l"] ** 2, lay["sig_t"] ** 2
        V[0] = sr2 * cx * cx + st2 * cy * cy
        V[1] = (sr2 - st2) * cx * cy
        V[2] = sr2 * cy * cy + st2 * cx * cx
        V[5] = 0.01 ** 2
    return V


# ------------------------------------------------------------------------------------------------------
# seeds (U18)
# ------------------------------------------------------------------------------------------------------
def three_point_seed(bz, h1, h2, h3, V1, inflate=100.0):
    """3-point helix through hits h1,h2,h3 (each (3,n)); state at h1. Returns par (6,n), cov (21,n), q (n)."""
    ax, ay, bx, by, cx, cy = h1[0], h1[1], h2[0], h2[1], h3[0], h3[1]
    d = 2 * (ax * (by - cy) + bx * (cy - ay) + cx * (ay - by))
    d = np.where(np.abs(d) < 1e-12, 1e-12, d)
    a2, b2, c2 = ax * ax + ay * ay, bx * bx + by * by, cx * cx + cy * cy
    ux = (a2 * (by - cy) + b2 * (cy - ay) + c2 * (ay - by)) / d
    uy = (a2 * (cx - bx) + b2 * (ax - cx) + c2 * (bx - ax)) / d
    rho = np.hypot(ax - ux, ay - uy)
    turn = (bx - ax) * (cy - by) - (by - ay) * (cx - bx)
    sg = np.where(turn >= 0, 1.0, -1.0)
    q = (-np.sign(bz) * sg).astype(np.int8)
    ipt = 1.0 / (KAPPA * abs(bz) * rho)
    u0x, u0y = ax - ux, ay - uy
    phi = np.arctan2(sg * u0x, -sg * u0y)
    u3x, u3y = cx - ux, cy - uy
    dpsi = np.abs(np.arctan2(u0x * u3y - u0y * u3x, u0x * u3x + u0y * u3y))
    theta = np.arctan2(rho * dpsi, h3[2] - h1[2])
    n = len(ax)
    par = np.stack([h1[0], h1[1], h1[2], ipt, phi, theta])
    cov = np.zeros((21, n))
    cov[0] = inflate * V1[0]; cov[1] = inflate * V1[1]; cov[2] = inflate * V1[2]
    cov[3] = inflate * V1[3]; cov[4] = inflate * V1[4]; cov[5] = inflate * V1[5]
    cov[9] = inflate * 0.04 ** 2
    cov[14] = inflate * 0.002 ** 2
    cov[20] = inflate * 0.002 ** 2
    return par, cov, q


# ------------------------------------------------------------------------------------------------------
# event assembly
# ------------------------------------------------------------------------------------------------------
def make_events(geom, seed, n_events, n_primary, n_secondary=0, n_noise=0, spectrum="loguniform",
                pt_range=(0.5, 10.0), n_hard=0, eta_max=1.0, eff=1.0, material=True, shuffle=True,
                seed_on_pixel=False, inflate=100.0, straggle=False, scatter=True, keep_truth=False, overlap_frac=0.0,
                n_modules_phi=64):
    """Returns dict(hits=..., truth_hits [mpl][n_part], seeds=..., ...). Particles 0..n_primary-1 of each event are
    'primary' (seed candidates), the rest 'secondary' (hits only). Draw order: per particle (pT, eta, phi, q, vx,
    vy, vz) as whole arrays, then `simulate`'s per-step draws, then noise (phi, l) per layer, then the shuffle."""
    rng = np.random.Generator(np.random.PCG64(seed))
    per_ev = n_primary + n_secondary
    n = n_events * per_ev
    ev_of = np.repeat(np.arange(n_events, dtype=np.int32), per_ev)
    local = np.tile(np.arange(per_ev), n_events)
    primary = local < n_primary
    u_pt, u_eta, u_phi, u_q = rng.random(n), rng.random(n), rng.random(n), rng.random(n)
    vx, vy, vz = rng.standard_normal(n) * 0.01, rng.standard_normal(n) * 0.01, rng.standard_normal(n) * 5.0
    if spectrum == "loguniform":
        pt = pt_range[0] * (pt_range[1] / pt_range[0]) ** u_pt
    else:  # pdf ~ pT^-3 above pt_range[0], truncated at pt_range[1]; the last n_hard primaries uniform 5-50 GeV
        pt = np.minimum(pt_range[0] / np.sqrt(1 - u_pt), pt_range[1])
        hard = primary & (local >= n_primary - n_hard)
        pt = np.where(hard, 5.0 + 45.0 * u_pt, pt)
    eta = (2 * u_eta - 1) * eta_max
    phi = (2 * u_phi - 1) * np.pi
    q = np.where(u_q < 0.5, -1, 1).astype(np.int8)
    theta = 2 * np.arctan(np.exp(-eta))
    plan_of = np.zeros(n, np.int8) if len(geom["plan_off"]) == 2 else np.where(eta >= 0, 0, 1).astype(np.int8)
    sim = simulate(geom, rng, ev_of, plan_of, q.astype(float), [vx, vy, vz, 1.0 / pt, phi, theta],
                   eff=eff, material=material, straggle=straggle, scatter=scatter, keep_truth=keep_truth,
                   keep_cross=overlap_frac > 0)
    hx, hy, hz, hl, final_state = sim[:5]
    mpl = hx.shape[0]
    nl = len(geom["layers"])
    # signal hits
    st_idx, p_idx = np.nonzero(hl >= 0)
    X = [hx[st_idx, p_idx]]; Y = [hy[st_idx, p_idx]]; Z = [hz[st_idx, p_idx]]
    LAY = [hl[st_idx, p_idx]]; EV = [ev_of[p_idx]]; PART = [p_idx.astype(np.int64)]; STEP = [st_idx.astype(np.int32)]
    # overlap hits: a fraction of the crossings is seen by a second, overlapping module of the same layer: an
    # independent measurement of the same true crossing point (drawn last but for the noise and the shuffle)
    SECOND = []
    if overlap_frac > 0:
        cross = sim[6]
        pick = rng.random(len(st_idx)) < overlap_frac
        g1, g2 = rng.standard_normal(len(st_idx)), rng.standard_normal(len(st_idx))
        for li, lay in enumerate(geom["layers"]):
            m = pick & (LAY[0] == li)
            if not m.any():
                continue
            cx_, cy_, cz_ = cross[0, st_idx[m], p_idx[m]], cross[1, st_idx[m], p_idx[m]], cross[2, st_idx[m], p_idx[m]]
            if lay["kind"] == 0:
                R = lay["pos"]
                ph = np.arctan2(cy_, cx_) + g1[m] * lay["sig_t"] / R
                X.append(R * np.cos(ph)); Y.append(R * np.sin(ph)); Z.append(cz_ + g2[m] * lay["sig_l"])
            else:
                rr = np.hypot(cx_, cy_)
                ph = np.arctan2(cy_, cx_) + g1[m] * lay["sig_t"] / rr
                rr = rr + g2[m] * lay["sig_l"]
                X.append(rr * np.cos(ph)); Y.append(rr * np.sin(ph)); Z.append(np.full(m.sum(), lay["pos"]))
            LAY.append(np.full(m.sum(), li, np.int32)); EV.append(ev_of[p_idx[m]]); PART.append(p_idx[m].astype(np.int64))
            STEP.append(np.full(m.sum(), -1, np.int32))                      # not a first hit: never a seed or truth_hits entry
            SECOND.append((st_idx[m], p_idx[m]))
    n_first = len(st_idx)
    # noise hits: n_noise per event spread evenly over layers
    if n_noise > 0:
        per_layer = n_noise // nl
        for li, lay in enumerate(geom["layers"]):
            m = per_layer * n_events
            ph = (2 * rng.random(m) - 1) * np.pi
            l2 = lay["lo"] + (lay["hi"] - lay["lo"]) * rng.random(m)
            if lay["kind"] == 0:
                X.append(lay["pos"] * np.cos(ph)); Y.append(lay["pos"] * np.sin(ph)); Z.append(l2)
            else:
                X.append(l2 * np.cos(ph)); Y.append(l2 * np.sin(ph)); Z.append(np.full(m, lay["pos"]))
            LAY.append(np.full(m, li, np.int32)); EV.append(np.repeat(np.arange(n_events, dtype=np.int32), per_layer))
            PART.append(np.full(m, -1, np.int64)); STEP.append(np.full(m, -1, np.int32))
    X, Y, Z = np.concatenate(X), np.concatenate(Y), np.concatenate(Z)
    LAY, EV, PART, STEP = np.concatenate(LAY), np.concatenate(EV), np.concatenate(PART), np.concatenate(STEP)
    nh = len(X)
    # module ids: n_modules_phi modules around every layer; the second hit of a crossing sits in the neighbouring module
    MOD = (np.floor((np.arctan2(Y, X) + np.pi) * n_modules_phi / (2 * np.pi)).astype(np.int64) % n_modules_phi)
    if SECOND:
        n_second = sum(len(a_) for a_, _ in SECOND)
        first_of = np.full((mpl, n), -1, np.int64)
        first_of[st_idx, p_idx] = np.arange(n_first)
        src = np.concatenate([first_of[a_, b_] for a_, b_ in SECOND])
        MOD[n_first:n_first + n_second] = (MOD[src] + 1) % n_modules_phi
    MOD = (LAY.astype(np.int64) * n_modules_phi + MOD).astype(np.int32)
    key = EV.astype(np.int64) * nl + LAY
    if shuffle:
        order = np.lexsort((rng.random(nh), key))
    else:
        order = np.argsort(key, kind="stable")
    X, Y, Z, LAY, EV, PART, STEP, key, MOD = X[order], Y[order], Z[order], LAY[order], EV[order], PART[order], STEP[order], key[order], MOD[order]
    counts = np.bincount(key, minlength=n_events * nl).reshape(n_events, nl)
    layer_off = np.zeros((n_events, nl + 1), np.int64)
    ev_start = np.concatenate([[0], np.cumsum(counts.sum(1))])
    layer_off[:, 0] = ev_start[:-1]
    layer_off[:, 1:] = ev_start[:-1, None] + np.cumsum(counts, 1)
    V = np.zeros((6, nh))
    for li, lay in enumerate(geom["layers"]):
        m = LAY == li
        if m.any():
            V[:, m] = hit_cov(lay, X[m], Y[m])
    truth_hits = np.full((mpl, n), -1, np.int32)
    sig = (PART >= 0) & (STEP >= 0)
    truth_hits[STEP[sig], PART[sig]] = np.nonzero(sig)[0].astype(np.int32)
    hits = dict(n_events=n_events, layer_off=layer_off.astype(np.int32).reshape(-1), x=X.astype(np.float32),
                y=Y.astype(np.float32), z=Z.astype(np.float32), V=V.astype(np.float32), module=MOD)
    # seeds: first three hits in plan order (optionally restricted to pixel layers)
    if seed_on_pixel:
        is_pix = np.zeros(nl, bool); is_pix[geom["pixel_layers"]] = True
        usable = (truth_hits >= 0) & is_pix[np.maximum(hl, 0)] & (hl >= 0)
    else:
        usable = truth_hits >= 0
    csum = np.cumsum(usable, 0)
    seedable = primary & (csum[-1] >= 3)
    sid = np.nonzero(seedable)[0]
    first3 = np.zeros((3, sid.size), np.int32)
    for k in range(3):
        stepk = np.argmax(usable[:, sid] & (csum[:, sid] == k + 1), 0)
        first3[k] = truth_hits[stepk, sid]
    H = [np.stack([hits["x"][first3[k]], hits["y"][first3[k]], hits["z"][first3[k]]]).astype(float) for k in range(3)]
    V1 = hits["V"][:, first3[0]].astype(float)
    par, cov, qs = three_point_seed(geom["bz"], H[0], H[1], H[2], V1, inflate)
    seeds = dict(par=par.astype(np.float32), cov=cov.astype(np.float32), q=qs, event=ev_of[sid].astype(np.int32),
                 hits=first3, plan=plan_of[sid].astype(np.int8), particle=sid.astype(np.int32),
                 track_hits=np.ascontiguousarray(truth_hits[:, sid]))
    truth = dict(pt=pt, eta=eta, phi=phi, q=q, vx=vx, vy=vy, vz=vz, theta=theta, event=ev_of, primary=primary,
                 final_state=final_state)
    if keep_truth:
        truth["states"] = sim[5]                          # (mpl, 6, n_particles): truth after each crossed layer
    return dict(geom=geom, hits=hits, truth_hits=truth_hits, hit_particle=PART.astype(np.int32), hit_layer=LAY.astype(np.int32),
                seeds=seeds, truth=truth, max_plan_len=mpl)


# ------------------------------------------------------------------------------------------------------
# the five BASELINE.json configs (scale < 1 shrinks counts for tests; geometry and distributions unchanged)
# ------------------------------------------------------------------------------------------------------
def config(i, scale=1.0, seed=0, overlap_frac=0.0):
    s = lambda v, lo=1: max(lo, int(round(v * scale)))
    if i == 0:
        g = geometry_barrel(10, 4.0, 40.0, 100.0, 0.02)
        return make_events(g, seed, 1, s(10000), shuffle=False), default_params()
    if i == 1:
        g = geometry_barrel(17, 4.0, 110.0, 150.0, np.linspace(0.01, 0.04, 17))
        return make_events(g, seed, 1, s(4000000), shuffle=False), default_params()
    if i == 2:
        g = geometry_barrel(17, 4.0, 110.0, 150.0, np.linspace(0.01, 0.04, 17))
        return make_events(g, seed, s(100), 1000, n_noise=20000), default_params(max_cand=6)
    if i == 3:
        g = geometry_barrel_endcap()
        return (make_events(g, seed, s(200), 1500, n_secondary=3900, n_noise=16000, spectrum="soft",
                            pt_range=(0.3, 50.0), n_hard=50, eta_max=2.5, eff=0.95, seed_on_pixel=True, overlap_frac=overlap_frac),
                default_params(max_cand=6, min_hits_keep=4))
    if i == 4:
        g = geometry_barrel_endcap()
        return (make_events(g, seed, s(64), 6000, n_secondary=13500, n_noise=60000, spectrum="soft",
                            pt_range=(0.3, 50.0), n_hard=0, eta_max=2.5, eff=0.95, seed_on_pixel=True),
                default_params(max_cand=8, min_hits_keep=4))
    raise ValueError(i)


# ------------------------------------------------------------------------------------------------------
# raw strip data for the clustering step. A toy stand-in for unpacked, calibrated
# silicon-strip ADC counts: no detector data is available here.
# ------------------------------------------------------------------------------------------------------
def make_strips(seed, n_modules, strips_per_module=512, occupancy=0.01, bad_frac=0.01, noise_mean=4.0):
    """Per strip: pedestal-subtracted ADC (uint16: Gaussian noise rounded and clipped at 0, plus charge deposits of
    1-5 strips with an exponential-tailed total charge), its expected noise (float32, per strip, ~N(noise_mean, 5 %)),
    a bad-strip flag (bad strips read 0). Modules of unequal length (every 7th module is half as long).
    Draw order: noise level, bad flags, noise samples, deposit positions, widths, charges, shares."""
    rng = np.random.Generator(np.random.PCG64(seed))
    lens = np.where(np.arange(n_modules) % 7 == 6, strips_per_module // 2, strips_per_module).astype(np.int64)
    off = np.concatenate([[0], np.cumsum(lens)]).astype(np.int32)
    n = int(off[-1])
    noise = (noise_mean * (1 + 0.05 * rng.standard_normal(n))).clip(0.5 * noise_mean).astype(np.float32)
    bad = (rng.random(n) < bad_frac).astype(np.uint8)
    sig = rng.standard_normal(n) * noise
    ndep = int(occupancy * n / 3)
    pos = rng.integers(0, n, ndep)
    width = rng.integers(1, 6, ndep)
    charge = 60.0 + rng.exponential(80.0, ndep)
    for k in range(5):
        m = width > k
        idx = np.minimum(pos[m] + k, n - 1)
        share = charge[m] / width[m] * (0.6 + 0.8 * rng.random(m.sum()))
        np.add.at(sig, idx, share)
    adc = np.clip(np.rint(sig), 0, 1023).astype(np.uint16)
    adc[bad != 0] = 0
    return dict(module_off=off, adc=adc, noise=noise, bad=bad)


def default_strip_params(**kw):
    p = dict(seed_thr=3.0, chan_thr=2.0, clus_thr=5.0, min_charge=30, max_holes=0, max_bad=1)
    p.update(kw)
    return p
