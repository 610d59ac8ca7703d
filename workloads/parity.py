"""Parity metrics between a float32 result and a float64 reference result (tolerances of BASELINE.json north_star,
made precise by readings U19/U20 of DESIGN.md §3). Pure numpy; used by the -m gpu tests and by bench.py's checks."""
import numpy as np

TOL_PAR, TOL_COV, TOL_CHI2 = 1e-4, 1e-3, 1e-3


def cidx(i, j):
    return i * (i + 1) // 2 + j if j <= i else j * (j + 1) // 2 + i


def unpack_cov(cov21):
    """(21, n) packed lower triangle -> (n, 6, 6)."""
    n = cov21.shape[1]
    C = np.zeros((n, 6, 6))
    for i in range(6):
        for j in range(6):
            C[:, i, j] = cov21[cidx(i, j)]
    return C


def local_frames(par, kind):
    """(n, 5, 6) maps global (x,y,z,ipt,phi,theta) to local (in-surface 1, in-surface 2, ipt, phi, theta): the surface
    normal is excluded because the transported covariance is singular along it (U2)."""
    n = par.shape[1]
    T = np.zeros((n, 5, 6))
    x, y = par[0], par[1]
    r = np.maximum(np.hypot(x, y), 1e-12)
    kind = np.broadcast_to(np.asarray(kind), (n,))
    b = kind == 0
    # barrel: tangential, z ; disk: x, y
    T[b, 0, 0], T[b, 0, 1] = (-y / r)[b], (x / r)[b]
    T[b, 1, 2] = 1.0
    T[~b, 0, 0] = 1.0
    T[~b, 1, 1] = 1.0
    T[:, 2, 3] = T[:, 3, 4] = T[:, 4, 5] = 1.0
    return T


def param_errors(par_gpu, par_ref, scale_pos):
    """Per-track worst |delta| / max(|v|, scale) over the six parameters (U19). phi is compared modulo 2 pi."""
    d = np.asarray(par_gpu, float) - par_ref
    d[4] = np.angle(np.exp(1j * d[4]))
    scale = np.stack([np.broadcast_to(scale_pos, d[0].shape)] * 3 + [np.abs(par_ref[3]), np.ones_like(d[0]),
                                                                    np.ones_like(d[0])])
    ref = np.abs(par_ref).copy()
    ref[4] = 1.0
    return np.max(np.abs(d) / np.maximum(ref, scale), axis=0)


def cov_errors(cov_gpu, cov_ref, par_ref, kind):
    """Per-track worst |dC_ij| / sqrt(C_ii C_jj) on the local 5x5 block (U19)."""
    T = local_frames(par_ref, kind)
    Cg = T @ unpack_cov(np.asarray(cov_gpu, float)) @ T.transpose(0, 2, 1)
    Cr = T @ unpack_cov(cov_ref) @ T.transpose(0, 2, 1)
    dg = np.sqrt(np.maximum(np.einsum("nii->ni", Cr), 1e-300))
    return np.max(np.abs(Cg - Cr) / (dg[:, :, None] * dg[:, None, :]), axis=(1, 2))


def chi2_errors(chi2_gpu, chi2_ref):
    return np.abs(np.asarray(chi2_gpu, float) - chi2_ref) / np.maximum(chi2_ref, 1.0)


def last_layer_of_fit(geom, plan, track_hits, nfit):
    """Layer index (and its kind / position scale) on which each fitted track's output state sits: the layer of
    its nfit-th hit in plan order. Tracks with nfit == 0 get the first layer of their plan."""
    plan_off, plan_layers = np.asarray(geom["plan_off"]), np.asarray(geom["plan_layers"])
    mpl, n = track_hits.shape
    has = track_hits >= 0
    cs = np.cumsum(has, 0)
    step = np.argmax(has & (cs == np.maximum(nfit, 1)[None]), 0)
    lay = plan_layers[plan_off[np.asarray(plan, int)] + step]
    kinds = np.array([l["kind"] for l in geom["layers"]])[lay]
    pos = np.array([abs(l["pos"]) for l in geom["layers"]])[lay]
    return lay, kinds, pos


def first_layer_of_backward_fit(geom, plan, track_hits, nfit):
    """Same for the backward fit: the layer of the nfit-th hit counted from the END of the hit list."""
    plan_off, plan_layers = np.asarray(geom["plan_off"]), np.asarray(geom["plan_layers"])
    has = track_hits >= 0
    cs = np.cumsum(has[::-1], 0)[::-1]
    step = np.argmax(has & (cs == np.maximum(nfit, 1)[None]), 0)
    lay = plan_layers[plan_off[np.asarray(plan, int)] + step]
    kinds = np.array([l["kind"] for l in geom["layers"]])[lay]
    pos = np.array([abs(l["pos"]) for l in geom["layers"]])[lay]
    return lay, kinds, pos
