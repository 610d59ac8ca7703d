"""Hand-placed events shared by the oracle pins (tests/test_oracle_build.py) and the -m gpu parity tests: inputs only,
with the expected results written by hand beside them (nothing here was produced by any implementation)."""
import numpy as np

from workloads import datagen


def tie_event():
    """Hand-placed event for the last two keys of the total order U14 (PAPER.md:41 'only the best ranking ones are
    cloned at each layer'): one straight-ish track through 5 barrel layers without material, one hit per layer, and
    the hit of layer 3 present TWICE (same position, same covariance, ids 3 and 4). Hit ids: layers 0,1,2 -> 0,1,2
    (the seed), layer 3 -> 3 and 4 (the twins), layer 4 -> 5. Both twins give children equal in (score, chi2) bit for
    bit, so only key 4 (lower hit id) orders them; the two candidates they make are then identical except for that
    id, so their children on layer 4 (both with hit 5) tie again and only key 3 (lower parent rank) orders them."""
    g = datagen.geometry_barrel(5, 4.0, 20.0, 100.0, 0.0)
    ev = datagen.make_events(g, 2, 1, 1, material=False)
    h, s = ev["hits"], ev["seeds"]
    assert s["par"].shape[1] == 1 and len(h["x"]) == 5
    ids = np.array([0, 1, 2, 3, 3, 4])
    hits = dict(n_events=1, x=h["x"][ids].copy(), y=h["y"][ids].copy(), z=h["z"][ids].copy(), V=np.ascontiguousarray(h["V"][:, ids]),
                layer_off=np.array([0, 1, 2, 3, 5, 6], np.int32))
    seeds = {k: np.ascontiguousarray(s[k]) for k in ("par", "cov", "q", "plan", "event", "hits")}
    assert list(seeds["hits"][:, 0]) == [0, 1, 2]
    return dict(geom=g, hits=hits, seeds=seeds), datagen.default_params(material_flags=0, min_hits_keep=4)


# expected hit lists, written by hand from U14 (not produced by any implementation)
TIE_EXPECTED = {1: [0, 1, 2, 3, 5],      # cap 1: the twins tie on layer 3, the lower id (3, not 4) is kept
                2: [0, 1, 2, 3, 5]}      # cap 2: both twins live on (ranks 0, 1 = ids 3, 4); on layer 4 their children
                                         # tie and the child of parent rank 0 ranks first, so the winner carries id 3


def nan_child_event(bad_layer=4):
    """One track through 6 disks (z = 10..60 cm, no material), one hit per disk, ids = layers. The hit on disk
    `bad_layer` carries V_xx = +inf (everything else as usual): its chi2 is finite (the x residual gets weight 0), so it
    is accepted, but the covariance update holds 0 * inf: the child is not finite (C9 / reading R1)."""
    layers = [datagen._disk_layer(10.0 * (k + 1), 1.0, 60.0, 0.0, 0.003, 0.01) for k in range(6)]
    g = dict(layers=layers, bz=3.8, n_phi_bins=63, n_eta_bins=40, plan_off=np.array([0, 6], np.int32),
             plan_layers=np.arange(6, dtype=np.int32), pixel_layers=np.arange(6), name="disks6")
    rng = np.random.Generator(np.random.PCG64(7))
    th = 2 * np.arctan(np.exp(-1.2))
    st0 = [np.array([0.01]), np.array([-0.02]), np.array([0.5]), np.array([1.0 / 2.0]), np.array([0.4]), np.array([th])]
    hx, hy, hz, hl, _ = datagen.simulate(g, rng, np.zeros(1, np.int32), np.zeros(1, np.int8), np.array([1.0]), st0, material=False)
    assert list(hl[:, 0]) == list(range(6))
    x, y, z = hx[:, 0], hy[:, 0], hz[:, 0]
    V = np.concatenate([datagen.hit_cov(layers[k], x[k:k + 1], y[k:k + 1]) for k in range(6)], axis=1).astype(np.float32)
    V[0, bad_layer] = np.inf; V[1, bad_layer] = 0.0                       # xx = inf, xy = 0
    hits = dict(n_events=1, x=x.astype(np.float32), y=y.astype(np.float32), z=z.astype(np.float32), V=V,
                layer_off=np.arange(7, dtype=np.int32))
    H = [np.stack([hits["x"][k:k + 1], hits["y"][k:k + 1], hits["z"][k:k + 1]]).astype(float) for k in range(3)]
    par, cov, q = datagen.three_point_seed(g["bz"], H[0], H[1], H[2], V[:, 0:1].astype(float))
    seeds = dict(par=par.astype(np.float32), cov=cov.astype(np.float32), q=q, event=np.zeros(1, np.int32),
                 hits=np.array([[0], [1], [2]], np.int32), plan=np.zeros(1, np.int8))
    return dict(geom=g, hits=hits, seeds=seeds), datagen.default_params(material_flags=0, min_hits_keep=4)
