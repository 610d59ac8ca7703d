"""Full-size bench workloads assembled from `datagen` chunks (bounded host memory, chunks generated in parallel
processes). No arithmetic of the method: concatenation, id offsets and permutations only.

Recipe: chunk k of a workload made with seed s comes from datagen with seed 16*s + k (fit) or
64*s + k (building, strips); chunks are concatenated in k order with hit ids, event ids and particle ids offset."""
import multiprocessing as mp
import os

import numpy as np

from . import datagen

BUILD_EVENTS = {2: 100, 3: 200, 4: 64}
BUILD_CHUNK = {2: 25, 3: 25, 4: 8}           # events per generated chunk
STRIP_EVENTS, STRIP_MODULES = 16, 15000


def _pool_map(fn, jobs):
    """jobs in parallel forked processes (generation is single-threaded numpy); falls back to a plain loop."""
    nproc = min(len(jobs), max(1, (os.cpu_count() or 2) - 1), 8)
    if nproc <= 1 or os.environ.get("MKF_BENCH_SERIAL"):
        return [fn(j) for j in jobs]
    try:
        with mp.get_context("fork").Pool(nproc) as pool:
            return pool.map(fn, jobs)
    except Exception:
        return [fn(j) for j in jobs]


def _fit_chunk(job):
    m, seed = job
    ev, prm = datagen.config(1, scale=m / 4000000.0, seed=seed)
    s = ev["seeds"]
    return ev["geom"], prm, ev["hits"], dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"], track_hits=s["track_hits"])


def make_fit_workload(seed, scale):
    """configs[1]: 4 M x scale helices as chunks of 1 M (seeds 16 seed + k), hits concatenated, ids offset. The fit
    does not use layer_off, so the whole workload is one 'event' with an all-zero layer_off.
    Returns geom, prm, hits, seeds, (hits, seeds) of the first chunk."""
    total = max(1, int(round(4000000 * scale)))
    chunk = 1000000
    jobs, done, k = [], 0, 0
    while done < total:
        m = min(chunk, total - done)
        jobs.append((m, seed * 16 + k)); done += m; k += 1
    res = _pool_map(_fit_chunk, jobs)
    geom, prm = res[0][0], res[0][1]
    parts, nh0 = [], 0
    for _, _, hits, s in res:
        th = s["track_hits"].copy()
        th[th >= 0] += nh0
        parts.append((hits, dict(s, track_hits=th)))
        nh0 += hits["x"].shape[0]
    hits = dict(n_events=1, layer_off=np.zeros(len(geom["layers"]) + 1, np.int32),
                x=np.concatenate([p[0]["x"] for p in parts]), y=np.concatenate([p[0]["y"] for p in parts]),
                z=np.concatenate([p[0]["z"] for p in parts]), V=np.concatenate([p[0]["V"] for p in parts], axis=1))
    seeds = {k2: np.ascontiguousarray(np.concatenate([p[1][k2] for p in parts], axis=-1)) for k2 in ("par", "cov", "q", "plan", "track_hits")}
    return geom, prm, hits, seeds, parts[0]


def shuffle_hit_order(hits, seeds, seed):
    """The same tracks and hits with the hit ids randomly permuted (one permutation over the whole hit array: the fit
    workload is a single all-layers 'event'): returns (hits, seeds) whose track_hits name the same hits at their new
    places. This is the memory order a fit meets when its hit lists come from track building."""
    nh = hits["x"].shape[0]
    rng = np.random.Generator(np.random.PCG64(1000003 + seed))
    perm = rng.permutation(nh).astype(np.int32)                 # new position -> old id
    inv = np.empty(nh, np.int32); inv[perm] = np.arange(nh, dtype=np.int32)
    h2 = dict(hits, x=hits["x"][perm], y=hits["y"][perm], z=hits["z"][perm], V=np.ascontiguousarray(hits["V"][:, perm]))
    th = seeds["track_hits"]
    th2 = np.where(th >= 0, inv[np.maximum(th, 0)], th).astype(np.int32)
    return h2, dict(seeds, track_hits=np.ascontiguousarray(th2))


def _build_chunk(job):
    which, n_ev, seed, ovl = job
    ev, prm = datagen.config(which, scale=n_ev / BUILD_EVENTS[which], seed=seed, **(dict(overlap_frac=ovl) if ovl else {}))
    s = ev["seeds"]
    keep = dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"], event=s["event"], hits=s["hits"], track_hits=s["track_hits"])
    return ev["geom"], prm, ev["hits"], keep


def make_build_workload(which, seed, scale, overlap_frac=0.0):
    """configs[2..4] as chunks of BUILD_CHUNK events (seeds 64 seed + k), concatenated: hit ids, event ids offset.
    At scale <= one chunk this is exactly datagen.config(which, scale, 64 seed). overlap_frac > 0 (configs[3] only):
    that fraction of the crossings is also seen by a neighbouring module; hits then carry `module`."""
    total = max(1, int(round(BUILD_EVENTS[which] * scale)))
    per = BUILD_CHUNK[which]
    jobs, done, k = [], 0, 0
    while done < total:
        m = min(per, total - done)
        jobs.append((which, m, seed * 64 + k, overlap_frac)); done += m; k += 1
    res = _pool_map(_build_chunk, jobs)
    geom, prm = res[0][0], res[0][1]
    nl = len(geom["layers"])
    X, Y, Z, V, LO, S, MOD = [], [], [], [], [], [], []
    nh0 = ev0 = 0
    for _, _, h, s in res:
        X.append(h["x"]); Y.append(h["y"]); Z.append(h["z"]); V.append(h["V"]); MOD.append(h["module"])
        LO.append(h["layer_off"].astype(np.int64) + nh0)
        s = dict(s, event=s["event"] + ev0, hits=s["hits"] + nh0, track_hits=np.where(s["track_hits"] >= 0, s["track_hits"] + nh0, s["track_hits"]))
        S.append(s)
        nh0 += h["x"].shape[0]; ev0 += h["n_events"]
    hits = dict(n_events=ev0, layer_off=np.concatenate(LO).astype(np.int32), x=np.concatenate(X), y=np.concatenate(Y), z=np.concatenate(Z),
                V=np.ascontiguousarray(np.concatenate(V, axis=1)))
    if overlap_frac:
        hits["module"] = np.concatenate(MOD).astype(np.int32)
    assert hits["layer_off"].shape[0] == ev0 * (nl + 1)
    seeds = {k2: np.ascontiguousarray(np.concatenate([s[k2] for s in S], axis=-1)) for k2 in S[0]}
    return dict(geom=geom, hits=hits, seeds=seeds), prm


def _strip_chunk(job):
    return datagen.make_strips(*job)


def make_strip_workload(seed, scale):
    """STRIP_EVENTS x scale events of STRIP_MODULES modules (about the module count of a strip tracker), one generated
    chunk per event (seeds 64 seed + k), concatenated: the batch is one flat module list."""
    n_ev = max(1, int(round(STRIP_EVENTS * scale))) if scale >= 1.0 / STRIP_EVENTS else 1
    n_mod = STRIP_MODULES if scale >= 1.0 / STRIP_EVENTS else max(8, int(round(STRIP_MODULES * STRIP_EVENTS * scale)))
    parts = _pool_map(_strip_chunk, [(64 * seed + k, n_mod) for k in range(n_ev)])
    off, base = [np.zeros(1, np.int32)], 0
    for p in parts:
        off.append((p["module_off"][1:].astype(np.int64) + base).astype(np.int32)); base += int(p["module_off"][-1])
    d = dict(module_off=np.concatenate(off), adc=np.concatenate([p["adc"] for p in parts]),
             noise=np.concatenate([p["noise"] for p in parts]), bad=np.concatenate([p["bad"] for p in parts]))
    return d, datagen.default_strip_params()
