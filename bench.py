"""bench.py — KF layer-steps/s of mkf_fit on BASELINE.json configs[1] (4 M helices x 17 barrel layers), or built
events/s of the building path on configs[2..4] (--workload build2|build3|build4).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl mkf|reference] [--workload fit|fitback|build2|build3|build4|strips]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P bench.py --gpus N ...

One JSON line on rank 0 (contract in DESIGN.md §8). A "step" is one pass of the whole path over the workload with
inputs resident in HBM; `e2e` is the same pass through the host-buffer C-ABI call (pinned host memory, copies
timed). Events/tracks are independent, so N > 1 shards them with no collective (weak scaling: every rank owns a
full-size workload generated from seed+rank).
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

ALGO_FLOP_PER_LAYER_STEP = 1000.0        # DESIGN.md §6 (SURVEY.md §8 d): propagate 150 + transport 420 + material 90 + update 340
ALGO_BYTES_PER_LAYER_STEP = 54.0         # hit 36 B + index 4 B + state in/out amortised 14 B
FP32_LANES_PER_SM, N_SM = 128, 148
# dram__bytes_read.sum + dram__bytes_write.sum of one mkf_fit_kernel launch on the full configs[1] workload, from
# the `ncu --set full` capture summarised in profiles/r1_fit_kernel_ncu.md (3.1226 GB + 0.4689 GB)
NCU_TRAFFIC_BYTES_FIT_FULL = 3.591e9


STRIP_BYTES_IN, STRIP_BYTES_PER_CLUSTER = 7, 20
# dram__bytes_read.sum + dram__bytes_write.sum of one sc_cluster_kernel launch on the full strips workload
# (profiles/r1_strips_kernel_ncu.md)
NCU_TRAFFIC_BYTES_STRIPS_FULL = 8.098e8


def peaks():
    p = dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")
    try:
        m = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        p.update(hbm_gbs=float(m["hbm_gbs"]), sm_max_mhz=float(m.get("sm_max_mhz", 1965.0)), source="measured")
    except Exception:
        pass
    p["fp32_tflops"] = N_SM * FP32_LANES_PER_SM * 2 * p["sm_max_mhz"] * 1e6 / 1e12
    return p


# ---------------------------------------------------------------------------------------------------------------
# workloads
# ---------------------------------------------------------------------------------------------------------------
def make_fit_workload(seed, scale):
    """configs[1]: generated as chunks of 1 M helices (bounded host memory), hits concatenated, ids offset."""
    from workloads import datagen
    total = max(1, int(round(4000000 * scale)))
    chunk = 1000000
    parts, nh0 = [], 0
    geom = prm = None
    done = 0
    k = 0
    while done < total:
        m = min(chunk, total - done)
        ev, prm = datagen.config(1, scale=m / 4000000.0, seed=seed * 16 + k)
        geom = ev["geom"]
        s = ev["seeds"]
        th = s["track_hits"].copy()
        th[th >= 0] += nh0
        parts.append((ev["hits"], dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"], track_hits=th)))
        nh0 += ev["hits"]["x"].shape[0]
        done += m
        k += 1
    hits = dict(n_events=1, layer_off=np.zeros(len(geom["layers"]) + 1, np.int32),
                x=np.concatenate([p[0]["x"] for p in parts]), y=np.concatenate([p[0]["y"] for p in parts]),
                z=np.concatenate([p[0]["z"] for p in parts]), V=np.concatenate([p[0]["V"] for p in parts], axis=1))
    seeds = {k2: np.ascontiguousarray(np.concatenate([p[1][k2] for p in parts], axis=-1)) for k2 in ("par", "cov", "q", "plan", "track_hits")}
    return geom, prm, hits, seeds, parts[0]


def make_build_workload(which, seed, scale):
    from workloads import datagen
    ev, prm = datagen.config(which, scale=scale, seed=seed)
    return ev, prm


# ---------------------------------------------------------------------------------------------------------------
# ranks: events / tracks are independent, so a rank owns its own workload and nothing but timings is exchanged
# ---------------------------------------------------------------------------------------------------------------
STRIP_EVENTS, STRIP_MODULES = 16, 15000


def make_strip_workload(seed, scale):
    """STRIP_EVENTS x scale events of STRIP_MODULES modules (about the module count of a strip tracker), generated one
    event at a time (seeds 64 seed + k) and concatenated: the batch is one flat module list."""
    from workloads import datagen
    n_ev = max(1, int(round(STRIP_EVENTS * scale))) if scale >= 1.0 / STRIP_EVENTS else 1
    n_mod = STRIP_MODULES if scale >= 1.0 / STRIP_EVENTS else max(8, int(round(STRIP_MODULES * STRIP_EVENTS * scale)))
    parts = [datagen.make_strips(64 * seed + k, n_mod) for k in range(n_ev)]
    off, base = [np.zeros(1, np.int32)], 0
    for p in parts:
        off.append((p["module_off"][1:].astype(np.int64) + base).astype(np.int32)); base += int(p["module_off"][-1])
    d = dict(module_off=np.concatenate(off), adc=np.concatenate([p["adc"] for p in parts]),
             noise=np.concatenate([p["noise"] for p in parts]), bad=np.concatenate([p["bad"] for p in parts]))
    return d, datagen.default_strip_params()


def oracle_strip_rate(d, sp, n_modules):
    from oracle import mkfo
    ns = int(d["module_off"][n_modules])
    t = time.perf_counter()
    r = mkfo.cluster_strips(d["module_off"][:n_modules + 1], d["adc"][:ns], d["noise"][:ns], d["bad"][:ns], **sp)
    dt = time.perf_counter() - t
    return ns / dt, dt, 1, r


def rank_seed(seed, rank):
    """Seed of the workload a rank owns (weak scaling: every rank generates a full-size workload of its own)."""
    return seed + rank


def aggregate(ms_total, units, world, device):
    """(max over ranks of the time, sum over ranks of the units). One all-reduce each; identity for world == 1."""
    if world == 1:
        return float(ms_total), float(units)
    import torch
    import torch.distributed as dist
    mx = torch.tensor([ms_total], dtype=torch.float64, device=device)
    sm = torch.tensor([units], dtype=torch.float64, device=device)
    dist.all_reduce(mx, op=dist.ReduceOp.MAX)
    dist.all_reduce(sm, op=dist.ReduceOp.SUM)
    return float(mx[0]), float(sm[0])


# ---------------------------------------------------------------------------------------------------------------
# clocks
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.samples, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "50"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        inside = [s for t, s in self.samples if t0 <= t <= t1]
        in_window = bool(inside)
        if not inside:                                   # timed region shorter than the sampling period: take the next samples
            for _ in range(40):
                if len(self.samples) >= 3:
                    break
                time.sleep(0.05)
            inside = [s for _, s in self.samples[-3:]]
        if self.proc:
            self.proc.terminate()
        mhz, mx, reasons = [], 0.0, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for s in inside:
            f = [x.strip() for x in s.split(",")]
            try:
                mhz.append(float(f[0])); mx = max(mx, float(f[1]))
            except Exception:
                continue
            for nme, v in zip(names, f[2:6]):
                if v.lower().startswith("active"):
                    reasons.add(nme)
        return dict(sm_mhz=float(np.median(mhz)) if mhz else None, sm_max_mhz=mx or None, reasons=sorted(reasons),
                    samples=len(mhz), in_timed_region=in_window)


# ---------------------------------------------------------------------------------------------------------------
# oracle legs (cpu_baseline of the mkf arm, and the whole --impl reference arm)
# ---------------------------------------------------------------------------------------------------------------
def oracle_fit_rate(geom, prm, hits, seeds, n_tracks, repeat=1, backward=False):
    from oracle import mkfo
    o = mkfo.Oracle(geom, prm)
    sl = slice(0, n_tracks)
    args = (hits, seeds["par"][:, sl], seeds["cov"][:, sl], seeds["q"][sl], seeds["plan"][sl], np.ascontiguousarray(seeds["track_hits"][:, sl]))
    t = time.perf_counter()
    for _ in range(repeat):
        r = o.fit_backward(*args) if backward else o.fit(*args)
    dt = (time.perf_counter() - t) / repeat
    return float(r["nfit"].sum()) / dt, dt, o.num_threads(), int(r["nfit"].sum()), r


def oracle_build_rate(ev, prm, n_events, dedup):
    from oracle import mkfo
    s = ev["seeds"]
    o = mkfo.Oracle(ev["geom"], prm)
    nl = len(ev["geom"]["layers"])
    h = ev["hits"]
    lo = h["layer_off"].reshape(-1, nl + 1)
    nh = int(lo[n_events - 1, nl])
    sub = dict(n_events=n_events, layer_off=np.ascontiguousarray(lo[:n_events]).reshape(-1), x=h["x"][:nh], y=h["y"][:nh], z=h["z"][:nh],
               V=np.ascontiguousarray(h["V"][:, :nh]))
    m = s["event"] < n_events
    t = time.perf_counter()
    idx = o.build_hit_index(sub)
    r = o.build_tracks(sub, idx, s["par"][:, m], s["cov"][:, m], s["q"][m], s["event"][m], np.ascontiguousarray(s["hits"][:, m]), s["plan"][m])
    if dedup:
        counts = np.bincount(s["event"][m], minlength=n_events)
        o.remove_duplicates(np.concatenate([[0], np.cumsum(counts)]).astype(np.int32), r["hit_ids"], r["nhits"], r["score"].astype(np.float32))
    dt = time.perf_counter() - t
    return n_events / dt, dt, o.num_threads(), r, m


# ---------------------------------------------------------------------------------------------------------------
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="mkf", choices=["mkf", "reference"])
    ap.add_argument("--workload", default="fit", choices=["fit", "fitback", "build2", "build3", "build4", "strips"])
    ap.add_argument("--scale", type=float, default=1.0, help="shrinks the workload (testing only; the JSON says so)")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=2)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    a = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    warm = max(a.warmup, 3)
    backward = a.workload == "fitback"
    is_fit = a.workload in ("fit", "fitback")
    is_strips = a.workload == "strips"
    metric = "KF layer-steps/s (propagate+update)" if is_fit else "clustered strips/s" if is_strips else "built events/s"
    unit = "layer-steps/s" if is_fit else "strips/s" if is_strips else "events/s"
    names = dict(fitback="configs[1] workload, backward fit (SURVEY f1): seeds = forward fit at the last hit, covariance x100",
                 fit="configs[1]: track fit, 4M helices x 17 barrel layers, MS + dE/dx, seeds from 3 hits, cov x100",
                 build2="configs[2]: building, barrel, 100 events x 1000 tracks + 20k noise hits, top 6",
                 build3="configs[3]: building, barrel+endcap, 200 events x 1500 seeds, ~80k hits/event",
                 strips="strip clustering (SURVEY f3, reading R8): %d events x %d modules of 512 / 256 strips, ~1 %% occupancy, "
                        "1 %% bad strips" % (STRIP_EVENTS, STRIP_MODULES),
                 build4="configs[4]: batched building + duplicate removal, 64 events x 6000 seeds, ~300k hits/event, top 8")
    cfg = dict(workload=names[a.workload], scale=a.scale, l2="inputs larger than L2 (no flush needed)", seed=a.seed)

    # ---- reference arm: the oracle on host cores, bounded sample ------------------------------------------------
    if a.impl == "reference":
        if rank != 0:
            return
        if is_fit:
            n_s = max(1, int(round(200000 * min(1.0, a.scale * 20))))
            geom, prm, hits, seeds, _ = make_fit_workload(a.seed, n_s / 4000000.0)
            rates = []
            for k in range(warm + a.steps):
                rate, dt, cores, steps, _ = oracle_fit_rate(geom, prm, hits, seeds, n_s)
                if k >= warm:
                    rates.append((rate, dt))
            sample = "first %d helices of the workload per step (%d layer-steps)" % (n_s, steps)
        elif is_strips:
            d, sp = make_strip_workload(a.seed, min(1.0, a.scale) * 4.0 / STRIP_EVENTS)
            rates = []
            for k in range(warm + a.steps):
                rate, dt, cores, _ = oracle_strip_rate(d, sp, len(d["module_off"]) - 1)
                if k >= warm:
                    rates.append((rate, dt))
            sample = "%d modules (%d strips) of the workload per step" % (len(d["module_off"]) - 1, len(d["adc"]))
        else:
            which = int(a.workload[-1])
            nev_full = {2: 100, 3: 200, 4: 64}[which]
            n_ev = max(1, min(4, int(round(nev_full * a.scale))))
            ev, prm = make_build_workload(which, a.seed, n_ev / nev_full)
            rates = []
            for k in range(warm + a.steps):
                rate, dt, cores, _, _ = oracle_build_rate(ev, prm, n_ev, which == 4)
                if k >= warm:
                    rates.append((rate, dt))
            sample = "%d events of the workload per step" % n_ev
        ms = 1e3 * float(np.mean([d for _, d in rates]))
        v = float(np.mean([r for r, _ in rates]))
        print(json.dumps(dict(metric=metric, value=v, unit=unit, n_gpus=a.gpus, steps=a.steps, warmup=warm, ms_per_step=ms,
                              higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic", config=cfg,
                              impl="reference", cpu_baseline=dict(value=v, unit=unit, cores=cores, kind="oracle", sample=sample),
                              e2e=dict(value=v, unit=unit, h2d_bytes_per_step=0, d2h_bytes_per_step=0), gpu_launches=0)))
        return

    # ---- mkf arm ------------------------------------------------------------------------------------------------
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl mkf needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl")
    from paper_2002_06295_b200 import binding as B

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    pk = peaks()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    if is_fit:
        geom, prm, hits, seeds, _ = make_fit_workload(rank_seed(a.seed, rank), a.scale)
        ctx = B.Context(geom, prm)
        dh = B.hits_to_device(hits)
        ds = B.to_device(seeds, ["par", "cov", "q", "plan", "track_hits"])
        n = seeds["par"].shape[1]
        out = B.alloc_fit_out(n)

        if backward:                                      # seeds of the backward fit: one untimed forward fit
            ctx.fit(dh, ds, ds["plan"], ds["track_hits"], out, out["chi2"], out["nfit"], out["status"])
            th = ds["track_hits"].clone()
            th[torch.cumsum((th >= 0).to(torch.int32), 0) > out["nfit"][None]] = -1
            ds = dict(ds, par=out["par"].clone(), cov=(100.0 * out["cov"]), track_hits=th.contiguous())
            seeds = {k: v.cpu().numpy() for k, v in ds.items()}

        def step():
            ctx.fit(dh, ds, ds["plan"], ds["track_hits"], out, out["chi2"], out["nfit"], out["status"], backward=backward)

        def units():
            return float(out["nfit"].sum().item())

        def e2e_step():
            if backward:                                  # no host entry point for the backward fit: pinned copies by torch
                hd = {k: (torch.from_numpy(v).cuda(non_blocking=True) if isinstance(v, np.ndarray) else v) for k, v in hits_p.items()}
                sd2 = {k: torch.from_numpy(v).cuda(non_blocking=True) for k, v in seeds_p.items()}
                ctx.fit(hd, sd2, sd2["plan"], sd2["track_hits"], out, out["chi2"], out["nfit"], out["status"], backward=True)
                res = [out[k].cpu() for k in ("par", "cov", "chi2", "nfit", "status")]
                h2d = sum(v.nbytes for v in hits_p.values() if isinstance(v, np.ndarray)) + sum(v.nbytes for v in seeds_p.values())
                return float(res[3].sum()), h2d, sum(t.numel() * t.element_size() for t in res)
            r = ctx.fit_host(hits_p, seeds_p, seeds_p["plan"], seeds_p["track_hits"])
            return float(r["nfit"].sum()), r["h2d_bytes"], r["d2h_bytes"]
    elif is_strips:
        from workloads import datagen
        ev_g, prm_g = datagen.config(0, scale=0.001)              # clustering uses no geometry; a context needs one
        ctx = B.Context(ev_g["geom"], prm_g)
        sd_host, sp = make_strip_workload(rank_seed(a.seed, rank), a.scale)
        n = len(sd_host["adc"])
        cap = n // 8
        sd = B.strips_to_device(sd_host)
        out = B.alloc_clusters(cap)
        ws = torch.empty(max(ctx.workspace_bytes(B.MKF_CALL_CLUSTER_STRIPS, 0, n, cap), 256), dtype=torch.uint8, device="cuda")

        def step():
            ctx.cluster_strips(sd, sp, out, ws)

        def units():
            return float(n)

        def e2e_step():
            r = ctx.cluster_strips_host(strips_p, sp, cap)
            return float(n), r["h2d_bytes"], r["d2h_bytes"]
    else:
        which = int(a.workload[-1])
        ev, prm = make_build_workload(which, rank_seed(a.seed, rank), a.scale)
        geom, hits, s = ev["geom"], ev["hits"], ev["seeds"]
        seeds = dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"], event=s["event"], hits=s["hits"])
        ctx = B.Context(geom, prm)
        dh = B.hits_to_device(hits)
        nh, nev, n = hits["x"].shape[0], hits["n_events"], s["par"].shape[1]
        idx, ws = B.alloc_hit_index(ctx, nev, nh)
        ds = B.to_device(seeds, ["par", "cov", "q", "plan", "event", "hits"])
        out = B.alloc_build_out(n, ctx.max_plan_len)
        dedup = which == 4
        if dedup:
            counts = np.bincount(s["event"], minlength=nev)
            toff = torch.from_numpy(np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)).cuda()
            keep = torch.empty(n, dtype=torch.uint8, device="cuda")
            nk = torch.empty(nev, dtype=torch.int32, device="cuda")
            ws2 = torch.empty(max(ctx.workspace_bytes(B.CALL_REMOVE_DUPLICATES, nev, nh, n), 256), dtype=torch.uint8, device="cuda")

        def step():
            ctx.build_hit_index(dh, idx, ws)
            ctx.build_tracks(dh, idx, ds, ds["event"], ds["hits"], ds["plan"], out, out["chi2"], out["score"], out["nhits"],
                             out["nmiss"], out["hit_ids"], out["status"])
            if dedup:
                ctx.remove_duplicates(nh, toff, out["hit_ids"], out["nhits"], out["score"], keep, nk, ws2)

        def units():
            return float(nev)

        def e2e_step():
            r = ctx.build_host(hits_p, seeds_p, seeds_p["event"], seeds_p["hits"], seeds_p["plan"], dedup=dedup)
            return float(nev), r["h2d_bytes"], r["d2h_bytes"]

    sampler = ClockSampler(local_rank) if rank == 0 else None
    for _ in range(warm):
        step()
    barrier()
    l0 = ctx.launch_count()
    t0 = time.time()
    ev0.record()
    for _ in range(a.steps):
        step()
    ev1.record()
    barrier()
    t1 = time.time()
    launches = ctx.launch_count() - l0
    ms_total = ev0.elapsed_time(ev1)
    u = units()
    clocks = sampler.stop(t0, t1) if sampler else None
    ms_total, u_all = aggregate(ms_total, u, world, "cuda")
    ms_step = ms_total / a.steps
    value = u_all / (ms_step * 1e-3)

    # ---- end to end through the host-buffer C-ABI call (pinned host memory) --------------------------------------
    def pin(d, keys):
        return {k: torch.from_numpy(np.ascontiguousarray(d[k])).pin_memory().numpy() for k in keys}
    if is_strips:
        strips_p = pin(sd_host, ["module_off", "adc", "noise", "bad"])
    else:
        hits_p = pin(hits, ["layer_off", "x", "y", "z", "V"]); hits_p["n_events"] = hits["n_events"]
        seeds_p = pin(seeds, list(seeds.keys()))
    e2e_step()                                            # warm the stream-ordered pool
    barrier()
    te = time.perf_counter()
    for _ in range(a.e2e_steps):
        eu, h2d, d2h = e2e_step()
    barrier()
    e2e_s = (time.perf_counter() - te) / a.e2e_steps
    e2e_s, eu = aggregate(e2e_s, eu, world, "cuda")
    e2e = dict(value=eu / e2e_s, unit=unit, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h), steps=a.e2e_steps,
               ms_per_step=1e3 * e2e_s, host_memory="pinned")

    if rank != 0:
        return
    # ---- roofline of the dominant kernel ----------------------------------------------------------------------------
    if is_fit:
        steps_per_launch = u                                  # one launch = one step = all layer-steps of this rank
        t_launch = ms_total / a.steps * 1e-3
        ach = ALGO_FLOP_PER_LAYER_STEP * steps_per_launch / t_launch / 1e12
        roof = dict(bound="alu", kernel="mkf_fit_backward_kernel" if backward else "mkf_fit_kernel", achieved=ach, peak=pk["fp32_tflops"], unit="TFLOP/s", frac=ach / pk["fp32_tflops"],
                    traffic=NCU_TRAFFIC_BYTES_FIT_FULL if (a.scale == 1.0 and not backward) else None,
                    algorithmic_bytes=ALGO_BYTES_PER_LAYER_STEP * steps_per_launch, peak_source="148 SM x 128 FP32 lanes x 2 flop x %.0f MHz (%s max clock)" % (pk["sm_max_mhz"], pk["source"]),
                    algorithmic_flop_per_layer_step=ALGO_FLOP_PER_LAYER_STEP,
                    hbm=dict(achieved=ALGO_BYTES_PER_LAYER_STEP * steps_per_launch / t_launch / 1e9, peak=pk["hbm_gbs"], unit="GB/s",
                             frac=ALGO_BYTES_PER_LAYER_STEP * steps_per_launch / t_launch / 1e9 / pk["hbm_gbs"]))
    elif is_strips:
        nclu = int(out["n_clusters"].item())
        algo = STRIP_BYTES_IN * u + STRIP_BYTES_PER_CLUSTER * nclu
        t_launch = ms_total / a.steps * 1e-3
        roof = dict(bound="hbm", kernel="sc_cluster_kernel", achieved=algo / t_launch / 1e9, peak=pk["hbm_gbs"], unit="GB/s",
                    frac=algo / t_launch / 1e9 / pk["hbm_gbs"], traffic=NCU_TRAFFIC_BYTES_STRIPS_FULL if a.scale == 1.0 else None,
                    algorithmic_bytes=algo, clusters=nclu, peak_source=pk["source"],
                    note="7 B per strip in (adc u16, noise f32, bad u8) + 20 B per cluster out; the timed step also holds one memset of the tile states")
    else:
        roof = dict(bound="hbm", kernel="mkf_build_kernel", achieved=None, peak=pk["hbm_gbs"], unit="GB/s", frac=None, traffic=None,
                    note="building is reported, not held to the 50% bar (BASELINE.json north_star); see DESIGN.md §6")
    # ---- cpu baseline: the oracle as it stands on a bounded sample ---------------------------------------------------
    cpu = None
    if not a.no_cpu_baseline:
        if is_fit:
            n_s = min(n, 1000000)
            rate, dt, cores, st, r = oracle_fit_rate(geom, prm, hits, seeds, n_s, backward=backward)
            cpu = dict(value=rate, unit=unit, cores=cores, kind="oracle", sample="first %d helices of the workload (%d layer-steps, %.1f s)" % (n_s, st, dt))
            # parity of the timed launch configuration on that same sample (the oracle results are already here)
            from workloads import parity
            g = {k: out[k][..., :n_s].cpu().numpy() for k in ("par", "cov", "chi2", "nfit", "status")}
            ok = r["nfit"] > 0
            where = parity.first_layer_of_backward_fit if backward else parity.last_layer_of_fit
            lay, kinds, pos = where(geom, seeds["plan"][:n_s], seeds["track_hits"][:, :n_s], r["nfit"])
            cpu["parity"] = dict(n=int(n_s), nfit_identical=bool(np.array_equal(g["nfit"], r["nfit"])),
                                 status_identical=bool(np.array_equal(g["status"].view(np.uint32), r["status"])),
                                 par_max=float(parity.param_errors(g["par"], r["par"], pos)[ok].max()),
                                 cov_max=float(parity.cov_errors(g["cov"], r["cov"], r["par"], kinds)[ok].max()),
                                 chi2_max=float(parity.chi2_errors(g["chi2"], r["chi2"])[ok].max()),
                                 tol=dict(par=parity.TOL_PAR, cov=parity.TOL_COV, chi2=parity.TOL_CHI2))
        elif is_strips:
            nm = len(sd_host["module_off"]) - 1
            rate, dt, cores, r = oracle_strip_rate(sd_host, sp, nm)
            cpu = dict(value=rate, unit=unit, cores=cores, kind="oracle", sample="the whole workload, %d strips (%.1f s)" % (n, dt))
            k = len(r["module"])
            g = {key: out[key][:k].cpu().numpy() for key in ("module", "first", "last", "charge", "bary")}
            cpu["parity"] = dict(n_clusters_oracle=k, n_clusters_identical=bool(k == nclu),
                                 identical=bool(k == nclu and all(np.array_equal(g[key].view(np.uint32), r[key].view(np.uint32)) for key in g)))
        else:
            n_ev = min(nev, 4)
            rate, dt, cores, r, m = oracle_build_rate(ev, prm, n_ev, dedup)
            cpu = dict(value=rate, unit=unit, cores=cores, kind="oracle", sample="first %d events of the workload (%.1f s)" % (n_ev, dt))
            hid = out["hit_ids"].cpu().numpy()[:, m]
            same = np.all(hid == r["hit_ids"], axis=0)
            cpu["parity"] = dict(n=int(m.sum()), hit_lists_identical=float(same.mean()),
                                 mismatches_with_margin_above_1e_3=int((r["margin"][~same] >= 1e-3).sum()),
                                 chi2_max=float((np.abs(out["chi2"].cpu().numpy()[m] - r["chi2"]) / np.maximum(r["chi2"], 1.0))[same].max()))
    print(json.dumps(dict(metric=metric, value=value, unit=unit, n_gpus=world, steps=a.steps, warmup=warm, ms_per_step=ms_step,
                          higher_is_better=True, scaling="weak", vs_baseline=None, dtype="u16/f32" if is_strips else "f32", data="synthetic", config=cfg,
                          clocks=clocks, e2e=e2e, gpu_launches=int(launches), roofline=roof, cpu_baseline=cpu, impl="mkf",
                          units_per_step=u_all)))


if __name__ == "__main__":
    main()
