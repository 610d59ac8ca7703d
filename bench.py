"""bench.py — the hot path of mkFit-style track reconstruction on one B200: KF layer-steps/s of mkf_fit on
BASELINE.json configs[1] (the headline line) and, in the same JSON line under `workloads`, every other workload:
the fit on hit lists in scattered order, the backward fit, track building on configs[2..4] (hit index + building
[+ duplicate removal]), the fit chained from a build, and strip clustering.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl mkf|reference] [--workload all|fit|fit_shuffled|fitback|build2|build3|build4|strips]
    python -m torch.distributed.run --nnodes=1 --nproc-per-node N --master-addr 127.0.0.1 --master-port P bench.py --gpus N ...

One JSON line on rank 0 (contract in DESIGN.md §8). A "step" is one pass of the whole path over the workload with
inputs resident in HBM; `e2e` is the same pass through the host-buffer C-ABI call (pinned host memory, copies
timed). Events/tracks are independent, so N > 1 shards them with no collective (weak scaling: every rank owns a
full-size workload generated from seed+rank); the `workloads` object is produced at N = 1 only.
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

from workloads import assemble                                    # noqa: E402
from workloads.assemble import make_fit_workload, make_build_workload, make_strip_workload, STRIP_EVENTS, STRIP_MODULES   # noqa: E402,F401

# ---- algorithmic work per unit ----------------------------------------------------------------------
ALGO_FLOP_PER_LAYER_STEP = 1000.0        # SURVEY.md §8 d: propagate 150 + transport 420 + material 90 + update 340
ALGO_BYTES_PER_LAYER_STEP = 54.0         # hit 36 B + index 4 B + state in/out amortised 14 B (hits read in id order)
ALGO_BYTES_PER_LAYER_STEP_REC = 66.0     # 48-byte hit record + 4 + 14 (hits gathered by scattered id)
FP32_LANES_PER_SM, N_SM = 128, 148
STRIP_BYTES_IN, STRIP_BYTES_PER_CLUSTER = 7, 20
HIT_INDEX_BYTES_PER_HIT = 100.0          # SURVEY.md §8 d: read 36, keys 8, sort passes, ids and offsets
# building (SURVEY.md §8 d): per candidate-layer-step 660 flop (propagate + transport + material), 70 flop per chi2
# evaluation, 340 per update; 16 B per hit position tested, 32 B per covariance read, 48 B per hit used in an update
BUILD_FLOP_STEP, BUILD_FLOP_CHI2, BUILD_FLOP_UPDATE = 660.0, 70.0, 340.0
BUILD_BYTES_POS, BUILD_BYTES_COV, BUILD_BYTES_UPD = 16.0, 32.0, 48.0


def peaks():
    p = dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")
    try:
        m = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        p.update(hbm_gbs=float(m["hbm_gbs"]), sm_max_mhz=float(m.get("sm_max_mhz", 1965.0)), source="measured")
    except Exception:
        pass
    p["fp32_tflops"] = N_SM * FP32_LANES_PER_SM * 2 * p["sm_max_mhz"] * 1e6 / 1e12
    p["fp32_source"] = "148 SM x 128 FP32 lanes x 2 flop x %.0f MHz (%s max clock; unit counts from the Blackwell guide)" % (p["sm_max_mhz"], p["source"])
    return p


def ncu_traffic(kernel, units):
    """dram__bytes_read + dram__bytes_write of one launch of `kernel` from the last `ncu --set full` capture, scaled
    from the units (layer-steps, events) of the captured launch to those of this run's launch (the kernels stream:
    traffic is linear in the units). profiles/traffic.json holds the captured bytes, units, commit and workload."""
    try:
        t = json.load(open(os.path.join(ROOT, "profiles", "traffic.json")))[kernel]
        return float(t["bytes"]) * float(units) / float(t["units"]), t.get("commit"), t.get("workload")
    except Exception:
        return None, None, None


# ---------------------------------------------------------------------------------------------------------------
# ranks: events / tracks are independent, so a rank owns its own workload and nothing but timings is exchanged
# ---------------------------------------------------------------------------------------------------------------
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
# clocks: one nvidia-smi sampler for the whole run, read back per timed window
# ---------------------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = "clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown," \
        "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap"

    def __init__(self, index):
        self.samples, self.proc = [], None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "10"], stdout=subprocess.PIPE,
                                         stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.samples.append((time.time(), line.strip()))

    def window(self, t0, t1):
        inside = [s for t, s in self.samples if t0 <= t <= t1]
        in_window = bool(inside)
        if not inside:                                   # timed region shorter than the sampling period: nearest samples
            for _ in range(10):
                if any(t > t1 for t, _ in self.samples):
                    break
                time.sleep(0.02)
            near = sorted(self.samples, key=lambda ts: abs(ts[0] - 0.5 * (t0 + t1)))[:3]
            inside = [s for _, s in near]
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

    def close(self):
        if self.proc:
            self.proc.terminate()


# ---------------------------------------------------------------------------------------------------------------
# oracle legs (cpu_baseline of the mkf arm, and the whole --impl reference arm)
# ---------------------------------------------------------------------------------------------------------------
def oracle_fit_rate(geom, prm, hits, seeds, n_tracks, repeat=1, backward=False):
    """Best of `repeat` runs of the oracle fit on the first n_tracks tracks."""
    from oracle import mkfo
    o = mkfo.Oracle(geom, prm)
    sl = slice(0, n_tracks)
    args = (hits, seeds["par"][:, sl], seeds["cov"][:, sl], seeds["q"][sl], seeds["plan"][sl], np.ascontiguousarray(seeds["track_hits"][:, sl]))
    best = None
    for _ in range(repeat):
        t = time.perf_counter()
        r = o.fit_backward(*args) if backward else o.fit(*args)
        dt = time.perf_counter() - t
        best = dt if best is None else min(best, dt)
    return float(r["nfit"].sum()) / best, best, o.num_threads(), int(r["nfit"].sum()), r


def sub_events(ev, n_events):
    """The first n_events events of a build workload (hits, seeds mask)."""
    nl = len(ev["geom"]["layers"])
    h, s = ev["hits"], ev["seeds"]
    lo = h["layer_off"].reshape(-1, nl + 1)
    nh = int(lo[n_events - 1, nl])
    sub = dict(n_events=n_events, layer_off=np.ascontiguousarray(lo[:n_events]).reshape(-1), x=h["x"][:nh], y=h["y"][:nh], z=h["z"][:nh],
               V=np.ascontiguousarray(h["V"][:, :nh]))
    return sub, s["event"] < n_events


def oracle_build_rate(ev, prm, n_events, dedup, repeat=1):
    from oracle import mkfo
    s = ev["seeds"]
    o = mkfo.Oracle(ev["geom"], prm)
    sub, m = sub_events(ev, n_events)
    best = None
    for _ in range(repeat):
        t = time.perf_counter()
        idx = o.build_hit_index(sub)
        r = o.build_tracks(sub, idx, s["par"][:, m], s["cov"][:, m], s["q"][m], s["event"][m], np.ascontiguousarray(s["hits"][:, m]), s["plan"][m])
        if dedup:
            counts = np.bincount(s["event"][m], minlength=n_events)
            r["dedup"] = o.remove_duplicates(np.concatenate([[0], np.cumsum(counts)]).astype(np.int32), r["hit_ids"], r["nhits"], r["score"].astype(np.float32))
        dt = time.perf_counter() - t
        best = dt if best is None else min(best, dt)
    return n_events / best, best, o.num_threads(), r, m


def oracle_strip_rate(d, sp, n_modules, repeat=1):
    from oracle import mkfo
    ns = int(d["module_off"][n_modules])
    best = None
    for _ in range(repeat):
        t = time.perf_counter()
        r = mkfo.cluster_strips(d["module_off"][:n_modules + 1], d["adc"][:ns], d["noise"][:ns], d["bad"][:ns], **sp)
        dt = time.perf_counter() - t
        best = dt if best is None else min(best, dt)
    return ns / best, best, 1, r


NAMES = dict(fit="configs[1]: track fit, 4M helices x 17 barrel layers, MS + dE/dx, seeds from 3 hits, cov x100; hits in id order (SoA planes)",
             fit_shuffled="configs[1] workload with the hit ids randomly permuted (the order a fit meets after track building); hits read as 48-byte records",
             fitback="configs[1] workload, backward fit (SURVEY f1): seeds = forward fit at the last hit, covariance x100",
             build2="configs[2]: building, barrel, 100 events x 1000 tracks + 20k noise hits, top 6",
             build3="configs[3]: building, barrel+endcap, 200 events x 1500 seeds, ~80k hits/event",
             build4="configs[4]: batched building + duplicate removal, 64 events x 6000 seeds, ~300k hits/event, top 8",
             strips="strip clustering (SURVEY f3, reading R8): %d events x %d modules of 512 / 256 strips, ~1 %% occupancy, 1 %% bad strips" % (STRIP_EVENTS, STRIP_MODULES))
METRIC = dict(fit=("KF layer-steps/s (propagate+update)", "layer-steps/s"), build=("built events/s", "events/s"), strips=("clustered strips/s", "strips/s"))


def kind_of(w):
    return "fit" if w.startswith("fit") else "strips" if w == "strips" else "build"


# ---------------------------------------------------------------------------------------------------------------
# the reference arm: the oracle alone on host cores, bounded sample per step
# ---------------------------------------------------------------------------------------------------------------
def reference_arm(a, warm):
    w = "fit" if a.workload == "all" else a.workload
    kind = kind_of(w)
    metric, unit = METRIC[kind]
    cfg = dict(workload=NAMES[w], scale=a.scale, l2="inputs larger than L2 (no flush needed)", seed=a.seed)
    if kind == "fit":
        n_s = max(1, int(round(200000 * min(1.0, a.scale * 20))))
        geom, prm, hits, seeds, _ = make_fit_workload(a.seed, n_s / 4000000.0)
        if w == "fit_shuffled":
            hits, seeds = assemble.shuffle_hit_order(hits, seeds, a.seed)
        if w == "fitback":
            from oracle import mkfo
            f = mkfo.Oracle(geom, prm).fit(hits, seeds["par"], seeds["cov"], seeds["q"], seeds["plan"], seeds["track_hits"])
            th = seeds["track_hits"].copy()
            th[np.cumsum(th >= 0, 0) > f["nfit"][None]] = -1
            seeds = dict(seeds, par=f["par"].astype(np.float32), cov=(100.0 * f["cov"]).astype(np.float32), track_hits=th)
        rates = []
        for k in range(warm + a.steps):
            rate, dt, cores, steps, _ = oracle_fit_rate(geom, prm, hits, seeds, n_s, backward=(w == "fitback"))
            if k >= warm:
                rates.append((rate, dt))
        sample = "first %d helices of the workload per step (%d layer-steps)" % (n_s, steps)
    elif kind == "strips":
        d, sp = make_strip_workload(a.seed, min(1.0, a.scale) * 4.0 / STRIP_EVENTS)
        rates = []
        for k in range(warm + a.steps):
            rate, dt, cores, _ = oracle_strip_rate(d, sp, len(d["module_off"]) - 1)
            if k >= warm:
                rates.append((rate, dt))
        sample = "%d modules (%d strips) of the workload per step" % (len(d["module_off"]) - 1, len(d["adc"]))
    else:
        which = int(w[-1])
        nev_full = assemble.BUILD_EVENTS[which]
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


# ---------------------------------------------------------------------------------------------------------------
# the mkf arm
# ---------------------------------------------------------------------------------------------------------------
class Runner:
    """Times one workload: W warm-up steps, K timed steps between CUDA events on torch's current stream (the stream the
    library launches on), barrier + synchronize on both sides, max over ranks."""

    def __init__(self, a, rank, local_rank, world, sampler):
        import torch
        self.torch, self.a, self.rank, self.local_rank, self.world, self.sampler = torch, a, rank, local_rank, world, sampler
        self.warm = max(a.warmup, 3)
        self.pk = peaks()
        self.cdev = "cpu" if os.environ.get("MKF_BENCH_BACKEND") == "gloo" else "cuda"     # where the collectives' tensors live

    def barrier(self, ranks=True):
        if self.world > 1 and ranks:
            import torch.distributed as dist
            dist.barrier()
        self.torch.cuda.synchronize()

    def timed(self, ctx, step, steps=None, warm=None, ranks=True):
        """ranks=False: a measurement only rank 0 makes (no barrier between the ranks: the others are not there)."""
        torch = self.torch
        steps = steps or self.a.steps
        for _ in range(self.warm if warm is None else warm):
            step()
        self.barrier(ranks)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        l0 = ctx.launch_count()
        t0 = time.time()
        e0.record()
        for _ in range(steps):
            step()
        e1.record()
        self.barrier(ranks)
        t1 = time.time()
        clocks = self.sampler.window(t0, t1) if self.sampler else None
        return e0.elapsed_time(e1), ctx.launch_count() - l0, clocks

    def e2e(self, fn, unit):
        """fn() -> (units, h2d bytes, d2h bytes): one untimed call (grows the context's arena once), then timed calls."""
        fn()
        self.barrier()
        te = time.perf_counter()
        for _ in range(self.a.e2e_steps):
            eu, h2d, d2h = fn()
        self.barrier()
        s = (time.perf_counter() - te) / self.a.e2e_steps
        s, eu = aggregate(s, eu, self.world, self.cdev)
        return dict(value=eu / s, unit=unit, h2d_bytes_per_step=int(h2d), d2h_bytes_per_step=int(d2h), steps=self.a.e2e_steps,
                    ms_per_step=1e3 * s, host_memory="pinned", h2d_gbs=h2d / s / 1e9,
                    note="H2D of all inputs, kernels and D2H of all outputs inside the timed region (wall clock around the synchronous call)")

    def pin(self, d, keys):
        torch = self.torch
        return {k: torch.from_numpy(np.ascontiguousarray(d[k])).pin_memory().numpy() for k in keys}


def run_fit(R, w, seed, workload=None):
    """fit | fit_shuffled | fitback on configs[1]. Returns the record (and keeps nothing on the device)."""
    import torch
    from paper_2002_06295_b200 import binding as B
    from workloads import parity
    a, pk = R.a, R.pk
    backward, shuffled = w == "fitback", w == "fit_shuffled"
    geom, prm, hits, seeds, _ = workload if workload is not None else make_fit_workload(seed, a.scale)
    if shuffled:
        hits, seeds = assemble.shuffle_hit_order(hits, seeds, seed)
    ctx = B.Context(geom, prm)
    dh = B.hits_to_device(hits)
    ds = B.to_device(seeds, ["par", "cov", "q", "plan", "track_hits"])
    n = seeds["par"].shape[1]
    out = B.alloc_fit_out(n)
    extra = {}
    if shuffled:                                           # the records are an input layout: packed once, outside the step
        dh["rec"] = torch.empty(12 * hits["x"].shape[0], dtype=torch.float32, device="cuda")
        ms_pack, _, _ = R.timed(ctx, lambda: ctx.pack_hits(dh, dh["rec"]), steps=5, warm=2)
        extra["pack_hits_ms"] = ms_pack / 5
        extra["pack_hits_gbs"] = 84.0 * hits["x"].shape[0] / (ms_pack / 5 * 1e-3) / 1e9
    if backward:                                           # seeds of the backward fit: one untimed forward fit
        ctx.fit(dh, ds, ds["plan"], ds["track_hits"], out, out["chi2"], out["nfit"], out["status"])
        th = ds["track_hits"].clone()
        th[torch.cumsum((th >= 0).to(torch.int32), 0) > out["nfit"][None]] = -1
        ds = dict(ds, par=out["par"].clone(), cov=(100.0 * out["cov"]), track_hits=th.contiguous())
        seeds = {k: v.cpu().numpy() for k, v in ds.items()}

    def step():
        ctx.fit(dh, ds, ds["plan"], ds["track_hits"], out, out["chi2"], out["nfit"], out["status"], backward=backward)

    ms_total, launches, clocks = R.timed(ctx, step)
    u = float(out["nfit"].sum().item())
    ms_total, u_all = aggregate(ms_total, u, R.world, R.cdev)
    ms_step = ms_total / a.steps
    rec = dict(workload=NAMES[w], metric=METRIC["fit"][0], unit=METRIC["fit"][1], value=u_all / (ms_step * 1e-3), ms_per_step=ms_step,
               steps=a.steps, warmup=R.warm, units_per_step=u_all, gpu_launches=int(launches), clocks=clocks, dtype="f32", **extra)
    # ---- end to end through the host-buffer C-ABI call ---------------------------------------------------------
    if not a.no_e2e:
        hits_p = R.pin(hits, ["layer_off", "x", "y", "z", "V"]); hits_p["n_events"] = hits["n_events"]
        seeds_p = R.pin(seeds, ["par", "cov", "q", "plan", "track_hits"])

        out_p = B.alloc_fit_out_host(n)

        def e2e_step():
            r = ctx.fit_host(hits_p, seeds_p, seeds_p["plan"], seeds_p["track_hits"], backward=backward, out=out_p)
            return float(r["nfit"].sum()), r["h2d_bytes"], r["d2h_bytes"]
        rec["e2e"] = R.e2e(e2e_step, METRIC["fit"][1])
        del hits_p, seeds_p, out_p
    # ---- f1: the two-filter smoother (mkf_fit_smooth, reading R14) on the first quarter of the tracks ----------------
    if w == "fit" and not a.no_chain:
        ns = max(1, n // 4)
        mpl = ds["track_hits"].shape[0]
        sds = {k: (v[..., :ns].contiguous() if k != "plan" and k != "q" else v[:ns].contiguous()) for k, v in ds.items()}
        par_s = torch.empty((mpl, 6, ns), dtype=torch.float32, device="cuda")
        cov_s = torch.empty((mpl, 21, ns), dtype=torch.float32, device="cuda")
        so = B.alloc_fit_out(ns)
        wss = torch.empty(max(ctx.workspace_bytes(B.CALL_FIT_SMOOTH, 0, 0, ns), 256), dtype=torch.uint8, device="cuda")

        def smooth_step():
            ctx.fit_smooth(dh, sds, sds["plan"], sds["track_hits"], par_s, cov_s, so["chi2"], so["nfit"], so["status"], wss)
        ms_s, _, clk_s = R.timed(ctx, smooth_step, steps=min(a.steps, 10))
        us = float(so["nfit"].sum().item())
        ts = ms_s / min(a.steps, 10) * 1e-3
        rec["smoother"] = dict(workload="mkf_fit_smooth on the first %d helices of configs[1]: forward pass, backward pass and the combined state at every fitted hit" % ns,
                               value=us / ts, unit="smoothed layer-steps/s", ms_per_step=ts * 1e3, units_per_step=us, clocks=clk_s,
                               out_bytes_per_layer_step=27 * 4, workspace_bytes=int(wss.numel()))
        del par_s, cov_s, wss, sds
    if R.rank != 0:
        return rec
    # ---- roofline of the kernel (the step is one launch) ---------------------------------------------------------
    t_launch = ms_step * 1e-3
    kernel = "mkf_fit_backward_kernel" if backward else "mkf_fit_kernel"
    bps = ALGO_BYTES_PER_LAYER_STEP_REC if shuffled else ALGO_BYTES_PER_LAYER_STEP
    ach = ALGO_FLOP_PER_LAYER_STEP * u / t_launch / 1e12
    traffic, tcommit, twl = ncu_traffic(kernel + ("/records" if shuffled else ""), u)
    rec["roofline"] = dict(bound="alu", kernel=kernel, achieved=ach, peak=pk["fp32_tflops"], unit="TFLOP/s", frac=ach / pk["fp32_tflops"],
                           traffic=traffic, traffic_commit=tcommit, algorithmic_bytes=bps * u,
                           peak_source=pk["fp32_source"], algorithmic_flop_per_layer_step=ALGO_FLOP_PER_LAYER_STEP,
                           note="algorithmic 1.0 kflop per layer-step (SURVEY §8d); the U-D kernels execute fewer: see profiles/ for the executed FP32 rate",
                           hbm=dict(achieved=bps * u / t_launch / 1e9, peak=pk["hbm_gbs"], unit="GB/s", frac=bps * u / t_launch / 1e9 / pk["hbm_gbs"],
                                    bytes_per_layer_step=bps, peak_source=pk["source"]))
    # ---- cpu baseline: the oracle as it stands on a bounded sample, best of 3, with the parity of that sample ------
    if not a.no_cpu_baseline:
        n_s = min(n, 1000000)
        rate, dt, cores, st, r = oracle_fit_rate(geom, prm, hits, seeds, n_s, repeat=3, backward=backward)
        cpu = dict(value=rate, unit=METRIC["fit"][1], cores=cores, kind="oracle", sample="first %d helices of the workload (%d layer-steps, best of 3: %.1f s)" % (n_s, st, dt))
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
        rec["cpu_baseline"] = cpu
    ctx.close()
    return rec


def run_build(R, w, seed):
    import torch
    from paper_2002_06295_b200 import binding as B
    a, pk = R.a, R.pk
    which = int(w[-1])
    ev, prm = make_build_workload(which, seed, a.scale)
    geom, hits, s = ev["geom"], ev["hits"], ev["seeds"]
    seeds = dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"], event=s["event"], hits=s["hits"])
    ctx = B.Context(geom, prm)
    dh = B.hits_to_device(hits)
    nh, nev, n = hits["x"].shape[0], hits["n_events"], s["par"].shape[1]
    idx, ws = B.alloc_hit_index(ctx, nev, nh)
    wsb = B.alloc_build_ws(ctx, nev, nh, n)
    ds = B.to_device(seeds, ["par", "cov", "q", "plan", "event", "hits"])
    out = B.alloc_build_out(n, ctx.max_plan_len)
    dedup = which == 4
    if dedup:
        counts = np.bincount(s["event"], minlength=nev)
        toff = torch.from_numpy(np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)).cuda()
        keep = torch.empty(n, dtype=torch.uint8, device="cuda")
        nk = torch.empty(nev, dtype=torch.int32, device="cuda")
        ws2 = torch.empty(max(ctx.workspace_bytes(B.CALL_REMOVE_DUPLICATES, nev, nh, n), 256), dtype=torch.uint8, device="cuda")

    def index():
        ctx.build_hit_index(dh, idx, ws)

    def tracks():
        ctx.build_tracks(dh, idx, ds, ds["event"], ds["hits"], ds["plan"], out, out["chi2"], out["score"], out["nhits"],
                         out["nmiss"], out["hit_ids"], out["status"], ws=wsb)

    def dd():
        ctx.remove_duplicates(nh, toff, out["hit_ids"], out["nhits"], out["score"], keep, nk, ws2)

    def step():
        index(); tracks()
        if dedup:
            dd()

    ms_total, launches, clocks = R.timed(ctx, step)
    ms_total, u_all = aggregate(ms_total, float(nev), R.world, R.cdev)
    ms_step = ms_total / a.steps
    rec = dict(workload=NAMES[w], metric=METRIC["build"][0], unit=METRIC["build"][1], value=u_all / (ms_step * 1e-3), ms_per_step=ms_step,
               steps=a.steps, warmup=R.warm, units_per_step=u_all, gpu_launches=int(launches), clocks=clocks, dtype="f32",
               n_hits=int(nh), n_seeds=int(n))
    # the parts of the step, timed alone (same inputs, same stream)
    ms_i, _, _ = R.timed(ctx, index, warm=1)
    ms_t, _, _ = R.timed(ctx, tracks, warm=1)
    parts = dict(hit_index_ms=ms_i / a.steps, build_tracks_ms=ms_t / a.steps)
    if dedup:
        ms_d, _, _ = R.timed(ctx, dd, warm=1)
        parts["remove_duplicates_ms"] = ms_d / a.steps
    rec["parts"] = parts
    if not a.no_e2e:
        hits_p = R.pin(hits, ["layer_off", "x", "y", "z", "V"]); hits_p["n_events"] = hits["n_events"]
        seeds_p = R.pin(seeds, list(seeds.keys()))

        out_p = B.alloc_build_out_host(n, ctx.max_plan_len)

        def e2e_step():
            r = ctx.build_host(hits_p, seeds_p, seeds_p["event"], seeds_p["hits"], seeds_p["plan"], dedup=dedup, out=out_p)
            return float(nev), r["h2d_bytes"], r["d2h_bytes"]
        rec["e2e"] = R.e2e(e2e_step, METRIC["build"][1])
        del hits_p, seeds_p
    if R.rank != 0:
        return rec
    # ---- work counters of one untimed pass -> algorithmic flop and bytes of mkf_build_tracks ------------------------
    cnt = torch.zeros(8, dtype=torch.int64, device="cuda")
    ctx.set_build_counters(cnt)
    tracks()
    torch.cuda.synchronize()
    ctx.set_build_counters(None)
    c = [int(v) for v in cnt.cpu().numpy()]
    cand_steps, pos_tests, chi2_evals, accepted, updates = c[0], c[1], c[2], c[3], c[4]
    t_b = parts["build_tracks_ms"] * 1e-3
    out_bytes = n * (27 * 4 + 5 * 4 + ctx.max_plan_len * 4)
    in_bytes = n * (27 * 4 + 1 + 1 + 4 + 12)
    algo_bytes = BUILD_BYTES_POS * pos_tests + BUILD_BYTES_COV * chi2_evals + BUILD_BYTES_UPD * updates + out_bytes + in_bytes
    algo_flop = BUILD_FLOP_STEP * cand_steps + BUILD_FLOP_CHI2 * chi2_evals + BUILD_FLOP_UPDATE * updates
    traffic, tcommit, twl = ncu_traffic("mkf_build_kernel/" + w, nev)
    rec["roofline"] = dict(bound="hbm", kernel="mkf_build_kernel", achieved=algo_bytes / t_b / 1e9, peak=pk["hbm_gbs"], unit="GB/s",
                           frac=algo_bytes / t_b / 1e9 / pk["hbm_gbs"], traffic=traffic, traffic_commit=tcommit,
                           algorithmic_bytes=algo_bytes, peak_source=pk["source"],
                           alu=dict(achieved=algo_flop / t_b / 1e12, peak=pk["fp32_tflops"], unit="TFLOP/s", frac=algo_flop / t_b / 1e12 / pk["fp32_tflops"],
                                    algorithmic_flop=algo_flop, peak_source=pk["fp32_source"]),
                           candidate_layer_steps=cand_steps, candidate_layer_steps_per_s=cand_steps / t_b,
                           hit_positions_tested=pos_tests, chi2_evaluations=chi2_evals, chi2_evaluations_per_s=chi2_evals / t_b,
                           hits_accepted=accepted, updates=updates,
                           note="algorithmic work of mkf_build_tracks from device counters of one untimed pass: 16 B per hit position tested + 32 B per "
                                "covariance read + 48 B per update + seeds in / tracks out; 660 flop per candidate-layer-step + 70 per chi2 + 340 per update "
                                "(SURVEY §8d). Building is latency-bound gathers: both fractions are reported, neither is held to the 50 % bar",
                           hit_index=dict(bound="hbm", achieved=HIT_INDEX_BYTES_PER_HIT * nh / (parts["hit_index_ms"] * 1e-3) / 1e9, peak=pk["hbm_gbs"], unit="GB/s",
                                          frac=HIT_INDEX_BYTES_PER_HIT * nh / (parts["hit_index_ms"] * 1e-3) / 1e9 / pk["hbm_gbs"],
                                          algorithmic_bytes=HIT_INDEX_BYTES_PER_HIT * nh, bytes_per_hit=HIT_INDEX_BYTES_PER_HIT))
    if not a.no_cpu_baseline:
        n_ev = min(nev, 4)
        rate, dt, cores, r, m = oracle_build_rate(ev, prm, n_ev, dedup, repeat=3 if which != 4 else 2)
        cpu = dict(value=rate, unit=METRIC["build"][1], cores=cores, kind="oracle", sample="first %d events of the workload (best of %d: %.1f s)" % (n_ev, 3 if which != 4 else 2, dt))
        hid = out["hit_ids"].cpu().numpy()[:, m]
        same = np.all(hid == r["hit_ids"], axis=0)
        par = dict(n=int(m.sum()), hit_lists_identical=float(same.mean()),
                   mismatches_with_margin_above_1e_3=int((r["margin"][~same] >= 1e-3).sum()),
                   chi2_max=float((np.abs(out["chi2"].cpu().numpy()[m] - r["chi2"]) / np.maximum(r["chi2"], 1.0))[same].max()),
                   oracle_chi2_evaluations=int(r["n_chi2_evals"]))
        if dedup:
            from oracle import mkfo
            k = int(m.sum())
            d = mkfo.Oracle(geom, prm).remove_duplicates(toff.cpu().numpy()[:n_ev + 1], hid, out["nhits"].cpu().numpy()[m], out["score"].cpu().numpy()[m])
            par["duplicate_removal_identical"] = bool(np.array_equal(d["keep"], keep.cpu().numpy()[:k]))
        cpu["parity"] = par
        rec["cpu_baseline"] = cpu
    # ---- f1: the fit chained from the build (hit lists as mkf_build_tracks wrote them; hits as 48-byte records) -----
    if which == 3 and not a.no_chain:
        dh["rec"] = torch.empty(12 * nh, dtype=torch.float32, device="cuda")
        ctx.pack_hits(dh, dh["rec"])
        fo = B.alloc_fit_out(n)
        th = out["hit_ids"].clone()

        def fit_step():
            ctx.fit(dh, ds, ds["plan"], th, fo, fo["chi2"], fo["nfit"], fo["status"])
        ms_f, _, clk = R.timed(ctx, fit_step, ranks=False)
        uf = float(fo["nfit"].sum().item())
        tf = ms_f / a.steps * 1e-3
        rec["chained_fit"] = dict(workload="mkf_fit over the hit lists mkf_build_tracks wrote for configs[3] (PAPER.md:25), hits as 48-byte records",
                                  value=uf / tf, unit="layer-steps/s", ms_per_step=ms_f / a.steps, units_per_step=uf, clocks=clk,
                                  roofline=dict(bound="alu", kernel="mkf_fit_kernel", achieved=ALGO_FLOP_PER_LAYER_STEP * uf / tf / 1e12, peak=pk["fp32_tflops"],
                                                unit="TFLOP/s", frac=ALGO_FLOP_PER_LAYER_STEP * uf / tf / 1e12 / pk["fp32_tflops"]))
    # ---- f2: overlap-hit recovery on the configs[3] recipe with a quarter of the crossings seen by a second module ----
    if which == 3 and not a.no_chain:
        rec["overlap_recovery"] = run_overlap(R, seed)
    ctx.close()
    return rec


def run_overlap(R, seed):
    """mkf_build_hit_index + mkf_build_tracks_overlap (reading R15) on 50 events x scale of the configs[3]
    recipe generated with overlap_frac = 0.25 (module ids from the generator)."""
    import torch
    from paper_2002_06295_b200 import binding as B
    a = R.a
    ev, prm = make_build_workload(3, seed, 0.25 * a.scale, overlap_frac=0.25)
    geom, hits, s = ev["geom"], ev["hits"], ev["seeds"]
    ctx = B.Context(geom, prm)
    dh = B.hits_to_device(hits, with_module=True)
    nh, nev, n = hits["x"].shape[0], hits["n_events"], s["par"].shape[1]
    idx, ws = B.alloc_hit_index(ctx, nev, nh)
    ds = B.to_device(dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"], event=s["event"], hits=s["hits"]), ["par", "cov", "q", "plan", "event", "hits"])
    out = B.alloc_build_out(n, ctx.max_plan_len)
    h2 = torch.empty((ctx.max_plan_len, n), dtype=torch.int32, device="cuda")
    wso = torch.empty(max(ctx.workspace_bytes(B.CALL_BUILD_TRACKS_OVERLAP, nev, nh, n), 256), dtype=torch.uint8, device="cuda")

    def step(h2=h2):
        ctx.build_hit_index(dh, idx, ws)
        ctx.build_tracks(dh, idx, ds, ds["event"], ds["hits"], ds["plan"], out, out["chi2"], out["score"], out["nhits"],
                         out["nmiss"], out["hit_ids"], out["status"], ws=wso, hit_ids2=h2)

    ms_o, launches, clk = R.timed(ctx, step, ranks=False)             # rank 0 alone gets here
    ms_p, _, _ = R.timed(ctx, lambda: step(None), warm=1, ranks=False)
    n2 = int((h2 >= 0).sum().item())
    ctx.close()
    return dict(workload="configs[3] recipe, %d events, overlap_frac 0.25: mkf_build_hit_index + mkf_build_tracks_overlap" % nev,
                value=nev / (ms_o / a.steps * 1e-3), unit="events/s", ms_per_step=ms_o / a.steps, units_per_step=float(nev), clocks=clk,
                gpu_launches=int(launches), n_hits=int(nh), n_seeds=int(n), second_hits_attached=n2,
                ms_per_step_without_recovery=ms_p / a.steps)


def run_strips(R, w, seed):
    import torch
    from paper_2002_06295_b200 import binding as B
    from workloads import datagen
    a, pk = R.a, R.pk
    ev_g, prm_g = datagen.config(0, scale=0.001)              # clustering uses no geometry; a context needs one
    ctx = B.Context(ev_g["geom"], prm_g)
    sd_host, sp = make_strip_workload(seed, a.scale)
    n = len(sd_host["adc"])
    cap = n // 8
    sd = B.strips_to_device(sd_host)
    out = B.alloc_clusters(cap)
    ws = torch.empty(max(ctx.workspace_bytes(B.MKF_CALL_CLUSTER_STRIPS, 0, n, cap), 256), dtype=torch.uint8, device="cuda")

    def step():
        ctx.cluster_strips(sd, sp, out, ws)

    ms_total, launches, clocks = R.timed(ctx, step)
    ms_total, u_all = aggregate(ms_total, float(n), R.world, R.cdev)
    ms_step = ms_total / a.steps
    rec = dict(workload=NAMES[w], metric=METRIC["strips"][0], unit=METRIC["strips"][1], value=u_all / (ms_step * 1e-3), ms_per_step=ms_step,
               steps=a.steps, warmup=R.warm, units_per_step=u_all, gpu_launches=int(launches), clocks=clocks, dtype="u16/f32")
    if not a.no_e2e:
        strips_p = R.pin(sd_host, ["module_off", "adc", "noise", "bad"])

        def e2e_step():
            r = ctx.cluster_strips_host(strips_p, sp, cap)
            return float(n), r["h2d_bytes"], r["d2h_bytes"]
        rec["e2e"] = R.e2e(e2e_step, METRIC["strips"][1])
    if R.rank != 0:
        return rec
    nclu = int(out["n_clusters"].item())
    algo = STRIP_BYTES_IN * float(n) + STRIP_BYTES_PER_CLUSTER * nclu
    t_launch = ms_step * 1e-3
    traffic, tcommit, _ = ncu_traffic("sc_cluster_kernel", n)
    rec["roofline"] = dict(bound="hbm", kernel="sc_cluster_kernel", achieved=algo / t_launch / 1e9, peak=pk["hbm_gbs"], unit="GB/s",
                           frac=algo / t_launch / 1e9 / pk["hbm_gbs"], traffic=traffic, traffic_commit=tcommit,
                           algorithmic_bytes=algo, clusters=nclu, peak_source=pk["source"],
                           note="7 B per strip in (adc u16, noise f32, bad u8) + 20 B per cluster out; the timed step also holds one memset of the tile states")
    if not a.no_cpu_baseline:
        nm = len(sd_host["module_off"]) - 1
        rate, dt, cores, r = oracle_strip_rate(sd_host, sp, nm, repeat=3)
        cpu = dict(value=rate, unit=METRIC["strips"][1], cores=cores, kind="oracle", sample="the whole workload, %d strips (best of 3: %.1f s)" % (n, dt))
        k = len(r["module"])
        g = {key: out[key][:k].cpu().numpy() for key in ("module", "first", "last", "charge", "bary")}
        cpu["parity"] = dict(n_clusters_oracle=k, n_clusters_identical=bool(k == nclu),
                             identical=bool(k == nclu and all(np.array_equal(g[key].view(np.uint32), r[key].view(np.uint32)) for key in g)))
        rec["cpu_baseline"] = cpu
    ctx.close()
    return rec


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="mkf", choices=["mkf", "reference"])
    ap.add_argument("--workload", default="all", choices=["all", "fit", "fit_shuffled", "fitback", "build2", "build3", "build4", "strips"],
                    help="all (default): the fit on configs[1] as the headline plus every other workload under `workloads`")
    ap.add_argument("--scale", type=float, default=1.0, help="shrinks the workload (testing only; the JSON says so)")
    ap.add_argument("--seed", type=int, default=0)
    ap.add_argument("--e2e-steps", type=int, default=3)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-chain", action="store_true")
    a = ap.parse_args()
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    warm = max(a.warmup, 3)
    if a.impl == "reference":
        if rank == 0:
            reference_arm(a, warm)
        return

    import torch
    if not torch.cuda.is_available():
        raise SystemExit("bench.py --impl mkf needs a CUDA device (there is no CPU fallback)")
    # MKF_BENCH_BACKEND=gloo with MKF_BENCH_ONE_GPU=1 runs every rank on GPU 0 with host-side collectives: a test of the
    # ranks' plumbing on a one-GPU box (tests/test_gpu_bench_ranks.py), never a measurement
    if os.environ.get("MKF_BENCH_ONE_GPU") == "1":
        local_rank = 0
    torch.cuda.set_device(local_rank)
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group(os.environ.get("MKF_BENCH_BACKEND", "nccl"))
    sampler = ClockSampler(local_rank) if rank == 0 else None
    R = Runner(a, rank, local_rank, world, sampler)
    seed = rank_seed(a.seed, rank)
    run = dict(fit=run_fit, fit_shuffled=run_fit, fitback=run_fit, build2=run_build, build3=run_build, build4=run_build, strips=run_strips)
    primary = "fit" if a.workload == "all" else a.workload
    t_start = time.time()
    others = {}
    if a.workload == "all":
        wl = make_fit_workload(seed, a.scale)                  # configs[1] is generated once for its three workloads
        head = run_fit(R, "fit", seed, workload=wl)
        if world == 1:
            saved = (a.no_e2e,)
            a.no_e2e = True                                    # the end-to-end number belongs to the headline; build4 and strips get their own below
            for w in ("fit_shuffled", "fitback"):
                others[w] = run_fit(R, w, seed, workload=wl)
                torch.cuda.empty_cache()
            del wl
            for w in ("build2", "build3"):
                others[w] = run[w](R, w, seed)
                torch.cuda.empty_cache()
            a.no_e2e = saved[0]
            for w in ("build4", "strips"):
                others[w] = run[w](R, w, seed)
                torch.cuda.empty_cache()
    else:
        head = run[primary](R, primary, seed)
    if sampler:
        sampler.close()
    if rank != 0:
        return
    kind = kind_of(primary)
    cfg = dict(workload=NAMES[primary], scale=a.scale, l2="inputs larger than L2 (no flush needed)", seed=a.seed)
    line = dict(metric=METRIC[kind][0], value=head["value"], unit=METRIC[kind][1], n_gpus=world, steps=a.steps, warmup=warm,
                ms_per_step=head["ms_per_step"], higher_is_better=True, scaling="weak", vs_baseline=None, dtype=head["dtype"], data="synthetic",
                config=cfg, clocks=head["clocks"], e2e=head.get("e2e"), gpu_launches=head["gpu_launches"], roofline=head.get("roofline"),
                cpu_baseline=head.get("cpu_baseline"), impl="mkf", units_per_step=head["units_per_step"])
    for k in ("parts", "chained_fit", "overlap_recovery", "smoother", "pack_hits_ms", "pack_hits_gbs", "n_hits", "n_seeds"):
        if k in head:
            line[k] = head[k]
    if others:
        others = dict(fit={k: v for k, v in head.items() if k != "e2e"}, **others)
        line["workloads"] = others
    line["bench_wall_s"] = time.time() - t_start
    print(json.dumps(line))


if __name__ == "__main__":
    main()
