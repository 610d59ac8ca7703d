"""Helpers for the -m gpu parity tests: run the CUDA path through the binding on datagen events."""
import numpy as np
import torch

from paper_2002_06295_b200 import binding as B


def gpu_fit(ev, prm, seeds=None, backward=False):
    s = seeds if seeds is not None else ev["seeds"]
    ctx = B.Context(ev["geom"], prm)
    hits = B.hits_to_device(ev["hits"])
    sd = B.to_device(s, ["par", "cov", "q", "plan", "track_hits"])
    n = s["par"].shape[1]
    out = B.alloc_fit_out(n)
    ctx.fit(hits, sd, sd["plan"], sd["track_hits"], out, out["chi2"], out["nfit"], out["status"], backward=backward)
    torch.cuda.synchronize()
    r = {k: v.cpu().numpy() for k, v in out.items()}
    r["status"] = r["status"].view(np.uint32)
    ctx.close()
    return r


def gpu_hit_index(ev, prm, packed=True):
    ctx = B.Context(ev["geom"], prm)
    hits = B.hits_to_device(ev["hits"])
    out, ws = B.alloc_hit_index(ctx, hits["n_events"], hits["x"].shape[0], packed=packed)
    ctx.build_hit_index(hits, out, ws)
    torch.cuda.synchronize()
    r = dict(bin_off=out["bin_off"].cpu().numpy().view(np.uint32), sorted_id=out["sorted_id"].cpu().numpy(),
             vmax=out["vmax"].cpu().numpy())
    if packed:
        r["packed"] = out["packed"].cpu().numpy()
    ctx.close()
    return r


def gpu_build(ev, prm, packed=True, dedup=False):
    s = ev["seeds"]
    ctx = B.Context(ev["geom"], prm)
    hits = B.hits_to_device(ev["hits"])
    nh = hits["x"].shape[0]
    idx, ws = B.alloc_hit_index(ctx, hits["n_events"], nh, packed=packed)
    ctx.build_hit_index(hits, idx, ws)
    sd = B.to_device(dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"], event=s["event"], hits=s["hits"]),
                     ["par", "cov", "q", "plan", "event", "hits"])
    n = s["par"].shape[1]
    out = B.alloc_build_out(n, ctx.max_plan_len)
    ctx.build_tracks(hits, idx, sd, sd["event"], sd["hits"], sd["plan"], out, out["chi2"], out["score"], out["nhits"],
                     out["nmiss"], out["hit_ids"], out["status"])
    r = None
    if dedup:
        counts = np.bincount(s["event"], minlength=hits["n_events"])
        toff = torch.from_numpy(np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)).cuda()
        keep = torch.empty(n, dtype=torch.uint8, device="cuda")
        nk = torch.empty(hits["n_events"], dtype=torch.int32, device="cuda")
        ws2 = torch.empty(max(ctx.workspace_bytes(B.CALL_REMOVE_DUPLICATES, hits["n_events"], nh, n), 256), dtype=torch.uint8, device="cuda")
        ctx.remove_duplicates(nh, toff, out["hit_ids"], out["nhits"], out["score"], keep, nk, ws2)
    torch.cuda.synchronize()
    r = {k: v.cpu().numpy() for k, v in out.items()}
    r["status"] = r["status"].view(np.uint32)
    if dedup:
        r["keep"] = keep.cpu().numpy(); r["n_kept"] = nk.cpu().numpy(); r["track_off"] = toff.cpu().numpy()
    r["launches"] = ctx.launch_count()
    ctx.close()
    return r


_strip_ctx = None


def strip_context():
    """Clustering uses no geometry; any context will do."""
    global _strip_ctx
    if _strip_ctx is None:
        from workloads import datagen
        ev, prm = datagen.config(0, scale=0.01)
        _strip_ctx = B.Context(ev["geom"], prm)
    return _strip_ctx


def gpu_cluster_strips(d, sp, capacity=None):
    """mkf_cluster_strips on the strips dict of datagen.make_strips; returns numpy arrays cut to the number found."""
    ctx = strip_context()
    n = int(d["adc"].shape[0])
    cap = n // 2 + 1 if capacity is None else capacity
    sd = B.strips_to_device(d)
    out = B.alloc_clusters(cap)
    nb = ctx.workspace_bytes(B.MKF_CALL_CLUSTER_STRIPS, 0, n, cap)
    ws = torch.empty(max(nb, 1), dtype=torch.uint8, device="cuda")
    ctx.cluster_strips(sd, sp, out, ws)
    torch.cuda.synchronize()
    k = int(out["n_clusters"].item())
    res = {key: out[key][:min(k, cap)].cpu().numpy() for key in ("module", "first", "last", "charge", "bary")}
    res["charge"] = res["charge"].view(np.uint32)
    res["n_clusters"] = k
    return res


def gpu_two_iterations(ev, prm, min_hits, max_chi2_ndf):
    """Iteration 1: index + build + duplicate removal on all seeds; mkf_mask_hits; iteration 2: masked index + build of the
    same seeds. Returns the numpy results of both iterations, the mask and the masked index."""
    s = ev["seeds"]
    ctx = B.Context(ev["geom"], prm)
    hits = B.hits_to_device(ev["hits"])
    nh, nev = hits["x"].shape[0], hits["n_events"]
    idx, ws = B.alloc_hit_index(ctx, nev, nh)
    ctx.build_hit_index(hits, idx, ws)
    sd = B.to_device(dict(par=s["par"], cov=s["cov"], q=s["q"], plan=s["plan"], event=s["event"], hits=s["hits"]),
                     ["par", "cov", "q", "plan", "event", "hits"])
    n = s["par"].shape[1]

    def build():
        out = B.alloc_build_out(n, ctx.max_plan_len)
        ctx.build_tracks(hits, idx, sd, sd["event"], sd["hits"], sd["plan"], out, out["chi2"], out["score"], out["nhits"],
                         out["nmiss"], out["hit_ids"], out["status"])
        return out
    o1 = build()
    counts = np.bincount(s["event"], minlength=nev)
    toff = torch.from_numpy(np.concatenate([[0], np.cumsum(counts)]).astype(np.int32)).cuda()
    keep = torch.empty(n, dtype=torch.uint8, device="cuda")
    nk = torch.empty(nev, dtype=torch.int32, device="cuda")
    ws2 = torch.empty(max(ctx.workspace_bytes(B.CALL_REMOVE_DUPLICATES, nev, nh, n), 256), dtype=torch.uint8, device="cuda")
    ctx.remove_duplicates(nh, toff, o1["hit_ids"], o1["nhits"], o1["score"], keep, nk, ws2)
    mask = torch.zeros(nh, dtype=torch.uint8, device="cuda")
    ctx.mask_hits(o1["hit_ids"], o1["nhits"], o1["chi2"], keep, min_hits, max_chi2_ndf, mask)
    r1 = {k: v.cpu().numpy() for k, v in o1.items()}
    r1["keep"] = keep.cpu().numpy()
    ctx.build_hit_index(hits, idx, ws, mask=mask)
    torch.cuda.synchronize()
    im = dict(bin_off=idx["bin_off"].cpu().numpy().view(np.uint32), vmax=idx["vmax"].cpu().numpy())
    im["sorted_id"] = idx["sorted_id"].cpu().numpy()[:int(im["bin_off"][-1])]
    o2 = build()
    torch.cuda.synchronize()
    r2 = {k: v.cpu().numpy() for k, v in o2.items()}
    ctx.close()
    return r1, mask.cpu().numpy(), im, r2
