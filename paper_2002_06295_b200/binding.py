"""Thin ctypes binding of libmkf.so (include/mkf.h): argument marshalling only — every step runs in the CUDA kernels.

Device calls take torch CUDA tensors (caller-owned; PyTorch is used for device memory and streams only) and enqueue
on torch's current stream without synchronising. Host calls (`fit_host`, `build_host`) take numpy arrays or CPU
tensors. There is no CPU fallback: a missing library or a missing CUDA device raises.
"""
import ctypes as C
import os

import numpy as np
import torch

from . import build as _build

OK, INVALID_ARG, CUDA_ERROR, WORKSPACE_TOO_SMALL, UNSUPPORTED = 0, -1, -2, -3, -4
PROP_UNREACHABLE, GRAZING, S_NOT_PD, NAN, STOPPED_ELOSS, TRUNCATED = 1, 2, 4, 8, 16, 32
CALL_BUILD_HIT_INDEX, CALL_FIT, CALL_BUILD_TRACKS, CALL_REMOVE_DUPLICATES = 0, 1, 2, 3
CALL_FIT_SMOOTH, CALL_BUILD_TRACKS_OVERLAP = 5, 6
STATIC_MAX_HITS = 1 << 20                      # MKF_STATIC_MAX_HITS of include/mkf.h

EXPORTS = ["mkf_create", "mkf_destroy", "mkf_last_error", "mkf_workspace_bytes", "mkf_launch_count", "mkf_max_plan_len",
           "mkf_build_hit_index", "mkf_fit", "mkf_fit_backward", "mkf_build_tracks", "mkf_remove_duplicates", "mkf_fit_host", "mkf_fit_backward_host", "mkf_build_host",
           "mkf_cluster_strips", "mkf_cluster_strips_host", "mkf_mask_hits", "mkf_build_hit_index_masked", "mkf_pack_hits", "mkf_set_build_counters", "mkf_fit_smooth", "mkf_build_tracks_overlap", "mkf_build_hit_index_static"]


class Layer(C.Structure):
    _fields_ = [("kind", C.c_int), ("pos", C.c_float), ("lo", C.c_float), ("hi", C.c_float), ("xx0", C.c_float),
                ("eta_lo", C.c_float), ("eta_hi", C.c_float)]


class Geometry(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("layers", C.POINTER(Layer)), ("bz", C.c_float), ("n_phi_bins", C.c_int),
                ("n_eta_bins", C.c_int), ("n_plans", C.c_int), ("plan_off", C.POINTER(C.c_int)),
                ("plan_layers", C.POINTER(C.c_int)), ("bz_layer", C.POINTER(C.c_float))]


class Params(C.Structure):
    _fields_ = [("chi2_cut", C.c_float), ("max_cand", C.c_int), ("max_consec_miss", C.c_int), ("min_hits_keep", C.c_int),
                ("score_hit", C.c_float), ("score_miss", C.c_float), ("graze_cos_min", C.c_float),
                ("material_flags", C.c_int), ("dup_frac", C.c_float)]


class Hits(C.Structure):
    _fields_ = [("n_events", C.c_int), ("n_hits", C.c_int), ("layer_off", C.c_void_p), ("x", C.c_void_p),
                ("y", C.c_void_p), ("z", C.c_void_p), ("V", C.c_void_p), ("rec", C.c_void_p), ("module", C.c_void_p)]


class HitIndex(C.Structure):
    _fields_ = [("bin_off", C.c_void_p), ("sorted_id", C.c_void_p), ("vmax", C.c_void_p), ("packed", C.c_void_p)]


class States(C.Structure):
    _fields_ = [("n", C.c_int), ("par", C.c_void_p), ("cov", C.c_void_p), ("q", C.c_void_p)]


class StripParams(C.Structure):
    _fields_ = [("seed_thr", C.c_float), ("chan_thr", C.c_float), ("clus_thr", C.c_float), ("min_charge", C.c_int),
                ("max_holes", C.c_int), ("max_bad", C.c_int)]


class Strips(C.Structure):
    _fields_ = [("n_modules", C.c_int), ("n_strips", C.c_int), ("module_off", C.c_void_p), ("adc", C.c_void_p),
                ("noise", C.c_void_p), ("bad", C.c_void_p)]


class Clusters(C.Structure):
    _fields_ = [("capacity", C.c_int), ("module", C.c_void_p), ("first", C.c_void_p), ("last", C.c_void_p),
                ("charge", C.c_void_p), ("bary", C.c_void_p), ("n_clusters", C.c_void_p)]


MKF_CALL_CLUSTER_STRIPS = 4


_lib = None


def lib():
    """Loads (building first if needed) libmkf.so. Raises if it cannot be built or loaded."""
    global _lib
    if _lib is None:
        path = _build.LIB if os.path.exists(_build.LIB) and os.environ.get("MKF_NO_REBUILD") else _build.build()
        L = C.CDLL(path)
        L.mkf_last_error.restype = C.c_char_p
        L.mkf_last_error.argtypes = [C.c_void_p]
        L.mkf_workspace_bytes.restype = C.c_size_t
        L.mkf_workspace_bytes.argtypes = [C.c_void_p, C.c_int, C.c_int, C.c_int, C.c_int]
        L.mkf_launch_count.restype = C.c_longlong
        L.mkf_launch_count.argtypes = [C.c_void_p]
        L.mkf_max_plan_len.argtypes = [C.c_void_p]
        L.mkf_destroy.restype = None
        L.mkf_destroy.argtypes = [C.c_void_p]
        L.mkf_create.argtypes = [C.POINTER(C.c_void_p), C.POINTER(Geometry), C.POINTER(Params)]
        vp, sz, i = C.c_void_p, C.c_size_t, C.c_int
        L.mkf_build_hit_index.argtypes = [vp, C.POINTER(Hits), C.POINTER(HitIndex), vp, sz, vp]
        L.mkf_build_hit_index_masked.argtypes = [vp, C.POINTER(Hits), vp, C.POINTER(HitIndex), vp, sz, vp]
        L.mkf_build_hit_index_static.argtypes = [vp, C.POINTER(Hits), C.POINTER(HitIndex), vp]
        L.mkf_mask_hits.argtypes = [vp, i, i, vp, i, vp, vp, vp, i, C.c_float, vp, vp]
        L.mkf_fit.argtypes = [vp, C.POINTER(Hits), C.POINTER(States), vp, vp, i, C.POINTER(States), vp, vp, vp, vp, sz, vp]
        L.mkf_fit_backward.argtypes = L.mkf_fit.argtypes
        L.mkf_fit_smooth.argtypes = [vp, C.POINTER(Hits), C.POINTER(States), vp, vp, i, vp, vp, vp, vp, vp, vp, sz, vp]
        L.mkf_pack_hits.argtypes = [vp, C.POINTER(Hits), vp, vp]
        L.mkf_set_build_counters.argtypes = [vp, vp]
        L.mkf_build_tracks.argtypes = [vp, C.POINTER(Hits), C.POINTER(HitIndex), C.POINTER(States), vp, vp, vp, i,
                                       C.POINTER(States), vp, vp, vp, vp, vp, vp, vp, sz, vp]
        L.mkf_build_tracks_overlap.argtypes = [vp, C.POINTER(Hits), C.POINTER(HitIndex), C.POINTER(States), vp, vp, vp, i,
                                               C.POINTER(States), vp, vp, vp, vp, vp, vp, vp, vp, sz, vp]
        L.mkf_remove_duplicates.argtypes = [vp, i, i, i, vp, vp, i, vp, vp, vp, vp, vp, sz, vp]
        ll = C.POINTER(C.c_longlong)
        L.mkf_cluster_strips.argtypes = [vp, C.POINTER(Strips), C.POINTER(StripParams), C.POINTER(Clusters), vp, sz, vp]
        L.mkf_cluster_strips_host.argtypes = [vp, C.POINTER(Strips), C.POINTER(StripParams), C.POINTER(Clusters), ll, ll]
        L.mkf_fit_host.argtypes = [vp, C.POINTER(Hits), C.POINTER(States), vp, vp, i, C.POINTER(States), vp, vp, vp, ll, ll]
        L.mkf_fit_backward_host.argtypes = L.mkf_fit_host.argtypes
        L.mkf_build_host.argtypes = [vp, C.POINTER(Hits), C.POINTER(States), vp, vp, vp, i, C.POINTER(States), vp, vp,
                                     vp, vp, vp, vp, vp, ll, ll]
        _lib = L
    return _lib


class MkfError(RuntimeError):
    pass


def _dev(t, dtype):
    if not (isinstance(t, torch.Tensor) and t.is_cuda and t.dtype == dtype and t.is_contiguous()):
        raise TypeError("expected a contiguous CUDA tensor of dtype %s" % dtype)
    return t.data_ptr()


def _host(a, dtype):
    if isinstance(a, torch.Tensor):
        a = a.numpy()
    if not (isinstance(a, np.ndarray) and a.dtype == dtype and a.flags["C_CONTIGUOUS"]):
        raise TypeError("expected a C-contiguous numpy array of dtype %s" % dtype)
    return a.ctypes.data


def _stream():
    return torch.cuda.current_stream().cuda_stream


class Context:
    """mkf_ctx: geometry + parameters (dicts as made by datagen). Methods carry the names of the C calls."""

    def __init__(self, geom, params):
        self.L = lib()
        lay = geom["layers"]
        self._layers = (Layer * len(lay))(*[Layer(int(l["kind"]), float(l["pos"]), float(l["lo"]), float(l["hi"]),
                                                 float(l["xx0"]), float(l["eta_lo"]), float(l["eta_hi"])) for l in lay])
        self._plan_off = np.ascontiguousarray(geom["plan_off"], np.int32)
        self._plan_layers = np.ascontiguousarray(geom["plan_layers"], np.int32)
        bzl = geom.get("bz_layer")
        self._bz_layer = np.ascontiguousarray(bzl, np.float32) if bzl is not None else None
        g = Geometry(len(lay), self._layers, float(geom["bz"]), int(geom["n_phi_bins"]), int(geom["n_eta_bins"]),
                     len(self._plan_off) - 1, self._plan_off.ctypes.data_as(C.POINTER(C.c_int)),
                     self._plan_layers.ctypes.data_as(C.POINTER(C.c_int)),
                     self._bz_layer.ctypes.data_as(C.POINTER(C.c_float)) if self._bz_layer is not None else None)
        p = Params(float(params["chi2_cut"]), int(params["max_cand"]), int(params["max_consec_miss"]),
                   int(params["min_hits_keep"]), float(params["score_hit"]), float(params["score_miss"]),
                   float(params["graze_cos_min"]), int(params["material_flags"]), float(params["dup_frac"]))
        h = C.c_void_p()
        rc = self.L.mkf_create(C.byref(h), C.byref(g), C.byref(p))
        if rc != OK:
            raise MkfError("mkf_create failed: %d" % rc)
        self.h = h
        self.n_layers = len(lay)
        self.n_bins = int(geom["n_phi_bins"]) * int(geom["n_eta_bins"])
        self.max_plan_len = int(self.L.mkf_max_plan_len(self.h))

    def close(self):
        if getattr(self, "h", None):
            self.L.mkf_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def _check(self, rc, what):
        if rc != OK:
            raise MkfError("%s failed (%d): %s" % (what, rc, self.L.mkf_last_error(self.h).decode()))

    def launch_count(self):
        return int(self.L.mkf_launch_count(self.h))

    def workspace_bytes(self, call_id, n_events, n_hits, n_seeds):
        return int(self.L.mkf_workspace_bytes(self.h, call_id, n_events, n_hits, n_seeds))

    # ---- marshalling helpers ------------------------------------------------------------------------------
    @staticmethod
    def hits_struct(h, ptr, i32=torch.int32, f32=torch.float32):
        rec, mod = h.get("rec"), h.get("module") if ptr is _dev else None
        return Hits(int(h["n_events"]), int(h["x"].shape[0]), ptr(h["layer_off"], i32), ptr(h["x"], f32), ptr(h["y"], f32),
                    ptr(h["z"], f32), ptr(h["V"], f32), ptr(rec, f32) if rec is not None else None,
                    ptr(mod, i32) if mod is not None else None)

    def pack_hits(self, hits, rec):
        """mkf_pack_hits: rec float32 CUDA tensor [n_hits * 12] receives the 48-byte hit records (mkf_hits.rec)."""
        hs = self.hits_struct(hits, _dev)
        rc = self.L.mkf_pack_hits(self.h, C.byref(hs), _dev(rec, torch.float32), _stream())
        self._check(rc, "mkf_pack_hits")

    # ---- the four calls -----------------------------------------------------------------------------------
    def build_hit_index(self, hits, out, ws, mask=None):
        """mask (uint8 CUDA tensor [n_hits] or None): mkf_build_hit_index_masked (reading R9).
        hits: dict of CUDA tensors (layer_off int32, x,y,z float32 [n], V float32 [6,n]); out: dict(bin_off int32
        [n_events*n_layers*n_bins+1] (unsigned offsets), sorted_id int32 [n], vmax float32 [n_events*n_layers*2],
        packed float32 [n*12 + 4] or None); ws: uint8 CUDA tensor."""
        hs = self.hits_struct(hits, _dev)
        packed = out.get("packed")
        idx = HitIndex(_dev(out["bin_off"], torch.int32), _dev(out["sorted_id"], torch.int32), _dev(out["vmax"], torch.float32),
                       _dev(packed, torch.float32) if packed is not None else None)
        wsp, wsn = (ws.data_ptr(), ws.numel()) if ws is not None else (None, 0)
        if mask is not None:
            rc = self.L.mkf_build_hit_index_masked(self.h, C.byref(hs), _dev(mask, torch.uint8), C.byref(idx), wsp, wsn, _stream())
        else:
            rc = self.L.mkf_build_hit_index(self.h, C.byref(hs), C.byref(idx), wsp, wsn, _stream())
        self._check(rc, "mkf_build_hit_index")

    build_hit_index_masked = build_hit_index

    def build_hit_index_static(self, hits, out):
        """mkf_build_hit_index_static: the plain hit index with its scratch inside the library (no workspace, no
        allocation; n_hits <= STATIC_MAX_HITS). hits, out as for build_hit_index."""
        hs = self.hits_struct(hits, _dev)
        packed = out.get("packed")
        idx = HitIndex(_dev(out["bin_off"], torch.int32), _dev(out["sorted_id"], torch.int32), _dev(out["vmax"], torch.float32),
                       _dev(packed, torch.float32) if packed is not None else None)
        rc = self.L.mkf_build_hit_index_static(self.h, C.byref(hs), C.byref(idx), _stream())
        self._check(rc, "mkf_build_hit_index_static")

    def mask_hits(self, hit_ids, nhits, chi2, keep, min_hits, max_chi2_ndf, mask):
        """mkf_mask_hits (reading R9): sets mask[h] = 1 for the hits of high-quality tracks; keep may be None."""
        rc = self.L.mkf_mask_hits(self.h, int(hit_ids.shape[1]), int(mask.shape[0]), _dev(hit_ids, torch.int32), int(hit_ids.shape[0]),
                                  _dev(nhits, torch.int32), _dev(chi2, torch.float32),
                                  _dev(keep, torch.uint8) if keep is not None else None, int(min_hits), float(max_chi2_ndf),
                                  _dev(mask, torch.uint8), _stream())
        self._check(rc, "mkf_mask_hits")

    def fit_backward(self, hits, seeds, plan, track_hits, out, chi2, nfit, status):
        """Outside-in fit (mkf_fit_backward); seeds sit on the layer of each track's last hit."""
        return self.fit(hits, seeds, plan, track_hits, out, chi2, nfit, status, backward=True)

    def fit(self, hits, seeds, plan, track_hits, out, chi2, nfit, status, backward=False):
        """seeds/out: dict(par float32 [6,n], cov float32 [21,n], q int8 [n]); plan int8 [n]; track_hits int32 [mpl,n]."""
        hs = self.hits_struct(hits, _dev)
        n = int(seeds["par"].shape[1])
        s = States(n, _dev(seeds["par"], torch.float32), _dev(seeds["cov"], torch.float32), _dev(seeds["q"], torch.int8))
        o = States(n, _dev(out["par"], torch.float32), _dev(out["cov"], torch.float32), _dev(seeds["q"], torch.int8))
        call = self.L.mkf_fit_backward if backward else self.L.mkf_fit
        rc = call(self.h, C.byref(hs), C.byref(s), _dev(plan, torch.int8), _dev(track_hits, torch.int32),
                            int(track_hits.shape[0]), C.byref(o), _dev(chi2, torch.float32), _dev(nfit, torch.int32),
                            _dev(status, torch.int32), None, 0, _stream())
        self._check(rc, "mkf_fit_backward" if backward else "mkf_fit")

    def set_build_counters(self, counters):
        """mkf_set_build_counters: int64 CUDA tensor [8] (zeroed by the caller) or None."""
        self._counters = counters                               # keep the tensor alive while the library holds its address
        self._check(self.L.mkf_set_build_counters(self.h, _dev(counters, torch.int64) if counters is not None else None), "mkf_set_build_counters")

    def fit_smooth(self, hits, seeds, plan, track_hits, par_s, cov_s, chi2, nfit, status, ws):
        """mkf_fit_smooth (reading R14): par_s float32 [mpl, 6, n], cov_s float32 [mpl, 21, n]."""
        hs = self.hits_struct(hits, _dev)
        n = int(seeds["par"].shape[1])
        s = States(n, _dev(seeds["par"], torch.float32), _dev(seeds["cov"], torch.float32), _dev(seeds["q"], torch.int8))
        rc = self.L.mkf_fit_smooth(self.h, C.byref(hs), C.byref(s), _dev(plan, torch.int8), _dev(track_hits, torch.int32),
                                   int(track_hits.shape[0]), _dev(par_s, torch.float32), _dev(cov_s, torch.float32),
                                   _dev(chi2, torch.float32), _dev(nfit, torch.int32), _dev(status, torch.int32),
                                   ws.data_ptr(), ws.numel(), _stream())
        self._check(rc, "mkf_fit_smooth")

    def build_tracks(self, hits, idx, seeds, seed_event, seed_hits, plan, out, chi2, score, nhits, nmiss, hit_ids, status, ws=None, hit_ids2=None):
        """hit_ids2 (int32 [mpl, n]) given: mkf_build_tracks_overlap (reading R15; hits must hold `module`)."""
        hs = self.hits_struct(hits, _dev)
        packed = idx.get("packed")
        ix = HitIndex(_dev(idx["bin_off"], torch.int32), _dev(idx["sorted_id"], torch.int32), _dev(idx["vmax"], torch.float32),
                      _dev(packed, torch.float32) if packed is not None else None)
        n = int(seeds["par"].shape[1])
        if ws is None:                                          # scratch for the call (kept for the next one of the same size)
            need = max(self.workspace_bytes(CALL_BUILD_TRACKS_OVERLAP if hit_ids2 is not None else CALL_BUILD_TRACKS,
                                            int(hits["n_events"]), int(hits["x"].shape[0]), n), 256)
            if getattr(self, "_build_ws", None) is None or self._build_ws.numel() < need:
                self._build_ws = torch.empty(need, dtype=torch.uint8, device=seeds["par"].device)
            ws = self._build_ws
        s = States(n, _dev(seeds["par"], torch.float32), _dev(seeds["cov"], torch.float32), _dev(seeds["q"], torch.int8))
        o = States(n, _dev(out["par"], torch.float32), _dev(out["cov"], torch.float32), _dev(seeds["q"], torch.int8))
        if hit_ids2 is not None:
            rc = self.L.mkf_build_tracks_overlap(self.h, C.byref(hs), C.byref(ix), C.byref(s), _dev(seed_event, torch.int32),
                                                 _dev(seed_hits, torch.int32), _dev(plan, torch.int8), int(hit_ids.shape[0]), C.byref(o),
                                                 _dev(chi2, torch.float32), _dev(score, torch.float32), _dev(nhits, torch.int32),
                                                 _dev(nmiss, torch.int32), _dev(hit_ids, torch.int32), _dev(hit_ids2, torch.int32),
                                                 _dev(status, torch.int32), ws.data_ptr(), ws.numel(), _stream())
        else:
            rc = self.L.mkf_build_tracks(self.h, C.byref(hs), C.byref(ix), C.byref(s), _dev(seed_event, torch.int32),
                                         _dev(seed_hits, torch.int32), _dev(plan, torch.int8), int(hit_ids.shape[0]), C.byref(o),
                                         _dev(chi2, torch.float32), _dev(score, torch.float32), _dev(nhits, torch.int32),
                                         _dev(nmiss, torch.int32), _dev(hit_ids, torch.int32), _dev(status, torch.int32),
                                         ws.data_ptr() if ws is not None else None, ws.numel() if ws is not None else 0, _stream())
        self._check(rc, "mkf_build_tracks")

    def remove_duplicates(self, n_hits, track_off, hit_ids, nhits, score, keep, n_kept, ws):
        n_events = int(track_off.shape[0]) - 1
        rc = self.L.mkf_remove_duplicates(self.h, n_events, int(hit_ids.shape[1]), int(n_hits), _dev(track_off, torch.int32),
                                          _dev(hit_ids, torch.int32), int(hit_ids.shape[0]), _dev(nhits, torch.int32),
                                          _dev(score, torch.float32), _dev(keep, torch.uint8), _dev(n_kept, torch.int32),
                                          ws.data_ptr(), ws.numel(), _stream())
        self._check(rc, "mkf_remove_duplicates")

    def cluster_strips(self, strips, prm, out, ws):
        """strips / out: dicts of CUDA tensors (strips_to_device, alloc_clusters); prm: dict (datagen.default_strip_params)."""
        n = int(strips["adc"].shape[0])
        s = Strips(int(strips["module_off"].shape[0]) - 1, n, _dev(strips["module_off"], torch.int32),
                   _dev(strips["adc"], torch.uint16), _dev(strips["noise"], torch.float32), _dev(strips["bad"], torch.uint8))
        o = Clusters(int(out["module"].shape[0]), _dev(out["module"], torch.int32), _dev(out["first"], torch.int32),
                     _dev(out["last"], torch.int32), _dev(out["charge"], torch.int32), _dev(out["bary"], torch.float32),
                     _dev(out["n_clusters"], torch.int32))
        sp = strip_params(prm)
        rc = self.L.mkf_cluster_strips(self.h, C.byref(s), C.byref(sp), C.byref(o), ws.data_ptr() if ws is not None else None,
                                       ws.numel() if ws is not None else 0, _stream())
        self._check(rc, "mkf_cluster_strips")

    def cluster_strips_host(self, strips, prm, capacity):
        """strips: dict of numpy arrays / CPU (pinned) tensors. Returns dict of numpy arrays cut to the number found."""
        i32, f32 = np.int32, np.float32
        n = int(strips["adc"].shape[0])
        s = Strips(int(strips["module_off"].shape[0]) - 1, n, _host(strips["module_off"], i32), _host(strips["adc"], np.uint16),
                   _host(strips["noise"], f32), _host(strips["bad"], np.uint8))
        out = dict(module=np.empty(capacity, i32), first=np.empty(capacity, i32), last=np.empty(capacity, i32),
                   charge=np.empty(capacity, np.uint32), bary=np.empty(capacity, f32))
        nc = np.zeros(1, i32)
        o = Clusters(capacity, out["module"].ctypes.data, out["first"].ctypes.data, out["last"].ctypes.data,
                     out["charge"].ctypes.data, out["bary"].ctypes.data, nc.ctypes.data)
        sp = strip_params(prm)
        h2d, d2h = C.c_longlong(0), C.c_longlong(0)
        rc = self.L.mkf_cluster_strips_host(self.h, C.byref(s), C.byref(sp), C.byref(o), C.byref(h2d), C.byref(d2h))
        self._check(rc, "mkf_cluster_strips_host")
        k = int(nc[0]) if int(nc[0]) <= capacity else 0          # overflow: only the count is defined (mkf.h)
        out = {key: v[:k] for key, v in out.items()}
        out["n_clusters"], out["h2d_bytes"], out["d2h_bytes"] = int(nc[0]), h2d.value, d2h.value
        return out

    # ---- host-buffer entry points -------------------------------------------------------------------------
    def fit_host(self, hits, seeds, plan, track_hits, backward=False, out=None):
        """All arguments numpy / CPU tensors; returns dict of numpy arrays plus the bytes copied each way.
        out (optional): preallocated result arrays (alloc_fit_out_host; pinned memory keeps the copies asynchronous)."""
        f32, i32, i8 = np.float32, np.int32, np.int8
        hs = self.hits_struct(hits, _host, i32, f32)
        n = int(seeds["par"].shape[1])
        out = dict(out) if out is not None else alloc_fit_out_host(n, pinned=False)
        s = States(n, _host(seeds["par"], f32), _host(seeds["cov"], f32), _host(seeds["q"], i8))
        o = States(n, out["par"].ctypes.data, out["cov"].ctypes.data, _host(seeds["q"], i8))
        h2d, d2h = C.c_longlong(0), C.c_longlong(0)
        call = self.L.mkf_fit_backward_host if backward else self.L.mkf_fit_host
        rc = call(self.h, C.byref(hs), C.byref(s), _host(plan, i8), _host(track_hits, i32),
                                 int(track_hits.shape[0]), C.byref(o), out["chi2"].ctypes.data, out["nfit"].ctypes.data,
                                 out["status"].ctypes.data, C.byref(h2d), C.byref(d2h))
        self._check(rc, "mkf_fit_host")
        out["h2d_bytes"], out["d2h_bytes"] = h2d.value, d2h.value
        return out

    def build_host(self, hits, seeds, seed_event, seed_hits, plan, dedup=False, out=None):
        f32, i32, i8 = np.float32, np.int32, np.int8
        hs = self.hits_struct(hits, _host, i32, f32)
        n = int(seeds["par"].shape[1])
        mpl = self.max_plan_len
        out = dict(out) if out is not None else alloc_build_out_host(n, mpl, pinned=False)
        keep = out.pop("keep") if dedup else None
        out.pop("keep", None)
        s = States(n, _host(seeds["par"], f32), _host(seeds["cov"], f32), _host(seeds["q"], i8))
        o = States(n, out["par"].ctypes.data, out["cov"].ctypes.data, _host(seeds["q"], i8))
        h2d, d2h = C.c_longlong(0), C.c_longlong(0)
        rc = self.L.mkf_build_host(self.h, C.byref(hs), C.byref(s), _host(seed_event, i32), _host(seed_hits, i32),
                                   _host(plan, i8), mpl, C.byref(o), out["chi2"].ctypes.data, out["score"].ctypes.data,
                                   out["nhits"].ctypes.data, out["nmiss"].ctypes.data, out["hit_ids"].ctypes.data,
                                   out["status"].ctypes.data, keep.ctypes.data if dedup else None, C.byref(h2d), C.byref(d2h))
        self._check(rc, "mkf_build_host")
        if dedup:
            out["keep"] = keep
        out["h2d_bytes"], out["d2h_bytes"] = h2d.value, d2h.value
        return out


def strip_params(p):
    return StripParams(p["seed_thr"], p["chan_thr"], p["clus_thr"], p["min_charge"], p["max_holes"], p["max_bad"])


def strips_to_device(d, device="cuda"):
    return dict(module_off=torch.from_numpy(d["module_off"]).to(device), adc=torch.from_numpy(d["adc"]).to(device),
                noise=torch.from_numpy(d["noise"]).to(device), bad=torch.from_numpy(d["bad"]).to(device))


def alloc_clusters(capacity, device="cuda"):
    i32 = torch.int32
    return dict(module=torch.empty(capacity, dtype=i32, device=device), first=torch.empty(capacity, dtype=i32, device=device),
                last=torch.empty(capacity, dtype=i32, device=device), charge=torch.empty(capacity, dtype=i32, device=device),
                bary=torch.empty(capacity, dtype=torch.float32, device=device),
                n_clusters=torch.zeros(1, dtype=i32, device=device))


# ---- convenience: allocate outputs on the device (still marshalling only) ---------------------------------------
def to_device(d, keys, device="cuda"):
    """Copies the named numpy arrays of dict d to CUDA tensors (int32/float32/int8 kept)."""
    return {k: torch.from_numpy(np.ascontiguousarray(d[k])).to(device) for k in keys}


def hits_to_device(hits, device="cuda", with_module=False):
    h = to_device(hits, ["layer_off", "x", "y", "z", "V"] + (["module"] if with_module else []), device)
    h["n_events"] = int(hits["n_events"])
    return h


def alloc_hit_index(ctx, n_events, n_hits, packed=True, device="cuda"):
    nseg = n_events * ctx.n_layers
    out = dict(bin_off=torch.empty(nseg * ctx.n_bins + 1, dtype=torch.int32, device=device),
               sorted_id=torch.empty(n_hits, dtype=torch.int32, device=device),
               vmax=torch.empty(nseg * 2, dtype=torch.float32, device=device),
               packed=torch.empty(n_hits * 12 + 4, dtype=torch.float32, device=device) if packed else None)
    ws = torch.empty(max(ctx.workspace_bytes(CALL_BUILD_HIT_INDEX, n_events, n_hits, 0), 256), dtype=torch.uint8, device=device)
    return out, ws


def _host_array(shape, dtype, pinned):
    if not pinned:
        return np.empty(shape, dtype)
    tdt = {np.float32: torch.float32, np.int32: torch.int32, np.uint8: torch.uint8}[dtype if dtype is not np.uint32 else np.int32]
    a = torch.empty(shape, dtype=tdt).pin_memory().numpy()
    return a.view(np.uint32) if dtype is np.uint32 else a


def alloc_fit_out_host(n, pinned=True):
    """Result arrays of fit_host in (pinned) host memory."""
    f32, i32 = np.float32, np.int32
    return dict(par=_host_array((6, n), f32, pinned), cov=_host_array((21, n), f32, pinned), chi2=_host_array(n, f32, pinned),
                nfit=_host_array(n, i32, pinned), status=_host_array(n, np.uint32, pinned))


def alloc_build_out_host(n, mpl, pinned=True):
    f32, i32 = np.float32, np.int32
    return dict(par=_host_array((6, n), f32, pinned), cov=_host_array((21, n), f32, pinned), chi2=_host_array(n, f32, pinned),
                score=_host_array(n, f32, pinned), nhits=_host_array(n, i32, pinned), nmiss=_host_array(n, i32, pinned),
                hit_ids=_host_array((mpl, n), i32, pinned), status=_host_array(n, np.uint32, pinned), keep=_host_array(n, np.uint8, pinned))


def alloc_build_ws(ctx, n_events, n_hits, n_seeds, device="cuda"):
    return torch.empty(max(ctx.workspace_bytes(CALL_BUILD_TRACKS, n_events, n_hits, n_seeds), 256), dtype=torch.uint8, device=device)


def alloc_fit_out(n, device="cuda"):
    return dict(par=torch.empty((6, n), dtype=torch.float32, device=device), cov=torch.empty((21, n), dtype=torch.float32, device=device),
                chi2=torch.empty(n, dtype=torch.float32, device=device), nfit=torch.empty(n, dtype=torch.int32, device=device),
                status=torch.empty(n, dtype=torch.int32, device=device))


def alloc_build_out(n, mpl, device="cuda"):
    f32, i32 = torch.float32, torch.int32
    return dict(par=torch.empty((6, n), dtype=f32, device=device), cov=torch.empty((21, n), dtype=f32, device=device),
                chi2=torch.empty(n, dtype=f32, device=device), score=torch.empty(n, dtype=f32, device=device),
                nhits=torch.empty(n, dtype=i32, device=device), nmiss=torch.empty(n, dtype=i32, device=device),
                hit_ids=torch.empty((mpl, n), dtype=i32, device=device), status=torch.empty(n, dtype=i32, device=device))
