"""ctypes binding of the float64 CPU oracle (oracle/mkfo.cpp). TEST INFRASTRUCTURE ONLY.

Builds oracle/libmkfo.so on first use with the host g++ (-O2, no fast-math, OpenMP if the compiler has it).
Inputs are numpy arrays (the same fp32 SoA arrays the CUDA library takes); outputs are numpy float64.
Shares nothing with paper_2002_06295_b200/ (own structs, own marshalling)."""
import ctypes as C
import os
import subprocess
import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_LIB = os.path.join(_HERE, "libmkfo.so")
_SRC = [os.path.join(_HERE, "mkfo.cpp"), os.path.join(_HERE, "mkfo.h")]


def build(force=False):
    """Compile the oracle. Returns the path of the shared library.
    MKFO_SANITIZE=1 in the environment builds oracle/libmkfo_san.so with -fsanitize=address,undefined instead (-O1 -g,
    no OpenMP); run the tests with LD_PRELOAD="$(gcc -print-file-name=libasan.so) $(gcc -print-file-name=libubsan.so)"
    and ASAN_OPTIONS=detect_leaks=0 (python itself leaks). DESIGN.md §2 records the outcome."""
    san = os.environ.get("MKFO_SANITIZE") == "1"
    out = os.path.join(_HERE, "libmkfo_san.so") if san else _LIB
    if not force and os.path.exists(out) and all(os.path.getmtime(out) >= os.path.getmtime(s) for s in _SRC):
        return out
    opt = ["-O1", "-g", "-fsanitize=address,undefined", "-fno-sanitize-recover=undefined", "-fno-omit-frame-pointer"] if san else ["-O2"]
    base = opt + ["-std=c++17", "-fPIC", "-shared", "-Wall", "-Wno-misleading-indentation", "-o", out, _SRC[0]]
    errs = []
    for cxx in ("/usr/bin/g++", "g++", "c++"):
        for omp in ([[]] if san else (["-fopenmp"], [])):
            r = subprocess.run([cxx] + omp + base, capture_output=True, text=True)
            if r.returncode == 0:
                return out
            errs.append(r.stderr[-500:])
    raise RuntimeError("oracle build failed:\n" + "\n".join(errs))


class Layer(C.Structure):
    _fields_ = [("kind", C.c_int), ("pos", C.c_float), ("lo", C.c_float), ("hi", C.c_float),
                ("xx0", C.c_float), ("eta_lo", C.c_float), ("eta_hi", C.c_float)]


class Geometry(C.Structure):
    _fields_ = [("n_layers", C.c_int), ("layers", C.POINTER(Layer)), ("bz", C.c_float),
                ("n_phi_bins", C.c_int), ("n_eta_bins", C.c_int), ("n_plans", C.c_int),
                ("plan_off", C.POINTER(C.c_int)), ("plan_layers", C.POINTER(C.c_int)), ("bz_layer", C.POINTER(C.c_float))]


class Params(C.Structure):
    _fields_ = [("chi2_cut", C.c_float), ("max_cand", C.c_int), ("max_consec_miss", C.c_int),
                ("min_hits_keep", C.c_int), ("score_hit", C.c_float), ("score_miss", C.c_float),
                ("graze_cos_min", C.c_float), ("material_flags", C.c_int), ("dup_frac", C.c_float)]


class Hits(C.Structure):
    _fields_ = [("n_events", C.c_int), ("n_hits", C.c_int), ("layer_off", C.POINTER(C.c_int)),
                ("x", C.POINTER(C.c_float)), ("y", C.POINTER(C.c_float)), ("z", C.POINTER(C.c_float)),
                ("V", C.POINTER(C.c_float))]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.mkfo_dedx.restype = C.c_double
        _lib.mkfo_dedx.argtypes = [C.c_double]
        _lib.mkfo_highland.restype = C.c_double
        _lib.mkfo_highland.argtypes = [C.c_double, C.c_double]
        _lib.mkfo_straggling_var.restype = C.c_double
        _lib.mkfo_straggling_var.argtypes = [C.c_double, C.c_double]
    return _lib


def _p(a, t):
    return a.ctypes.data_as(C.POINTER(t))


def _f32(a):
    return np.ascontiguousarray(a, dtype=np.float32)


def _i32(a):
    return np.ascontiguousarray(a, dtype=np.int32)


def _i8(a):
    return np.ascontiguousarray(a, dtype=np.int8)


def _dp(a):
    return a.ctypes.data_as(C.POINTER(C.c_double))


class Oracle:
    """Holds geometry + params (dicts from the datagen module) in C structs and exposes the mkfo_* calls."""

    def __init__(self, geom, params):
        self.L = lib()
        lay = geom["layers"]
        self._layers = (Layer * len(lay))(*[Layer(int(l["kind"]), float(l["pos"]), float(l["lo"]), float(l["hi"]),
                                                 float(l["xx0"]), float(l["eta_lo"]), float(l["eta_hi"])) for l in lay])
        self._plan_off = _i32(geom["plan_off"])
        self._plan_layers = _i32(geom["plan_layers"])
        self._bz_layer = _f32(geom["bz_layer"]) if geom.get("bz_layer") is not None else None      # R13 field hook
        self.g = Geometry(len(lay), self._layers, float(geom["bz"]), int(geom["n_phi_bins"]), int(geom["n_eta_bins"]),
                          len(self._plan_off) - 1, _p(self._plan_off, C.c_int), _p(self._plan_layers, C.c_int),
                          _p(self._bz_layer, C.c_float) if self._bz_layer is not None else None)
        self.p = Params(float(params["chi2_cut"]), int(params["max_cand"]), int(params["max_consec_miss"]),
                        int(params["min_hits_keep"]), float(params["score_hit"]), float(params["score_miss"]),
                        float(params["graze_cos_min"]), int(params["material_flags"]), float(params["dup_frac"]))
        self.n_layers = len(lay)
        self.nbins = int(geom["n_phi_bins"]) * int(geom["n_eta_bins"])
        self.max_plan_len = int(np.max(np.diff(self._plan_off)))

    # -- hits marshalling: keeps the arrays alive on the returned struct
    def hits(self, h):
        keep = dict(lo=_i32(h["layer_off"]), x=_f32(h["x"]), y=_f32(h["y"]), z=_f32(h["z"]), V=_f32(h["V"]))
        s = Hits(int(h["n_events"]), int(keep["x"].shape[0]), _p(keep["lo"], C.c_int), _p(keep["x"], C.c_float),
                 _p(keep["y"], C.c_float), _p(keep["z"], C.c_float), _p(keep["V"], C.c_float))
        s._keep = keep
        return s

    def build_hit_index(self, h, mask=None):
        """mask (uint8[n_hits], reading R9): hits with mask != 0 are left out; sorted_id is then cut to the hits placed."""
        hs = self.hits(h)
        nseg = hs.n_events * self.n_layers
        bin_off = np.zeros(nseg * self.nbins + 1, np.uint32)
        sorted_id = np.zeros(hs.n_hits, np.int32)
        vmax = np.zeros(nseg * 2, np.float32)
        if mask is not None:
            mask = np.ascontiguousarray(mask, np.uint8)
            assert mask.shape[0] == hs.n_hits
        rc = self.L.mkfo_build_hit_index_masked(C.byref(self.g), C.byref(hs), _p(mask, C.c_ubyte) if mask is not None else None,
                                                _p(bin_off, C.c_uint), _p(sorted_id, C.c_int), _p(vmax, C.c_float))
        assert rc == 0
        return dict(bin_off=bin_off, sorted_id=sorted_id[:int(bin_off[-1])], vmax=vmax)

    def fit(self, h, par, cov, q, plan, track_hits):
        hs = self.hits(h)
        par, cov, q, plan, th = _f32(par), _f32(cov), _i8(q), _i8(plan), _i32(track_hits)
        n = par.shape[1]
        mpl = th.shape[0]
        out = dict(par=np.zeros((6, n)), cov=np.zeros((21, n)), chi2=np.zeros(n), nfit=np.zeros(n, np.int32),
                   status=np.zeros(n, np.uint32))
        rc = self.L.mkfo_fit(C.byref(self.g), C.byref(self.p), C.byref(hs), n, _p(par, C.c_float), _p(cov, C.c_float),
                             _p(q, C.c_byte), _p(plan, C.c_byte), _p(th, C.c_int), mpl, _dp(out["par"]),
                             _dp(out["cov"]), _dp(out["chi2"]), _p(out["nfit"], C.c_int), _p(out["status"], C.c_uint))
        assert rc == 0
        return out

    def fit_backward(self, h, par, cov, q, plan, track_hits):
        hs = self.hits(h)
        par, cov, q, plan, th = _f32(par), _f32(cov), _i8(q), _i8(plan), _i32(track_hits)
        n = par.shape[1]
        out = dict(par=np.zeros((6, n)), cov=np.zeros((21, n)), chi2=np.zeros(n), nfit=np.zeros(n, np.int32),
                   status=np.zeros(n, np.uint32))
        rc = self.L.mkfo_fit_backward(C.byref(self.g), C.byref(self.p), C.byref(hs), n, _p(par, C.c_float),
                                      _p(cov, C.c_float), _p(q, C.c_byte), _p(plan, C.c_byte), _p(th, C.c_int), th.shape[0],
                                      _dp(out["par"]), _dp(out["cov"]), _dp(out["chi2"]), _p(out["nfit"], C.c_int),
                                      _p(out["status"], C.c_uint))
        assert rc == 0
        return out

    def fit_smooth(self, h, par, cov, q, plan, track_hits):
        """R14: par_s (mpl, 6, n), cov_s (mpl, 21, n) smoothed states per plan step (zero where no fitted hit)."""
        hs = self.hits(h)
        par, cov, q, plan, th = _f32(par), _f32(cov), _i8(q), _i8(plan), _i32(track_hits)
        n = par.shape[1]
        mpl = th.shape[0]
        out = dict(par_s=np.zeros((mpl, 6, n)), cov_s=np.zeros((mpl, 21, n)), chi2=np.zeros(n), nfit=np.zeros(n, np.int32),
                   status=np.zeros(n, np.uint32))
        rc = self.L.mkfo_fit_smooth(C.byref(self.g), C.byref(self.p), C.byref(hs), n, _p(par, C.c_float), _p(cov, C.c_float),
                                    _p(q, C.c_byte), _p(plan, C.c_byte), _p(th, C.c_int), mpl, _dp(out["par_s"]),
                                    _dp(out["cov_s"]), _dp(out["chi2"]), _p(out["nfit"], C.c_int), _p(out["status"], C.c_uint))
        assert rc == 0
        return out

    def build_tracks(self, h, idx, par, cov, q, seed_event, seed_hits, plan, brute_force=False, max_plan_len=None, module=None):
        """module (int32[n_hits], reading R15): overlap-hit recovery; the result then also holds hit_ids2."""
        hs = self.hits(h)
        par, cov, q, plan = _f32(par), _f32(cov), _i8(q), _i8(plan)
        se, sh = _i32(seed_event), _i32(seed_hits)
        n = par.shape[1]
        mpl = self.max_plan_len if max_plan_len is None else max_plan_len
        out = dict(par=np.zeros((6, n)), cov=np.zeros((21, n)), chi2=np.zeros(n), score=np.zeros(n),
                   nhits=np.zeros(n, np.int32), nmiss=np.zeros(n, np.int32), hit_ids=np.zeros((mpl, n), np.int32),
                   status=np.zeros(n, np.uint32), margin=np.zeros(n))
        nev = C.c_longlong(0)
        bo = np.ascontiguousarray(idx["bin_off"], np.uint32)
        si = _i32(idx["sorted_id"])
        vm = _f32(idx["vmax"])
        args = [C.byref(self.g), C.byref(self.p), C.byref(hs), _p(bo, C.c_uint), _p(si, C.c_int),
                _p(vm, C.c_float), int(bool(brute_force)), n, _p(par, C.c_float),
                _p(cov, C.c_float), _p(q, C.c_byte), _p(se, C.c_int), _p(sh, C.c_int),
                _p(plan, C.c_byte), mpl, _dp(out["par"]), _dp(out["cov"]), _dp(out["chi2"]),
                _dp(out["score"]), _p(out["nhits"], C.c_int), _p(out["nmiss"], C.c_int),
                _p(out["hit_ids"], C.c_int), _p(out["status"], C.c_uint), _dp(out["margin"]), C.byref(nev)]
        if module is not None:
            mod = _i32(module)
            assert mod.shape[0] == hs.n_hits
            out["hit_ids2"] = np.zeros((mpl, n), np.int32)
            rc = self.L.mkfo_build_tracks_overlap(*args, _p(mod, C.c_int), _p(out["hit_ids2"], C.c_int))
        else:
            rc = self.L.mkfo_build_tracks(*args)
        assert rc == 0
        out["n_chi2_evals"] = nev.value
        return out

    def remove_duplicates(self, track_off, hit_ids, nhits, score):
        to, hi, nh, sc = _i32(track_off), _i32(hit_ids), _i32(nhits), _f32(score)
        n_events = to.shape[0] - 1
        n = hi.shape[1]
        keep = np.zeros(n, np.uint8)
        n_kept = np.zeros(n_events, np.int32)
        rc = self.L.mkfo_remove_duplicates(C.byref(self.p), n_events, _p(to, C.c_int), _p(hi, C.c_int), hi.shape[0],
                                           _p(nh, C.c_int), _p(sc, C.c_float), _p(keep, C.c_ubyte), _p(n_kept, C.c_int))
        assert rc == 0
        return dict(keep=keep, n_kept=n_kept)

    def window(self, layer, u, Cm, vmax):
        u = np.ascontiguousarray(u, np.float64)
        Cm = np.ascontiguousarray(Cm, np.float64)
        vm = np.ascontiguousarray(vmax, np.float64)
        o = [C.c_int(0) for _ in range(4)]
        self.L.mkfo_window(C.byref(self.g), C.byref(self.p), int(layer), _dp(u), _dp(Cm), _dp(vm), *[C.byref(v) for v in o])
        return tuple(v.value for v in o)

    def num_threads(self):
        return int(self.L.mkfo_num_threads())


# ---- single-step functions (for the pins) ---------------------------------------------------------------
def propagate(kind, pos, bz, q, u, Cm=None):
    """Returns (rc, u1, F, C1, s)."""
    L = lib()
    u = np.ascontiguousarray(u, np.float64)
    u1, F, C1, s = np.zeros(6), np.zeros((6, 6)), np.zeros((6, 6)), C.c_double(0)
    Cp = _dp(np.ascontiguousarray(Cm, np.float64)) if Cm is not None else None
    rc = L.mkfo_propagate(int(kind), C.c_double(pos), C.c_double(bz), int(q), _dp(u), Cp, _dp(u1), _dp(F), _dp(C1),
                          C.byref(s))
    return rc, u1, F, C1, s.value


def propagate_dir(kind, pos, bz, q, dirn, u, Cm=None):
    """Returns (rc, u1, F, C1, s); dirn = +1 forward, -1 backward."""
    L = lib()
    u = np.ascontiguousarray(u, np.float64)
    u1, F, C1, s = np.zeros(6), np.zeros((6, 6)), np.zeros((6, 6)), C.c_double(0)
    Cp = _dp(np.ascontiguousarray(Cm, np.float64)) if Cm is not None else None
    rc = L.mkfo_propagate_dir(int(kind), C.c_double(pos), C.c_double(bz), int(q), int(dirn), _dp(u), Cp, _dp(u1), _dp(F),
                              _dp(C1), C.byref(s))
    return rc, u1, F, C1, s.value


def material_dir(kind, xx0, flags, dirn, u, Cm):
    u = np.array(u, np.float64)
    Cm = np.array(Cm, np.float64)
    th0, dE = C.c_double(0), C.c_double(0)
    rc = lib().mkfo_material_dir(int(kind), C.c_double(xx0), int(flags), int(dirn), _dp(u), _dp(Cm), C.byref(th0), C.byref(dE))
    return rc, u, Cm, th0.value, dE.value


def helix_step(bz, q, u, s):
    u = np.ascontiguousarray(u, np.float64)
    u1 = np.zeros(6)
    lib().mkfo_helix_step(C.c_double(bz), int(q), _dp(u), C.c_double(s), _dp(u1))
    return u1


def material(kind, xx0, flags, u, Cm):
    u = np.array(u, np.float64)
    Cm = np.array(Cm, np.float64)
    th0, dE = C.c_double(0), C.c_double(0)
    rc = lib().mkfo_material(int(kind), C.c_double(xx0), int(flags), _dp(u), _dp(Cm), C.byref(th0), C.byref(dE))
    return rc, u, Cm, th0.value, dE.value


def smooth_combine(kind, u_f, C_f, u_b, C_b):
    """R14: weighted mean of a forward and a backward estimate on a surface. Returns (rc, u_s, C_s)."""
    u_s, C_s = np.zeros(6), np.zeros((6, 6))
    a = [np.ascontiguousarray(x, np.float64) for x in (u_f, C_f, u_b, C_b)]
    rc = lib().mkfo_smooth_combine(int(kind), _dp(a[0]), _dp(a[1]), _dp(a[2]), _dp(a[3]), _dp(u_s), _dp(C_s))
    return rc, u_s, C_s


def dedx(p):
    return lib().mkfo_dedx(float(p))


def highland(p, t):
    return lib().mkfo_highland(float(p), float(t))


def straggling_var(p, t):
    return lib().mkfo_straggling_var(float(p), float(t))


def chi2(u, Cm, m, V6):
    c2 = C.c_double(0)
    rc = lib().mkfo_chi2(_dp(np.ascontiguousarray(u, np.float64)), _dp(np.ascontiguousarray(Cm, np.float64)),
                         _dp(np.ascontiguousarray(m, np.float64)), _dp(np.ascontiguousarray(V6, np.float64)), C.byref(c2))
    return rc, c2.value


def update(u, Cm, m, V6):
    u = np.array(u, np.float64)
    Cm = np.array(Cm, np.float64)
    c2 = C.c_double(0)
    rc = lib().mkfo_update(_dp(u), _dp(Cm), _dp(np.ascontiguousarray(m, np.float64)),
                           _dp(np.ascontiguousarray(V6, np.float64)), C.byref(c2))
    return rc, u, Cm, c2.value


def cluster_strips(module_off, adc, noise, bad, seed_thr=3.0, chan_thr=2.0, clus_thr=5.0, min_charge=0, max_holes=0, max_bad=1):
    """R8: returns dict(module, first, last, charge, bary) of the kept clusters, ordered by (module, first strip)."""
    mo = _i32(module_off)
    adc = np.ascontiguousarray(adc, np.uint16); noise = _f32(noise); bad = np.ascontiguousarray(bad, np.uint8)
    n = adc.shape[0]
    om, of, ol = np.zeros(n, np.int32), np.zeros(n, np.int32), np.zeros(n, np.int32)
    oc, ob = np.zeros(n, np.uint32), np.zeros(n, np.float32)
    L = lib()
    k = L.mkfo_cluster_strips(mo.shape[0] - 1, _p(mo, C.c_int), _p(adc, C.c_ushort), _p(noise, C.c_float), _p(bad, C.c_ubyte),
                              C.c_float(seed_thr), C.c_float(chan_thr), C.c_float(clus_thr), int(min_charge), int(max_holes),
                              int(max_bad), _p(om, C.c_int), _p(of, C.c_int), _p(ol, C.c_int), _p(oc, C.c_uint), _p(ob, C.c_float))
    return dict(module=om[:k].copy(), first=of[:k].copy(), last=ol[:k].copy(), charge=oc[:k].copy(), bary=ob[:k].copy())


def mask_hits(n_hits, hit_ids, nhits, chi2, keep=None, min_hits=8, max_chi2_ndf=5.0, mask=None):
    """Reading R9: mask[h] = 1 for the hits of high-quality tracks. Returns the mask."""
    L = lib()
    hi = np.ascontiguousarray(hit_ids, np.int32)
    n = hi.shape[1]
    nh, c2 = np.ascontiguousarray(nhits, np.int32), np.ascontiguousarray(chi2, np.float32)
    mask = np.zeros(n_hits, np.uint8) if mask is None else np.ascontiguousarray(mask, np.uint8).copy()
    if keep is not None:
        keep = np.ascontiguousarray(keep, np.uint8)
    rc = L.mkfo_mask_hits(n, int(n_hits), _p(hi, C.c_int), hi.shape[0], _p(nh, C.c_int), _p(c2, C.c_float),
                          _p(keep, C.c_ubyte) if keep is not None else None, int(min_hits), C.c_float(max_chi2_ndf), _p(mask, C.c_ubyte))
    assert rc == 0
    return mask
