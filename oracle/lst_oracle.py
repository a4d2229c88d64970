"""ctypes loader for the CPU oracle (oracle/lst_oracle.c).  TEST INFRASTRUCTURE ONLY.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
import this.  It never imports, links or calls anything of the CUDA path.
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "lst_oracle.c")
_HDR = os.path.join(_HERE, "lst_oracle.h")
_SO = os.path.join(_HERE, "liblst_oracle.so")

MD, LS, T3, T5, PT3, PT5, TC = range(7)
PLS_KEEP = -1
LEVEL_NAMES = ("MD", "LS", "T3", "T5", "PT3", "PT5", "TC")


class Config(C.Structure):
    _fields_ = [(n, C.c_double) for n in (
        "kB", "pt_min", "n_sigma", "z0max", "d0max", "chi2max", "dr2max", "map_kscale", "map_z0",
        "ec_md_sys", "modez_slack", "seed_sig_phi", "seed_sig_pt", "seed_sig_z")] + [
        ("sig_t", C.c_double * 4), ("sig_z", C.c_double * 4), ("sig_r", C.c_double * 4),
        ("dup_t5_shared", C.c_int32), ("dup_pt5_shared", C.c_int32), ("dup_pt3_shared", C.c_int32),
        ("s0_enabled", C.c_int32), ("start_layer_mask", C.c_uint32)]


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (-O2, no fast-math, no intrinsics).  LST_ORACLE_SO (tests only:
    tests/test_oracle_mutations.py) names an already built library to load instead."""
    if os.environ.get("LST_ORACLE_SO"):
        return os.environ["LST_ORACLE_SO"]
    stale = (not os.path.exists(_SO)) or any(
        os.path.getmtime(p) > os.path.getmtime(_SO) for p in (_SRC, _HDR))
    if force or stale:
        subprocess.check_call(["gcc", "-O2", "-std=c11", "-fPIC", "-shared", "-Wall", "-Wextra",
                               "-fno-fast-math", "-o", _SO, _SRC, "-lm"])
    return _SO


_lib = None


def lib():
    global _lib
    if _lib is None:
        L = C.CDLL(build())
        vp, u32, i32 = C.c_void_p, C.c_uint32, C.c_int
        L.lsto_default_config.argtypes = [C.POINTER(Config)]
        L.lsto_build_module_map.argtypes = [u32] + [vp] * 8 + [C.POINTER(Config), C.POINTER(vp), C.POINTER(vp)]
        L.lsto_free.argtypes = [vp]
        L.lsto_create.restype = vp
        L.lsto_create.argtypes = [u32, vp, vp, vp, vp, C.POINTER(Config)]
        L.lsto_destroy.argtypes = [vp]
        L.lsto_load_event.argtypes = [vp, u32, vp, vp, vp, vp, u32, vp, vp, vp, vp, vp, vp]
        L.lsto_set_truncation.argtypes = [vp, vp, vp]
        L.lsto_set_s0_fixpoint.argtypes = [vp, i32]
        L.lsto_build_md.argtypes = [vp]
        for f in ("lsto_build_ls", "lsto_build_t3", "lsto_build_t5", "lsto_dedup"):
            getattr(L, f).argtypes = [vp, i32]
        L.lsto_link_pixel.argtypes = [vp, u32, u32]
        L.lsto_link_pixel_indexed.argtypes = [vp, u32, u32]
        L.lsto_test_cuts.argtypes = [C.POINTER(Config), i32, vp, vp, vp, vp, vp, i32, C.POINTER(i32)]
        L.lsto_test_inject.argtypes = [vp, u32, vp, u32, vp, u32, vp, vp, u32, vp, vp, u32, vp, vp]
        L.lsto_count.restype = u32
        L.lsto_count.argtypes = [vp, i32]
        L.lsto_arity.restype = u32
        L.lsto_arity.argtypes = [i32]
        L.lsto_get.argtypes = [vp, i32, vp, vp, vp, vp]
        L.lsto_get_t5_kin.argtypes = [vp, vp]
        L.lsto_get_keep.argtypes = [vp, i32, vp]
        L.lsto_eval.argtypes = [vp, i32, vp, u32, C.POINTER(C.c_double)]
        L.lsto_test_helpers.argtypes = [vp, vp, vp, C.c_double, vp]
        L.lsto_test_kasa.argtypes = [C.POINTER(Config), vp, vp, vp, C.c_double, C.POINTER(C.c_double),
                                     C.POINTER(C.c_double)]
        _lib = L
    return _lib


def default_config() -> Config:
    c = Config()
    lib().lsto_default_config(C.byref(c))
    return c


def _p(a):
    return a.ctypes.data_as(C.c_void_p)


def build_module_map(geom, cfg: Config | None = None):
    """C2 module map of a lstgen.Geometry -> (row_offsets u32[n+1], cols u32[nnz])."""
    cfg = cfg or default_config()
    off, cols = C.c_void_p(), C.c_void_p()
    n = geom.n_modules
    arrs = [np.ascontiguousarray(a) for a in (geom.category, geom.logical_layer, geom.rmin, geom.rmax,
                                              geom.phic, geom.half_phi, geom.zmin, geom.zmax)]
    rc = lib().lsto_build_module_map(n, *[_p(a) for a in arrs], C.byref(cfg), C.byref(off), C.byref(cols))
    assert rc == 0
    o = np.ctypeslib.as_array(C.cast(off, C.POINTER(C.c_uint32)), shape=(n + 1,)).copy()
    nnz = int(o[-1])
    c = np.ctypeslib.as_array(C.cast(cols, C.POINTER(C.c_uint32)), shape=(max(nnz, 1),)).copy()[:nnz]
    lib().lsto_free(off)
    lib().lsto_free(cols)
    return o, c


class Oracle:
    """One detector (+ module map) and, after load(), one event."""

    def __init__(self, geom, map_offsets, map_cols, cfg: Config | None = None):
        self.cfg = cfg or default_config()
        self._cat = np.ascontiguousarray(geom.category, dtype=np.uint8)
        self._lay = np.ascontiguousarray(geom.logical_layer, dtype=np.uint8)
        self._off = np.ascontiguousarray(map_offsets, dtype=np.uint32)
        self._cols = np.ascontiguousarray(map_cols, dtype=np.uint32)
        cols = self._cols if self._cols.size else np.zeros(1, np.uint32)
        self._h = lib().lsto_create(geom.n_modules, _p(self._cat), _p(self._lay), _p(self._off), _p(cols),
                                    C.byref(self.cfg))
        self.n_seeds = 0

    def close(self):
        if self._h:
            lib().lsto_destroy(self._h)
            self._h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    def set_truncation(self, phic, caps=None):
        """Occupancy-truncation mode: azimuth hit order + per-bucket caps [6, 16] (or None)."""
        ph = np.ascontiguousarray(phic, dtype=np.float32)
        cp = np.ascontiguousarray(caps, dtype=np.uint32).reshape(6, 16) if caps is not None else None
        rc = lib().lsto_set_truncation(self._h, _p(ph), _p(cp) if cp is not None else None)
        assert rc == 0

    def set_s0_fixpoint(self, on=True):
        """Greedy (fix-point) S0 for the T5 collection instead of the non-greedy rule."""
        assert lib().lsto_set_s0_fixpoint(self._h, int(on)) == 0

    def load(self, ev):
        f = lambda a, dt: np.ascontiguousarray(a, dtype=dt)
        x, y, z, det = f(ev.x, np.float32), f(ev.y, np.float32), f(ev.z, np.float32), f(ev.det, np.uint32)
        sp, se, sf, sz = (f(a, np.float32) for a in (ev.seed_pt, ev.seed_eta, ev.seed_phi, ev.seed_z0))
        sq, sid = f(ev.seed_q, np.int8), f(ev.seed_hit_ids, np.uint32)
        rc = lib().lsto_load_event(self._h, len(x), _p(x), _p(y), _p(z), _p(det), len(sp), _p(sp), _p(se),
                                   _p(sf), _p(sz), _p(sq), _p(sid))
        if rc != 0:
            raise ValueError("oracle: invalid event (det out of range)")
        self.n_seeds = len(sp)

    def run(self, upto: int = TC, brute: bool = False, seed_range=None, pixel_indexed: bool = False):
        """Build the levels up to `upto`.  brute: all-pairs loops instead of the index-driven ones
        (module map, joins, cleaning).  Pixel linking is all pairs unless pixel_indexed (identical
        output through a per-module first-anchor window)."""
        L, b = lib(), int(brute)
        L.lsto_build_md(self._h)
        if upto >= LS:
            L.lsto_build_ls(self._h, b)
        if upto >= T3:
            L.lsto_build_t3(self._h, b)
        if upto >= T5:
            L.lsto_build_t5(self._h, b)
        if upto >= PT3:
            s0, s1 = seed_range if seed_range is not None else (0, self.n_seeds)
            (L.lsto_link_pixel_indexed if pixel_indexed else L.lsto_link_pixel)(self._h, s0, s1)
        if upto >= TC:
            L.lsto_dedup(self._h, b)
        return self

    def count(self, level: int) -> int:
        return int(lib().lsto_count(self._h, level))

    def get(self, level: int):
        """dict(hits [n, arity] u32, parents [n,2] u32, f [n,4] f64, margin [n] f64)."""
        n, ar = self.count(level), int(lib().lsto_arity(level))
        hits = np.zeros((n, max(ar, 1)), np.uint32)
        par = np.zeros((n, 2), np.uint32)
        f = np.zeros((n, 4), np.float64)
        m = np.zeros(n, np.float64)
        lib().lsto_get(self._h, level, _p(hits) if ar else None, _p(par), _p(f), _p(m))
        return dict(hits=hits[:, :ar], parents=par, f=f, margin=m)

    def t5_kin(self):
        out = np.zeros((self.count(T5), 3), np.float64)
        lib().lsto_get_t5_kin(self._h, _p(out))
        return out

    def keep(self, level: int):
        n = self.n_seeds if level == PLS_KEEP else self.count(level)
        k = np.zeros(max(n, 1), np.uint8)
        rc = lib().lsto_get_keep(self._h, level, _p(k))
        assert rc == 0
        return k[:n].astype(bool)

    def dedup(self, brute: bool = False):
        lib().lsto_dedup(self._h, int(brute))
        return self

    def inject(self, md_hits, t3_md=(), t5_md=(), t5_kin=(), pt3_po=(), pt3_chi2=(), pt5_po=(), pt5_chi2=()):
        """Test hook: replace the object collections of the loaded event by hand-built ones
        (lsto_test_inject) so that dedup() can be pinned on constructed cases."""
        u = lambda a, w: np.ascontiguousarray(np.asarray(a, dtype=np.uint32).reshape(-1, w))
        d = lambda a, w: np.ascontiguousarray(np.asarray(a, dtype=np.float64).reshape(-1, w))
        md, t3, t5, k5 = u(md_hits, 2), u(t3_md, 3), u(t5_md, 5), d(t5_kin, 4)
        p3, c3, p5, c5 = u(pt3_po, 2), d(pt3_chi2, 1), u(pt5_po, 2), d(pt5_chi2, 1)
        assert len(t5) == len(k5) and len(p3) == len(c3) and len(p5) == len(c5)
        rc = lib().lsto_test_inject(self._h, len(md), _p(md), len(t3), _p(t3), len(t5), _p(t5), _p(k5),
                                    len(p3), _p(p3), _p(c3), len(p5), _p(p5), _p(c5))
        if rc != 0:
            raise ValueError("oracle inject: index out of range")
        return self

    def eval(self, level: int, hits, seed: int = 0):
        """Evaluate one candidate given original hit indices -> (passed, margin)."""
        h = np.ascontiguousarray(hits, dtype=np.uint32)
        m = C.c_double(0.0)
        rc = lib().lsto_eval(self._h, level, _p(h), int(seed), C.byref(m))
        if rc < 0:
            raise ValueError("oracle eval: bad arguments")
        return bool(rc), m.value


def helpers(A, B, Cc, k=0.0):
    """C0 helpers on double inputs -> dict (test hook)."""
    a, b, c = (np.ascontiguousarray(v, dtype=np.float64) for v in (A, B, Cc))
    out = np.zeros(7)
    lib().lsto_test_helpers(_p(a), _p(b), _p(c), float(k), _p(out))
    return dict(sd=out[0], dphi=out[1], chord=out[2], dr=out[3], kappa3=out[4], arc=out[5], wrap=out[6])


def kasa(x, y, cat, kc, cfg: Config | None = None):
    """Weighted Kasa circle fit of 5 points (test hook) -> (ok, R, chi2)."""
    cfg = cfg or default_config()
    x, y = (np.ascontiguousarray(v, dtype=np.float64) for v in (x, y))
    cat = np.ascontiguousarray(cat, dtype=np.int32)
    R, c2 = C.c_double(0), C.c_double(0)
    ok = lib().lsto_test_kasa(C.byref(cfg), _p(x), _p(y), _p(cat), float(kc), C.byref(R), C.byref(c2))
    return bool(ok), R.value, c2.value



CUT_LE, CUT_POS, CUT_GUARD = 0, 1, 2


def cuts(level: int, pts, cats, aux=None, cfg: Config | None = None):
    """Test hook (lsto_test_cuts): one selection function on DOUBLE inputs.
    Returns (passed, f[8], trace) with trace = [(kind, v, thr), ...] in evaluation order."""
    cfg = cfg or default_config()
    pts = np.ascontiguousarray(pts, dtype=np.float64).reshape(-1)
    cats = np.ascontiguousarray(cats, dtype=np.int32).reshape(-1)
    aux = np.ascontiguousarray(aux if aux is not None else np.zeros(8), dtype=np.float64).reshape(-1)
    f, tr, n = np.zeros(8), np.zeros(3 * 64), C.c_int32(0)
    rc = lib().lsto_test_cuts(C.byref(cfg), int(level), _p(pts), _p(cats), _p(aux), _p(f), _p(tr), len(tr), C.byref(n))
    if rc < 0:
        raise ValueError("oracle cuts: bad level")
    assert 3 * n.value <= len(tr)
    return bool(rc), f, [tuple(tr[3 * k:3 * k + 3]) for k in range(n.value)]
