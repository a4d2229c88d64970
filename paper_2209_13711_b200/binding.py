"""Thin ctypes binding of include/lst.h (argument marshalling only).

Every step of the hot path runs inside liblst_b200.so (hand-written CUDA for sm_100a).  PyTorch is
used for device memory (the per-slot workspace), streams and nothing else.  There is no CPU
fallback: importing works without a GPU (the library loads and exports its symbols), but creating
a context without the library or without a CUDA device raises.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SO = os.path.join(_HERE, "liblst_b200.so")

LST_OK, LST_EINVAL, LST_ENOMEM, LST_ECUDA, LST_ESTATE = 0, -1, -2, -3, -4
LST_MD, LST_LS, LST_T3, LST_T5, LST_PT3, LST_PT5, LST_TC = range(7)
LST_NLEVEL = 7
LEVEL_NAMES = ("MD", "LS", "T3", "T5", "PT3", "PT5", "TC")

EXPORTS = ("lst_default_config", "lst_build_module_map", "lst_free", "lst_create", "lst_destroy",
           "lst_workspace_bytes", "lst_bind_workspace", "lst_load_event", "lst_run", "lst_get_objects",
           "lst_get_counts", "lst_launches_per_run", "lst_run_timed", "lst_strerror", "lst_run_batch", "lst_batch_events", "lst_get_fixpoint_unsettled")
TEST_EXPORTS = ("lst_host_eval", "lst_host_ls_window", "lst_test_get_hit_index")      # include/lst_test.h
STATIC_EXPORTS = ("lst_index_hits_static",)                  # include/lst_static.h
LST_STATIC_MAX_HITS, LST_STATIC_MAX_DETS = 1 << 18, 1 << 16


class lst_config(C.Structure):
    _fields_ = [(n, C.c_double) for n in (
        "kB", "pt_min", "n_sigma", "z0max", "d0max", "chi2max", "dr2max", "map_kscale", "map_z0",
        "ec_md_sys", "modez_slack", "seed_sig_phi", "seed_sig_pt", "seed_sig_z")] + [
        ("sig_t", C.c_double * 4), ("sig_z", C.c_double * 4), ("sig_r", C.c_double * 4),
        ("dup_t5_shared", C.c_int32), ("dup_pt5_shared", C.c_int32), ("dup_pt3_shared", C.c_int32),
        ("s0_enabled", C.c_int32), ("start_layer_mask", C.c_uint32)] + [
        (n, C.c_float) for n in (
            "cap_md_per_hit", "cap_ls_per_hit", "cap_t3_per_hit", "cap_t5_per_hit", "cap_pt3_per_seed",
            "cap_pt5_per_seed", "cap_mdcand_per_hit", "cap_lscand_per_hit", "cap_t3cand_per_hit",
            "cap_t5cand_per_hit")] + [("use_cuda_graph", C.c_int32), ("enum_pruning", C.c_int32), ("use_pdl", C.c_int32),
                                   ("batch_events", C.c_int32), ("trunc_cap", (C.c_uint32 * 16) * 6),
                                   ("store_half", C.c_int32), ("s0_fixpoint_passes", C.c_int32)]


class lst_geometry(C.Structure):
    _fields_ = [("n_modules", C.c_uint32), ("category", C.c_void_p), ("logical_layer", C.c_void_p),
                ("rmin", C.c_void_p), ("rmax", C.c_void_p), ("phic", C.c_void_p), ("half_phi", C.c_void_p),
                ("zmin", C.c_void_p), ("zmax", C.c_void_p)]


class lst_module_map(C.Structure):
    _fields_ = [("row_offsets", C.c_void_p), ("cols", C.c_void_p)]


class lst_hits(C.Structure):
    _fields_ = [("n", C.c_uint32), ("x", C.c_void_p), ("y", C.c_void_p), ("z", C.c_void_p),
                ("det", C.c_void_p), ("on_device", C.c_int)]


class lst_pixel_seeds(C.Structure):
    _fields_ = [("n", C.c_uint32), ("pt", C.c_void_p), ("eta", C.c_void_p), ("phi", C.c_void_p),
                ("z0", C.c_void_p), ("q", C.c_void_p), ("hit_ids", C.c_void_p), ("on_device", C.c_int)]


class lst_objects(C.Structure):
    _fields_ = [("n", C.c_uint32), ("arity", C.c_uint32), ("hit_idx", C.c_void_p), ("parents", C.c_void_p),
                ("f", C.c_void_p), ("keep", C.c_void_p), ("on_device", C.c_int)]


class LstError(RuntimeError):
    def __init__(self, status, where):
        self.status = status
        super().__init__("%s: %s (%d)" % (where, lib().lst_strerror(status).decode(), status))


_lib = None


def lib():
    """Load liblst_b200.so (built by paper_2209_13711_b200.build); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(_SO):
            raise ImportError("liblst_b200.so is not built: run `python -m paper_2209_13711_b200.build` "
                              "(there is no CPU fallback)")
        L = C.CDLL(_SO)
        vp, u32 = C.c_void_p, C.c_uint32
        L.lst_default_config.argtypes = [C.POINTER(lst_config)]
        L.lst_default_config.restype = None
        L.lst_build_module_map.argtypes = [C.POINTER(lst_geometry), C.POINTER(lst_config), C.POINTER(vp), C.POINTER(vp)]
        L.lst_free.argtypes = [vp]
        L.lst_free.restype = None
        L.lst_create.argtypes = [C.POINTER(lst_geometry), C.POINTER(lst_module_map), C.POINTER(lst_config), u32, u32,
                                 u32, C.POINTER(vp)]
        L.lst_destroy.argtypes = [vp]
        L.lst_destroy.restype = None
        L.lst_workspace_bytes.argtypes = [vp]
        L.lst_workspace_bytes.restype = C.c_size_t
        L.lst_bind_workspace.argtypes = [vp, u32, vp, C.c_size_t]
        L.lst_load_event.argtypes = [vp, u32, C.POINTER(lst_hits), C.POINTER(lst_pixel_seeds), vp]
        L.lst_run.argtypes = [vp, u32, vp]
        L.lst_run_batch.argtypes = [vp, u32, vp]
        L.lst_batch_events.argtypes = [vp]
        L.lst_batch_events.restype = u32
        L.lst_get_fixpoint_unsettled.argtypes = [vp, u32, C.POINTER(u32)]
        L.lst_get_objects.argtypes = [vp, u32, C.c_int, C.c_int, C.POINTER(lst_objects)]
        L.lst_get_counts.argtypes = [vp, u32, vp, vp]
        L.lst_launches_per_run.argtypes = [vp]
        L.lst_launches_per_run.restype = u32
        L.lst_run_timed.argtypes = [vp, u32, vp, u32, vp, vp, C.POINTER(u32)]
        L.lst_strerror.argtypes = [C.c_int]
        L.lst_strerror.restype = C.c_char_p
        L.lst_host_eval.argtypes = [C.POINTER(lst_config), C.c_int, u32, vp, vp, vp, vp, vp, vp]
        L.lst_host_ls_window.argtypes = [C.POINTER(lst_config), u32, vp, vp, vp, vp, vp, vp]
        L.lst_test_get_hit_index.argtypes = [vp, u32, vp, vp, vp, C.POINTER(u32)]
        L.lst_index_hits_static.argtypes = [vp, vp, vp, vp, u32, vp, u32, vp, vp, vp, vp, vp, C.c_char_p, C.c_size_t]
        _lib = L
    return _lib


def _check(rc, where):
    if rc != LST_OK:
        raise LstError(rc, where)


def _p(a):
    return C.c_void_p(a.ctypes.data) if a is not None else None


def lst_default_config() -> lst_config:
    c = lst_config()
    lib().lst_default_config(C.byref(c))
    return c


class _GeomArrays:
    """Keeps contiguous numpy copies alive while a lst_geometry points at them."""

    def __init__(self, geom):
        f = lambda a, dt: np.ascontiguousarray(a, dtype=dt)
        self.arr = [f(geom.category, np.uint8), f(geom.logical_layer, np.uint8)] + [
            f(getattr(geom, n), np.float32) for n in ("rmin", "rmax", "phic", "half_phi", "zmin", "zmax")]
        self.c = lst_geometry(int(self.arr[0].shape[0]), *[a.ctypes.data for a in self.arr])


def lst_build_module_map(geom, cfg: lst_config | None = None):
    """C2 module map (host) -> (row_offsets u32[n+1], cols u32[nnz])."""
    ga = _GeomArrays(geom)
    off, cols = C.c_void_p(), C.c_void_p()
    _check(lib().lst_build_module_map(C.byref(ga.c), C.byref(cfg) if cfg is not None else None, C.byref(off),
                                      C.byref(cols)), "lst_build_module_map")
    n = ga.c.n_modules
    o = np.ctypeslib.as_array(C.cast(off, C.POINTER(C.c_uint32)), shape=(n + 1,)).copy()
    nnz = int(o[-1])
    c = np.ctypeslib.as_array(C.cast(cols, C.POINTER(C.c_uint32)), shape=(max(nnz, 1),)).copy()[:nnz]
    lib().lst_free(off)
    lib().lst_free(cols)
    return o, c


def lst_host_eval(level, pts, cats, aux=None, cfg: lst_config | None = None):
    """Test hook: the CUDA path's per-candidate arithmetic compiled for the host -> (pass, pre, f[n,3])."""
    pts = np.ascontiguousarray(pts, dtype=np.float32)
    cats = np.ascontiguousarray(cats, dtype=np.uint8)
    n = pts.shape[0]
    aux = np.ascontiguousarray(aux, dtype=np.float64) if aux is not None else None
    ok, pre, f = np.zeros(n, np.uint8), np.zeros(n, np.uint8), np.zeros((n, 3), np.float64)
    _check(lib().lst_host_eval(C.byref(cfg) if cfg is not None else None, level, n, _p(pts), _p(cats), _p(aux),
                               _p(ok), _p(pre), _p(f)), "lst_host_eval")
    return ok.astype(bool), pre.astype(bool), f


def lst_host_ls_window(row, row_cat, box, box_cat, cfg: lst_config | None = None):
    """Test hook: ls_row_window on the host -> (live [n] bool, w [n] f32)."""
    row = np.ascontiguousarray(row, dtype=np.float32)
    box = np.ascontiguousarray(box, dtype=np.float32)
    rc, bc = (np.ascontiguousarray(a, dtype=np.uint8) for a in (row_cat, box_cat))
    n = row.shape[0]
    live, w = np.zeros(n, np.uint8), np.zeros(n, np.float32)
    _check(lib().lst_host_ls_window(C.byref(cfg) if cfg is not None else None, n, _p(row), _p(rc), _p(box), _p(bc),
                                    _p(live), _p(w)), "lst_host_ls_window")
    return live.astype(bool), w


def lst_index_hits_static(x, y, z, det, phic, det_off, hit_orig, hit_xyzr, n_rejected, stream=None, n_hits=None,
                          n_dets=None):
    """include/lst_static.h: step a0 with the library's fixed scratch array, for callers that may not
    allocate GPU memory.  Every array is a torch CUDA tensor the CALLER made (inputs x, y, z f32 and
    det i32 / u32 bits of n_hits elements, phic f32 of n_dets / 2; outputs det_off [n_dets + 1],
    hit_orig [n_hits], hit_xyzr [n_hits, 4] f32, n_rejected [1]); this wrapper only passes their
    addresses on and allocates nothing itself.  Nothing is synchronised: the work is enqueued on
    `stream` (default: the legacy default stream).  Events above LST_STATIC_MAX_HITS / _DETS raise
    LstStaticError with the library's message.  Calls share one scratch array per GPU: keep them on
    one stream (or order them with events), and make the first call on a GPU before any stream capture."""
    n_hits = int(x.shape[0]) if n_hits is None else int(n_hits)
    n_dets = 2 * int(phic.shape[0]) if n_dets is None else int(n_dets)
    ptr = lambda t: C.c_void_p(t.data_ptr()) if t is not None else None
    err = C.create_string_buffer(384)
    rc = lib().lst_index_hits_static(ptr(x), ptr(y), ptr(z), ptr(det), n_hits, ptr(phic), n_dets, ptr(det_off),
                                     ptr(hit_orig), ptr(hit_xyzr), ptr(n_rejected),
                                     C.c_void_p(stream.cuda_stream if stream is not None else 0), err, len(err))
    if rc != LST_OK:
        raise LstStaticError(rc, err.value.decode())


class LstStaticError(RuntimeError):
    def __init__(self, status, text):
        self.status = status
        super().__init__("%s (%d)" % (text, status))


class LST:
    """One detector on one GPU with n_slots event slots (include/lst.h).  Methods are the C calls."""

    def __init__(self, geom, map_offsets, map_cols, cfg: lst_config | None = None, n_slots: int = 1,
                 max_hits: int = 1 << 18, max_seeds: int = 1 << 13, device: str = "cuda:0"):
        import torch
        if not torch.cuda.is_available():
            raise RuntimeError("paper_2209_13711_b200 needs a CUDA device (no CPU fallback)")
        self._torch = torch
        self.device = torch.device(device)
        self.cfg = cfg if cfg is not None else lst_default_config()
        self.n_slots, self.max_hits, self.max_seeds = n_slots, max_hits, max_seeds
        ga = _GeomArrays(geom)
        self._n_modules_src = ga.arr[0]
        off = np.ascontiguousarray(map_offsets, dtype=np.uint32)
        cols = np.ascontiguousarray(map_cols, dtype=np.uint32)
        cols_ = cols if cols.size else np.zeros(1, np.uint32)
        mm = lst_module_map(off.ctypes.data, cols_.ctypes.data)
        self._h = C.c_void_p()
        with torch.cuda.device(self.device):
            _check(lib().lst_create(C.byref(ga.c), C.byref(mm), C.byref(self.cfg), n_slots, max_hits, max_seeds,
                                    C.byref(self._h)), "lst_create")
            self.workspace_bytes = int(lib().lst_workspace_bytes(self._h))
            self._ws = []
            for s in range(n_slots):
                w = torch.empty(self.workspace_bytes + 256, dtype=torch.uint8, device=self.device)
                ptr = (w.data_ptr() + 255) & ~255
                _check(lib().lst_bind_workspace(self._h, s, C.c_void_p(ptr), self.workspace_bytes), "lst_bind_workspace")
                self._ws.append(w)
        self._keep = {}

    def close(self):
        if getattr(self, "_h", None) and self._h.value:
            lib().lst_destroy(self._h)
            self._h = C.c_void_p()
            self._ws = []

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    @staticmethod
    def _stream_ptr(stream):
        return C.c_void_p(stream.cuda_stream if stream is not None else 0)

    def lst_load_event(self, slot, x, y, z, det, seeds=None, stream=None):
        """x, y, z (f32), det (u32): numpy arrays (host) or torch CUDA tensors.  seeds: None or a tuple
        (pt, eta, phi, z0 f32, q i8, hit_ids u32[n,4]) of the same kind."""
        torch = self._torch
        on_dev = isinstance(x, torch.Tensor)
        if on_dev:
            ptr = lambda a: C.c_void_p(a.data_ptr())
            arrs = [x, y, z, det]
            n = int(x.shape[0])
        else:
            f = lambda a, dt: np.ascontiguousarray(a, dtype=dt)
            arrs = [f(x, np.float32), f(y, np.float32), f(z, np.float32), f(det, np.uint32)]
            ptr = _p
            n = int(arrs[0].shape[0])
        h = lst_hits(n, *[ptr(a) for a in arrs], int(on_dev))
        sp = None
        sarrs = None
        if seeds is not None and len(seeds[0]) > 0:
            if on_dev:
                sarrs = list(seeds)
            else:
                dts = (np.float32, np.float32, np.float32, np.float32, np.int8, np.uint32)
                sarrs = [np.ascontiguousarray(a, dtype=dt) for a, dt in zip(seeds, dts)]
            sp = lst_pixel_seeds(int(sarrs[0].shape[0]), *[ptr(a) for a in sarrs], int(on_dev))
        self._keep[slot] = (arrs, sarrs)    # keep host arrays alive until the copy has run
        _check(lib().lst_load_event(self._h, slot, C.byref(h), C.byref(sp) if sp is not None else None,
                                    self._stream_ptr(stream)), "lst_load_event")

    def lst_run(self, slot, stream=None):
        _check(lib().lst_run(self._h, slot, self._stream_ptr(stream)), "lst_run")

    def lst_run_batch(self, group, stream=None):
        _check(lib().lst_run_batch(self._h, group, self._stream_ptr(stream)), "lst_run_batch")

    def lst_get_fixpoint_unsettled(self, slot):
        n = C.c_uint32(0)
        _check(lib().lst_get_fixpoint_unsettled(self._h, slot, C.byref(n)), "lst_get_fixpoint_unsettled")
        return int(n.value)

    def lst_run_timed(self, slot, stream=None):
        """-> list of (kernel name, ms) of one un-graphed, event-bracketed pass of the chain."""
        cap = 96
        names = (C.c_char_p * cap)()
        ms = np.zeros(cap, np.float32)
        n = C.c_uint32(0)
        _check(lib().lst_run_timed(self._h, slot, self._stream_ptr(stream), cap, C.cast(names, C.c_void_p), _p(ms),
                                   C.byref(n)), "lst_run_timed")
        k = min(int(n.value), cap)
        return [(names[i].decode(), float(ms[i])) for i in range(k)]

    def lst_get_counts(self, slot):
        cnt = np.zeros(LST_NLEVEL, np.uint32)
        cand = np.zeros(18, np.uint64)
        _check(lib().lst_get_counts(self._h, slot, _p(cnt), _p(cand)), "lst_get_counts")
        return cnt, cand

    def lst_get_objects(self, slot, level):
        """Host copy of one level: dict(hits [n, arity], parents [n, 2], f [n, 4], keep [n] or None)."""
        o = lst_objects()
        _check(lib().lst_get_objects(self._h, slot, level, 1, C.byref(o)), "lst_get_objects")
        n, ar = int(o.n), int(o.arity)

        def arr(ptr, shape, ct, dt):
            if n == 0 or not ptr:
                return np.zeros(shape, dt)
            return np.ctypeslib.as_array(C.cast(ptr, C.POINTER(ct)), shape=shape).copy()

        keep = arr(o.keep, (n,), C.c_uint8, np.uint8).astype(bool) if o.keep else None
        return dict(hits=arr(o.hit_idx, (n, ar), C.c_uint32, np.uint32),
                    parents=arr(o.parents, (n, 2), C.c_uint32, np.uint32),
                    f=arr(o.f, (n, 4), C.c_float, np.float32), keep=keep)

    def lst_test_get_hit_index(self, slot):
        """Test hook (include/lst_test.h): (det_off, hit_orig, hit_xyzr [n, 4]) step a0 left in the slot."""
        n = C.c_uint32(0)
        _check(lib().lst_test_get_hit_index(self._h, slot, None, None, None, C.byref(n)), "lst_test_get_hit_index")
        n = int(n.value)
        n_det = 2 * len(self._n_modules_src)
        det_off, orig, xyzr = np.zeros(n_det + 1, np.uint32), np.zeros(max(n, 1), np.uint32), np.zeros((max(n, 1), 4), np.float32)
        _check(lib().lst_test_get_hit_index(self._h, slot, _p(det_off), _p(orig), _p(xyzr), None), "lst_test_get_hit_index")
        return det_off, orig[:n], xyzr[:n]

    def launches_per_run(self):
        return int(lib().lst_launches_per_run(self._h))
