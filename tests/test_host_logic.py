"""CPU-only checks of the product's host logic (no GPU, no compute kernels):
  * the C-ABI library loads and exports every symbol include/lst.h declares;
  * the host module-map builder equals the oracle's (independent implementations of reading C2);
  * the CUDA path's per-candidate arithmetic (lst_math.cuh, compiled for the host through the
    lst_host_eval test hook) takes the same decisions as the oracle on exhaustively enumerated
    candidates, its fp32 pre-filter never rejects an accepted candidate, and its derived floats
    agree to rounding.
"""
import os
import re

import numpy as np
import pytest

import lstgen
from oracle import lst_oracle as O
from paper_2209_13711_b200 import binding as B
from paper_2209_13711_b200 import build as lst_build

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module", autouse=True)
def _built():
    lst_build.build()


def _declared(header):
    hdr = open(os.path.join(ROOT, "include", header)).read()
    hdr = re.sub(r"/\*.*?\*/", "", hdr, flags=re.S)
    return set(re.findall(r"\b(lst_[a-z_0-9]+)\s*\(", hdr))


def test_library_exports_every_declared_symbol():
    declared = _declared("lst.h")
    assert {"lst_create", "lst_load_event", "lst_run", "lst_get_objects"} <= declared
    L = B.lib()
    for name in sorted(declared):
        assert hasattr(L, name), name
    assert declared == set(B.EXPORTS)
    # the test hooks live in their own header and are not part of the product API
    hooks = _declared("lst_test.h")
    assert hooks == set(B.TEST_EXPORTS) and not (hooks & declared)
    for name in sorted(hooks):
        assert hasattr(L, name), name
    # the allocation-free entry point has a header of its own
    static = _declared("lst_static.h")
    assert static == set(B.STATIC_EXPORTS) and not (static & (declared | hooks))
    for name in sorted(static):
        assert hasattr(L, name), name
    hdr = open(os.path.join(ROOT, "include", "lst_static.h")).read()
    assert "LST_STATIC_MAX_HITS %du" % B.LST_STATIC_MAX_HITS in hdr and "LST_STATIC_MAX_DETS %du" % B.LST_STATIC_MAX_DETS in hdr


def test_default_config_matches_oracle_config():
    a, b = B.lst_default_config(), O.default_config()
    for name, _ in O.Config._fields_:
        va, vb = getattr(a, name), getattr(b, name)
        if hasattr(va, "__len__"):
            assert list(va) == list(vb), name
        else:
            assert va == vb, name


@pytest.mark.parametrize("barrel_only", [True, False])
def test_module_map_builder_equals_oracle(barrel_only, geom_barrel, geom_full, map_barrel, map_full):
    geom, (off_o, cols_o) = (geom_barrel, map_barrel) if barrel_only else (geom_full, map_full)
    off, cols = B.lst_build_module_map(geom)
    assert np.array_equal(off, off_o)
    assert np.array_equal(cols, cols_o)
    assert int(np.diff(off).max()) <= 512


def test_invalid_arguments_are_rejected_without_gpu(geom_barrel):
    import ctypes as C
    L = B.lib()
    assert L.lst_build_module_map(None, None, None, None) == B.LST_EINVAL
    assert L.lst_workspace_bytes(None) == 0
    assert L.lst_strerror(B.LST_ENOMEM).decode().startswith("workspace")
    out = C.c_void_p()
    assert L.lst_create(None, None, None, 1, 10, 10, C.byref(out)) == B.LST_EINVAL


# ----------------------------------------------------------------------------- arithmetic vs oracle
def _oracle(geom, mp, ev, upto=O.T5):
    o = O.Oracle(geom, mp[0], mp[1])
    o.load(ev)
    o.run(upto=upto)
    return o


@pytest.fixture(scope="module")
def small_full(geom_full, map_full):
    ev = lstgen.make_event(geom_full, "cfg3", n_particles=1500)
    return ev, _oracle(geom_full, map_full, ev)


def _md_candidates(geom, ev):
    det = ev.det.astype(np.int64)
    order = np.argsort(det, kind="stable")
    pairs = []
    sd = det[order]
    mods = np.unique(sd >> 1)
    for m in mods:
        lo = order[np.searchsorted(sd, 2 * m):np.searchsorted(sd, 2 * m + 1)]
        up = order[np.searchsorted(sd, 2 * m + 1):np.searchsorted(sd, 2 * m + 2)]
        if len(lo) and len(up):
            a, b = np.meshgrid(lo, up, indexing="ij")
            pairs.append(np.stack([a.ravel(), b.ravel()], 1))
    return np.concatenate(pairs)


def test_md_arithmetic_equals_oracle(geom_full, small_full):
    ev, o = small_full
    pairs = _md_candidates(geom_full, ev)
    xyz = np.stack([ev.x, ev.y, ev.z], 1)
    pts = np.concatenate([xyz[pairs[:, 0]], xyz[pairs[:, 1]]], 1)
    cat = geom_full.category[(ev.det[pairs[:, 0]] >> 1)]
    cats = np.stack([cat, cat], 1)
    ok, pre, f = B.lst_host_eval(B.LST_MD, pts, cats)
    md = o.get(O.MD)
    want = set(map(tuple, md["hits"].tolist()))
    got = set(map(tuple, pairs[ok].tolist()))
    assert got == want and len(want) > 1000
    assert not (ok & ~pre).any(), "fp32 pre-filter rejected an accepted MD"
    assert pre.mean() < 0.5                      # and it does filter
    idx = {t: i for i, t in enumerate(map(tuple, pairs.tolist()))}
    sel = np.array([idx[t] for t in map(tuple, md["hits"].tolist())])
    assert np.allclose(f[sel, 0], md["f"][:, 1], rtol=1e-12, atol=0)     # kappa
    assert np.allclose(f[sel, 1], md["f"][:, 2], rtol=1e-12, atol=0)     # sigma kappa
    assert np.allclose(f[sel, 2], md["f"][:, 0], rtol=1e-12, atol=1e-18)  # dphi


def _md_tables(geom, ev, o):
    md = o.get(O.MD)
    anchor = md["hits"][:, 0].astype(np.int64)
    xyz = np.stack([ev.x, ev.y, ev.z], 1)[anchor]
    mod = md["parents"][:, 0].astype(np.int64)
    return md, xyz, mod, geom.category[mod]


def test_ls_arithmetic_equals_oracle(geom_full, map_full, small_full):
    ev, o = small_full
    md, xyz, mod, cat = _md_tables(geom_full, ev, o)
    off, cols = map_full
    n_md = len(mod)
    mstart = np.searchsorted(mod, np.arange(geom_full.n_modules + 1))
    ii, oo = [], []
    for i in range(n_md):
        for B_ in cols[off[mod[i]]:off[mod[i] + 1]]:
            a, b = mstart[B_], mstart[B_ + 1]
            if b > a:
                ii.append(np.full(b - a, i)); oo.append(np.arange(a, b))
    ii, oo = np.concatenate(ii), np.concatenate(oo)
    pts = np.concatenate([xyz[ii], xyz[oo]], 1)
    cats = np.stack([cat[ii], cat[oo]], 1)
    aux = np.stack([md["f"][ii, 1], md["f"][ii, 2], md["f"][oo, 1], md["f"][oo, 2]], 1)
    ok, pre, f = B.lst_host_eval(B.LST_LS, pts, cats, aux)
    ls = o.get(O.LS)
    want = set(map(tuple, ls["parents"].tolist()))
    got = set(zip(ii[ok].tolist(), oo[ok].tolist()))
    assert got == want and len(want) > 1000
    assert not (ok & ~pre).any(), "fp32 pre-filter rejected an accepted LS"
    assert pre.mean() < 0.3
    # the fp32 pre-filter sees fp32-rounded kappa_MD on the GPU as well (aux cast inside the hook)
    idx = {t: k for k, t in enumerate(zip(ii.tolist(), oo.tolist()))}
    sel = np.array([idx[t] for t in map(tuple, ls["parents"].tolist())])
    assert np.allclose(f[sel, 0], ls["f"][:, 1], rtol=1e-11, atol=0)
    assert np.allclose(f[sel, 2], ls["f"][:, 0], rtol=1e-11, atol=1e-18)
    assert (cats[:, 1] >= 2).sum() > 1000 and (cats[:, 1] < 2).sum() > 1000     # both modes exercised


def test_t3_t5_arithmetic_equals_oracle(geom_full, small_full):
    ev, o = small_full
    md, xyz, mod, cat = _md_tables(geom_full, ev, o)
    ls, t3, t5 = o.get(O.LS), o.get(O.T3), o.get(O.T5)
    lp = ls["parents"].astype(np.int64)
    first = np.searchsorted(lp[:, 0], np.arange(len(mod) + 1))
    # T3 candidates: LS a, LS b with inner(b) == outer(a)
    aa, bb = [], []
    for a in range(len(lp)):
        s, e = first[lp[a, 1]], first[lp[a, 1] + 1]
        if e > s:
            aa.append(np.full(e - s, a)); bb.append(np.arange(s, e))
    aa, bb = np.concatenate(aa), np.concatenate(bb)
    m = np.stack([lp[aa, 0], lp[aa, 1], lp[bb, 1]], 1)
    pts = xyz[m].reshape(len(m), 9)
    ok, pre, f = B.lst_host_eval(B.LST_T3, pts, cat[m])
    want = set(map(tuple, t3["parents"].tolist()))
    got = set(zip(aa[ok].tolist(), bb[ok].tolist()))
    assert got == want and len(want) > 500
    assert not (ok & ~pre).any(), "fp32 pre-filter rejected an accepted T3"
    print("T3 pre-filter keeps %.3f of the candidates, %.3f pass" % (pre.mean(), ok.mean()))
    assert pre.mean() < 0.9                      # and it does filter
    idx = {t: k for k, t in enumerate(zip(aa.tolist(), bb.tolist()))}
    sel = np.array([idx[t] for t in map(tuple, t3["parents"].tolist())])
    assert np.allclose(f[sel, 0], t3["f"][:, 1], rtol=1e-9, atol=0)      # kappa3
    assert np.allclose(f[sel, 1], t3["f"][:, 2], rtol=1e-9, atol=0)
    assert np.allclose(f[sel, 2], t3["f"][:, 0], rtol=1e-9, atol=1e-15)  # beta
    # T5 candidates: T3 a, T3 b with first MD of b == third MD of a
    tp = t3["parents"].astype(np.int64)
    tm = np.stack([lp[tp[:, 0], 0], lp[tp[:, 0], 1], lp[tp[:, 1], 1]], 1)
    tfirst = np.searchsorted(tm[:, 0], np.arange(len(mod) + 1))
    aa, bb = [], []
    for a in range(len(tm)):
        s, e = tfirst[tm[a, 2]], tfirst[tm[a, 2] + 1]
        if e > s:
            aa.append(np.full(e - s, a)); bb.append(np.arange(s, e))
    aa, bb = np.concatenate(aa), np.concatenate(bb)
    m5 = np.concatenate([tm[aa], tm[bb][:, 1:]], 1)
    pts = xyz[m5].reshape(len(m5), 15)
    aux = np.stack([t3["f"][aa, 1], t3["f"][aa, 2], t3["f"][bb, 1], t3["f"][bb, 2]], 1)
    ok, _, f = B.lst_host_eval(B.LST_T5, pts, cat[m5], aux)
    want = set(map(tuple, t5["parents"].tolist()))
    got = set(zip(aa[ok].tolist(), bb[ok].tolist()))
    assert got == want and len(want) > 100
    idx = {t: k for k, t in enumerate(zip(aa.tolist(), bb.tolist()))}
    sel = np.array([idx[t] for t in map(tuple, t5["parents"].tolist())])
    assert np.allclose(f[sel, 0], t5["f"][:, 0], rtol=1e-9)              # R
    assert np.allclose(f[sel, 1], t5["f"][:, 1], rtol=1e-6, atol=1e-9)   # chi2
    assert np.allclose(f[sel, 2], o.t5_kin()[:, 1], rtol=1e-9, atol=1e-12)  # eta


def test_ls_row_window_never_excludes_an_accepted_pair(geom_full, map_full, small_full):
    """The per-(inner MD, connected module) window of the LS enumeration (ls_row_window, run on the
    host): for every LS the oracle accepts, the module box test is live and the pair's azimuth
    difference lies inside the window; and the window does restrict (most module pairs are cut)."""
    ev, o = small_full
    md, xyz, mod, cat = _md_tables(geom_full, ev, o)
    ls = o.get(O.LS)["parents"].astype(np.int64)
    rt = np.hypot(xyz[:, 0].astype(np.float64), xyz[:, 1].astype(np.float64)).astype(np.float32)
    z = xyz[:, 2].astype(np.float32)
    nm = geom_full.n_modules
    box = np.zeros((nm, 4), np.float32)
    box[:, 0] = box[:, 2] = np.inf
    box[:, 1] = box[:, 3] = -np.inf
    np.minimum.at(box[:, 0], mod, rt); np.maximum.at(box[:, 1], mod, rt)
    np.minimum.at(box[:, 2], mod, z); np.maximum.at(box[:, 3], mod, z)
    i, oo = ls[:, 0], ls[:, 1]
    live, w = B.lst_host_ls_window(np.stack([rt[i], z[i]], 1), cat[i], box[mod[oo]], cat[oo])
    assert live.all()
    phi = np.arctan2(xyz[:, 1].astype(np.float64), xyz[:, 0].astype(np.float64))
    dphi = np.abs(np.remainder(phi[oo] - phi[i] + np.pi, 2 * np.pi) - np.pi)
    assert (dphi <= w.astype(np.float64) - 1e-4).all()          # inside, with the 2e-4 margin to spare
    assert (w < 3.2).mean() > 0.8
    # all (row, connected module with MDs) pairs: a good part is dropped by the pointing cone alone
    off, cols = map_full
    has = np.bincount(mod, minlength=nm) > 0
    rows, mods = [], []
    for r in range(0, len(mod), 7):
        Bs = cols[off[mod[r]]:off[mod[r] + 1]]
        Bs = Bs[has[Bs]]
        rows.append(np.full(len(Bs), r)); mods.append(Bs)
    rows, mods = np.concatenate(rows), np.concatenate(mods).astype(np.int64)
    live, w = B.lst_host_ls_window(np.stack([rt[rows], z[rows]], 1), cat[rows], box[mods], geom_full.category[mods])
    assert 0.3 < live.mean() < 0.95
