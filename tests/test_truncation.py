"""Occupancy-truncated memory mode: "a bucket keeps the K first objects
of its canonical order".  CPU part: the oracle's truncation mode pinned against an independent numpy
restatement of the rule at the MD level and against properties at every level.  GPU part (-m gpu):
the CUDA path with lst_config.trunc_cap against the oracle in the same mode, every level."""
import numpy as np
import pytest

import lstgen
from oracle import lst_oracle as O

CAPS = np.zeros((6, 16), np.uint32)
CAPS[O.MD, :] = 5
CAPS[O.LS, :] = 12
CAPS[O.T3, :] = 10
CAPS[O.T5, :] = 6
CAPS[O.PT3, 0] = 3
CAPS[O.PT5, 0] = 2


def _run(geom, mp, ev, caps, order=True, upto=O.TC):
    o = O.Oracle(geom, mp[0], mp[1])
    if order:
        o.set_truncation(geom.phic, caps)
    o.load(ev)
    o.run(upto=upto, pixel_indexed=True)
    return o


def _keys(o, lvl):
    d = o.get(lvl)
    h = d["hits"].astype(np.int64)
    if lvl in (O.PT3, O.PT5):
        h = np.concatenate([d["parents"][:, :1].astype(np.int64), h], 1)
    return [tuple(r) for r in h.tolist()]


def test_azimuth_order_alone_changes_no_set(geom_barrel, map_barrel):
    ev = lstgen.make_event(geom_barrel, "cfg2s")
    a, b = _run(geom_barrel, map_barrel, ev, None, order=False), _run(geom_barrel, map_barrel, ev, None, order=True)
    for lvl in (O.MD, O.LS, O.T3, O.T5, O.PT3, O.PT5, O.TC):
        assert a.count(lvl) == b.count(lvl) > 0
        if lvl != O.TC:
            assert set(_keys(a, lvl)) == set(_keys(b, lvl))
    # ... and the MDs of a module now ascend in the azimuth of their lower hit relative to the module centre
    md = b.get(O.MD)
    mod = md["parents"][:, 0].astype(np.int64)
    lo = md["hits"][:, 0].astype(np.int64)
    rel = np.arctan2(ev.y[lo].astype(np.float64), ev.x[lo].astype(np.float64)) - np.asarray(geom_barrel.phic, np.float64)[mod]
    rel = np.remainder(rel + np.pi, 2 * np.pi) - np.pi
    assert np.all(np.diff(mod) >= 0) and np.all(np.diff(rel)[np.diff(mod) == 0] >= 0)


def test_md_cap_is_the_first_k_of_a_numpy_restatement(geom_barrel, map_barrel):
    """MD level, typed independently: group the EXACT mini-doublets by module, order them by (azimuth
    of the lower hit relative to the module centre, its index, the same of the upper hit), keep K."""
    ev = lstgen.make_event(geom_barrel, "cfg2")
    caps = np.zeros((6, 16), np.uint32)
    caps[O.MD, :] = 2
    exact = _run(geom_barrel, map_barrel, ev, None, order=False, upto=O.MD).get(O.MD)
    got = set(_keys(_run(geom_barrel, map_barrel, ev, caps, upto=O.MD), O.MD))
    phic = np.asarray(geom_barrel.phic, np.float64)
    x, y = ev.x.astype(np.float64), ev.y.astype(np.float64)
    want, over = set(), 0
    mod = exact["parents"][:, 0].astype(np.int64)
    for m in np.unique(mod):
        rows = exact["hits"][mod == m].astype(np.int64)
        rel = lambda h: np.remainder(np.arctan2(y[h], x[h]) - phic[m] + np.pi, 2 * np.pi) - np.pi
        order = sorted(range(len(rows)), key=lambda k: (rel(rows[k, 0]), rows[k, 0], rel(rows[k, 1]), rows[k, 1]))
        over += len(rows) > 2
        want |= {tuple(rows[k].tolist()) for k in order[:2]}
    assert over > 20, "the cap must bite for the pin to mean something"
    assert got == want


def test_caps_at_every_level_keep_the_first_k_of_a_numpy_restatement(geom_barrel, map_barrel):
    """WHICH objects a full bucket keeps, at every level, typed independently of the oracle's truncation code
    and cascaded from the EXACT collections (acceptance depends only on the object's own constituents, so the
    truncated level = the exact level restricted to kept constituents, then cut per bucket):
      MD   order inside a module: (azimuth of the lower hit relative to the module centre, its index, the same of
           the upper hit); global MD order = (module, that)
      LS   candidates row-major over (inner MD, outer MD) in MD order; bucket = module of the inner MD
      T3   row-major over (first LS, second LS) in LS order; T5 likewise over T3s; bucket = module of the first MD
      pT3 / pT5: per pixel seed, the T3 / T5 in their own order."""
    ev = lstgen.make_event(geom_barrel, "cfg2s")
    exact, tr = _run(geom_barrel, map_barrel, ev, None, order=False), _run(geom_barrel, map_barrel, ev, CAPS)
    lay = np.asarray(geom_barrel.logical_layer, np.int64)
    phic = np.asarray(geom_barrel.phic, np.float64)
    x, y, det = ev.x.astype(np.float64), ev.y.astype(np.float64), ev.det.astype(np.int64)
    rel = lambda h: float(np.remainder(np.arctan2(y[h], x[h]) - phic[det[h] >> 1] + np.pi, 2 * np.pi) - np.pi)

    def first_k(cands, key, bucket, cap):
        """cands: tuples; keep per bucket the cap(bucket) first in key order -> (kept set, rank of every kept one)"""
        kept, n_in = [], {}
        for t in sorted(cands, key=key):
            b = bucket(t)
            if n_in.get(b, 0) < cap(b):
                n_in[b] = n_in.get(b, 0) + 1
                kept.append(t)
        return {t: r for r, t in enumerate(kept)}          # ranks follow the key order: usable as the next level's order

    hits = lambda lvl: [tuple(r) for r in exact.get(lvl)["hits"].astype(np.int64).tolist()]
    mod_of = lambda t: int(det[t[0]] >> 1)
    cap_mod = lambda lvl: (lambda m: int(CAPS[lvl, lay[m]]))
    md = first_k(hits(O.MD), lambda t: (mod_of(t), rel(t[0]), t[0], rel(t[1]), t[1]), mod_of, cap_mod(O.MD))
    ls = first_k([t for t in hits(O.LS) if t[0:2] in md and t[2:4] in md], lambda t: (md[t[0:2]], md[t[2:4]]), mod_of, cap_mod(O.LS))
    t3 = first_k([t for t in hits(O.T3) if t[0:4] in ls and t[2:6] in ls], lambda t: (ls[t[0:4]], ls[t[2:6]]), mod_of, cap_mod(O.T3))
    t5 = first_k([t for t in hits(O.T5) if t[0:6] in t3 and t[4:10] in t3], lambda t: (t3[t[0:6]], t3[t[4:10]]), mod_of, cap_mod(O.T5))
    want = {O.MD: set(md), O.LS: set(ls), O.T3: set(t3), O.T5: set(t5)}
    for lvl, below, cap in ((O.PT3, t3, int(CAPS[O.PT3, 0])), (O.PT5, t5, int(CAPS[O.PT5, 0]))):
        d = exact.get(lvl)
        cands = [(int(p), *h) for p, h in zip(d["parents"][:, 0].tolist(), d["hits"].astype(np.int64).tolist()) if tuple(h) in below]
        want[lvl] = set(first_k(cands, lambda t: (t[0], below[t[1:]]), lambda t: t[0], lambda b: cap))
    for lvl in (O.MD, O.LS, O.T3, O.T5, O.PT3, O.PT5):
        got = set(_keys(tr, lvl))
        assert len(want[lvl]) < exact.count(lvl), "level %s: the cap must bite" % O.LEVEL_NAMES[lvl]
        assert got == want[lvl], "level %s: %d kept objects differ from the restatement" % (O.LEVEL_NAMES[lvl], len(got ^ want[lvl]))


def test_caps_at_every_level_properties(geom_barrel, map_barrel):
    ev = lstgen.make_event(geom_barrel, "cfg2s")
    exact, tr = _run(geom_barrel, map_barrel, ev, None, order=False), _run(geom_barrel, map_barrel, ev, CAPS)
    lay = np.asarray(geom_barrel.logical_layer, np.int64)
    first_mod = None
    for lvl in (O.MD, O.LS, O.T3, O.T5, O.PT3, O.PT5):
        ke, kt = set(_keys(exact, lvl)), _keys(tr, lvl)
        assert set(kt) <= ke and len(set(kt)) == len(kt), "a truncated level is a subset of the exact one"
        assert 0 < len(kt) < len(ke), "level %s: the caps must bite" % O.LEVEL_NAMES[lvl]
        d = tr.get(lvl)
        if lvl in (O.PT3, O.PT5):
            _, cnt = np.unique(d["parents"][:, 0], return_counts=True)
            assert cnt.max() <= CAPS[lvl, 0]
        else:
            # bucket = module of the first MD = module of the first hit
            m = ev.det[d["hits"][:, 0].astype(np.int64)].astype(np.int64) >> 1
            u, cnt = np.unique(m, return_counts=True)
            assert np.all(cnt <= CAPS[lvl, lay[u]])
            assert np.all(np.diff(m) >= 0), "objects stay grouped by the module of their first MD"
    assert tr.count(O.TC) > 0


@pytest.mark.gpu
@pytest.mark.parametrize("cfg_name", ["cfg2s", "cfg4", "cfg4h"])
def test_gpu_truncated_mode_matches_oracle_truncated_mode(geom_barrel, map_barrel, geom_full, map_full, cfg_name):
    """The CUDA path with lst_config.trunc_cap against the oracle in the same mode: identical object
    sets at every level (the objects a full bucket keeps are decided by the canonical order, i.e. by the
    fp32 azimuth keys of the hits on the GPU and fp64 ones in the oracle: a pair of hits of one sensor
    closer than ~1e-6 rad in azimuth could flip; none does on these seeded events), TC included."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2209_13711_b200 import binding as B
    geom, mp = (geom_barrel, map_barrel) if cfg_name == "cfg2s" else (geom_full, map_full)
    caps = CAPS.copy()
    if cfg_name == "cfg4":
        caps[O.MD, :], caps[O.LS, :], caps[O.T3, :], caps[O.T5, :] = 8, 30, 24, 8
        caps[O.PT3, 0], caps[O.PT5, 0] = 6, 3
    ev = lstgen.make_event(geom, cfg_name, seed=1000 if cfg_name == "cfg4h" else None)
    if cfg_name == "cfg4h":
        # the bench size (event 0 of the bench batch) with caps chosen the way the bench chooses them: a quantile
        # of the per-module / per-seed occupancy measured in exact mode (0.99, so that every level bites on ONE event)
        from paper_2209_13711_b200 import occupancy
        ex = B.LST(geom, mp[0], mp[1], n_slots=1, max_hits=ev.n_hits, max_seeds=max(ev.n_seeds, 1))
        caps = occupancy.caps_from_sample(geom, [ev], occupancy.run_sample(ex, [ev]), 0.99)
        ex.close()
    o = _run(geom, mp, ev, caps)
    cfg = B.lst_default_config()
    for l in range(6):
        for k in range(16):
            cfg.trunc_cap[l][k] = int(caps[l, k])
    lst = B.LST(geom, mp[0], mp[1], cfg=cfg, n_slots=1, max_hits=ev.n_hits, max_seeds=max(ev.n_seeds, 1))
    lst.lst_load_event(0, ev.x, ev.y, ev.z, ev.det, (ev.seed_pt, ev.seed_eta, ev.seed_phi, ev.seed_z0, ev.seed_q, ev.seed_hit_ids))
    lst.lst_run(0)
    cnt, _ = lst.lst_get_counts(0)
    exact = _run(geom, mp, ev, None, order=False)
    for lvl in (O.MD, O.LS, O.T3, O.T5, O.PT3, O.PT5):
        got = lst.lst_get_objects(0, lvl)
        h = got["hits"].astype(np.int64)
        if lvl in (O.PT3, O.PT5):
            h = np.concatenate([got["parents"][:, :1].astype(np.int64), h], 1)
        kg = set(map(tuple, h.tolist()))
        assert kg == set(_keys(o, lvl)), "level %s differs from the oracle's truncated mode" % O.LEVEL_NAMES[lvl]
        assert 0 < len(kg) < exact.count(lvl), "level %s: the caps must bite" % O.LEVEL_NAMES[lvl]
    assert cnt[O.TC] == o.count(O.TC) > 0
    # keep flags object by object, the TC list entry by entry and its floats (the comparison of the exact mode)
    import test_gpu_parity as G
    assert G.compare_cleaning(o, lst, ev) == o.count(O.TC)
    lst.close()


@pytest.mark.gpu
def test_gpu_calibration_separates_resizing_from_truncation_and_a_busier_event_is_refused_loudly(geom_full, map_full):
    """occupancy.calibrate on a small sample: the report holds the exact mode at the default factors, the exact
    mode with sample-sized factors (the control) and the truncated mode with sample-sized factors, and quotes
    control / truncated as the truncation gain.  Then an event four times busier than anything in the sample
    runs with the calibrated capacities: the truncated mode caps a BUCKET, the capacities stay global, so the
    event must be refused with LST_ENOMEM naming the stage (include/lst.h) - never a silently smaller result -
    and the slot must serve the next event normally."""
    import torch
    if not torch.cuda.is_available():
        pytest.skip("no CUDA device")
    from paper_2209_13711_b200 import binding as B
    from paper_2209_13711_b200 import occupancy
    calib = [lstgen.make_event(geom_full, "cfg4", seed=7000 + k, n_particles=1500) for k in range(3)]
    cfg_t, rep = occupancy.calibrate(geom_full, map_full[0], map_full[1], calib, quantile=0.99)
    ws_d, ws_s, ws_t = (rep[k] for k in ("workspace_bytes_exact_defaults", "workspace_bytes_exact_sample_sized",
                                         "workspace_bytes_truncated"))
    assert ws_t <= ws_s < ws_d
    assert rep["footprint_ratio"] == round(ws_s / ws_t, 3) and rep["footprint_ratio_vs_defaults"] == round(ws_d / ws_t, 2)
    kept = rep["objects_kept_fraction"]
    assert all(0.0 < kept[n] <= 1.0 for n in ("md", "ls", "t3", "t5", "tc")) and kept["ls"] < 1.0

    busy = lstgen.make_event(geom_full, "cfg4", seed=7100)                  # 6 000 particles
    mh_cal = max(e.n_hits for e in calib)
    assert busy.n_hits > 3 * mh_cal
    scale = mh_cal / busy.n_hits           # same capacities as calibrated, in a context that can load the busy event
    for name in ("cap_md_per_hit", "cap_ls_per_hit", "cap_t3_per_hit", "cap_t5_per_hit", "cap_mdcand_per_hit",
                 "cap_lscand_per_hit", "cap_t3cand_per_hit", "cap_t5cand_per_hit"):
        setattr(cfg_t, name, getattr(cfg_t, name) * scale)
    seeds = lambda e: (e.seed_pt, e.seed_eta, e.seed_phi, e.seed_z0, e.seed_q, e.seed_hit_ids)
    ms = max(busy.n_seeds, max(e.n_seeds for e in calib))
    lst = B.LST(geom_full, map_full[0], map_full[1], cfg=cfg_t, n_slots=1, max_hits=busy.n_hits, max_seeds=ms)
    lst.lst_load_event(0, calib[0].x, calib[0].y, calib[0].z, calib[0].det, seeds(calib[0]))
    lst.lst_run(0)
    want, _ = lst.lst_get_counts(0)
    assert want[O.TC] > 0
    lst.lst_load_event(0, busy.x, busy.y, busy.z, busy.det, seeds(busy))
    lst.lst_run(0)
    with pytest.raises(B.LstError) as e:
        lst.lst_get_counts(0)
    assert e.value.status == B.LST_ENOMEM and "capacity exceeded" in str(e.value)
    lst.lst_load_event(0, calib[0].x, calib[0].y, calib[0].z, calib[0].det, seeds(calib[0]))
    lst.lst_run(0)
    again, _ = lst.lst_get_counts(0)
    assert np.array_equal(again, want), "the slot recovers after a refused event"
    lst.close()
