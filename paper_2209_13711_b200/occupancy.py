"""Occupancy-truncated memory mode: calibration helper.

The paper fixes its array sizes by truncating object occupancies at the 99.9 % / 99.99 % quantile
measured on a sample.  Here: run a sample of events in exact mode through the C-ABI, take per level
and logical layer the quantile of the per-module occupancy (per seed for pT3 / pT5) as
`lst_config.trunc_cap`, run the sample again with the caps and size the capacity factors
(`lst_config.cap_*`) from the truncated occupancies.  Marshalling and numpy bookkeeping only: every
event goes through lst_load_event / lst_run / lst_get_objects.
"""
from __future__ import annotations

import math

import numpy as np

from . import binding as B

LEVELS = (B.LST_MD, B.LST_LS, B.LST_T3, B.LST_T5, B.LST_PT3, B.LST_PT5)
HEADROOM = 1.3          # object capacities: largest occupancy of the sample x this
CAND_HEADROOM = 1.6     # work-item capacities (the items of a module waste up to half of their 1024 candidates)
LIST_HEADROOM = 2.0     # candidate lists: largest number of pre-filter survivors of the sample x this.  The survivors
                        # of the pixel stages fluctuate far more from event to event than the object counts do (an
                        # unseen event of the same workload reached 1.4 x the maximum of a 16-event sample)


def _seeds(ev):
    return (ev.seed_pt, ev.seed_eta, ev.seed_phi, ev.seed_z0, ev.seed_q, ev.seed_hit_ids) if ev.n_seeds else None


def run_sample(lst, events):
    """-> per event (counts [7], cand [18], {level: bucket id of every object})."""
    out = []
    for ev in events:
        lst.lst_load_event(0, ev.x, ev.y, ev.z, ev.det, _seeds(ev))
        lst.lst_run(0)
        cnt, cand = lst.lst_get_counts(0)
        buckets = {}
        for lvl in LEVELS:
            o = lst.lst_get_objects(0, lvl)
            if lvl in (B.LST_PT3, B.LST_PT5):
                buckets[lvl] = o["parents"][:, 0].astype(np.int64)            # the pixel seed
            else:                                                              # module of the first MD = of the first hit
                buckets[lvl] = np.asarray(ev.det, np.int64)[o["hits"][:, 0].astype(np.int64)] >> 1
        out.append((cnt.copy(), cand.copy(), buckets))
    return out


def caps_from_sample(geom, events, sample, quantile):
    """trunc_cap [6, 16]: per level and logical layer the `quantile` of the occupancy of a module of
    that layer (all modules of the layer x all events, empty ones included); per seed for pT3 / pT5."""
    lay = np.asarray(geom.logical_layer, np.int64)
    caps = np.zeros((6, 16), np.uint32)
    for lvl in LEVELS:
        if lvl in (B.LST_PT3, B.LST_PT5):
            occ = np.concatenate([np.bincount(s[2][lvl], minlength=ev.n_seeds) for ev, s in zip(events, sample)])
            caps[lvl, 0] = max(1, int(math.ceil(np.quantile(occ, quantile)))) if occ.size else 1
        else:
            per_mod = np.stack([np.bincount(s[2][lvl], minlength=geom.n_modules) for s in sample])   # [events, modules]
            for L in np.unique(lay):
                occ = per_mod[:, lay == L].ravel()
                if occ.max(initial=0) > 0:
                    caps[lvl, L] = max(1, int(math.ceil(np.quantile(occ, quantile))))
    return caps


def config_with_caps(caps, base=None):
    cfg = base if base is not None else B.lst_default_config()
    for l in range(6):
        for k in range(16):
            cfg.trunc_cap[l][k] = int(caps[l, k])
    return cfg


def size_factors(cfg, sample, max_hits, max_seeds):
    """Capacity factors from the largest occupancies of the (truncated) sample, times HEADROOM."""
    cnt = np.stack([s[0] for s in sample]).astype(np.float64).max(0)
    cand = np.stack([s[1] for s in sample]).astype(np.float64).max(0)
    # an object capacity also sizes the stage's candidate list (2 x capacity + 4096 entries), which holds the
    # pre-filter survivors of the UNtruncated enumeration: cand[6 + stage], stages MD, LS, T3, T5, pT5, pT3
    surv = {B.LST_MD: cand[6], B.LST_LS: cand[7], B.LST_T3: cand[8], B.LST_T5: cand[9], B.LST_PT5: cand[10], B.LST_PT3: cand[11]}
    f = lambda lvl, n: float(max(HEADROOM * cnt[lvl], 0.5 * LIST_HEADROOM * surv[lvl]) / max(n, 1))
    cfg.cap_md_per_hit, cfg.cap_ls_per_hit = f(B.LST_MD, max_hits), f(B.LST_LS, max_hits)
    cfg.cap_t3_per_hit, cfg.cap_t5_per_hit = f(B.LST_T3, max_hits), f(B.LST_T5, max_hits)
    cfg.cap_pt3_per_seed, cfg.cap_pt5_per_seed = f(B.LST_PT3, max_seeds), f(B.LST_PT5, max_seeds)
    fc = lambda v: float(CAND_HEADROOM * v / max(max_hits, 1))
    cfg.cap_mdcand_per_hit, cfg.cap_lscand_per_hit = fc(cand[0]), fc(cand[1])
    cfg.cap_t3cand_per_hit, cfg.cap_t5cand_per_hit = fc(cand[2]), fc(cand[3])
    return cfg


def calibrate(geom, map_offsets, map_cols, events, quantile=0.999, device="cuda:0"):
    """-> (cfg for the truncated mode, report dict).  `events`: the calibration sample (keep it disjoint from
    the events that are later timed or served: the capacities are fitted to this sample with HEADROOM /
    CAND_HEADROOM, and an event that exceeds them is reported as LST_ENOMEM, see include/lst.h).

    The report separates the two effects that shrink a workspace: re-sizing the capacity factors from a
    sample (available to the exact mode as well) and the truncation itself.  It therefore holds THREE
    workspaces: exact mode at the default factors, exact mode with sample-sized factors (the control), and
    truncated mode with sample-sized factors.  `footprint_ratio` is control / truncated: the gain that is
    due to truncation alone; `footprint_ratio_vs_defaults` includes the re-sizing."""
    mh, ms = max(e.n_hits for e in events), max(max(e.n_seeds for e in events), 1)
    mk = lambda cfg: B.LST(geom, map_offsets, map_cols, cfg=cfg, n_slots=1, max_hits=mh, max_seeds=ms, device=device)
    same = lambda a, b: all(np.array_equal(x[0], y[0]) for x, y in zip(a, b))
    exact = mk(None)
    ws_exact = exact.workspace_bytes
    s_exact = run_sample(exact, events)
    exact.close()
    # control: the exact mode with capacities sized from the same sample, same headroom
    sized = mk(size_factors(B.lst_default_config(), s_exact, mh, ms))
    ws_exact_sized = sized.workspace_bytes
    assert same(s_exact, run_sample(sized, events))      # (an overflow would raise LST_ENOMEM)
    sized.close()
    caps = caps_from_sample(geom, events, s_exact, quantile)
    # pass 1: the caps with the default capacities -> truncated occupancies; pass 2: capacities sized from them
    lst = mk(config_with_caps(caps))
    s_tr = run_sample(lst, events)
    lst.close()
    cfg = size_factors(config_with_caps(caps), s_tr, mh, ms)
    lst = mk(cfg)
    ws_tr = lst.workspace_bytes
    assert same(s_tr, run_sample(lst, events))           # must reproduce pass 1
    lst.close()
    tot_e = np.stack([s[0] for s in s_exact]).astype(np.float64).sum(0)
    tot_t = np.stack([s[0] for s in s_tr]).astype(np.float64).sum(0)
    names = ("md", "ls", "t3", "t5", "pt3", "pt5", "tc")
    report = {
        "quantile": quantile, "events": len(events),
        "workspace_bytes_exact_defaults": int(ws_exact), "workspace_bytes_exact_sample_sized": int(ws_exact_sized),
        "workspace_bytes_truncated": int(ws_tr),
        "footprint_ratio": round(ws_exact_sized / ws_tr, 3),
        "footprint_ratio_vs_defaults": round(ws_exact / ws_tr, 2),
        "footprint_note": "footprint_ratio = exact mode with sample-sized capacities / truncated mode with sample-sized "
                          "capacities (truncation alone); _vs_defaults also counts the re-sizing of the default factors",
        "objects_kept_fraction": {n: round(float(tot_t[k] / max(tot_e[k], 1.0)), 5) for k, n in enumerate(names)},
        "caps_per_layer": {names[l]: [int(v) for v in caps[l]] for l in range(4)},
        "caps_per_seed": {"pt3": int(caps[B.LST_PT3, 0]), "pt5": int(caps[B.LST_PT5, 0])},
    }
    return cfg, report
