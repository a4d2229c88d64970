"""Physics-sanity harness on SYNTHETIC truth.

The paper's efficiency / fake-rate / duplicate-rate figures (Figs. 12-16) are
measured on CMS simulation, which is not available here; this module computes the same three
quantities for the track candidates of the synthetic events, whose truth (particle of every hit and
of every pixel seed) comes from lstgen.  Definitions (restated):
  * a track candidate is MATCHED to a particle if at least `min_frac` (75 %) of its hits - outer-
    tracker hits and the four pixel hits of its seed - come from that particle; otherwise it is FAKE;
  * efficiency = fraction of the denominator particles matched by at least one track candidate,
    denominator = prompt or displaced particles with pT > 0.8 GeV inside the acceptance that left
    hits in both sensors of at least `min_modules` modules (reconstructable);
  * fake rate = fraction of track candidates that are fake;
  * duplicate rate = fraction of matched track candidates whose particle is also matched by
    another, earlier candidate of the list.
Inputs are the arrays lst_get_objects(LST_TC) returns (or the oracle's TC list in the same layout);
nothing here runs on the hot path.
"""
from __future__ import annotations

import numpy as np

PAD = 0xFFFFFFFF
TC_T5, TC_PT3, TC_PT5, TC_PLS = 3, 4, 5, 6


def match_track_candidates(ev, tc_hits, tc_type, min_frac=0.75):
    """tc_hits [n, 14] u32: ten outer-tracker hit indices (padded with 0xFFFFFFFF) + the four pixel-hit
    ids of the seed (padded for a T5); tc_type [n].  -> (pid [n] i64, -1 = fake; n_hits [n])."""
    tc_hits = np.asarray(tc_hits, dtype=np.int64).reshape(-1, 14)
    n = tc_hits.shape[0]
    seed_of = {tuple(r): k for k, r in enumerate(np.asarray(ev.seed_hit_ids, np.int64).tolist())}
    hit_pid = np.asarray(ev.pid, np.int64)
    out = np.full(n, -1, np.int64)
    nh = np.zeros(n, np.int64)
    for i in range(n):
        ot = tc_hits[i, :10]
        pids = hit_pid[ot[ot != PAD]].tolist()
        pix = tuple(tc_hits[i, 10:].tolist())
        if pix[0] != PAD:
            sp = int(ev.seed_pid[seed_of[pix]])
            pids += [sp] * 4
        nh[i] = len(pids)
        if not pids:
            continue
        vals, cnt = np.unique(np.asarray(pids), return_counts=True)
        k = int(np.argmax(cnt))
        if vals[k] >= 0 and cnt[k] >= min_frac * len(pids):
            out[i] = vals[k]
    return out, nh


def reconstructable(ev, min_modules=5, pt_min=0.8, eta_max=2.4):
    """Boolean mask over the particles: pT, acceptance, and both sensors hit in >= min_modules modules."""
    P = ev.particles
    npart = len(P["pt"])
    det, pid = np.asarray(ev.det, np.int64), np.asarray(ev.pid, np.int64)
    ok = pid >= 0
    key = pid[ok] * (1 << 32) + (det[ok] >> 1)
    lo = np.unique(key[(det[ok] & 1) == 0])
    up = np.unique(key[(det[ok] & 1) == 1])
    both = np.intersect1d(lo, up)
    nmod = np.bincount((both >> 32).astype(np.int64), minlength=npart)
    return (P["pt"] > pt_min) & (np.abs(P["eta"]) < eta_max) & (nmod >= min_modules)


def rates(ev, tc_hits, tc_type, tc_pt=None, tc_eta=None, min_frac=0.75, min_modules=5,
          pt_edges=(0.8, 1.0, 1.5, 2.0, 3.0, 5.0, 10.0, 1e9), eta_edges=(0.0, 0.4, 0.8, 1.2, 1.6, 2.0, 2.4),
          rv_edges=(0.0, 0.1, 1.0, 2.5, 5.0, 10.0)):
    """Efficiency, fake rate and duplicate rate of one event's track candidates (see module docstring).
    Returns a dict of overall numbers and of (numerator, denominator) arrays per bin, so that several
    events can be added before dividing."""
    P = ev.particles
    pid, _ = match_track_candidates(ev, tc_hits, tc_type, min_frac)
    den = reconstructable(ev, min_modules)
    found = np.zeros(len(P["pt"]), bool)
    found[pid[pid >= 0]] = True
    rv = np.hypot(P["vx"], P["vy"])

    def binned(x, edges, sel_num, sel_den):
        num, d = np.histogram(x[sel_num], bins=edges)[0], np.histogram(x[sel_den], bins=edges)[0]
        return num.astype(np.int64), d.astype(np.int64)

    prompt = ~np.asarray(P["sec"], bool)
    out = {
        "n_tc": int(len(pid)), "n_fake": int((pid < 0).sum()),
        "n_den": int(den.sum()), "n_found": int((den & found).sum()),
        "n_den_prompt": int((den & prompt).sum()), "n_found_prompt": int((den & prompt & found).sum()),
        "eff_vs_pt": binned(P["pt"], pt_edges, den & found, den),
        "eff_vs_abs_eta": binned(np.abs(P["eta"]), eta_edges, den & found, den),
        "eff_vs_rv": binned(rv, rv_edges, den & found, den),
    }
    matched = pid >= 0
    first = np.zeros(len(pid), bool)
    _, idx = np.unique(pid[matched], return_index=True)
    first[np.nonzero(matched)[0][idx]] = True
    out["n_matched"] = int(matched.sum())
    out["n_duplicate"] = int((matched & ~first).sum())
    if tc_pt is not None:
        tc_pt, tc_eta = np.asarray(tc_pt, np.float64), np.abs(np.asarray(tc_eta, np.float64))
        out["fake_vs_pt"] = binned(tc_pt, pt_edges, pid < 0, np.ones(len(pid), bool))
        out["fake_vs_abs_eta"] = binned(tc_eta, eta_edges, pid < 0, np.ones(len(pid), bool))
        out["dup_vs_pt"] = binned(tc_pt, pt_edges, matched & ~first, matched)
    return out


def add(a, b):
    """Sum of two rates() results (counts and (num, den) pairs)."""
    if a is None:
        return b
    out = {}
    for k, v in a.items():
        out[k] = (v[0] + b[k][0], v[1] + b[k][1]) if isinstance(v, tuple) else v + b[k]
    return out


def summary(r):
    """Overall rates of an accumulated rates() result, JSON-friendly."""
    frac = lambda n, d: round(float(n) / d, 5) if d else None
    s = {"track_candidates": r["n_tc"], "efficiency": frac(r["n_found"], r["n_den"]),
         "efficiency_prompt": frac(r["n_found_prompt"], r["n_den_prompt"]), "fake_rate": frac(r["n_fake"], r["n_tc"]),
         "duplicate_rate": frac(r["n_duplicate"], r["n_matched"]), "denominator_particles": r["n_den"]}
    for k in ("eff_vs_pt", "eff_vs_abs_eta", "eff_vs_rv", "fake_vs_pt", "fake_vs_abs_eta", "dup_vs_pt"):
        if k in r:
            s[k] = [frac(n, d) for n, d in zip(r[k][0].tolist(), r[k][1].tolist())]
    return s
