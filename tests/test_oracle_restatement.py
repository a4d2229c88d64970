"""The oracle's selection functions against a third transcription of SURVEY.md 8(c) (plain numpy,
tests/survey_restatement.py, typed from the survey's formulas, not from either C file): on ~1e4
candidates per level sampled from a smeared full-detector event, every cut VARIABLE and every
THRESHOLD the oracle evaluates (its trace, oracle.cuts) equals the restatement's, the decisions
are equal, and so are the stored / derived quantities.  A sign flip, a swapped sigma index, a
dropped tolerance term or a transposed operand made in the oracle but not in the survey's formula
fails here; the one-hot tolerance pins of test_oracle_pins2.py cover the survey-vs-intent side.
"""
import numpy as np
import pytest

import lstgen
from oracle import lst_oracle as O

import survey_restatement as S

G = S.Cfg()
RTOL = 1e-9
N_SAMPLE = 10000


def _close(a, b, what):
    a, b = np.asarray(a, float), np.asarray(b, float)
    bad = ~(np.abs(a - b) <= RTOL * np.maximum(np.abs(a), np.abs(b)) + 1e-13)
    assert not bad.any(), "%s: %d of %d differ, first %r vs %r" % (what, bad.sum(), len(a), a[bad][:1], b[bad][:1])


@pytest.fixture(scope="module")
def event(geom_full, map_full):
    ev = lstgen.make_event(geom_full, "cfg4", n_particles=1500)
    o = O.Oracle(geom_full, map_full[0], map_full[1])
    o.load(ev)
    o.run(upto=O.PT5, pixel_indexed=True)
    xyz = np.stack([ev.x, ev.y, ev.z], 1).astype(np.float64)
    md = o.get(O.MD)
    mod = md["parents"][:, 0].astype(np.int64)
    return dict(ev=ev, o=o, xyz=xyz, md=md, mod=mod, cat=geom_full.category[mod].astype(np.int64),
                anchor=xyz[md["hits"][:, 0].astype(np.int64)])


def _sample(rng, n_total, must):
    """must (indices of accepted candidates) + random others, <= N_SAMPLE."""
    must = np.asarray(must, dtype=np.int64)
    if len(must) > N_SAMPLE // 2:
        must = rng.choice(must, N_SAMPLE // 2, replace=False)
    rest = rng.choice(n_total, min(n_total, N_SAMPLE - len(must)), replace=False)
    return np.unique(np.concatenate([must, rest]))


def test_md_cuts_equal_restatement(geom_full, event):
    ev, xyz = event["ev"], event["xyz"]
    det = ev.det.astype(np.int64)
    order = np.argsort(det, kind="stable")
    sdet = det[order]
    pairs = []
    for m in np.unique(sdet >> 1):
        lo = order[np.searchsorted(sdet, 2 * m):np.searchsorted(sdet, 2 * m + 1)]
        up = order[np.searchsorted(sdet, 2 * m + 1):np.searchsorted(sdet, 2 * m + 2)]
        if len(lo) and len(up):
            a, b = np.meshgrid(lo, up, indexing="ij")
            pairs.append(np.stack([a.ravel(), b.ravel()], 1))
    pairs = np.concatenate(pairs)
    acc = set(map(tuple, event["md"]["hits"].astype(np.int64).tolist()))
    must = [i for i, p in enumerate(map(tuple, pairs.tolist())) if p in acc]
    sel = _sample(np.random.default_rng(1), len(pairs), must)
    pairs = pairs[sel]
    L, U = xyz[pairs[:, 0]], xyz[pairs[:, 1]]
    cat = geom_full.category[det[pairs[:, 0]] >> 1].astype(np.int64)
    ok, cuts, out, ec = S.md(G, L, U, cat)
    n_ok = 0
    for i in range(len(pairs)):
        p, f, tr = O.cuts(O.MD, [L[i], U[i]], [cat[i]])
        assert p == bool(ok[i]), (i, tr)
        names = ["E1", "E2"] if ec[i] else ["B1sign", "B1", "B2"]
        assert len(tr) == len(names)
        for (kind, v, thr), nm in zip(tr, names):
            _close([v], [cuts[nm][0][i]], "MD %s v" % nm)
            if cuts[nm][1] is not None:
                assert kind == O.CUT_LE
                _close([thr], [cuts[nm][1][i]], "MD %s thr" % nm)
            else:
                assert kind == O.CUT_POS
        _close(f[:3], [out["dphi"][i], out["kappa"][i], out["sigk"][i]], "MD out")
        n_ok += p
    assert n_ok > 1000 and ec.sum() > 500 and (~ec).sum() > 500
    assert {tuple(x) for x, k in zip(pairs.tolist(), ok) if k} == {tuple(pairs[j]) for j in range(len(pairs)) if tuple(pairs[j]) in acc}


def _ls_candidates(event, map_full):
    off, cols = map_full
    mod = event["mod"]
    mstart = np.searchsorted(mod, np.arange(int(mod.max()) + 2))
    ii, oo = [], []
    for i in range(len(mod)):
        for B in cols[off[mod[i]]:off[mod[i] + 1]]:
            if B + 1 < len(mstart) and mstart[B + 1] > mstart[B]:
                ii.append(np.full(mstart[B + 1] - mstart[B], i)); oo.append(np.arange(mstart[B], mstart[B + 1]))
    return np.concatenate(ii), np.concatenate(oo)


def test_ls_cuts_equal_restatement(map_full, event):
    md, A_, cat = event["md"], event["anchor"], event["cat"]
    ii, oo = _ls_candidates(event, map_full)
    acc = set(map(tuple, event["o"].get(O.LS)["parents"].astype(np.int64).tolist()))
    must = [k for k, t in enumerate(zip(ii.tolist(), oo.tolist())) if t in acc]
    sel = _sample(np.random.default_rng(2), len(ii), must)
    ii, oo = ii[sel], oo[sel]
    ki, ski, ko, sko = md["f"][ii, 1], md["f"][ii, 2], md["f"][oo, 1], md["f"][oo, 2]
    ok, cuts, out, mz = S.ls(G, A_[ii], A_[oo], cat[ii], cat[oo], ki, ski, ko, sko)
    n_ok = 0
    for k in range(len(ii)):
        p, f, tr = O.cuts(O.LS, [A_[ii[k]], A_[oo[k]]], [cat[ii[k]], cat[oo[k]]], [ki[k], ski[k], ko[k], sko[k]])
        assert p == bool(ok[k]), (k, tr)
        names = ["L1", "dot", "den", "L2", "L3i", "L3o"] if mz[k] else ["L1", "dot", "L2", "L3i", "L3o"]
        assert len(tr) == len(names), tr
        for (kind, v, thr), nm in zip(tr, names):
            _close([v], [cuts[nm][0][k]], "LS %s v" % nm)
            if cuts[nm][1] is not None:
                _close([thr], [cuts[nm][1][k]], "LS %s thr" % nm)
        _close(f[:3], [out["dphi"][k], out["kappa"][k], out["sigk"][k]], "LS out")
        n_ok += p
    assert n_ok > 1000 and mz.sum() > 1000 and (~mz).sum() > 1000
    assert (ok & mz).sum() > 200 and (ok & ~mz).sum() > 200
    assert {(a, b) for a, b, k in zip(ii.tolist(), oo.tolist(), ok) if k} == acc & set(zip(ii.tolist(), oo.tolist()))


def _join(first_of, last_of, n_md):
    """Candidate pairs (a, b) with first_of[b] == last_of[a]; objects grouped by first_of ascending."""
    start = np.searchsorted(first_of, np.arange(n_md + 1))
    aa, bb = [], []
    for a in range(len(last_of)):
        s, e = start[last_of[a]], start[last_of[a] + 1]
        if e > s:
            aa.append(np.full(e - s, a)); bb.append(np.arange(s, e))
    return np.concatenate(aa), np.concatenate(bb)


def test_t3_t5_cuts_equal_restatement(event):
    o, A_, cat = event["o"], event["anchor"], event["cat"]
    n_md = len(cat)
    lp = o.get(O.LS)["parents"].astype(np.int64)
    t3, t5 = o.get(O.T3), o.get(O.T5)
    aa, bb = _join(lp[:, 0], lp[:, 1], n_md)
    acc = set(map(tuple, t3["parents"].astype(np.int64).tolist()))
    must = [k for k, t in enumerate(zip(aa.tolist(), bb.tolist())) if t in acc]
    sel = _sample(np.random.default_rng(3), len(aa), must)
    aa, bb = aa[sel], bb[sel]
    m = np.stack([lp[aa, 0], lp[aa, 1], lp[bb, 1]], 1)
    ok, cuts, out = S.t3(G, A_[m[:, 0]], A_[m[:, 1]], A_[m[:, 2]], cat[m[:, 0]], cat[m[:, 1]], cat[m[:, 2]])
    for k in range(len(m)):
        p, f, tr = O.cuts(O.T3, A_[m[k]], cat[m[k]])
        assert p == bool(ok[k]), (k, tr)
        assert len(tr) == 3
        for (kind, v, thr), nm in zip(tr, ("T3-1", "T3-2", "T3-3")):
            _close([v], [cuts[nm][0][k]], "T3 %s v" % nm)
            _close([thr], [cuts[nm][1][k]], "T3 %s thr" % nm)
        _close(f[:3], [out["beta"][k], out["kappa3"][k], out["sigk3"][k]], "T3 out")
    assert ok.sum() > 500 and (~ok).sum() > 200
    modes = (cat[m] >= 2).any(1)
    assert modes.sum() > 300 and (~modes).sum() > 300
    # ---- T5
    tp = t3["parents"].astype(np.int64)
    tm = np.stack([lp[tp[:, 0], 0], lp[tp[:, 0], 1], lp[tp[:, 1], 1]], 1)
    aa, bb = _join(tm[:, 0], tm[:, 2], n_md)
    acc = set(map(tuple, t5["parents"].astype(np.int64).tolist()))
    must = [k for k, t in enumerate(zip(aa.tolist(), bb.tolist())) if t in acc]
    sel = _sample(np.random.default_rng(4), len(aa), must)
    aa, bb = aa[sel], bb[sel]
    m5 = np.concatenate([tm[aa], tm[bb][:, 1:]], 1)
    aux = np.stack([t3["f"][aa, 1], t3["f"][aa, 2], t3["f"][bb, 1], t3["f"][bb, 2]], 1)
    ok, cuts, out = S.t5(G, A_[m5], cat[m5], *aux.T)
    names = ["T5-1", "mid T3-1", "mid T3-2", "mid T3-3", None, "T5-3", None]
    for k in range(len(m5)):
        p, f, tr = O.cuts(O.T5, A_[m5[k]], cat[m5[k]], aux[k])
        assert p == bool(ok[k]), (k, tr)
        assert len(tr) == len(names)
        for (kind, v, thr), nm in zip(tr, names):
            if nm is None:
                assert kind == O.CUT_POS
                continue
            _close([v], [cuts[nm][0][k]], "T5 %s v" % nm)
            _close([thr], [cuts[nm][1][k]], "T5 %s thr" % nm)
        if p:
            _close(f[:5], [out["R"][k], out["chi2"][k], out["pt"][k], out["eta"][k], out["phi"][k]], "T5 out")
    assert ok.sum() > 100 and (~ok).sum() > 100


@pytest.mark.parametrize("five", [False, True])
def test_pixel_cuts_equal_restatement(geom_full, event, five):
    o, ev, A_, cat, mod = event["o"], event["ev"], event["anchor"], event["cat"], event["mod"]
    lp = o.get(O.LS)["parents"].astype(np.int64)
    tp = o.get(O.T3)["parents"].astype(np.int64)
    tm = np.stack([lp[tp[:, 0], 0], lp[tp[:, 0], 1], lp[tp[:, 1], 1]], 1)
    if five:
        fp = o.get(O.T5)["parents"].astype(np.int64)
        om = np.concatenate([tm[fp[:, 0]], tm[fp[:, 1]][:, 1:]], 1)
        acc = o.get(O.PT5)["parents"].astype(np.int64)
    else:
        om = tm
        acc = o.get(O.PT3)["parents"].astype(np.int64)
    rng = np.random.default_rng(5)
    # accepted pairs, the same seeds against random objects, and random pairs
    k = min(len(acc), N_SAMPLE // 3)
    a = acc[rng.choice(len(acc), k, replace=False)]
    b = np.stack([a[:, 0], rng.integers(0, len(om), k)], 1)
    c = np.stack([rng.integers(0, ev.n_seeds, k), rng.integers(0, len(om), k)], 1)
    # hard negatives: an accepted seed against other objects starting at the same MD
    first = {}
    for j, f0 in enumerate(om[:, 0].tolist()):
        first.setdefault(f0, []).append(j)
    d = np.array([(p, j) for p, ob in a[:k // 2].tolist() for j in first[om[ob, 0]][:3]], dtype=np.int64)
    pairs = np.unique(np.concatenate([a, b, c, d]), axis=0)
    sp, se, sf, sz = (np.asarray(v, np.float64)[pairs[:, 0]] for v in (ev.seed_pt, ev.seed_eta, ev.seed_phi, ev.seed_z0))
    sq = ev.seed_q.astype(np.float64)[pairs[:, 0]]
    objs = om[pairs[:, 1]]
    lay = geom_full.logical_layer[mod[objs[:, 0]]].astype(np.int64)
    ok, cuts, out = S.px(G, A_[objs], cat[objs], sp, se, sf, sz, sq, lay)
    accset = set(map(tuple, acc.tolist()))
    n_acc = 0
    for i in range(len(pairs)):
        p, f, tr = O.cuts(O.PT5 if five else O.PT3, A_[objs[i]], cat[objs[i]], [sp[i], se[i], sf[i], sz[i], sq[i], lay[i]])
        assert p == bool(ok[i]) == (tuple(pairs[i]) in accset), (i, tr)
        if lay[i] not in G.start_layers:
            continue
        n = objs.shape[1]
        assert len(tr) == 3 * n
        for q in range(n):
            for (kind, v, thr), nm in zip(tr[3 * q:3 * q + 3], ("s%d" % q, "phi%d" % q, "zeta%d" % q)):
                _close([v], [cuts[nm][0][i]], "px %s v" % nm)
                if cuts[nm][1] is not None:
                    _close([thr], [cuts[nm][1][i]], "px %s thr" % nm)
        if p:
            _close([f[0]], [out["chi2"][i]], "px chi2")
            n_acc += 1
    assert n_acc > 300 and (~ok).sum() > 1000
