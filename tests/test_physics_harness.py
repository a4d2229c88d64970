"""Physics-sanity harness on the oracle's track candidates: hand-checkable cases and
the magnitudes the paper quotes as context (efficiency plateau ~90 % and up, duplicate
rate of a few per cent; the synthetic events have no material effects, so efficiency is higher)."""
import numpy as np

import lstgen
from oracle import lst_oracle as O
from paper_2209_13711_b200 import physics as PH
from helpers import track_event


def _oracle_tc(geom, mp, ev):
    """The oracle's TC list in the layout of lst_get_objects(LST_TC): [n, 14] hits, types, pt, eta."""
    o = O.Oracle(geom, mp[0], mp[1])
    o.load(ev)
    o.run(upto=O.TC, pixel_indexed=True)
    tc = o.get(O.TC)
    objs = {lvl: o.get(lvl) for lvl in (O.T5, O.PT3, O.PT5)}
    ids = np.asarray(ev.seed_hit_ids, np.int64)
    rows = []
    for t, i in tc["parents"].tolist():
        ot, pix = [PH.PAD] * 10, [PH.PAD] * 4
        if t == O.TC:
            pix = ids[i].tolist()
        else:
            h = objs[t]["hits"][i].tolist()
            ot[:len(h)] = h
            if t != O.T5:
                pix = ids[objs[t]["parents"][i, 0]].tolist()
        rows.append(ot + pix)
    return np.asarray(rows, np.int64).reshape(-1, 14), tc["parents"][:, 0], tc["f"][:, 0], tc["f"][:, 1]


def test_single_clean_track_is_found_once_and_nothing_is_fake(geom_barrel, map_barrel):
    ev, _ = track_event(geom_barrel, pt=[3.0, 2.0], eta=[0.1, -0.3], phi=[0.4, 2.0], q=[1, -1], seeds=True)
    hits, typ, pt, eta = _oracle_tc(geom_barrel, map_barrel, ev)
    r = PH.rates(ev, hits, typ, pt, eta)
    assert r["n_den"] == 2 and r["n_found"] == 2 and r["n_fake"] == 0
    pid, nh = PH.match_track_candidates(ev, hits, typ)
    assert set(pid.tolist()) == {0, 1} and np.all(nh >= 10)
    assert r["n_duplicate"] == len(pid) - 2          # every candidate beyond the first of a particle is a duplicate


def test_a_candidate_of_mixed_hits_is_fake(geom_barrel, map_barrel):
    ev, _ = track_event(geom_barrel, pt=[3.0, 3.0], eta=[0.1, 0.12], phi=[0.4, 0.45], q=[1, 1], seeds=False)
    pid = np.asarray(ev.pid)
    a, b = np.nonzero(pid == 0)[0], np.nonzero(pid == 1)[0]
    mixed = np.concatenate([a[:5], b[:5], [PH.PAD] * 4])          # 5 + 5 hits: no particle reaches 75 %
    pure = np.concatenate([a[:10], [PH.PAD] * 4])
    m, _ = PH.match_track_candidates(ev, np.stack([mixed, pure]), np.array([3, 3]))
    assert m.tolist() == [-1, 0]


def test_rates_on_config2_with_seeds(geom_barrel, map_barrel):
    ev = lstgen.make_event(geom_barrel, "cfg2s")
    hits, typ, pt, eta = _oracle_tc(geom_barrel, map_barrel, ev)
    s = PH.summary(PH.rates(ev, hits, typ, pt, eta))
    assert s["denominator_particles"] > 50
    assert s["efficiency_prompt"] >= 0.95, s
    assert s["fake_rate"] <= 0.30 and s["duplicate_rate"] <= 0.30, s
    assert len(s["eff_vs_pt"]) == 7 and len(s["eff_vs_rv"]) == 5
