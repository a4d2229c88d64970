"""Test helpers: tiny events for the pins, set comparison of object collections."""
from __future__ import annotations

import numpy as np

import lstgen
from lstgen import events as E


def track_event(geom, pt, eta, phi, q, vz=0.0, smear=False, seeds=False):
    """Noise-free event made of the given prompt particles (lists or scalars)."""
    as_list = lambda v: list(v) if np.ndim(v) else [v]
    pt, eta, phi, q = map(as_list, (pt, eta, phi, q))
    vz = as_list(vz) if np.ndim(vz) else [vz] * len(pt)
    P = E.particles_from_lists(pt, eta, phi, q, vz=vz)
    rng = np.random.Generator(np.random.Philox(key=12345))
    x, y, z, det, pid = E.simulate(geom, P, rng, smear=smear, noise_frac=0.0, shuffle=False)
    sd = E.make_seeds(P, rng, smear=False, fake_frac=0.0) if seeds else None
    ev = E.pack_event(x, y, z, det, pid, P, sd)
    return ev, (x, y, z, det, pid)


def modules_with_both_sensors(det):
    det = np.asarray(det, dtype=np.int64)
    mods = det >> 1
    lo = set(mods[(det & 1) == 0].tolist())
    up = set(mods[(det & 1) == 1].tolist())
    return sorted(lo & up)


def tuple_set(hits):
    """Set of hit-index tuples of an [n, arity] array."""
    return set(map(tuple, np.asarray(hits, dtype=np.int64).tolist()))


def permute_event(ev, perm):
    """Event with hit order permuted: new hit j = old hit perm[j]."""
    import dataclasses
    return dataclasses.replace(ev, x=ev.x[perm].copy(), y=ev.y[perm].copy(), z=ev.z[perm].copy(),
                               det=ev.det[perm].copy(), pid=ev.pid[perm].copy())
