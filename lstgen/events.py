"""Seeded synthetic events: particles -> helices -> sensor hits (+ pixel seeds).

Recipe (BASELINE.json configs 1-5):
  * particles: pT = 0.5 (1-U)^(-1/2) GeV (dN/dpT ~ pT^-3 above 0.5 GeV) or uniform in a range,
    eta, phi uniform, q = +-1, vertex N(0, 15 um) in x,y and N(0, 5 cm) in z; a fraction are
    secondaries: vertex r ~ U(0, 10 cm), azimuth uniform, direction = vertex azimuth + N(0, 0.25);
  * helix in B = 3.8 T along z, outgoing arc only (turning angle < pi), first crossing of every
    sensor plane; local coordinates smeared by N(0, pitch/sqrt(12)) and clipped to the sensor;
  * noise hits uniform over modules, sensors and sensor area; hit order shuffled;
  * pixel seeds (configs 4-5): one per primary with |eta| < 2.4 and pT > 0.8 GeV, parameters
    smeared (1 % pT, 1 mrad phi, 0.5 mm z0), plus 30 % fakes with uniform parameters; every
    seed owns 4 pixel-hit ids; a fifth of the fakes borrow 2 ids from a true seed.

RNG: numpy Philox keyed by the event seed; draw order = the order of the statements below.
Nothing here evaluates any LST selection.
"""
from __future__ import annotations

import dataclasses
import math

import numpy as np

from . import geometry as G

B_FIELD_T = 3.8
K_B = 0.00299792458 * B_FIELD_T          # GeV / cm: pT = K_B * R


@dataclasses.dataclass
class Event:
    x: np.ndarray          # f32 [n_hits]
    y: np.ndarray
    z: np.ndarray
    det: np.ndarray        # u32 [n_hits]  2*module + sensor (0 = lower, 1 = upper)
    pid: np.ndarray        # i32 [n_hits]  truth particle (-1 noise); diagnostics only
    particles: dict
    seed_pt: np.ndarray    # f32 [n_seeds]
    seed_eta: np.ndarray
    seed_phi: np.ndarray
    seed_z0: np.ndarray
    seed_q: np.ndarray     # i8
    seed_hit_ids: np.ndarray  # u32 [n_seeds, 4]  pixel-hit id space
    seed_pid: np.ndarray   # i32  truth particle (-1 fake)

    @property
    def n_hits(self) -> int:
        return int(self.x.shape[0])

    @property
    def n_seeds(self) -> int:
        return int(self.seed_pt.shape[0])


CONFIGS = {
    # name: barrel_only, n_particles, spectrum, pt_range, eta_max, f_secondary, noise, seeds, rng seed
    "cfg1": dict(barrel_only=True, n=10, spectrum=False, pt_range=(1.0, 10.0), eta_max=0.8,
                 f_sec=0.0, noise=0.0, seeds=False, seed=1),
    "cfg2": dict(barrel_only=True, n=500, spectrum=True, pt_range=None, eta_max=0.8,
                 f_sec=0.0, noise=0.01, seeds=False, seed=2),
    # config 2 with pixel seeds: small enough for the oracle's all-pairs (brute) linking and cleaning
    "cfg2s": dict(barrel_only=True, n=500, spectrum=True, pt_range=None, eta_max=0.8,
                  f_sec=0.0, noise=0.01, seeds=True, seed=22),
    "cfg3": dict(barrel_only=False, n=6000, spectrum=True, pt_range=None, eta_max=2.4,
                 f_sec=0.15, noise=0.02, seeds=False, seed=3),
    "cfg3h": dict(barrel_only=False, n=13500, spectrum=True, pt_range=None, eta_max=2.4,
                  f_sec=0.15, noise=0.02, seeds=False, seed=3),
    "cfg4": dict(barrel_only=False, n=6000, spectrum=True, pt_range=None, eta_max=2.4,
                 f_sec=0.15, noise=0.02, seeds=True, seed=4),
    "cfg4h": dict(barrel_only=False, n=13500, spectrum=True, pt_range=None, eta_max=2.4,
                  f_sec=0.15, noise=0.02, seeds=True, seed=4),
}


def _wrap(a):
    return (a + np.pi) % (2.0 * np.pi) - np.pi


def make_particles(rng, n, eta_max, spectrum=True, pt_range=None, f_sec=0.0):
    if spectrum:
        pt = 0.5 * (1.0 - rng.random(n)) ** -0.5
    else:
        pt = rng.uniform(pt_range[0], pt_range[1], n)
    eta = rng.uniform(-eta_max, eta_max, n)
    phi = rng.uniform(-np.pi, np.pi, n)
    q = np.where(rng.random(n) < 0.5, -1, 1).astype(np.int64)
    vx = rng.normal(0.0, 0.0015, n)
    vy = rng.normal(0.0, 0.0015, n)
    vz = rng.normal(0.0, 5.0, n)
    sec = rng.random(n) < f_sec
    rv = rng.uniform(0.0, 10.0, n)
    pv = rng.uniform(-np.pi, np.pi, n)
    dv = rng.normal(0.0, 0.25, n)
    vx = np.where(sec, rv * np.cos(pv), vx)
    vy = np.where(sec, rv * np.sin(pv), vy)
    phi = np.where(sec, _wrap(pv + dv), phi)
    return dict(pt=pt, eta=eta, phi=phi, q=q, vx=vx, vy=vy, vz=vz, sec=sec)


def particles_from_lists(pt, eta, phi, q, vx=None, vy=None, vz=None):
    n = len(pt)
    z = np.zeros(n)
    return dict(pt=np.asarray(pt, float), eta=np.asarray(eta, float), phi=np.asarray(phi, float),
                q=np.asarray(q, np.int64),
                vx=z.copy() if vx is None else np.asarray(vx, float),
                vy=z.copy() if vy is None else np.asarray(vy, float),
                vz=z.copy() if vz is None else np.asarray(vz, float),
                sec=np.zeros(n, bool))


def _barrel_hits(geom, P, rng, smear, out):
    om = -P["q"] * K_B / P["pt"]
    for l, R in enumerate(G.BARREL_R):
        cat = G.CAT_BPS if l < 3 else G.CAT_B2S
        gap = G.GAP_OF_CAT[cat]
        nphi = geom.barrel_nphi[l]
        base = geom.barrel_base[l]
        sig_t = G.PITCH_T[cat] / math.sqrt(12.0)
        sig_l = G.PITCH_L[cat] / math.sqrt(12.0)
        # candidate modules: the 3 nearest the prompt-approximation azimuth at radius R
        phi_at_R = _wrap(P["phi"] + np.arcsin(np.clip(om * R / 2.0, -1.0, 1.0)))
        ip0 = np.round(phi_at_R / (2.0 * np.pi / nphi)).astype(np.int64)
        for dip in (-1, 0, 1):
            ip = (ip0 + dip) % nphi
            phic = 2.0 * np.pi * ip / nphi
            cphi, sphi = np.cos(phic), np.sin(phic)
            nv = P["vx"] * cphi + P["vy"] * sphi
            uv = -P["vx"] * sphi + P["vy"] * cphi
            a0 = _wrap(P["phi"] - phic)
            for sens, off in ((0, -gap / 2.0), (1, gap / 2.0)):
                S = np.sin(a0) + om * (R + off - nv)
                ok = np.abs(S) <= 1.0
                a1 = np.arcsin(np.clip(S, -1.0, 1.0))
                s = (a1 - a0) / om
                ok &= (s > 0.0) & (np.abs(om * s) < np.pi)
                u = uv - (np.cos(a1) - np.cos(a0)) / om
                zz = P["vz"] + s * np.sinh(P["eta"])
                iz = np.floor((zz + 120.0) / 10.0).astype(np.int64)
                ok &= (np.abs(u) <= G.HALF_MODULE) & (iz >= 0) & (iz < G.BARREL_NZ)
                idx = np.nonzero(ok)[0]
                zc = -115.0 + 10.0 * iz[idx]
                uu = u[idx]
                vv = zz[idx] - zc
                if smear:
                    uu = np.clip(uu + rng.normal(0.0, sig_t, len(idx)), -G.HALF_MODULE, G.HALF_MODULE)
                    vv = np.clip(vv + rng.normal(0.0, sig_l, len(idx)), -G.HALF_MODULE, G.HALF_MODULE)
                cp, sp = cphi[idx], sphi[idx]
                x = (R + off) * cp - uu * sp
                y = (R + off) * sp + uu * cp
                mod = base + iz[idx] * nphi + ip[idx]
                out.append((x, y, zc + vv, 2 * mod + sens, idx))


def _endcap_hits(geom, P, rng, smear, out):
    om = -P["q"] * K_B / P["pt"]
    sh = np.sinh(P["eta"])
    sh = np.where(np.abs(sh) < 1e-12, 1e-12, sh)
    rnphi = np.asarray(geom.ring_nphi)
    rbase = np.asarray(geom.ring_base)
    for side in (0, 1):
        sgn = 1.0 if side == 0 else -1.0
        for d, Z in enumerate(G.DISK_Z):
            dbase = geom.n_barrel + (side * 5 + d) * geom.n_per_disk
            for sens in (0, 1):
                for cat in (G.CAT_EPS, G.CAT_E2S):
                    gap = G.GAP_OF_CAT[cat]
                    sig_t = G.PITCH_T[cat] / math.sqrt(12.0)
                    sig_l = G.PITCH_L[cat] / math.sqrt(12.0)
                    zp = sgn * (Z + (gap / 2.0 if sens else -gap / 2.0))
                    s = (zp - P["vz"]) / sh
                    ok = (s > 0.0) & (np.abs(om * s) < np.pi)
                    a = P["phi"] + om * s
                    x = P["vx"] + (np.sin(a) - np.sin(P["phi"])) / om
                    y = P["vy"] - (np.cos(a) - np.cos(P["phi"])) / om
                    r = np.hypot(x, y)
                    ph = np.arctan2(y, x) % (2.0 * np.pi)
                    k = np.floor((r - G.RING_RLO) / G.D_RING).astype(np.int64)
                    ok &= (k >= 0) & (k < G.N_RING)
                    kk = np.clip(k, 0, G.N_RING - 1)
                    ok &= (kk < G.N_PS_RINGS) == (cat == G.CAT_EPS)
                    idx = np.nonzero(ok)[0]
                    kk = kk[idx]
                    nph = rnphi[kk]
                    w = 2.0 * np.pi / nph
                    ip = np.minimum(np.floor(ph[idx] / w).astype(np.int64), nph - 1)
                    rr, pp = r[idx], ph[idx]
                    if smear:
                        pp = pp + rng.normal(0.0, sig_t, len(idx)) / rr
                        rr = rr + rng.normal(0.0, sig_l, len(idx))
                        rlo = G.RING_RLO + kk * G.D_RING
                        rr = np.clip(rr, rlo, rlo + G.D_RING)
                        pp = np.clip(pp, ip * w, (ip + 1) * w)
                    mod = dbase + rbase[kk] + ip
                    out.append((rr * np.cos(pp), rr * np.sin(pp), np.full(len(idx), zp),
                                2 * mod + sens, idx))


def _noise_hits(geom, rng, n_noise):
    nm = geom.n_modules
    mods = rng.integers(0, nm, n_noise)
    sens = rng.integers(0, 2, n_noise)
    u = rng.uniform(-1.0, 1.0, n_noise)
    v = rng.uniform(-1.0, 1.0, n_noise)
    cat = geom.category[mods].astype(np.int64)
    gap = np.asarray(G.GAP_OF_CAT)[cat]
    is_ec = cat >= 2
    phic = geom.phic[mods].astype(np.float64)
    # barrel: flat sensor at normal distance rmin (+gap for the upper one)
    rn = geom.rmin[mods].astype(np.float64) + np.where(sens == 1, gap, 0.0)
    ub = u * G.HALF_MODULE
    xb = rn * np.cos(phic) - ub * np.sin(phic)
    yb = rn * np.sin(phic) + ub * np.cos(phic)
    zb = 0.5 * (geom.zmin[mods] + geom.zmax[mods]).astype(np.float64) + v * G.HALF_MODULE
    # endcap: annular sector at |z| of the sensor plane
    r = geom.rmin[mods] + 0.5 * (v + 1.0) * (geom.rmax[mods] - geom.rmin[mods]).astype(np.float64)
    ph = phic + u * geom.half_phi[mods].astype(np.float64)
    zl = geom.zmin[mods].astype(np.float64)
    ze = zl + np.sign(zl) * np.where(sens == 1, gap, 0.0)
    x = np.where(is_ec, r * np.cos(ph), xb)
    y = np.where(is_ec, r * np.sin(ph), yb)
    z = np.where(is_ec, ze, zb)
    return x, y, z, 2 * mods + sens, np.full(n_noise, -1, dtype=np.int64)


def simulate(geom, P, rng, smear=True, noise_frac=0.0, shuffle=True):
    """Hits of the particles P in `geom` (+ noise); returns x, y, z, det, pid (float64/int64)."""
    out = []
    _barrel_hits(geom, P, rng, smear, out)
    if not geom.barrel_only:
        _endcap_hits(geom, P, rng, smear, out)
    cols = [np.concatenate([o[c] for o in out]) if out else np.zeros(0) for c in range(5)]
    x, y, z, det, pid = cols
    n_noise = int(round(noise_frac * len(x)))
    if n_noise > 0:
        nx, ny, nz, nd, npid = _noise_hits(geom, rng, n_noise)
        x, y, z = np.concatenate([x, nx]), np.concatenate([y, ny]), np.concatenate([z, nz])
        det, pid = np.concatenate([det, nd]), np.concatenate([pid, npid])
    if shuffle and len(x) > 0:
        perm = rng.permutation(len(x))
        x, y, z, det, pid = x[perm], y[perm], z[perm], det[perm], pid[perm]
    return x, y, z, det.astype(np.int64), pid.astype(np.int64)


def make_seeds(P, rng, smear=True, fake_frac=0.3):
    sel = np.nonzero((~P["sec"]) & (np.abs(P["eta"]) < 2.4) & (P["pt"] > 0.8))[0]
    nt = len(sel)
    if smear:
        pt = P["pt"][sel] * (1.0 + 0.01 * rng.normal(0.0, 1.0, nt))
        phi = _wrap(P["phi"][sel] + 0.001 * rng.normal(0.0, 1.0, nt))
        z0 = P["vz"][sel] + 0.05 * rng.normal(0.0, 1.0, nt)
    else:
        pt, phi, z0 = P["pt"][sel].copy(), P["phi"][sel].copy(), P["vz"][sel].copy()
    eta = P["eta"][sel].copy()
    q = P["q"][sel].copy()
    pid = sel.astype(np.int64)
    nf = int(round(fake_frac * nt))
    if nf > 0:
        pt = np.concatenate([pt, rng.uniform(0.8, 10.0, nf)])
        eta = np.concatenate([eta, rng.uniform(-2.4, 2.4, nf)])
        phi = np.concatenate([phi, rng.uniform(-np.pi, np.pi, nf)])
        z0 = np.concatenate([z0, rng.uniform(-15.0, 15.0, nf)])
        q = np.concatenate([q, np.where(rng.random(nf) < 0.5, -1, 1)])
        pid = np.concatenate([pid, np.full(nf, -1, dtype=np.int64)])
    n = nt + nf
    hit_ids = (4 * np.arange(n, dtype=np.int64)[:, None] + np.arange(4)[None, :])
    if nf > 0 and nt > 0:
        borrow = rng.random(nf) < 0.2
        donor = rng.integers(0, nt, nf)
        for j in np.nonzero(borrow)[0]:
            hit_ids[nt + j, 0:2] = hit_ids[donor[j], 0:2]
    if n > 0:
        perm = rng.permutation(n)
        pt, eta, phi, z0, q, pid, hit_ids = (a[perm] for a in (pt, eta, phi, z0, q, pid, hit_ids))
    return pt, eta, phi, z0, q, hit_ids, pid


def pack_event(x, y, z, det, pid, P, seeds=None) -> Event:
    if seeds is None:
        e = np.zeros(0)
        seeds = (e, e, e, e, np.zeros(0, np.int64), np.zeros((0, 4), np.int64), np.zeros(0, np.int64))
    spt, seta, sphi, sz0, sq, sids, spid = seeds
    f32 = lambda a: np.ascontiguousarray(a, dtype=np.float32)
    return Event(
        x=f32(x), y=f32(y), z=f32(z), det=np.ascontiguousarray(det, dtype=np.uint32),
        pid=np.ascontiguousarray(pid, dtype=np.int32), particles=P,
        seed_pt=f32(spt), seed_eta=f32(seta), seed_phi=f32(sphi), seed_z0=f32(sz0),
        seed_q=np.ascontiguousarray(sq, dtype=np.int8),
        seed_hit_ids=np.ascontiguousarray(sids, dtype=np.uint32).reshape(-1, 4),
        seed_pid=np.ascontiguousarray(spid, dtype=np.int32),
    )


def make_event(geom, config: str, seed: int | None = None, n_particles: int | None = None) -> Event:
    """One event of a named BASELINE.json config (`cfg1` ... `cfg4h`); `seed` overrides the
    config's own (config 5 = cfg4 / cfg4h with seeds 1000..1063)."""
    c = CONFIGS[config]
    assert geom.barrel_only == c["barrel_only"], "geometry does not match the config"
    rng = np.random.Generator(np.random.Philox(key=c["seed"] if seed is None else seed))
    n = c["n"] if n_particles is None else n_particles
    P = make_particles(rng, n, c["eta_max"], c["spectrum"], c["pt_range"], c["f_sec"])
    x, y, z, det, pid = simulate(geom, P, rng, smear=True, noise_frac=c["noise"])
    seeds = make_seeds(P, rng) if c["seeds"] else None
    return pack_event(x, y, z, det, pid, P, seeds)
