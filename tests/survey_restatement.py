"""A third, independent transcription of the selection arithmetic, typed from SURVEY.md section 8(c)
(C0-C6) in vectorised numpy -- NOT from oracle/lst_oracle.c and not from csrc/lst_math.cuh.

Each function takes arrays of candidates and returns
    cuts : dict  name -> (v, thr)   arrays; the predicate is  v <= thr  ("sign" cuts: v > 0, thr = None)
    out  : dict  name -> array      the stored / derived quantities
so that tests can compare every cut variable and every threshold with the oracle's trace
(oracle.cuts) one by one, not only the final decision.  Points are arrays [N, 3] (x, y, z) in
double precision; cat arrays hold the module category 0 bPS, 1 b2S, 2 ePS, 3 e2S.
"""
from __future__ import annotations

import numpy as np

S12 = np.sqrt(12.0)


class Cfg:
    """SURVEY.md Appendix B defaults."""
    kB = 0.00299792458 * 3.8
    pt_min = 0.8
    n_sigma = 4.0
    z0max = 15.0
    d0max = 2.5
    chi2max = 18.42
    ec_md_sys = 0.3
    modez_slack = 0.15
    seed_sig_phi, seed_sig_pt, seed_sig_z = 0.001, 0.01, 0.05
    sig_t = np.array([0.01, 0.009, 0.01, 0.009]) / S12
    sig_z = np.array([0.15, 5.0, 0.0, 0.0]) / S12
    sig_r = np.array([0.0, 0.0, 0.15, 5.0]) / S12
    start_layers = (0, 1, 6, 7, 11, 12)

    @property
    def kmax(self):
        return self.kB / (2.0 * self.pt_min)


# ----------------------------------------------------------------------------- C0
def rt(P):
    return np.sqrt(P[:, 0] ** 2 + P[:, 1] ** 2)


def cross(ax, ay, bx, by):
    return ax * by - ay * bx


def sd(A, B):
    D = B - A
    return cross(A[:, 0], A[:, 1], D[:, 0], D[:, 1]) / (rt(A) * rt(B))


def dphi(A, B):
    D = B - A
    return np.arctan2(cross(A[:, 0], A[:, 1], D[:, 0], D[:, 1]), A[:, 0] * B[:, 0] + A[:, 1] * B[:, 1])


def chord(A, B):
    return np.hypot(B[:, 0] - A[:, 0], B[:, 1] - A[:, 1])


def dr(A, B):
    D = B - A
    return (2.0 * (A[:, 0] * D[:, 0] + A[:, 1] * D[:, 1]) + D[:, 0] ** 2 + D[:, 1] ** 2) / (rt(A) + rt(B))


def kappa3(A, B, C):
    ab, bc, ac = B - A, C - B, C - A
    return cross(ab[:, 0], ab[:, 1], bc[:, 0], bc[:, 1]) / (
        np.hypot(ab[:, 0], ab[:, 1]) * np.hypot(bc[:, 0], bc[:, 1]) * np.hypot(ac[:, 0], ac[:, 1]))


def arc(r, k):
    """s(r; kappa) = r if |kappa r| <= 1e-4 else asin(clamp(kappa r)) / kappa."""
    kr = k * r
    with np.errstate(divide="ignore", invalid="ignore"):
        big = np.arcsin(np.clip(kr, -1.0, 1.0)) / k
    return np.where(np.abs(kr) <= 1e-4, r, big)


def wrap(a):
    return np.remainder(a + np.pi, 2.0 * np.pi) - np.pi


# ----------------------------------------------------------------------------- C1
def md(g, L, U, cat):
    cat = np.asarray(cat)
    rl, ru = rt(L), rt(U)
    dz = U[:, 2] - L[:, 2]
    sdv, cxy, drv = sd(L, U), chord(L, U), dr(L, U)
    st = g.sig_t[cat]
    tolphi = g.n_sigma * st * (1.0 / rl + 1.0 / ru)
    ec = cat >= 2
    azl = np.abs(L[:, 2])
    with np.errstate(divide="ignore", invalid="ignore"):
        b1 = (np.abs(dz - L[:, 2] * drv / rl), g.z0max * drv / rl + 2.0 * g.n_sigma * g.sig_z[cat])
        b2 = (np.abs(sdv), g.kmax * cxy + tolphi)
        e1 = (np.abs(drv - rl * dz / L[:, 2]),
              rl * np.abs(dz) * g.z0max / (azl * (azl - g.z0max)) + 2.0 * g.n_sigma * g.sig_r[cat])
        e2 = (np.abs(sdv), np.abs(dz) * np.arcsin(np.minimum(1.0, g.kmax * rl)) / (azl - g.z0max) + tolphi)
        cpred = np.where(ec, np.abs(dz) * rl / azl, cxy)
        out = dict(kappa=sdv / cpred, sigk=st * (1.0 / rl + 1.0 / ru) / cpred, dphi=np.arcsin(np.clip(sdv, -1, 1)))
    cuts = dict(B1sign=(drv, None), B1=b1, B2=b2, E1=e1, E2=e2)
    ok_b = (drv > 0) & (b1[0] <= b1[1]) & (b2[0] <= b2[1])
    ok_e = (e1[0] <= e1[1]) & (e2[0] <= e2[1]) & (azl - g.z0max > 1e-9)
    ok = np.where(ec, ok_e, ok_b) & (cpred > 1e-9)
    return ok, cuts, out, ec


# ----------------------------------------------------------------------------- C3
def ls(g, A, B, ci, co, ki, ski, ko, sko):
    ci, co = np.asarray(ci), np.asarray(co)
    ri, ro = rt(A), rt(B)
    ns = g.n_sigma
    dz = B[:, 2] - A[:, 2]
    drv, sdv, cxy, dph = dr(A, B), sd(A, B), chord(A, B), dphi(A, B)
    modeZ = co >= 2
    N = ri * dz - A[:, 2] * drv
    E = ri * g.sig_z[co] + ro * g.sig_z[ci] + np.abs(B[:, 2]) * g.sig_r[ci] + np.abs(A[:, 2]) * g.sig_r[co]
    l1 = (np.abs(N), g.z0max * np.abs(drv) + ns * E)
    tphi = g.sig_t[ci] / ri + g.sig_t[co] / ro
    tolphi = ns * tphi
    dot = A[:, 0] * B[:, 0] + A[:, 1] * B[:, 1]
    # mode R
    l2r = (np.abs(sdv), g.kmax * cxy + tolphi)
    with np.errstate(divide="ignore", invalid="ignore"):
        k_r, sk_r = sdv / cxy, tphi / cxy
        # mode Z
        rbar, zbar = 0.5 * (ri + ro), 0.5 * (np.abs(A[:, 2]) + np.abs(B[:, 2]))
        adz = np.abs(dz)
        Sbar = np.arcsin(np.minimum(1.0, g.kmax * (rbar + ns * (g.sig_r[ci] + g.sig_r[co]) / 2.0))) / g.kmax
        den = zbar - g.z0max - ns * g.sig_z[ci] / 2.0
        l2z = (np.abs(dph), g.kmax * (adz + ns * g.sig_z[ci]) * Sbar / den + tolphi)
        lever = zbar / (adz * rbar)
        k_z, sk_z = dph * lever, tphi * lever
        slack_z = np.abs(k_z) * (g.z0max / zbar + g.modez_slack + ns * (g.sig_r[ci] + g.sig_r[co]) / (ri + ro)
                                 + ns * g.sig_z[ci] / adz)
    kls = np.where(modeZ, k_z, k_r)
    sk = np.where(modeZ, sk_z, sk_r)
    slack = np.where(modeZ, slack_z, 0.0)
    l3i = (np.abs(ki - kls), ns * (ski + sk) + slack + np.where(ci >= 2, g.ec_md_sys * np.abs(kls), 0.0))
    l3o = (np.abs(ko - kls), ns * (sko + sk) + slack + np.where(co >= 2, g.ec_md_sys * np.abs(kls), 0.0))
    l2 = (np.where(modeZ, l2z[0], l2r[0]), np.where(modeZ, l2z[1], l2r[1]))
    ok = (l1[0] <= l1[1]) & (dot > 0) & (l2[0] <= l2[1]) & (l3i[0] <= l3i[1]) & (l3o[0] <= l3o[1])
    ok &= np.where(modeZ, (den > 1e-9) & (adz > 1e-9), cxy > 1e-9)
    cuts = dict(L1=l1, dot=(dot, None), den=(den, None), L2=l2, L3i=l3i, L3o=l3o)
    return ok, cuts, dict(kappa=kls, sigk=sk, dphi=dph), modeZ


# ----------------------------------------------------------------------------- C4
def sig_perp(g, P, cat):
    return g.sig_t[cat] + g.sig_r[cat] * np.minimum(1.0, g.kmax * rt(P))


def t3(g, P1, P2, P3, c1, c2, c3):
    c1, c2, c3 = map(np.asarray, (c1, c2, c3))
    ns = g.n_sigma
    modeZ = (c1 >= 2) | (c2 >= 2) | (c3 >= 2)
    a, b, c13 = chord(P1, P2), chord(P2, P3), chord(P1, P3)
    k3 = kappa3(P1, P2, P3)
    sk3 = (sig_perp(g, P2, c2) + (b * sig_perp(g, P1, c1) + a * sig_perp(g, P3, c3)) / c13) / (a * b)
    t31 = (np.abs(k3), g.kmax + ns * sk3)
    D12, D23 = P2 - P1, P3 - P2
    beta = np.arctan2(cross(D12[:, 0], D12[:, 1], D23[:, 0], D23[:, 1]), D12[:, 0] * D23[:, 0] + D12[:, 1] * D23[:, 1])
    d12, d23 = dphi(P1, P2), dphi(P2, P3)
    d13 = d12 + d23
    k13 = np.sin(d13) / c13
    r1, r2, r3 = rt(P1), rt(P2), rt(P3)
    L1 = np.where(modeZ, P1[:, 2], arc(r1, k13))
    L2 = np.where(modeZ, P2[:, 2], arc(r2, k13))
    L3 = np.where(modeZ, P3[:, 2], arc(r3, k13))
    sL1 = np.where(modeZ, g.sig_z[c1], 0.0)
    sL2 = np.where(modeZ, g.sig_z[c2], 0.0)
    sL3 = np.where(modeZ, g.sig_z[c3], 0.0)
    Nphi = d12 * (L3 - L2) - d23 * (L2 - L1)
    Nrho = (1.0 / r2 - 1.0 / r1) * (L3 - L2) - (1.0 / r3 - 1.0 / r2) * (L2 - L1)
    Ephi = (g.sig_t[c1] / r1 * np.abs(L3 - L2) + g.sig_t[c2] / r2 * np.abs(L3 - L1) + g.sig_t[c3] / r3 * np.abs(L2 - L1)
            + sL1 * np.abs(d23) + sL2 * np.abs(d13) + sL3 * np.abs(d12))
    t32 = (np.abs(Nphi), g.d0max * np.abs(Nrho) + ns * Ephi)
    s1 = r1 * (1.0 + (k3 * r1) ** 2 / 6.0)
    s2 = r2 * (1.0 + (k3 * r2) ** 2 / 6.0)
    s3 = r3 * (1.0 + (k3 * r3) ** 2 / 6.0)
    z1, z2, z3 = P1[:, 2], P2[:, 2], P3[:, 2]
    N = (s2 - s1) * (z3 - z1) - (s3 - s1) * (z2 - z1)
    Ez = (g.sig_z[c3] * np.abs(s2 - s1) + g.sig_z[c2] * np.abs(s3 - s1) + g.sig_z[c1] * np.abs(s3 - s2)
          + g.sig_r[c2] * np.abs(z3 - z1) + g.sig_r[c3] * np.abs(z2 - z1) + g.sig_r[c1] * np.abs(z3 - z2))
    t33 = (np.abs(N), ns * Ez)
    ok = (t31[0] <= t31[1]) & (t32[0] <= t32[1]) & (t33[0] <= t33[1])
    return ok, {"T3-1": t31, "T3-2": t32, "T3-3": t33}, dict(kappa3=k3, sigk3=sk3, beta=beta)


# ----------------------------------------------------------------------------- C5
def kasa(g, P, cats, kc):
    """P: [N, 5, 3]; weighted algebraic circle fit, geometric residuals."""
    x, y = P[:, :, 0], P[:, :, 1]
    r = np.sqrt(x ** 2 + y ** 2)
    sig2 = g.sig_t[cats] ** 2 + (g.sig_r[cats] * np.minimum(1.0, kc[:, None] * r)) ** 2
    w = 1.0 / sig2
    sw = w.sum(1)
    u = x - ((w * x).sum(1) / sw)[:, None]
    v = y - ((w * y).sum(1) / sw)[:, None]
    zeta = u ** 2 + v ** 2
    Suu, Suv, Svv = (w * u * u).sum(1), (w * u * v).sum(1), (w * v * v).sum(1)
    Suz, Svz, Sz = (w * u * zeta).sum(1), (w * v * zeta).sum(1), (w * zeta).sum(1)
    det = Suu * Svv - Suv ** 2
    # [Suu Suv; Suv Svv] [B C]^T = -[Suz Svz]^T
    Bc = (-Suz * Svv + Svz * Suv) / det
    Cc = (-Svz * Suu + Suz * Suv) / det
    cx, cy = -Bc / 2.0, -Cc / 2.0
    R = np.sqrt((Bc ** 2 + Cc ** 2) / 4.0 + Sz / sw)
    e = np.hypot(u - cx[:, None], v - cy[:, None]) - R[:, None]
    return R, (w * e ** 2).sum(1), det


def t5(g, P, cats, k3a, sk3a, k3b, sk3b):
    """P: [N, 5, 3] anchors; returns cuts incl. the middle triplet's."""
    cats = np.asarray(cats)
    t51 = (np.abs(k3a - k3b), g.n_sigma * (sk3a + sk3b))
    okm, cm, _ = t3(g, P[:, 1], P[:, 2], P[:, 3], cats[:, 1], cats[:, 2], cats[:, 3])
    k135 = kappa3(P[:, 0], P[:, 2], P[:, 4])
    R, chi2, det = kasa(g, P, cats, np.abs(k135))
    k5 = np.sign(k135) / (2.0 * R)
    r1, r5 = rt(P[:, 0]), rt(P[:, 4])
    den = arc(r5, k5) - arc(r1, k5)
    out = dict(R=R, chi2=chi2, pt=g.kB * R,
               phi=wrap(np.arctan2(P[:, 0, 1], P[:, 0, 0]) - np.arcsin(np.clip(k5 * r1, -1, 1))),
               eta=np.arcsinh((P[:, 4, 2] - P[:, 0, 2]) / den))
    ok = (t51[0] <= t51[1]) & okm & (det > 0) & (chi2 <= g.chi2max) & (den > 1e-9)
    cuts = {"T5-1": t51, "mid T3-1": cm["T3-1"], "mid T3-2": cm["T3-2"], "mid T3-3": cm["T3-3"],
            "T5-3": (chi2, np.full_like(chi2, g.chi2max))}
    return ok, cuts, out


# ----------------------------------------------------------------------------- C6
def px(g, P, cats, pt, eta, phi, z0, q, first_layer):
    """P: [N, n, 3] anchors of the OT object; seed arrays [N]."""
    cats = np.asarray(cats)
    n = P.shape[1]
    kp = -q * g.kB / (2.0 * pt)
    sh = np.sinh(eta)
    ok = np.isin(first_layer, g.start_layers)
    cuts, tot = {}, 0.0
    for k in range(n):
        h, c = P[:, k], cats[:, k]
        r = rt(h)
        ec = c >= 2
        with np.errstate(divide="ignore", invalid="ignore"):
            s = np.where(ec, (h[:, 2] - z0) / sh, arc(r, kp))
            dph = wrap(np.arctan2(h[:, 1], h[:, 0]) - (phi + kp * s))
            sphi = g.seed_sig_phi + g.seed_sig_pt * np.abs(kp) * s + g.sig_t[c] / r
            rp = np.where(np.abs(kp * s) <= 1e-4, s, np.sin(kp * s) / kp)
            dzt = np.where(ec, r - rp, h[:, 2] - (z0 + sh * s))
            szt = np.where(ec, g.seed_sig_z / np.abs(sh) + g.sig_r[c], g.seed_sig_z + g.sig_z[c])
        cuts["s%d" % k] = (s, None)
        cuts["phi%d" % k] = (np.abs(dph), g.n_sigma * sphi)
        cuts["zeta%d" % k] = (np.abs(dzt), g.n_sigma * szt)
        ok = ok & (s > 0) & (np.abs(dph) <= g.n_sigma * sphi) & (np.abs(dzt) <= g.n_sigma * szt)
        tot = tot + (dph / sphi) ** 2 + (dzt / szt) ** 2
    return ok, cuts, dict(chi2=tot / (2.0 * n))


# ----------------------------------------------------------------------------- C2 module map
# SURVEY.md 8(c) C2 (Fig. 4), typed from the survey's bullet list.  One point is derived
# rather than copied: for an endcap target the survey takes "the hull over corners of (z_B - z0)/(z_A - z0)
# (only where side (z_A - z0) > 0)".  Over the box z0 in [-z0', z0'] x z_A in [zlo_A, zhi_A] that ratio is
# monotone in each variable, so its hull over the ADMISSIBLE part of the box is spanned by the admissible
# corners -- unless a corner is inadmissible, in which case the admissible part reaches z_A - z0 -> 0+ and the
# ratio has no upper bound there.  Hence: fewer than four admissible corners => upper end = +infinity.
MAP_KSCALE, MAP_Z0, MAP_D0MAX = 1.25, 20.0, 2.5


def map_next_layers(L):
    """barrel l -> barrel l + 1 and disk 1 of either side; disk d -> disk d + 1 of the same side; no skips."""
    if L < 6:
        return ([L + 1] if L + 1 < 6 else []) + [6, 11]
    if 6 <= L < 10 or 11 <= L < 15:
        return [L + 1]
    return []


def module_map(geom, kscale=MAP_KSCALE, z0p=MAP_Z0, d0max=MAP_D0MAX, cfg=Cfg()):
    """-> (row_offsets [n + 1], cols) of the C2 map, columns ascending inside a row."""
    f = lambda a: np.asarray(a, np.float64)
    lay = np.asarray(geom.logical_layer, np.int64)
    rmin, rmax, phic, hphi, zmin, zmax = map(f, (geom.rmin, geom.rmax, geom.phic, geom.half_phi, geom.zmin, geom.zmax))
    n = len(lay)
    kp = kscale * cfg.kmax
    by_layer = {L: np.nonzero(lay == L)[0] for L in range(16)}
    target_is_endcap = lay >= 6
    off, cols = np.zeros(n + 1, np.int64), []
    for A in range(n):
        cand = [by_layer[L] for L in map_next_layers(int(lay[A]))]
        Bs = np.sort(np.concatenate(cand)) if cand else np.zeros(0, np.int64)
        if Bs.size:
            aA = np.arcsin(min(1.0, kp * rmin[A]))
            aB = np.arcsin(np.minimum(1.0, kp * rmax[Bs]))
            d = phic[Bs] - phic[A]
            d = np.abs(d - 2 * np.pi * np.round(d / (2 * np.pi)))
            ok_phi = d <= hphi[A] + hphi[Bs] + aB - aA + d0max * np.maximum(0.0, 1.0 / rmin[A] - 1.0 / rmax[Bs])
            rho_lo, rho_hi = rmin[Bs] / rmax[A], aB / aA
            ok_rz = np.zeros(Bs.size, bool)
            bar = ~target_is_endcap[Bs]
            # barrel target: hull of z0 + (z_A - z0) rho over the 8 corners against [zlo_B, zhi_B]
            zp = np.stack([z0 + (zA - z0) * rho for z0 in (-z0p, z0p) for zA in (zmin[A], zmax[A]) for rho in (rho_lo, rho_hi)])
            ok_rz[bar] = ((zp.min(0) <= zmax[Bs]) & (zp.max(0) >= zmin[Bs]))[bar]
            # endcap target: hull of (z_B - z0) / (z_A - z0) over the admissible corners against [rho_lo, rho_hi]
            zB = zmin[Bs]
            side = np.where(zB > 0, 1.0, -1.0)
            lo, hi, nvalid = np.full(Bs.size, np.inf), np.full(Bs.size, -np.inf), np.zeros(Bs.size, np.int64)
            for z0 in (-z0p, z0p):
                for zA in (zmin[A], zmax[A]):
                    den = zA - z0
                    adm = side * den > 0.0
                    q = np.where(adm, (zB - z0) / (den if den != 0.0 else 1.0), np.nan)
                    lo = np.where(adm, np.minimum(lo, q), lo)
                    hi = np.where(adm, np.maximum(hi, q), hi)
                    nvalid += adm
            hi = np.where(nvalid < 4, np.inf, hi)
            ec_ok = (nvalid > 0) & (lo <= rho_hi) & (hi >= rho_lo)
            ok_rz[~bar] = ec_ok[~bar]
            cols.append(Bs[ok_phi & ok_rz])
        off[A + 1] = off[A] + (len(cols[-1]) if Bs.size else 0)
    return off, (np.concatenate(cols) if cols else np.zeros(0, np.int64))
