"""Do the pins actually pin?  Single-token mutations of oracle/lst_oracle.c (a swapped sigma index,
a dropped tolerance term, a wrong factor, a flipped sign, an off-by-one threshold, survivors-only
semantics dropped ...) are compiled into a scratch library and the pin tests are run against it
(LST_ORACLE_SO): every mutant must be caught, and by the pin named for that function.  This is the
evidence for DESIGN.md section 3's "pinned" column; it is not a product test.
"""
import os
import subprocess
import sys
from concurrent.futures import ThreadPoolExecutor

import pytest

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "lst_oracle.c")

# (what, original text, mutated text, the pin expected to catch it)
MUTANTS = [
    ("MD B1: factor 2 of the z tolerance", "g->z0max * drv / l->rt + 2.0 * g->n_sigma * g->sig_z[cat]",
     "g->z0max * drv / l->rt + 1.0 * g->n_sigma * g->sig_z[cat]", "test_md_b1_terms"),
    ("MD E1: z0max term dropped", "l->rt * fabs(dz) * g->z0max / (azl * (azl - g->z0max)) + 2.0", "2.0", "test_md_e1_terms"),
    ("MD E2: asin dropped", "fabs(dz) * asin(min2(1.0, c->kmax * l->rt)) / (azl - g->z0max) + tolphi",
     "fabs(dz) * (c->kmax * l->rt) / (azl - g->z0max) + tolphi", "test_md_e2_edge_closed_form"),
    ("MD: phi tolerance uses one radius", "double tolphi = g->n_sigma * st * (1.0 / l->rt + 1.0 / u->rt);",
     "double tolphi = g->n_sigma * st * (2.0 / l->rt);", "test_md_"),
    ("MD: exported dphi without asin", "out->dphi = asin(clamp1(sdv));", "out->dphi = clamp1(sdv);", "test_md_"),
    ("LS L1: sigma_z indices swapped", "A->rt * g->sig_z[co] + B->rt * g->sig_z[ci]",
     "A->rt * g->sig_z[ci] + B->rt * g->sig_z[co]", "test_ls_l1_terms"),
    ("LS L1: sigma_r(o) term dropped", " + fabs(A->z) * g->sig_r[co];", ";", "test_ls_l1_terms"),
    ("LS L2 mode Z: sigma_z(i) missing in the lever", "c->kmax * (adz + ns * g->sig_z[ci]) * Sbar / den", "c->kmax * adz * Sbar / den",
     "test_ls_l2_"),
    ("LS mode Z: sigma_kappa without the lever", "sigkls = tphi * lever;", "sigkls = tphi / cxy;", "test_ls_l2_"),
    ("LS L3: z0max / zbar slack dropped", "fabs(kls) * (g->z0max / zbar + g->modez_slack", "fabs(kls) * (g->modez_slack",
     "test_ls_l2_and_l3_terms"),
    ("LS L3: endcap systematic keyed on the wrong stub",
     "(is_endcap(ci) ? g->ec_md_sys * fabs(kls) : 0.0));\n  cut_le(&r, fabs(o->kappa",
     "(is_endcap(co) ? g->ec_md_sys * fabs(kls) : 0.0));\n  cut_le(&r, fabs(o->kappa", "test_ls_l2_and_l3_terms"),
    ("LS L3: tolerance four times too tight", "ns * (i->sigk + sigkls) + slack", "0.25 * ns * (i->sigk + sigkls) + slack",
     "test_ls_l2_and_l3_terms"),
    ("T3-1: a and b swapped in sigma_kappa3", "(b * sig_perp(c, P1) + a * sig_perp(c, P3))",
     "(a * sig_perp(c, P1) + b * sig_perp(c, P3))", "test_t3_"),
    ("T3-2: lever resolutions swapped", "sL1 * fabs(d23) + sL2 * fabs(d13) + sL3 * fabs(d12)",
     "sL1 * fabs(d12) + sL2 * fabs(d13) + sL3 * fabs(d23)", "test_t3_terms"),
    ("T3-2: d0max allowance dropped", "g->d0max * fabs(Nrho) + ns * Ephi", "ns * Ephi", "test_t3_terms"),
    ("T3-3: sigma_r indices swapped", "g->sig_r[P2->cat] * fabs(P3->z - P1->z) + g->sig_r[P3->cat] * fabs(P2->z - P1->z)",
     "g->sig_r[P3->cat] * fabs(P3->z - P1->z) + g->sig_r[P2->cat] * fabs(P2->z - P1->z)", "test_t3_terms"),
    ("T3-3: sign of the second product", "double Nz = (s2 - s1) * (P3->z - P1->z) - (s3 - s1) * (P2->z - P1->z);",
     "double Nz = (s2 - s1) * (P3->z - P1->z) + (s3 - s1) * (P2->z - P1->z);", "test_t3_"),
    ("T3: beta with swapped operands", "double beta = atan2(cross2(d12x, d12y, d23x, d23y), dot2(d12x, d12y, d23x, d23y));",
     "double beta = atan2(cross2(d23x, d23y, d12x, d12y), dot2(d12x, d12y, d23x, d23y));", "test_t3_beta"),
    ("T5-1: max instead of sum", "g->n_sigma * (sk3a + sk3b)", "g->n_sigma * max2(sk3a, sk3b)", "test_t5_1_radius_match_threshold"),
    ("T5-3: weights 1/sigma instead of 1/sigma^2", "w[k] = 1.0 / (st * st + sr * sr);", "w[k] = 1.0 / (st + sr);", "test_t5_chi2"),
    ("C6: pT term of sigma_phi dropped", "g->seed_sig_phi + g->seed_sig_pt * fabs(kp) * s + g->sig_t[h->cat] / h->rt",
     "g->seed_sig_phi + g->sig_t[h->cat] / h->rt", "test_px_windows_terms"),
    ("C6: endcap sigma_zeta without 1/|sinh eta|", "szt = g->seed_sig_z / fabs(sh) + g->sig_r[h->cat];",
     "szt = g->seed_sig_z + g->sig_r[h->cat];", "test_px_windows_terms"),
    ("C6: chi2_pix normalisation", "*chi2 = sum / (2.0 * n);", "*chi2 = sum / (1.0 * n);", "test_px_windows_terms"),
    ("C2: displacement allowance dropped", " + g->d0max * max2(0.0, 1.0 / rminA - 1.0 / rmaxB))) return 0;", ")) return 0;",
     "test_map_c2_"),
    ("C2: curvature margin 1.0 instead of map_kscale", "double kp = g->map_kscale * g->kB / (2.0 * g->pt_min);",
     "double kp = 1.0 * g->kB / (2.0 * g->pt_min);", "test_map_c2_"),
    ("C2: barrel may skip a layer", "if (L < 6) { if (L + 1 < 6) out[n++] = L + 1; out[n++] = 6;",
     "if (L < 6) { if (L + 2 < 6) out[n++] = L + 2; out[n++] = 6;", "test_map_c2_"),
    ("C2: unbounded end applied to the lower end", "if (nvalid < 4) hi = INFINITY;", "if (nvalid < 4) lo = -INFINITY;", "test_map_c2_"),
    ("C2: z0 margin 15 instead of map_z0", "double z0s[2] = {-g->map_z0, g->map_z0}", "double z0s[2] = {-g->z0max, g->z0max}", "test_map_c2_"),
    ("C2: rho_lo from the wrong radii", "double rho_lo = rminB / rmaxA, rho_hi = aB / aA;", "double rho_lo = rminB / rminA, rho_hi = aB / aA;",
     "test_map_c2_"),
    ("S0: > instead of >= (indexed)", "if (shared_ot(&o[a], &o[b]) >= min_shared && beats",
     "if (shared_ot(&o[a], &o[b]) > min_shared && beats", "test_s0_"),
    ("S0: > instead of >= (all pairs)", "|| shared_ot(&o[a], &o[b]) >= min_shared;", "|| shared_ot(&o[a], &o[b]) > min_shared;",
     "test_s0_"),
    ("S1-S3: Delta R^2 cut 10 % tighter", "return (d < c->cfg.dr2max) || shared_ot", "return (d < 0.9 * c->cfg.dr2max) || shared_ot",
     "test_s1_s2_s3"),
    ("S1: compares with removed pT5 too", "if (c->keep_pt5[b] && cross_dup(c, &op3[a], &op5[b], &m)) { k3[a] = 0; break; }",
     "if (cross_dup(c, &op3[a], &op5[b], &m)) { k3[a] = 0; break; }", "test_s1_s2_s3"),
    ("S2: ignores the surviving pT3", "for (uint32_t b = 0; b < np3 && !dup; ++b) if (c->keep_pt3[b] && cross_dup(c, &o5[a], &op3[b], &m)) dup = 1;",
     ";", "test_s"),
    ("S3: earlier-unused-pLS rule dropped", "if (dr2_f(&A, &Bq) < c->cfg.dr2max) dup = 1;", "if (0) dup = 1;", "test_s1_s2_s3"),
    ("S3: shared pixel hit ignored", "|| shared_ot(a, b) >= 1 || shared_pix(a, b) >= 1;", "|| shared_ot(a, b) >= 1;", "test_s1_s2_s3"),
]


def _run(k, tmp):
    what, a, b, pin = MUTANTS[k]
    src = open(SRC).read()
    assert src.count(a) >= 1, "mutation target vanished: " + what
    c = os.path.join(tmp, "mut%d.c" % k)
    so = os.path.join(tmp, "mut%d.so" % k)
    with open(c, "w") as f:
        f.write(src.replace(a, b, 1))
    subprocess.check_call(["gcc", "-O1", "-std=c11", "-fPIC", "-shared", "-w", "-I", os.path.join(ROOT, "oracle"),
                           "-o", so, c, "-lm"])
    env = dict(os.environ, LST_ORACLE_SO=so)
    r = subprocess.run([sys.executable, "-m", "pytest", "-x", "-q", "-p", "no:cacheprovider",
                        os.path.join(ROOT, "tests", "test_oracle_pins2.py")], cwd=ROOT, env=env, capture_output=True, text=True)
    failed = [ln for ln in r.stdout.splitlines() if ln.startswith("FAILED")]
    return what, pin, r.returncode, failed


def test_every_mutant_is_caught_by_its_pin(tmp_path):
    with ThreadPoolExecutor(max_workers=min(8, os.cpu_count() or 2)) as ex:
        results = list(ex.map(lambda k: _run(k, str(tmp_path)), range(len(MUTANTS))))
    survived = [w for w, pin, rc, failed in results if rc == 0]
    assert not survived, "mutants not caught by any pin: %s" % survived
    for what, pin, rc, failed in results:
        assert failed and pin in failed[0], "%s: expected a %s* pin to fail first, got %s" % (what, pin, failed[:1])
