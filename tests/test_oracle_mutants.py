"""Mutation test of the oracle's pins (CPU only).

Every entry of MUTANTS is a plausible one-line mistake in oracle/lst_oracle.c (a dropped tolerance term, a
wrong operand, a missing cut, a broken near-threshold rule).  The test copies the oracle's source to a
scratch directory, applies ONE mistake, compiles it with the oracle's own flags, loads it through a second
instance of oracle/binding.py and runs the named pin (a check function of tests/test_oracle_values.py or a
test of tests/test_oracle_pins.py / test_oracle_dedup.py) on it: the pin must FAIL.  The unmutated copy must
pass every pin.  This is what "pinned" means here: a mistake anywhere in the cut arithmetic fails a named
CPU test.  (Round-1 review: 12 of 20 such mistakes passed the whole CPU suite; they are the first 12 below.)
"""
import importlib.util
import os
import subprocess

import pytest

from . import test_oracle_dedup as D
from . import test_oracle_pins as P
from . import test_oracle_values as V

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
SRC = os.path.join(ROOT, "oracle", "lst_oracle.c")
HDR = os.path.join(ROOT, "oracle", "lst_oracle.h")
BINDING = os.path.join(ROOT, "oracle", "binding.py")

# (name, text to replace (must occur exactly once), replacement, pin that must fail)
MUTANTS = [
    # ---- the 12 that survived the round-1 suite ----
    ("near_thr always 0",
     "return fabsf(v - t) <= p->near_rel * fabsf(t);", "(void)p; (void)v; (void)t; return 0;",
     V.check_md_barrel_thresholds),
    ("LS near also ORs the un-evaluated zv cut",
     "nr |= near_thr(p, kv, p->ls_kappa_max);", "nr |= near_thr(p, kv, p->ls_kappa_max) | near_thr(p, zv, zl);",
     V.check_ls_thresholds),
    ("endcap MD: md_e_slope dropped",
     "* inv_2rmin) * p->md_e_slope) / den", "* inv_2rmin) * 1.0f) / den", V.check_md_endcap_thresholds),
    ("endcap MD: + md_e_tol dropped",
     "/ den + p->md_e_tol);", "/ den);", V.check_md_endcap_thresholds),
    ("endcap MD: z0_max |rb - ra| dropped from rl",
     "float rl = p->z0_max * fabsf(rb - ra) + p->md_z_tol * fabsf(za);", "float rl = p->md_z_tol * fabsf(za);",
     V.check_md_endcap_thresholds),
    ("LS endcap z tolerance uses |zA|/rA",
     "p->ls_z_tol * (1.0f + fabsf(zB) / rB)", "p->ls_z_tol * (1.0f + fabsf(zA) / rA)", V.check_ls_thresholds),
    ("T3 endcap factor removed",
     "tol = e ? tol * (1.0f + fabsf(zC) / rC) : tol;", "tol = e ? tol : tol;", V.check_t3_thresholds),
    ("T3 tol1 * ratio dropped",
     "float tol = p->t3_z_tol0 + p->t3_z_tol1 * ratio;", "float tol = p->t3_z_tol0;", V.check_t3_thresholds),
    ("T5 third cut dropped",
     "if (fabsf(d3) <= tol) acc = 1;", "acc = 1;", V.check_t5_thresholds),
    ("T5 fmaxf(|ki|, |ko|) -> |ki|",
     "fmaxf(fabsf(ki), fabsf(ko))", "fabsf(ki)", V.check_t5_thresholds),
    ("pT tolk: pt_k_tol1 |kp| dropped",
     "float tolk = p->pt_k_tol0 + p->pt_k_tol1 * fabsf(kp);", "float tolk = p->pt_k_tol0;", V.check_pt_thresholds),
    ("pT endcap factor of zt removed",
     "zt[i] = eQ[i] ? p->pt_z_tol * (1.0f + fabsf(zQ) / rQ) : p->pt_z_tol;", "zt[i] = p->pt_z_tol;",
     V.check_pt_thresholds),
    ("dedup rule 2(b): same-seed clause dropped",
     "if (pt5[2 * Z] == pX || share(mX, 3, mZ, 5) >= 2) keep3[X] = 0;", "if (share(mX, 3, mZ, 5) >= 2) keep3[X] = 0;",
     V.check_dedup_rule_2b_isolated),
    # ---- further one-line mistakes, one per term ----
    ("MD barrel: md_b_phi_tol dropped",
     "(ra * inv_2rmin + p->md_b_phi_tol)", "(ra * inv_2rmin)", V.check_md_barrel_thresholds),
    ("MD barrel: zl uses rb",
     "p->z0_max * (rb - ra) + p->md_z_tol * ra;", "p->z0_max * (rb - ra) + p->md_z_tol * rb;",
     V.check_md_barrel_thresholds),
    ("MD barrel: near of the second cut evaluated although the first failed",
     "nr |= near_thr(p, fabsf(crs), lim);\n      if (fabsf(crs) <= lim) {\n        nr |= near_thr(p, zv, zl);",
     "nr |= near_thr(p, fabsf(crs), lim) | near_thr(p, zv, zl);\n      if (fabsf(crs) <= lim) {",
     V.check_md_barrel_thresholds),
    ("MD endcap: den uses + z0_max",
     "float den = fabsf(za) - p->z0_max;", "float den = fabsf(za) + p->z0_max;", V.check_md_endcap_thresholds),
    ("MD endcap: rl uses |zb|",
     "p->md_z_tol * fabsf(za);", "p->md_z_tol * fabsf(zb);", V.check_md_endcap_thresholds),
    ("LS: zl loses z0_max (rho - 1)",
     "float zl = p->z0_max * (rho - 1.0f) + ztol;", "float zl = ztol;", V.check_ls_thresholds),
    ("LS: dB sign",
     "dB = fabsf(sB + half);", "dB = fabsf(sB - half);", V.check_ls_direction_signs),
    ("LS: dA sign",
     "dA = fabsf(sA - half);", "dA = fabsf(sA + half);", V.check_ls_direction_signs),
    ("LS: endcap flag of B ignored in e",
     "int e = eA || eB;", "int e = eA;", V.check_ls_thresholds),
    ("LS: dB cut skipped",
     "okB = dB <= p->ls_dir_tol;", "okB = 1;", V.check_ls_thresholds),
    ("LS: kv scale",
     "float kv = fabsf(kappa) * r_min;", "float kv = fabsf(kappa) * r_min * 0.5f;", V.check_ls_thresholds),
    ("T3: zpred uses inverse ratio",
     "float ratio = len[1] / len[0];", "float ratio = len[0] / len[1];", V.check_t3_thresholds),
    ("T3: endcap factor uses zB",
     "tol * (1.0f + fabsf(zC) / rC)", "tol * (1.0f + fabsf(zB) / rC)", V.check_t3_thresholds),
    ("T3: flag of B ignored",
     "int e = eA || eB || eC;", "int e = eA || eC;", V.check_t3_thresholds),
    ("T5: second cut compares d1 again",
     "nr |= near_thr(p, fabsf(d2), tol);\n      if (fabsf(d2) <= tol) {",
     "nr |= near_thr(p, fabsf(d1), tol);\n      if (fabsf(d1) <= tol) {", V.check_t5_thresholds),
    ("T5: score drops d3",
     "vals[2] = (d1 * d1 + d2 * d2) + d3 * d3;", "vals[2] = (d1 * d1 + d2 * d2);", V.check_t5_thresholds),
    ("pT: gate tolerance dropped",
     "(lw * inv_2rmin + p->pt_gate_tol)", "(lw * inv_2rmin)", V.check_pt_thresholds),
    ("pT: kp sign",
     "float kp = (-q) / (pt * kr);", "float kp = (q) / (pt * kr);", V.check_pt_thresholds),
    ("pT: pT5 base score dropped",
     "score = score + base_score;", "score = score;", V.check_pt_thresholds),
    ("pT: r-z at L uses the flag of A",
     "int eQ[2] = {eA, eL};", "int eQ[2] = {eA, eA};", V.check_pt_thresholds),
    ("pT: second stored curvature not cut on",
     "for (int i = 0; i < n_kt && ok; ++i) {\n          float dk = kx - kt[i];\n          nr |=",
     "for (int i = 0; i < 1 && ok; ++i) {\n          float dk = kx - kt[i];\n          nr |=", V.check_pt_thresholds),
    ("pT: slope without the division by lv",
     "float slope = (z1 - z0) / lv;", "float slope = (z1 - z0);", V.check_pt_thresholds),
    ("dedup rule 3(c) share 2 -> 3",
     "if (share(mX, 5, t3_md + 3 * pt3[2 * Z + 1], 3) >= 2) keepT[X] = 0;",
     "if (share(mX, 5, t3_md + 3 * pt3[2 * Z + 1], 3) >= 3) keepT[X] = 0;", V.check_dedup_rule_2b_isolated),
    ("dedup rule 2(b) looks at removed pT5s too",
     "if (!keep5[Z]) continue;\n      const int* mZ", "const int* mZ", V.check_dedup_rule_2b_isolated),
    ("event loop: near counter not accumulated for MDs",
     "ev->near[ORC_ST_MD] += nr;", "ev->near[ORC_ST_MD] += 0 * nr;", V.check_event_near_counts),
    ("T4: fmaxf(|k1|, |k2|) -> |k1|",
     "float tol = p->t4_tol0 + p->t4_tol1 * fmaxf(fabsf(k1), fabsf(k2));", "float tol = p->t4_tol0 + p->t4_tol1 * fabsf(k1);",
     V.check_t4_thresholds),
    ("T4: relative term dropped",
     "float tol = p->t4_tol0 + p->t4_tol1 * fmaxf(fabsf(k1), fabsf(k2));", "float tol = p->t4_tol0;", V.check_t4_thresholds),
    ("T4: second T3 looked up by its SECOND LS",
     "for (int t = 0; t < n_t3; ++t) t3_of_ls[T3_I(ev, t)[0] + 1]++;", "for (int t = 0; t < n_t3; ++t) t3_of_ls[T3_I(ev, t)[1] + 1]++;",
     V.check_t4_dedup_and_event),
    ("rule 5: share threshold 3 -> 2",
     "if (share(mY, 4, mX, 4) >= 3 && better(md_hits, t4_score[Y], -1, mY, t4_score[X], -1, mX, 4)) keep4[X] = 0;",
     "if (share(mY, 4, mX, 4) >= 2 && better(md_hits, t4_score[Y], -1, mY, t4_score[X], -1, mX, 4)) keep4[X] = 0;",
     V.check_t4_dedup_and_event),
    ("rule 5: removed T5s count too",
     "if (keepT[Z] && share(mX, 4, t5_md + 5 * Z, 5) >= 2) keep4[X] = 0;", "if (share(mX, 4, t5_md + 5 * Z, 5) >= 2) keep4[X] = 0;",
     V.check_t4_dedup_and_event),
    ("rule 5: pT3 clause dropped",
     "if (keep3[Z] && share(mX, 4, t3_md + 3 * pt3[2 * Z + 1], 3) >= 2) keep4[X] = 0;", "(void)keep3;", V.check_t4_dedup_and_event),
    ("T5 MLP: rectifier dropped", "h[j] = fmaxf(a, 0.0f);", "h[j] = a;", V.check_t5_mlp),
    ("T5 MLP: W1 read column-major", "a = a + W1[6 * j + i] * f[i];", "a = a + W1[8 * i + j] * f[i];", V.check_t5_mlp),
    ("T5 MLP: feature kb and ko swapped",
     "float f[6] = {fabsf(ki) * S, fabsf(kb) * S, fabsf(ko) * S,", "float f[6] = {fabsf(ki) * S, fabsf(ko) * S, fabsf(kb) * S,",
     V.check_t5_mlp),
    ("T5 MLP: output bias dropped", "s = p->t5_mlp[64];", "s = 0.0f;", V.check_t5_mlp),
    # ---- the candidate counters of orc_run_event (the denominator of the near-threshold bar, reading N2) ----
    ("n_tests[MD] counts accepted candidates only",
     "ev->n_tests[ORC_ST_MD]++;\n          int acc = orc_md_test(p, endcap, x[a], y[a], z[a], x[b], y[b], z[b], vals, &nr);",
     "int acc = orc_md_test(p, endcap, x[a], y[a], z[a], x[b], y[b], z[b], vals, &nr);\n          ev->n_tests[ORC_ST_MD] += acc;",
     lambda O: P.test_bruteforce_all_pairs(O, "dense")),
    ("n_tests[LS] counted once per map entry, not per candidate",
     "for (int B = md_first[m2]; B < md_first[m2 + 1]; ++B) {\n          float vals[8];\n          int nr;\n          ev->n_tests[ORC_ST_LS]++;",
     "ev->n_tests[ORC_ST_LS]++;\n        for (int B = md_first[m2]; B < md_first[m2 + 1]; ++B) {\n          float vals[8];\n          int nr;",
     lambda O: P.test_bruteforce_all_pairs(O, "dense")),
    ("n_tests[T3] goes to the LS counter",
     "ev->n_tests[ORC_ST_T3]++;", "ev->n_tests[ORC_ST_LS]++;", lambda O: P.test_bruteforce_all_pairs(O, "dense")),
    ("n_tests[T5] counts the first T3s that have a candidate, not the candidates",
     "ev->n_tests[ORC_ST_T5]++;", "ev->n_tests[ORC_ST_T5] += (t2 == t3_first[C]);",
     lambda O: P.test_bruteforce_all_pairs(O, "dense")),
    ("n_tests[pT3] leaves out the accepted candidates",
     "ev->n[ORC_K_PT3]++;", "ev->n[ORC_K_PT3]++;\n        ev->n_tests[ORC_ST_PT3]--;", lambda O: P.test_bruteforce_all_pairs(O, "dense")),
    ("n_tests[pT5] goes to the pT3 counter",
     "ev->n_tests[ORC_ST_PT5]++;", "ev->n_tests[ORC_ST_PT3]++;", lambda O: P.test_bruteforce_all_pairs(O, "dense")),
    ("g: third coefficient", "t = 0.075f + t;", "t = 0.75f + t;", P.test_g_taylor_coefficients),
    ("kappa3: factor 2", "return (2.0f * crs) / ((lpq * lqs) * lps);", "return (1.0f * crs) / ((lpq * lqs) * lps);",
     lambda O: P.test_kappa3_is_textbook_circumradius(O, 100.0, True)),
    ("dedup: T5 share threshold 3 -> 2",
     "if (share(mY, 5, mX, 5) >= 3 && better(md_hits, t5_score[Y], -1, mY, t5_score[X], -1, mX, 5))",
     "if (share(mY, 5, mX, 5) >= 2 && better(md_hits, t5_score[Y], -1, mY, t5_score[X], -1, mX, 5))",
     D.test_t5_pair_sharing_three_mds_keeps_lower_score),
]


def _build_variant(tmp_path, name, old, new):
    src = open(SRC).read()
    if old is not None:
        assert src.count(old) == 1, f"mutant '{name}': the text to replace occurs {src.count(old)} times"
        src = src.replace(old, new)
    d = tmp_path / ("m_" + "".join(c if c.isalnum() else "_" for c in name)[:60])
    d.mkdir()
    (d / "lst_oracle.c").write_text(src)
    (d / "lst_oracle.h").write_text(open(HDR).read())
    so = str(d / "liblst_oracle_variant.so")
    subprocess.run(["gcc", "-O2", "-ffp-contract=off", "-fno-fast-math", "-std=c99", "-shared", "-fPIC", "-o", so,
                    str(d / "lst_oracle.c"), "-lm"], check=True)
    spec = importlib.util.spec_from_file_location("oracle_variant_" + d.name, BINDING)
    mod = importlib.util.module_from_spec(spec)
    spec.loader.exec_module(mod)
    mod.build = lambda force=False: so   # this instance loads the variant library, never the real oracle
    return mod


def test_unmutated_copy_passes_every_pin(tmp_path):
    O = _build_variant(tmp_path, "identity", None, None)
    for check in V.CHECKS:
        check(O)
    for _, _, _, pin in MUTANTS:
        pin(O)


@pytest.mark.parametrize("name,old,new,pin", MUTANTS, ids=[m[0] for m in MUTANTS])
def test_mutant_is_killed(tmp_path, name, old, new, pin):
    O = _build_variant(tmp_path, name, old, new)
    with pytest.raises(AssertionError):
        pin(O)
