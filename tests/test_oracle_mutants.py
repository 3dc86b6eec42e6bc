"""Mutation check of the oracle pins.  CPU only.

A pin is only worth something if a plausible mistake in oracle/lst_oracle.cpp makes it fail.  This test builds
deliberately broken copies of the oracle (one textual mutation each: a dropped tolerance term, a deleted condition,
a changed coefficient, a wrong index, a flipped tie rule), routes the pins of tests/test_oracle_terms.py and
tests/test_oracle_pins.py through each copy, and requires that at least one of the named pins FAILS.  The unmutated
source must pass the same pins (that is what the ordinary tests check).

The mutant libraries are compiled into a temporary directory; nothing here is used by any other test.
"""
import os
import subprocess
import tempfile
from concurrent.futures import ThreadPoolExecutor

import pytest

from oracle import lst_oracle as O
import test_oracle_terms as T
import test_oracle_order as TO

SRC = open(os.path.join(os.path.dirname(O.__file__), "lst_oracle.cpp")).read()

# (name, text in the source, replacement, pins expected to notice; "geo"/"barrel" = which geometry fixture the pin takes)
MUTANTS = [
    # ---- ls_eval
    ("L2 without A.dr*|B.z|", "rhs = rhs + A.dr * rabs(B.z);", "", [("pin_ls_L2_terms", None)]),
    ("L2 without B.dr*|A.z|", "rhs = rhs + B.dr * rabs(A.z);", "", [("pin_ls_L2_terms", None)]),
    ("L2 without A.dz*sB", "rhs = rhs + A.dz * sB;", "", [("pin_ls_L2_terms", None)]),
    ("L2 without B.dz*sA", "rhs = rhs + B.dz * sA;", "", [("pin_ls_L2_terms", None)]),
    ("L2 A.dz*sA instead of A.dz*sB", "rhs = rhs + A.dz * sB;", "rhs = rhs + A.dz * sA;", [("pin_ls_L2_terms", None)]),
    ("L2 A.dr*|A.z| instead of A.dr*|B.z|", "rhs = rhs + A.dr * rabs(B.z);", "rhs = rhs + A.dr * rabs(A.z);", [("pin_ls_L2_terms", None)]),
    ("L2 with radii instead of arc lengths", "const R sA = A.r * arcfac<R>(ta * ta);\n  const R sB = B.r * arcfac<R>(tb * tb);",
     "const R sA = A.r;\n  const R sB = B.r;", [("pin_ls_L2_uses_arc_length", None)]),
    ("L3 outer-MD test deleted", "if (!(rabs(B.c - c) <= (B.w + B.f * ac) * lo.f[CUT_L3])) return false;", "", [("pin_ls_curvature_L1_L3", None)]),
    ("L3 inner-MD test deleted", "if (!(rabs(A.c - c) <= (A.w + A.f * ac) * lo.f[CUT_L3])) return false;", "", [("pin_ls_curvature_L1_L3", None)]),
    ("L3 inner without f*|c|", "(A.w + A.f * ac)", "(A.w)", [("pin_ls_curvature_L1_L3", None)]),
    ("L3 outer without f*|c|", "(B.w + B.f * ac)", "(B.w)", [("pin_ls_curvature_L1_L3", None)]),
    ("c_ls sign", "const R c = (R(-2.0f) * cr) / ((A.r * B.r) * d);", "const R c = (R(2.0f) * cr) / ((A.r * B.r) * d);", [("pin_ls_curvature_L1_L3", None)]),
    # ---- triplet_eval / t3_eval
    ("T2 without (B.dr+C.dr)*|zab|", "rhs = rhs + (B.dr + C.dr) * rabs(zab);", "", [("pin_triplet_T2_terms", None)]),
    ("T2 without (A.dr+B.dr)*|zbc|", "rhs = rhs + (A.dr + B.dr) * rabs(zbc);", "", [("pin_triplet_T2_terms", None)]),
    ("T2 first term zeroed", "R rhs = (A.dz + B.dz) * sbc;", "R rhs = R(0.0f);", [("pin_triplet_T2_terms", None)]),
    ("T2 without (B.dz+C.dz)*sab", "rhs = rhs + (B.dz + C.dz) * sab;", "", [("pin_triplet_T2_terms", None)]),
    ("T2 without 0.05*(sab+sbc)", "rhs = rhs + R(0.05f) * (sab + sbc);", "", [("pin_triplet_T2_terms", None)]),
    ("T2 (B.dz+C.dz)*sbc", "rhs = rhs + (B.dz + C.dz) * sab;", "rhs = rhs + (B.dz + C.dz) * sbc;", [("pin_triplet_T2_terms", None)]),
    ("second T3 condition deleted", "if (!(rabs(c_bc - k) <= R(C_TOL3_F) * lo.f[CUT_T3])) return false;", "", [("pin_t3_curvature_consistency", None)]),
    ("first T3 condition deleted", "if (!(rabs(c_ab - k) <= R(C_TOL3_F) * lo.f[CUT_T3])) return false;                 // T3", "", [("pin_t3_curvature_consistency", None)]),
    # ---- md_eval
    ("endcap M2 factor 0.15 -> 0.05", "R(0.15f) * Ls", "R(0.05f) * Ls", [("pin_md_endcap_terms", None)]),
    ("endcap M3 factor 1.3 -> 1.0", "R(1.3f) * Ls * S", "R(1.0f) * Ls * S", [("pin_md_endcap_terms", None)]),
    ("endcap f 0.3 -> 0", "f = R(0.3f);", "f = R(0.0f);", [("pin_md_endcap_terms", None)]),
    ("barrel M2 without the Z0 term", "const R rhs2 = drho * R(Z0_MAX_F) / r1 + l2tol;", "const R rhs2 = l2tol;", [("pin_md_barrel_terms", None)]),
    ("barrel M1 deleted", "if (!(drho > R(0.0f))) return false;", "", [("pin_md_barrel_terms", None)]),
    # ---- pls_anchor
    ("dZ without dr*|cot|", "R dZ = m.dz + m.dr * rabs(p.cot);", "R dZ = m.dz;", [("pin_pls_longitudinal_terms", None)]),
    ("dZ without 0.003*s*sec", "dZ = dZ + R(0.003f) * (s * p.sec);", "", [("pin_pls_longitudinal_terms", None)]),
    ("dZ without 0.05", "dZ = dZ + R(0.05f);", "", [("pin_pls_longitudinal_terms", None)]),
    ("dZ with s instead of s*sec", "dZ = dZ + R(0.003f) * (s * p.sec);", "dZ = dZ + R(0.003f) * s;", [("pin_pls_longitudinal_terms", None)]),
    ("z prediction with r instead of s", "const R s = m.r * arcfac<R>(t * t);", "const R s = m.r;", [("pin_pls_longitudinal_terms", None)]),
    ("dT without the curvature term", "dT = dT + R(0.03f) * (r2 * p.h);", "", [("pin_pls_transverse_terms", None)]),
    ("dT without 0.02", "dT = dT + R(0.02f);", "", [("pin_pls_transverse_terms", None)]),
    ("chi2 without the z term", "*chi2 = *chi2 + b * b;", "", [("pin_pls_chi2_golden", None)]),
    ("chi2 without the transverse term", "*chi2 = *chi2 + a * a;", "", [("pin_pls_chi2_golden", None)]),
    # ---- run_chain
    ("a1: endcap MDs given dz = DL as well", "d.dz = subdet[m] == 0 ? R(DL_F[mtype[m]]) : R(0.0f);", "d.dz = R(DL_F[mtype[m]]);",
     [("pin_chain_anchor_tolerances_endcap", "geo")]),
    ("a1: endcap MDs given dr = 0", "d.dr = subdet[m] == 0 ? R(0.0f) : R(DL_F[mtype[m]]);", "d.dr = R(0.0f);",
     [("pin_chain_anchor_tolerances_endcap", "geo")]),
    ("a1: barrel MDs given dr = DL as well", "d.dr = subdet[m] == 0 ? R(0.0f) : R(DL_F[mtype[m]]);", "d.dr = R(DL_F[mtype[m]]);",
     [("pin_chain_anchor_tolerances_barrel", "geo")]),
    ("a4: bridge evaluated on (a,c,d)", "triplet_eval<R>(res->md[u.b], res->md[u.c], res->md[v.b], lo.f[CUT_Q1]", "triplet_eval<R>(res->md[u.a], res->md[u.c], res->md[v.b], lo.f[CUT_Q1]",
     [("pin_chain_t5_curvature_indices", "geo")]),
    ("a6: best5 tie rule < -> <=", "if (res->best5_pls[t] < 0 || chi < chi5[t])", "if (res->best5_pls[t] < 0 || chi <= chi5[t])", [("pin_tc_tie_rules", "barrel")]),
    ("a6: best3 tie rule < -> <=", "if (best3[x] < 0 || chi < chi3[x])", "if (best3[x] < 0 || chi <= chi3[x])", [("pin_tc_tie_rules", "barrel")]),
    ("a6: win5 tie rule < -> <=", "chi5[t] < chi5[win5[p]]", "chi5[t] <= chi5[win5[p]]", [("pin_tc_tie_rules", "barrel")]),
    ("a6: win3 tie rule < -> <=", "chi3[x] < chi3[win3[p]]", "chi3[x] <= chi3[win3[p]]", [("pin_tc_tie_rules", "barrel")]),
    ("a6: T3 used with 2 of 3 MDs", "if (found == 3) t3_used[x] = 1;", "if (found >= 2) t3_used[x] = 1;", [("pin_tc_used_and_free_rules", "barrel")]),
    ("a6: pT3 pass not skipping pLS that own a pT5", "      if (win5[p] >= 0) continue;\n      R chi = R(0.0f);", "      R chi = R(0.0f);", [("pin_tc_used_and_free_rules", "barrel")]),
    ("a6: T3-used test never fires", "if (found == 3) t3_used[x] = 1;", "", [("pin_tc_used_and_free_rules", "barrel")]),
    # ---- f1 duplicate cleaning
    ("f1: more than half -> at least half", "if (2 * shared > nh[x]) keep[x] = 0;", "if (2 * shared >= nh[x]) keep[x] = 0;", [("pin_clean_rule_by_hand", None)]),
    ("f1: fraction of Y's hits instead of X's", "if (2 * shared > nh[x]) keep[x] = 0;", "if (2 * shared > nh[y]) keep[x] = 0;", [("pin_clean_rule_by_hand", None)]),
    ("f1: rank ignores the type", "  if (y.type != x.type) return y.type < x.type;\n", "", [("pin_clean_rule_by_hand", None)]),
    ("f1: rank ignores chi2", "  if (qy != qx) return qy < qx;\n", "", [("pin_clean_rule_by_hand", None)]),
    ("f1: chi2 order reversed", "  if (qy != qx) return qy < qx;", "  if (qy != qx) return qy > qx;", [("pin_clean_rule_by_hand", None)]),
    ("f1: ties to the later row", "  return iy < ix;", "  return iy > ix;", [("pin_clean_rule_by_hand", None)]),
    ("f1: greedy (dropped candidates no longer drop others)", "        if (y == x || !better_rank(tc[y], q[y], y, tc[x], q[x], x)) continue;",
     "        if (y == x || !keep[y] || !better_rank(tc[y], q[y], y, tc[x], q[x], x)) continue;", [("pin_clean_rule_by_hand", None)]),
    ("f1: pT3 ranked with the T5's chi2", "      if (c.type == 2) chi = res->chi3[c.obj];", "      if (c.type == 2) chi = res->chi5[0];", [("pin_clean_all_pairs", "geo")]),
    ("f3: hidden layers beyond the first skipped", "  for (int l = 1; l < n_hidden; ++l) {", "  for (int l = 1; l < 1; ++l) {", [("pin_dnn_variants", "geo")]),
    ("f3: 38 features: anchor order a,b,c,d,e,e", "const int order[6] = {0, 1, 2, 2, 3, 4};", "const int order[6] = {0, 1, 2, 3, 4, 4};", [("pin_dnn_variants", "geo")]),
    ("f3: 38 features: layer not fed", "x[4 + 5 * i + 4] = float(layer[q]) * 0.1f;", "x[4 + 5 * i + 4] = 0.0f;", [("pin_dnn_variants", "geo")]),
    ("f3: 38 features: T5 pT from c_in only", "const float c5 = 0.5f * (cin + cout);", "const float c5 = cin;", [("pin_dnn_variants", "geo")]),
    # ---- build order of the lists (SPEC.md 4.0-4.5 "Order" clauses) and the two branches no config event reaches
    ("a0: hits of a sensor in reverse arrival order", "res->hit_orig[cur[key[i]]++] = i;",
     "res->hit_orig[res->sensor_start[key[i] + 1] - 1 - (cur[key[i]]++ - res->sensor_start[key[i]])] = i;", [("pin_build_order", "geo")]),
    ("a1: upper hit outer loop, lower hit inner", "    for (int32_t i = ss[2 * m]; i < ss[2 * m + 1]; ++i) {\n      for (int32_t j = ss[2 * m + 1]; j < ss[2 * m + 2]; ++j) {",
     "    for (int32_t j = ss[2 * m + 1]; j < ss[2 * m + 2]; ++j) {\n      for (int32_t i = ss[2 * m]; i < ss[2 * m + 1]; ++i) {", [("pin_build_order", "geo")]),
    ("a2: CSR row walked last column first", "for (int32_t e = rowptr[m]; e < rowptr[m + 1]; ++e) {", "for (int32_t e = rowptr[m + 1] - 1; e >= rowptr[m]; --e) {", [("pin_build_order", "geo")]),
    ("a3: partner LS loop descending", "for (int32_t l1 = res->ls_start[s0.b]; l1 < res->ls_start[s0.b + 1]; ++l1) {",
     "for (int32_t l1 = res->ls_start[s0.b + 1] - 1; l1 >= res->ls_start[s0.b]; --l1) {", [("pin_build_order", "geo")]),
    ("a4: partner T3 loop descending", "for (int32_t i1 = res->t3_start[u.c]; i1 < res->t3_start[u.c + 1]; ++i1) {",
     "for (int32_t i1 = res->t3_start[u.c + 1] - 1; i1 >= res->t3_start[u.c]; --i1) {", [("pin_build_order", "geo")]),
    ("radius feature clamped at 1e4", "const float rad = std::fmin(1.0f / ac, 1.0e5f);   // c = 0 -> +inf -> clamped",
     "const float rad = std::fmin(1.0f / ac, 1.0e4f);", [("pin_radius_clamp", None)]),
    ("pT feature clamped at 1e4", "  const float rad = std::fmin(1.0f / ac, 1.0e5f);\n  return std::log10(KAPPA_F * rad);",
     "  const float rad = std::fmin(1.0f / ac, 1.0e4f);\n  return std::log10(KAPPA_F * rad);", [("pin_radius_clamp", None)]),
    ("md_eval: S without the cap at 1", "const R S = std::fmin(R(1.0f), r2 * R(C_HALF_F));", "const R S = r2 * R(C_HALF_F);", [("pin_md_sagitta_cap", None)]),
    ("a6: T5 match accepts a chi2 that is not a number", "      if (!ok || !chi2_is_a_number<R>(chi)) continue;   // T5 match", "      if (!ok) continue;", [("pin_match_needs_a_chi2_that_is_a_number", "geo")]),
    ("a6: T3 match accepts a chi2 that is not a number", "      if (!ok || !chi2_is_a_number<R>(chi)) continue;   // T3 match", "      if (!ok) continue;", [("pin_match_needs_a_chi2_that_is_a_number", "geo")]),
    ("f1: upper hits left out of the tuples", "hits[10 * i + 2 * k + 1] = ho[res->md[mds[k]].hit_up];", "hits[10 * i + 2 * k + 1] = ho[res->md[mds[k]].hit_lo];", [("pin_clean_all_pairs", "geo")]),
]


def _build(i, workdir):
    name, old, new, _ = MUTANTS[i]
    assert SRC.count(old) == 1, f"mutation '{name}' does not apply exactly once (the source moved on: update MUTANTS)"
    src = os.path.join(workdir, f"m{i}.cpp")
    lib = os.path.join(workdir, f"m{i}.so")
    with open(src, "w") as f:
        f.write(SRC.replace(old, new))
    subprocess.check_call(["g++", "-O1", "-std=c++17", "-ffp-contract=off", "-fno-fast-math", "-shared", "-fPIC", "-o", lib, src])
    return lib


@pytest.fixture(scope="module")
def mutant_libs():
    with tempfile.TemporaryDirectory() as d:
        with ThreadPoolExecutor(max_workers=os.cpu_count() or 4) as ex:
            libs = list(ex.map(lambda i: _build(i, d), range(len(MUTANTS))))
        yield libs


def _endcap_eff_pin(geo):
    e_ls, e_t3 = T.pin_smeared_endcap_efficiency(geo)
    assert e_ls >= T.ENDCAP_EFF_LS and e_t3 >= T.ENDCAP_EFF_T3, (e_ls, e_t3)


def test_every_mutant_is_noticed(mutant_libs, geo_full, geo_barrel):
    survivors = []
    for (name, _, _, pins), lib in zip(MUTANTS, mutant_libs):
        killed = False
        with O.use_library(lib):
            for pin, fixture in pins:
                fn = getattr(T, pin, None) or getattr(TO, pin)
                try:
                    fn() if fixture is None else fn(geo_full if fixture == "geo" else geo_barrel)
                except AssertionError:
                    killed = True
                    break
        if not killed:
            survivors.append(name)
    assert not survivors, f"mutants that no pin noticed: {survivors}"


def test_endcap_efficiency_notices_dropped_dr_terms(mutant_libs, geo_full):
    """per-cut truth efficiency on smeared forward tracks: dropping the delta-r terms must crater it"""
    idx = [i for i, m in enumerate(MUTANTS) if m[0] in ("L2 without B.dr*|A.z|", "T2 without (B.dr+C.dr)*|zab|", "a1: endcap MDs given dr = 0")]
    assert len(idx) == 3
    for i in idx:
        with O.use_library(mutant_libs[i]):
            with pytest.raises(AssertionError):
                _endcap_eff_pin(geo_full)
    _endcap_eff_pin(geo_full)        # and the real oracle passes
