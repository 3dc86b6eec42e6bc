"""GPU-vs-oracle comparison used by the `-m gpu` tests and __graft_entry__.smoke().
Bars (SPEC.md 5 / BASELINE.json north_star): index tuples and cut payloads bit-exact, features 1e-6
relative (+1e-7), scores 1e-5 absolute, |score - 0.5| <= 1e-5 excluded from pass/fail."""
import numpy as np
import canon
from oracle import lst_oracle as O

FEAT_RTOL, FEAT_ATOL, SCORE_ATOL = 1e-6, 1e-7, 1e-5


def f32(a):
    return np.asarray(a, dtype=np.float64).astype(np.float32)


def bits_equal(a, b):
    """Same fp32 bit patterns, except that a NaN equals any NaN: IEEE 754 leaves the sign and payload of a GENERATED NaN to the
    implementation (x86 produces 0xFFC00000, the GPU 0x7FFFFFFF).  Only reachable with non-finite input coordinates (an upper hit
    at x = inf gives c_md = inf / inf by SPEC.md 4.1 on both sides); every finite value, +-0 and +-inf must still match bit for bit."""
    a = np.ascontiguousarray(a, dtype=np.float32).ravel(); b = np.ascontiguousarray(b, dtype=np.float32).ravel()
    if a.shape != b.shape:
        return False
    both_nan = np.isnan(a) & np.isnan(b)
    return bool(np.array_equal(a.view(np.uint32)[~both_nan], b.view(np.uint32)[~both_nan]))


def compare(geo, weights, ev, gpu, check_order=True, dnn=(23, 2)):
    """`gpu` = LST.fetch(slot) dict.  Returns a dict of counts; raises AssertionError on any mismatch."""
    r = O.run(geo, weights, ev, dnn=dnn)
    g = gpu
    assert g["status"] == r.flags, (g["status"], r.flags)
    # a0
    assert np.array_equal(g["hit"]["orig"], r.hit_orig)
    # MD
    assert canon.same_set(g["md"]["hits"], r.md_hits), "MD sets differ"
    if check_order:
        assert np.array_equal(g["md"]["hits"], r.md_hits)
        assert np.array_equal(g["md"]["modt"] >> 2, r.md_mod)
        assert bits_equal(g["md"]["cw"], r.md_real[:, :2]), "c_md / w_md not bit-exact"
        assert bits_equal(g["md"]["anchor"], r.md_real[:, 2:6])
    # LS
    assert canon.same_set(canon.ls_tuples(g["md"]["hits"], g["ls"]["ab"]), canon.ls_tuples(r.md_hits, r.ls)), "LS sets differ"
    assert np.array_equal(g["ls"]["ab"], r.ls) and bits_equal(g["ls"]["c"], r.ls_c)
    # T3
    assert canon.same_set(canon.t3_tuples(g["md"]["hits"], g["t3"]["abc"][:, :3]), canon.t3_tuples(r.md_hits, r.t3[:, :3])), "T3 sets differ"
    assert np.array_equal(g["t3"]["abc"][:, :3], r.t3[:, :3]) and np.array_equal(g["t3"]["abc"][:, 3], r.t3[:, 3])
    assert np.array_equal(g["t3"]["l1"], r.t3[:, 4]) and bits_equal(g["t3"]["k"], r.t3_k)
    # T5 candidates
    assert canon.same_set(canon.t5_tuples(g["md"]["hits"], g["t5c"]["md"]), canon.t5_tuples(r.md_hits, r.t5c[:, :5])), "T5 candidate sets differ"
    assert np.array_equal(g["t5c"]["md"], r.t5c[:, :5]) and np.array_equal(g["t5c"]["t3"], r.t5c[:, 5:7])
    assert bits_equal(g["t5c"]["curv"], r.t5c_curv)
    n5c = len(r.t5c)
    n_border = n_flip = 0
    if n5c:
        fa, fb = g["t5c"]["feat"].astype(np.float64), r.t5c_feat
        tol = FEAT_RTOL * np.maximum(np.abs(fa), np.abs(fb)) + FEAT_ATOL
        assert np.all(np.abs(fa - fb) <= tol), f"features off by {np.max(np.abs(fa - fb) - tol)}"
        ds = np.abs(g["t5c"]["score"].astype(np.float64) - r.t5c_score)
        assert ds.max() <= SCORE_ATOL, f"score off by {ds.max()}"
        border = np.abs(r.t5c_score - 0.5) <= SCORE_ATOL
        n_border = int(border.sum())
        gp, op = g["t5c"]["pass"].astype(np.int8), r.t5c[:, 7].astype(np.int8)
        assert np.array_equal(gp[~border], op[~border]), "DNN decisions differ away from the threshold"
        flip = border & (gp != op)
        n_flip = int(flip.sum())
        if n_flip:   # replay the oracle with the GPU's decision on the borderline candidates only
            ov = -np.ones(n5c, np.int8); ov[flip] = gp[flip]
            r = O.run(geo, weights, ev, t5_override=ov, dnn=dnn)
    # T5 list, matching, TC
    assert np.array_equal(g["t5"]["cand"], r.t5)
    assert np.array_equal(g["match5"]["best5_pls"], r.best5_pls)
    m = r.best5_pls >= 0
    assert bits_equal(g["match5"]["chi2"][m], r.chi5[m]), "chi2 not bit-exact"
    assert np.array_equal(g["tc"]["tc"].reshape(-1, 3), r.tc), "TC lists differ"
    ta = canon.tc_tuples(g["md"]["hits"], g["t3"]["abc"][:, :3], g["t5c"]["md"][g["t5"]["cand"]], g["tc"]["tc"].reshape(-1, 3))
    tb = canon.tc_tuples(r.md_hits, r.t3[:, :3], r.t5c[r.t5][:, :5], r.tc)
    assert canon.same_set(ta, tb)
    # f1: hit tuples and rank chi2 of every candidate, keep flags, cleaned list (SPEC.md 4.7)
    assert np.array_equal(g["tcx"]["hits"].reshape(-1, 12)[:, :10], r.tc_hits), "TC hit tuples differ"
    assert np.array_equal(g["tcx"]["q"].view(np.uint32), r.tc_q), "rank chi2 not bit-exact"
    assert np.array_equal(g["tcx"]["keep"], r.tc_keep), "duplicate-cleaning flags differ"
    assert np.array_equal(g["tcc"]["tc"].reshape(-1, 3), r.tcc), "cleaned TC lists differ"
    assert g["counts"]["tcc"] == len(r.tcc)
    c = g["counts"]
    for k in ("md", "ls", "t3", "t5c", "t5", "tc"):
        assert c[k] == r.counts[k], (k, c[k], r.counts[k])
    tcb = np.bincount(r.tc[:, 0], minlength=4) if len(r.tc) else np.zeros(4, int)
    assert [c["pt5"], c["t5tc"], c["pt3"], c["plstc"]] == tcb.tolist()
    out = dict(r.counts); out.update(border=n_border, flips=n_flip, tcc=len(r.tcc))
    return out


def compare_graph(geo, weights, ev, g):
    """`g` = LST.fetch_graph(slot): the exported MD / LS graph against the oracle's (SPEC.md 4.8)."""
    r = O.run(geo, weights, ev, last_stage="ls")
    o = r.graph
    assert np.array_equal(g["rowptr"], o["rowptr"]) and np.array_equal(g["col"], o["col"]) and np.array_equal(g["node_hits"], o["node_hits"])
    assert bits_equal(g["edge_c"], o["edge_c"])
    assert bits_equal(g["node_feat"][:, :4], o["node_feat"][:, :4]) and bits_equal(g["node_feat"][:, 6:], o["node_feat"][:, 6:])
    a, b = g["node_feat"][:, 4:6].astype(np.float64), o["node_feat"][:, 4:6]
    assert np.all(np.abs(a - b) <= FEAT_RTOL * np.maximum(np.abs(a), np.abs(b)) + FEAT_ATOL)
    return len(o["col"])
