"""Canonical forms for comparing object sets independent of internal order (SPEC.md 5):
every object is expanded to its tuple of ORIGINAL hit indices and rows are sorted
lexicographically.  Pure index bookkeeping, shared by oracle-vs-oracle and GPU-vs-oracle tests."""
import numpy as np


def lexsort_rows(a):
    a = np.asarray(a)
    if a.shape[0] == 0:
        return a, np.zeros(0, dtype=np.int64)
    order = np.lexsort(a.T[::-1])
    return a[order], order


def md_tuples(md_hits):
    return np.asarray(md_hits, dtype=np.int64).reshape(-1, 2)


def ls_tuples(md_hits, ls):
    md = md_tuples(md_hits)
    ls = np.asarray(ls).reshape(-1, 2)
    return np.concatenate([md[ls[:, 0]], md[ls[:, 1]]], axis=1) if len(ls) else np.zeros((0, 4), np.int64)


def t3_tuples(md_hits, t3_md):
    md = md_tuples(md_hits)
    t = np.asarray(t3_md).reshape(-1, 3)
    return np.concatenate([md[t[:, i]] for i in range(3)], axis=1) if len(t) else np.zeros((0, 6), np.int64)


def t5_tuples(md_hits, t5_md):
    md = md_tuples(md_hits)
    t = np.asarray(t5_md).reshape(-1, 5)
    return np.concatenate([md[t[:, i]] for i in range(5)], axis=1) if len(t) else np.zeros((0, 10), np.int64)


def tc_tuples(md_hits, t3_md, t5_md_of_t5list, tc):
    """TC rows -> (type, pls, 10 hit indices padded with -1)."""
    tc = np.asarray(tc).reshape(-1, 3)
    out = -np.ones((len(tc), 12), dtype=np.int64)
    t5h = t5_tuples(md_hits, t5_md_of_t5list)
    t3h = t3_tuples(md_hits, t3_md)
    for i, (ty, p, o) in enumerate(tc):
        out[i, 0], out[i, 1] = ty, p
        if ty in (0, 1):
            out[i, 2:12] = t5h[o]
        elif ty == 2:
            out[i, 2:8] = t3h[o]
    return out


def same_set(a, b):
    a, _ = lexsort_rows(a)
    b, _ = lexsort_rows(b)
    return a.shape == b.shape and bool(np.array_equal(a, b))
