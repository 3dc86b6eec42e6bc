"""Pins for the BUILD ORDER of the oracle's lists, and for two branches no event of the configs reaches.  CPU only.

PAPER.md:45-60 (Table 1) fixes only the sequence of the steps; the order of the objects inside each list is a SPEC.md
reading (4.0 "stable", 4.1 "Order: (m, i, j)", 4.2 "row order", 4.3 / 4.4 "Order (l0, l1)" / "(u, v)").  That order is
load-bearing: capacity overflow keeps "the first cap objects in build order", the duplicate cleaning ranks T5s by row,
and the pLS winners break ties on the object index.  The set comparisons of the other pin files cannot see it, so the
checks here are written from the "Order" clauses with numpy only -- no oracle predicate, none of the oracle's own
range tables as input -- on an event in which 3000 hits appear twice (same position and sensor, different original
index), so that the stable sort of 4.0 decides which copy comes first in every later list.
"""
import dataclasses

import numpy as np

from lstgen import config_event, xavier_weights
from oracle import lst_oracle as O
import test_oracle_terms as T

N_DUP = 3000


def _event_with_duplicated_hits(geo):
    ev = config_event(geo, 1)                         # PU50
    cat = lambda a: np.concatenate([a, a[:N_DUP]])
    return dataclasses.replace(ev, x=cat(ev.x), y=cat(ev.y), z=cat(ev.z), key=cat(ev.key), hit_particle=cat(ev.hit_particle))


def _strictly_increasing(*cols):
    """rows of the table with these columns are strictly increasing in lexicographic order"""
    t = np.stack([np.asarray(c, dtype=np.int64) for c in cols], axis=1)
    d = t[1:] - t[:-1]
    first = np.argmax(d != 0, axis=1)                  # first column that differs (0 if none does)
    lead = d[np.arange(len(d)), first]
    return bool((lead > 0).all())


def pin_build_order(geo):
    ev = _event_with_duplicated_hits(geo)
    n_orig = ev.n_hits - N_DUP
    r = O.run(geo, xavier_weights(2), ev)
    M = int(geo.n_modules)
    key = ev.key.astype(np.int64)
    rowptr, col = np.asarray(geo.conn_rowptr, np.int64), np.asarray(geo.conn_col, np.int64)

    # 4.0: hit_orig is THE stable sort of the in-range keys (ties in a sensor stay in arrival order)
    inr = np.flatnonzero(key < 2 * M)
    expect = inr[np.argsort(key[inr], kind="stable")]
    assert np.array_equal(r.hit_orig, expect)
    assert np.array_equal(r.sensor_start, np.searchsorted(key[expect], np.arange(2 * M + 1)))
    pos = np.full(ev.n_hits, -1, np.int64)
    pos[expect] = np.arange(expect.size)               # sorted position of every original hit, from numpy's sort

    # 4.1: MD rows strictly increasing in (module, sorted position of the lower hit, of the upper hit)
    lo, up, mod = r.md_hits[:, 0], r.md_hits[:, 1], r.md_mod.astype(np.int64)
    assert np.array_equal(key[lo], 2 * mod) and np.array_equal(key[up], 2 * mod + 1)
    assert _strictly_increasing(mod, pos[lo], pos[up])
    # the duplicated hits really decide something: MDs built on a copy exist, and a copy always follows its original
    assert (lo >= n_orig).sum() > 200 and (up >= n_orig).sum() > 200
    assert (pos[n_orig:] > pos[:N_DUP]).all()
    n_md = len(mod)
    # within a module the lower hit is the outer loop: some module must hold MDs of >= 2 lower hits with upper hits not in step
    same = mod[1:] == mod[:-1]
    assert (same & (pos[lo][1:] > pos[lo][:-1]) & (pos[up][1:] < pos[up][:-1])).any()

    # 4.2: LS rows strictly increasing in (a, rank of module(b) in the CSR row of module(a), b); ls_start = first row per a
    a, b = r.ls[:, 0].astype(np.int64), r.ls[:, 1].astype(np.int64)
    rank = np.empty(len(a), np.int64)
    for i in range(len(a)):
        row = col[rowptr[mod[a[i]]]:rowptr[mod[a[i]] + 1]]
        hit = np.flatnonzero(row == mod[b[i]])
        assert hit.size == 1                           # an LS only joins CSR-connected modules
        rank[i] = hit[0]
    assert _strictly_increasing(a, rank, b)
    assert ((a[1:] == a[:-1]) & (rank[1:] > rank[:-1])).sum() > 100      # rows really span several columns
    assert np.array_equal(r.graph["rowptr"], np.searchsorted(a, np.arange(n_md + 1)))

    # 4.3: T3 rows strictly increasing in (first LS, second LS); the MDs are those of the two LSs sharing the middle MD
    l0, l1 = r.t3[:, 3].astype(np.int64), r.t3[:, 4].astype(np.int64)
    assert _strictly_increasing(l0, l1)
    assert ((l0[1:] == l0[:-1])).sum() > 50
    assert np.array_equal(r.t3[:, 0], a[l0]) and np.array_equal(r.t3[:, 1], b[l0])
    assert np.array_equal(r.t3[:, 1], a[l1]) and np.array_equal(r.t3[:, 2], b[l1])

    # 4.4 / 4.5: T5-candidate rows strictly increasing in (inner T3, outer T3); the T5 list = passing candidates ascending
    u, v = r.t5c[:, 5].astype(np.int64), r.t5c[:, 6].astype(np.int64)
    assert _strictly_increasing(u, v)
    assert ((u[1:] == u[:-1])).sum() > 20
    assert np.array_equal(r.t3[u, 2], r.t3[v, 0])
    assert np.array_equal(r.t5c[:, :5], np.stack([r.t3[u, 0], r.t3[u, 1], r.t3[u, 2], r.t3[v, 1], r.t3[v, 2]], axis=1))
    assert np.array_equal(r.t5, np.flatnonzero(r.t5c[:, 7]))
    assert 0 < len(r.t5) < len(u)


def pin_radius_clamp():
    """SPEC.md 4.5: x[20..22] = log10f(fminf(1/|c|, 1e5)).  c = 0 gives 1/|c| = +inf, clamped to 1e5: the feature is exactly 5;
    c = 1e-6 (radius 1e6 cm, beyond the clamp) gives 5 as well; c = 2e-5 (radius 5e4 cm, inside) gives log10(5e4)."""
    ax, ay, az, ar = [np.array([30., 40., 50., 60., 70.], np.float32)] + [np.zeros(5, np.float32)] * 2 + [np.array([30., 40., 50., 60., 70.], np.float32)]
    x = O.features(ax, ay, az, ar, 0.0, 1.0e-6, 2.0e-5)
    assert x[20] == np.float32(5.0) and x[21] == np.float32(5.0)
    assert abs(float(x[22]) - np.log10(5.0e4)) < 1e-6
    x38 = O.features38(ax, ay, az, ar, np.arange(1, 6), 0.0, -1.0e-6, 2.0e-5)
    assert x38[1] == np.float32(5.0) and x38[37] == np.float32(5.0)                 # radius of the inner T3, bridge radius
    assert abs(float(x38[0]) - np.log10(0.0114 * 1.0e5)) < 1e-6                     # pT of the inner T3 at the clamp


def pin_md_sagitta_cap():
    """SPEC.md 4.1: S = fmin(1, r2 * C_HALF), the sine of the largest bend angle at radius r2; it saturates at r2 = 1 / 0.007125 =
    140.35 cm, beyond every module of the configs, so only a hand-made pair reaches the branch.  Endcap PS pair: lower hit
    (150, 0, 200), upper hit (150.3, y2, 200.4): Ls = 0.4 * 150 / 200 = 0.3, drho = 0.3 (M2 holds), dt = y2, r2 * C_HALF = 1.071.
    M3 with the cap: |dt| <= 1.3 * 0.3 * 1 + 0.01225 = 0.40225; without it the bound would be 1.3 * 0.3 * 1.071 + 0.01225 = 0.4299."""
    h1 = (150.0, 0.0, 200.0)
    ok_in, _ = O.md_eval(h1, (150.3, 0.39, 200.4), 1, 0)
    ok_between, _ = O.md_eval(h1, (150.3, 0.415, 200.4), 1, 0)
    ok_out, _ = O.md_eval(h1, (150.3, 0.44, 200.4), 1, 0)
    assert ok_in and not ok_between and not ok_out


def pin_match_needs_a_chi2_that_is_a_number(geo):
    """SPEC.md 4.6 [R20]: a pair only matches if its finished chi2 is a number below infinity.
    Single pair: straight seed along +x (pT = 1000 GeV), anchor at (50, 0, 0.1).  With pz = 0 it matches (|zres| = 0.1 <= 0.2).  With
    pz = +-inf: cot = sec = inf, dZ = inf, |zres| = |0.1 - inf| = inf <= dZ holds, but b = inf / inf = NaN -> no match.  NaN: no match.
    (An anchor with delta_r = 0, i.e. a barrel MD, rejects such a seed by itself: 0 * inf = NaN in dZ.  Endcap MDs have delta_r > 0.)
    Without the clause an infinite seed "matches" all-endcap objects with chi2 = NaN and, if it comes first, keeps them
    (`chi < NaN` is false for every later seed)."""
    ok, chi = O.pls_match(T._seed(0.0, 0.0), 1, T.A9(50.0, 0.0, 0.1))
    assert ok and 0.0 < chi < 2.0
    for pz in (np.inf, -np.inf, np.nan):
        assert not O.pls_match([T.PT_STRAIGHT, 0.0, pz, 0.0], 1, T.A9(50.0, 0.0, 0.1))[0]
    # chain: every seed of a PU50 event preceded by a copy with pz = +-inf.  The copies must match nothing (all of them end as plain
    # pLS candidates) and the real seeds must get exactly the rows they get without the copies.
    ev = config_event(geo, 1)
    r0 = O.run(geo, xavier_weights(2), ev)
    two = lambda a: np.repeat(a, 2)
    pz = two(ev.pls_pz).copy()
    pz[0::2] = np.where(pz[0::2] >= 0, np.inf, -np.inf).astype(np.float32)
    ev2 = dataclasses.replace(ev, pls_px=two(ev.pls_px), pls_py=two(ev.pls_py), pls_pz=pz, pls_z0=two(ev.pls_z0), pls_q=two(ev.pls_q),
                              pls_particle=two(ev.pls_particle))
    r = O.run(geo, xavier_weights(2), ev2)
    tc = r.tc
    copies = tc[(tc[:, 1] >= 0) & (tc[:, 1] % 2 == 0)]
    assert len(copies) == ev.n_pls and (copies[:, 0] == 3).all()
    real = tc[~((tc[:, 1] >= 0) & (tc[:, 1] % 2 == 0))].copy()
    real[:, 1] = np.where(real[:, 1] >= 0, real[:, 1] // 2, -1)
    assert np.array_equal(real, r0.tc)
    assert np.array_equal(np.where(r.best5_pls >= 0, r.best5_pls // 2, -1), r0.best5_pls) and (r.best5_pls[r.best5_pls >= 0] % 2 == 1).all()
    assert np.isfinite(r.chi5).all() and np.isfinite(r.chi3).all()
    # the event has what the clause is about: T5s / T3s whose anchors are all endcap MDs (delta_r * |cot| = inf, not 0 * inf = NaN)
    sub = np.asarray(geo.subdet)[r.md_mod]
    assert (sub[r.t5c[r.t5][:, :5]].min(axis=1) == 1).sum() > 20


def test_build_order(geo_full): pin_build_order(geo_full)
def test_match_needs_a_chi2_that_is_a_number(geo_full): pin_match_needs_a_chi2_that_is_a_number(geo_full)
def test_radius_clamp(): pin_radius_clamp()
def test_md_sagitta_cap(): pin_md_sagitta_cap()
