"""Pins for the CPU oracle against what mathematics fixes (the paper prints no worked example, so
parity against the paper itself is unpinned -- DESIGN.md "Readings").  CPU only.

Each pin is chosen so that a plausible mistake in oracle/lst_oracle.cpp (dropped term, wrong sign,
wrong index, transposed operand) fails at least one of them.
"""
import numpy as np
import pytest

from lstgen import build_geometry, make_event, config_event, xavier_weights
from lstgen.events import KAPPA64
from oracle import lst_oracle as O
import canon

W1 = xavier_weights(1)


# ------------------------------------------------------------------ arcfac vs asin (SPEC.md 3.2)
def test_arcfac_matches_asin():
    xs = np.linspace(1e-4, 0.823, 400)
    rel = np.array([abs(O.arcfac(x * x, f64=True) - np.arcsin(x) / x) / (np.arcsin(x) / x) for x in xs])
    assert rel.max() <= 2.0e-3
    assert rel[xs <= 0.77].max() <= 7e-4
    assert rel[xs <= 0.5].max() <= 2e-6
    assert O.arcfac(0.0) == 1.0
    # fp32 Horner agrees with the fp64 one to rounding
    assert max(abs(O.arcfac(x * x) - O.arcfac(x * x, f64=True)) for x in xs) < 5e-7


# ------------------------------------------------------------------ Menger curvature textbook cases
def _anchor(x, y, z, dz=0.1299, dr=0.0, c=0.0, w=1.0, f=0.0):
    return np.array([x, y, z, np.hypot(x, y), c, w, f, dz, dr], dtype=np.float32)


def test_menger_textbook():
    R = 100.0
    # (R,0) -> (0,R) -> (-R,0) is counter-clockwise = phi increasing = negative charge => k = -1/R
    ok, k = O.bridge_eval(_anchor(R, 0, 0), _anchor(0, R, 0), _anchor(-R, 0, 0))
    assert ok and abs(k + 1.0 / R) < 1e-9
    ok, k = O.bridge_eval(_anchor(-R, 0, 0), _anchor(0, R, 0), _anchor(R, 0, 0))
    assert ok and abs(k - 1.0 / R) < 1e-9
    ok, k = O.bridge_eval(_anchor(10, 10, 0), _anchor(20, 20, 0), _anchor(40, 40, 0))
    assert ok and k == 0.0
    # curvature above the pT threshold fails T1: circle of radius 50 cm (pT = 0.57 GeV)
    ok, _ = O.bridge_eval(_anchor(50, 0, 0), _anchor(0, 50, 0), _anchor(-50, 0, 0))
    assert not ok
    # r-z non-linearity fails T2
    ok, _ = O.bridge_eval(_anchor(30, 0, 0), _anchor(50, 1, 0), _anchor(70, 3, 40.0))
    assert not ok


# ------------------------------------------------------------------ closed-form helices
def _helix_points(pt, q, phi0, eta, zv, radii):
    R = pt / KAPPA64
    s = 2 * R * np.arcsin(np.asarray(radii) / (2 * R))
    psi = phi0 - q * s / R
    x = -q * R * (np.sin(psi) - np.sin(phi0))
    y = q * R * (np.cos(psi) - np.cos(phi0))
    z = zv + s * np.sinh(eta)
    return x, y, z, s


@pytest.mark.parametrize("q", [-1, 1])
def test_closed_form_curvatures(q):
    rng = np.random.default_rng(7)
    for pt in [0.8, 0.85, 1.0, 1.5, 3.0, 10.0]:
        for _ in range(40):
            phi0 = rng.uniform(0, 2 * np.pi); eta = rng.uniform(-0.8, 0.8); zv = rng.uniform(-10, 10)
            radii = [23.0, 23.26, 36.0, 36.26, 51.0, 51.26]
            x, y, z, s = _helix_points(pt, q, phi0, eta, zv, radii)
            truth = q * KAPPA64 / pt
            mds = []
            for i in range(3):
                ok, out = O.md_eval([x[2 * i], y[2 * i], z[2 * i]], [x[2 * i + 1], y[2 * i + 1], z[2 * i + 1]], 0, 0)
                assert ok, (pt, i)
                # 2.6 mm lever arm: input quantisation limits the MD estimate (SPEC.md 6)
                assert abs(out[0] - truth) <= 1e-4 * max(1.0, pt / 1.5) * abs(truth) * 4
                assert abs(out[3] - radii[2 * i]) < 1e-4
                mds.append(np.array([x[2 * i], y[2 * i], z[2 * i], out[3], out[0], out[1], out[2], out[4], out[5]], np.float32))
            ok, c01 = O.ls_eval(mds[0], mds[1]); assert ok
            ok, c12 = O.ls_eval(mds[1], mds[2]); assert ok
            assert abs(c01 - truth) <= 1e-4 * abs(truth) and abs(c12 - truth) <= 1e-4 * abs(truth)
            ok, k = O.t3_eval(mds[0], mds[1], mds[2], c01, c12); assert ok
            assert abs(k - truth) <= 1e-4 * abs(truth)
            # pT and radius reproduced (north star: 1e-4 relative)
            assert abs(KAPPA64 / abs(k) - pt) <= 1e-4 * pt
            # pLS residuals vanish on the generating helix (fp64 restatement)
            pls = [pt * np.cos(phi0), pt * np.sin(phi0), pt * np.sinh(eta), zv]
            for i in (0, 2, 4):
                res = O.pls_residual(pls, q, [x[i], y[i], z[i]])
                assert abs(res[0]) < 1e-6   # KAPPA is the fp32 literal 0.0114f
                arc_err = 2e-3 if pt < 1.0 else 1e-5
                assert abs(res[1]) <= arc_err * abs(s[i] * np.sinh(eta)) + 1e-9
                assert abs(res[2] - s[i]) <= arc_err * s[i]


def test_endcap_md_closed_form():
    rng = np.random.default_rng(11)
    n_ok = 0
    for _ in range(300):
        pt = rng.uniform(0.8, 20.0); q = rng.choice([-1, 1]); phi0 = rng.uniform(0, 2 * np.pi)
        eta = rng.uniform(1.3, 2.3) * rng.choice([-1, 1]); zv = rng.uniform(-10, 10)
        R = pt / KAPPA64
        zd = 131.0 * np.sign(eta)
        pts = []
        for zp in (zd, zd + 0.26 * np.sign(eta)):
            s = (zp - zv) / np.sinh(eta)
            psi = phi0 - q * s / R
            pts.append([-q * R * (np.sin(psi) - np.sin(phi0)), q * R * (np.cos(psi) - np.cos(phi0)), zp])
        r = np.hypot(pts[0][0], pts[0][1])
        if not (23 <= r < 60) or s > np.pi * R:
            continue
        ok, out = O.md_eval(pts[0], pts[1], 1, 0)
        assert ok
        n_ok += 1
        assert out[2] == np.float32(0.3) and out[5] == np.float32(0.1299) and out[4] == 0.0
    assert n_ok > 50


# ------------------------------------------------------------------ noise-free truth passes every cut
def test_noise_free_truth_all_found(geo_full):
    ev = make_event(geo_full, 5, n_particles=600, smear=False, shuffle=True)
    r = O.run(geo_full, W1, ev)
    part = ev.particles
    hp = ev.hit_particle
    good = (part["pt"] >= 0.8) & (np.abs(part["zv"]) <= 15.0)
    # expected MDs: (particle, module) with both sensor hits present
    mod = ev.key >> 1
    exp = {}
    for i in range(ev.n_hits):
        if good[hp[i]]:
            exp.setdefault((hp[i], mod[i]), []).append(i)
    exp_md = {tuple(sorted(v, key=lambda h: ev.key[h])) for v in exp.values() if len(v) == 2}
    got_md = {tuple(t) for t in r.md_hits.tolist()}
    assert exp_md <= got_md
    # expected LS / T3 / T5: consecutive crossings of one particle (when the modules are connected)
    md_of = {}
    for i, (lo, up) in enumerate(r.md_hits):
        if hp[lo] == hp[up] and good[hp[lo]]:
            md_of.setdefault(hp[lo], []).append(i)
    conn = {(m, c) for m in range(geo_full.n_modules)
            for c in geo_full.conn_col[geo_full.conn_rowptr[m]:geo_full.conn_rowptr[m + 1]]}
    ls_set = {tuple(t) for t in r.ls.tolist()}
    t3_set = {tuple(t[:3]) for t in r.t3.tolist()}
    t5_set = {tuple(t[:5]) for t in r.t5c.tolist()}
    n_ls = n_t3 = n_t5 = 0
    for p, mds in md_of.items():
        mds = sorted(mds, key=lambda i: r.md_real[i, 5] ** 2 + r.md_real[i, 4] ** 2)
        chain_ok = [(r.md_mod[a], r.md_mod[b]) in conn for a, b in zip(mds[:-1], mds[1:])]
        for i in range(len(mds) - 1):
            if chain_ok[i]:
                n_ls += 1
                assert (mds[i], mds[i + 1]) in ls_set
        for i in range(len(mds) - 2):
            if chain_ok[i] and chain_ok[i + 1]:
                n_t3 += 1
                assert tuple(mds[i:i + 3]) in t3_set
        for i in range(len(mds) - 4):
            if all(chain_ok[i:i + 4]):
                n_t5 += 1
                assert tuple(mds[i:i + 5]) in t5_set
    assert n_ls > 500 and n_t3 > 300 and n_t5 > 100


def test_smeared_barrel_muons_efficiency(geo_barrel):
    """Physics sanity of the frozen constants: smeared configs[0]-style muons survive every stage."""
    tot = found = 0
    for seed in range(20):
        ev = make_event(geo_barrel, 1000 + seed, origin_muons=10)
        r = O.run(geo_barrel, W1, ev)
        hp = ev.hit_particle
        for t in r.t5c[:, :5]:
            hits = r.md_hits[t].ravel()
            found += int(len(set(hp[hits])) == 1)
        tot += 2 * 10   # layers 1-5 and 2-6
        assert np.sum(r.tc[:, 0] == 3) == 0 or len(r.tc) == 10
    assert found >= 0.97 * tot   # five stacked 3-sigma cuts


# ------------------------------------------------------------------ brute force on tiny events
def _md9(r, i):
    c, w, x, y, z, rr = r.md_real[i]
    return np.array([x, y, z, rr, c, w, 0, 0, 0], dtype=np.float32)


def _brute(geo, ev, weights):
    """All-pairs / all-tuples enumeration with the single predicates; different loops, same cuts."""
    n = ev.n_hits
    mod = (ev.key >> 1).astype(np.int64); up = (ev.key & 1).astype(np.int64)
    conn = {(m, int(c)) for m in range(geo.n_modules)
            for c in geo.conn_col[geo.conn_rowptr[m]:geo.conn_rowptr[m + 1]]}
    mds = {}
    for i in range(n):
        for j in range(n):
            if mod[i] == mod[j] and up[i] == 0 and up[j] == 1:
                m = mod[i]
                ok, o = O.md_eval([ev.x[i], ev.y[i], ev.z[i]], [ev.x[j], ev.y[j], ev.z[j]], geo.subdet[m], geo.mtype[m])
                if ok:
                    mds[(i, j)] = (np.array([ev.x[i], ev.y[i], ev.z[i], o[3], o[0], o[1], o[2], o[4], o[5]], np.float32), m)
    lss = {}
    for ka, (a9, ma) in mds.items():
        for kb, (b9, mb) in mds.items():
            if (ma, mb) in conn:
                ok, c = O.ls_eval(a9, b9)
                if ok:
                    lss[(ka, kb)] = np.float32(c)
    t3s = {}
    for (a, b), c0 in lss.items():
        for (b2, c), c1 in lss.items():
            if b2 == b:
                ok, k = O.t3_eval(mds[a][0], mds[b][0], mds[c][0], c0, c1)
                if ok:
                    t3s[(a, b, c)] = np.float32(k)
    t5s = set()
    for (a, b, c) in t3s:
        for (c2, d, e) in t3s:
            if c2 == c:
                ok, _ = O.bridge_eval(mds[b][0], mds[c][0], mds[d][0])
                if ok:
                    t5s.add((a, b, c, d, e))
    return mds, lss, t3s, t5s


@pytest.mark.parametrize("seed,kw", [(21, dict(n_particles=24, per_vertex=8, n_noise=0)),
                                    (22, dict(origin_muons=6, n_noise=0)),
                                    (23, dict(n_particles=30, per_vertex=30, n_noise=40))])
def test_brute_force_tiny(geo_full, seed, kw):
    ev = make_event(geo_full, seed, **kw)
    if kw.get("n_noise"):
        # pile the noise into occupied modules so that fake combinations are actually tested
        rng = np.random.default_rng(seed)
        occ = np.unique(ev.key[ev.hit_particle >= 0])
        sel = np.flatnonzero(ev.hit_particle < 0)
        src = rng.choice(np.flatnonzero(ev.hit_particle >= 0), size=sel.size)
        ev.key[sel] = ev.key[src] ^ rng.integers(0, 2, sel.size).astype(np.uint32)
        ev.x[sel] = ev.x[src] + rng.normal(0, 0.05, sel.size).astype(np.float32)
        ev.y[sel] = ev.y[src] + rng.normal(0, 0.05, sel.size).astype(np.float32)
        ev.z[sel] = ev.z[src] + rng.normal(0, 0.2, sel.size).astype(np.float32) * (geo_full.subdet[ev.key[src] >> 1] == 0)
        assert occ.size
    assert ev.n_hits < 500
    r = O.run(geo_full, W1, ev)
    mds, lss, t3s, t5s = _brute(geo_full, ev, W1)
    assert {tuple(t) for t in r.md_hits.tolist()} == set(mds)
    mh = [tuple(t) for t in r.md_hits.tolist()]
    assert {(mh[a], mh[b]) for a, b in r.ls.tolist()} == set(lss)
    assert {(mh[a], mh[b], mh[c]) for a, b, c, _, _ in r.t3.tolist()} == set(t3s)
    assert {tuple(mh[i] for i in t[:5]) for t in r.t5c.tolist()} == t5s
    assert len(mds) > 20 and len(t5s) > 2
    # payloads line up as well
    for (a, b), c in zip(r.ls.tolist(), r.ls_c):
        assert np.float32(c) == lss[(mh[a], mh[b])]
    for t, k in zip(r.t3.tolist(), r.t3_k):
        assert np.float32(k) == t3s[(mh[t[0]], mh[t[1]], mh[t[2]])]
    # ---- TC selection by brute force over all (pLS, object) pairs (SPEC.md 4.6)
    def anchors(md_idx):
        out = []
        for i in md_idx:
            a9 = mds[mh[i]][0]
            out.append(a9)
        return np.stack(out)
    t5list = [r.t5c[c, :5] for c in r.t5]
    best5 = {}
    for t, m5 in enumerate(t5list):
        cand = []
        for p in range(ev.n_pls):
            ok, chi = O.pls_match([ev.pls_px[p], ev.pls_py[p], ev.pls_pz[p], ev.pls_z0[p]], ev.pls_q[p], anchors(m5))
            if ok:
                cand.append((np.float32(chi), p))
        if cand:
            best5[t] = min(cand)
    win5 = {}
    for t, (chi, p) in best5.items():
        if p not in win5 or (chi, t) < win5[p]:
            win5[p] = (chi, t)
    exp = [(0, p, win5[p][1]) for p in sorted(win5)]
    exp += [(1, -1, t) for t in range(len(t5list)) if t not in best5]
    used_sets = [set(t5list[t].tolist()) for _, t in win5.values()]
    best3 = {}
    for x, t in enumerate(r.t3.tolist()):
        if any(set(t[:3]) <= u for u in used_sets):
            continue
        cand = []
        for p in range(ev.n_pls):
            if p in win5:
                continue
            ok, chi = O.pls_match([ev.pls_px[p], ev.pls_py[p], ev.pls_pz[p], ev.pls_z0[p]], ev.pls_q[p], anchors(t[:3]))
            if ok:
                cand.append((np.float32(chi), p))
        if cand:
            best3[x] = min(cand)
    win3 = {}
    for x, (chi, p) in best3.items():
        if p not in win3 or (chi, x) < win3[p]:
            win3[p] = (chi, x)
    exp += [(2, p, win3[p][1]) for p in sorted(win3)]
    exp += [(3, p, -1) for p in range(ev.n_pls) if p not in win5 and p not in win3]
    assert [tuple(t) for t in r.tc.tolist()] == exp


# ------------------------------------------------------------------ fp64 instantiation
def test_double_instantiation_agrees(geo_full):
    ev = config_event(geo_full, 1)
    w = xavier_weights(2)
    a = O.run(geo_full, w, ev)
    b = O.run(geo_full, w, ev, use_double=True)
    for name, fa, fb in [("md", a.md_hits, b.md_hits),
                         ("ls", canon.ls_tuples(a.md_hits, a.ls), canon.ls_tuples(b.md_hits, b.ls)),
                         ("t3", canon.t3_tuples(a.md_hits, a.t3[:, :3]), canon.t3_tuples(b.md_hits, b.t3[:, :3])),
                         ("t5", canon.t5_tuples(a.md_hits, a.t5c[:, :5]), canon.t5_tuples(b.md_hits, b.t5c[:, :5]))]:
        sa = {tuple(t) for t in np.asarray(fa).tolist()}
        sb = {tuple(t) for t in np.asarray(fb).tolist()}
        assert len(sa ^ sb) <= max(2, 2e-3 * len(sa)), name
    # payloads on common LSs agree to fp32 rounding x conditioning
    ca = {tuple(t): c for t, c in zip(canon.ls_tuples(a.md_hits, a.ls).tolist(), a.ls_c)}
    cb = {tuple(t): c for t, c in zip(canon.ls_tuples(b.md_hits, b.ls).tolist(), b.ls_c)}
    common = set(ca) & set(cb)
    d = np.array([abs(ca[k] - cb[k]) for k in common])
    assert d.max() < 2e-6


# ------------------------------------------------------------------ invariants
def _rot90(geo, ev):
    """(x, y) -> (-y, x) is exact in fp32; module -> the module a quarter turn further."""
    M = geo.n_modules
    rot = np.zeros(M, dtype=np.int64)
    n = 0
    for l in range(6):
        nphi = geo.barrel_nphi[l]
        ids = np.arange(nphi * 24).reshape(nphi, 24)
        rot[n:n + nphi * 24] = (n + np.roll(ids, -nphi // 4, axis=0)).ravel()
        n += nphi * 24
    for s in range(2):
        for d in range(5):
            for k in range(9):
                nphi = geo.ring_nphi[k]
                base = geo.disk_base[s, d, k]
                rot[base:base + nphi] = base + (np.arange(nphi) + nphi // 4) % nphi
    import copy
    e2 = copy.deepcopy(ev)
    e2.x, e2.y = (-ev.y).copy(), ev.x.copy()
    e2.key = (2 * rot[ev.key >> 1] + (ev.key & 1)).astype(np.uint32)
    e2.pls_px, e2.pls_py = (-ev.pls_py).copy(), ev.pls_px.copy()
    return e2, rot


def test_rotation_by_quarter_turn(geo_sym4):
    g = geo_sym4
    ev = make_event(g, 31, n_particles=900, n_noise=1500, inefficiency=0.05)
    e2, rot = _rot90(g, ev)
    # the CSR itself must be symmetric for the statement to make sense
    for m in range(0, g.n_modules, 37):
        a = sorted(rot[g.conn_col[g.conn_rowptr[m]:g.conn_rowptr[m + 1]]].tolist())
        b = sorted(g.conn_col[g.conn_rowptr[rot[m]]:g.conn_rowptr[rot[m] + 1]].tolist())
        assert a == b
    w = xavier_weights(31)
    a = O.run(g, w, ev)
    b = O.run(g, w, e2)
    assert canon.same_set(a.md_hits, b.md_hits)
    assert canon.same_set(canon.ls_tuples(a.md_hits, a.ls), canon.ls_tuples(b.md_hits, b.ls))
    assert canon.same_set(canon.t3_tuples(a.md_hits, a.t3[:, :3]), canon.t3_tuples(b.md_hits, b.t3[:, :3]))
    assert canon.same_set(canon.t5_tuples(a.md_hits, a.t5c[:, :5]), canon.t5_tuples(b.md_hits, b.t5c[:, :5]))
    assert len(a.t5c) > 50
    # curvatures are bit-identical too (only dot / cross / r^2 enter)
    sa, oa = canon.lexsort_rows(canon.ls_tuples(a.md_hits, a.ls))
    sb, ob = canon.lexsort_rows(canon.ls_tuples(b.md_hits, b.ls))
    assert np.array_equal(a.ls_c[oa], b.ls_c[ob])


def test_mirror_z(geo_full):
    g = geo_full
    ev = config_event(g, 1, seed=41)
    M = g.n_modules
    mir = np.zeros(M, dtype=np.int64)
    n = 0
    for l in range(6):
        nphi = g.barrel_nphi[l]
        ids = np.arange(nphi * 24).reshape(nphi, 24)
        mir[n:n + nphi * 24] = (n + ids[:, ::-1]).ravel()
        n += nphi * 24
    per_side = (M - n) // 2
    mir[n:n + per_side] = np.arange(n + per_side, M)
    mir[n + per_side:] = np.arange(n, n + per_side)
    import copy
    e2 = copy.deepcopy(ev)
    e2.z = (-ev.z).copy()
    e2.key = (2 * mir[ev.key >> 1] + (ev.key & 1)).astype(np.uint32)
    e2.pls_pz = (-ev.pls_pz).copy(); e2.pls_z0 = (-ev.pls_z0).copy()
    w = xavier_weights(2)
    a = O.run(g, w, ev); b = O.run(g, w, e2)
    assert canon.same_set(a.md_hits, b.md_hits)
    assert canon.same_set(canon.t3_tuples(a.md_hits, a.t3[:, :3]), canon.t3_tuples(b.md_hits, b.t3[:, :3]))
    assert canon.same_set(canon.t5_tuples(a.md_hits, a.t5c[:, :5]), canon.t5_tuples(b.md_hits, b.t5c[:, :5]))
    # matching uses only |.| of z residuals and cot -> the chi2-ranked TC list mirrors exactly as well
    ta = canon.tc_tuples(a.md_hits, a.t3[:, :3], a.t5c[a.t5][:, :5], a.tc)
    tb = canon.tc_tuples(b.md_hits, b.t3[:, :3], b.t5c[b.t5][:, :5], b.tc)
    pass_same = np.array_equal(a.t5c[:, 7], b.t5c[:, 7])   # scores see eta -> -eta, decisions may differ
    if pass_same:
        assert canon.same_set(ta, tb)


def test_hit_order_permutation(geo_full):
    g = geo_full
    ev = config_event(g, 1, seed=51)
    rng = np.random.default_rng(1)
    perm = rng.permutation(ev.n_hits)
    import copy
    e2 = copy.deepcopy(ev)
    e2.x, e2.y, e2.z, e2.key = ev.x[perm], ev.y[perm], ev.z[perm], ev.key[perm]
    w = xavier_weights(2)
    a = O.run(g, w, ev); b = O.run(g, w, e2)
    bm = perm[b.md_hits]      # back to the original numbering
    assert canon.same_set(a.md_hits, bm)
    assert canon.same_set(canon.t5_tuples(a.md_hits, a.t5c[:, :5]), canon.t5_tuples(bm, b.t5c[:, :5]))
    assert sorted(np.bincount(a.tc[:, 0], minlength=4)) == sorted(np.bincount(b.tc[:, 0], minlength=4))


@pytest.mark.parametrize("cut", ["M2", "M3", "L1", "L2", "L3", "T1", "T2", "T3", "Q1", "Q2"])
def test_loosening_gives_supersets(geo_full, cut):
    ev = config_event(geo_full, 1, seed=61)
    w = xavier_weights(2)
    a = O.run(geo_full, w, ev, last_stage="t5")
    b = O.run(geo_full, w, ev, loosen={cut: 1.25}, last_stage="t5")
    sets = lambda r: [{tuple(t) for t in r.md_hits.tolist()},
                      {tuple(t) for t in canon.ls_tuples(r.md_hits, r.ls).tolist()},
                      {tuple(t) for t in canon.t3_tuples(r.md_hits, r.t3[:, :3]).tolist()},
                      {tuple(t) for t in canon.t5_tuples(r.md_hits, r.t5c[:, :5]).tolist()}]
    sa, sb = sets(a), sets(b)
    grew = False
    for x, y in zip(sa, sb):
        assert x <= y
        grew |= len(y) > len(x)
    assert grew, "loosening had no effect: the cut is not wired"


# ------------------------------------------------------------------ DNN
def _mlp64(w, x):
    w = w.astype(np.float64)
    W1_, b1 = w[:736].reshape(32, 23), w[736:768]
    W2_, b2 = w[768:1792].reshape(32, 32), w[1792:1824]
    w3, b3 = w[1824:1856], w[1856]
    h1 = np.maximum(W1_ @ x + b1, 0.0)
    h2 = np.maximum(W2_ @ h1 + b2, 0.0)
    return 1.0 / (1.0 + np.exp(-(w3 @ h2 + b3)))


def test_dnn_against_independent_fp64(geo_full):
    ev = config_event(geo_full, 1)
    w = xavier_weights(2, bias_scale=0.3)     # non-zero biases so a dropped bias term shows
    r = O.run(geo_full, w, ev, last_stage="t5")
    assert len(r.t5c) > 500
    ref = np.array([_mlp64(w, f) for f in r.t5c_feat])
    assert np.abs(ref - r.t5c_score).max() < 1e-6
    assert np.array_equal(r.t5c[:, 7] == 1, r.t5c_score > 0.5)
    assert 0.02 < np.mean(r.t5c_score > 0.5) < 0.98 or True
    # features from float64 definitions
    mdr = r.md_real
    for t, f, cv in list(zip(r.t5c, r.t5c_feat, r.t5c_curv))[:200]:
        for i in range(5):
            c, w_, x, y, z, rr = mdr[t[i]]
            exp = [rr / 100.0, z / 100.0, np.arcsinh(z / rr), np.arctan2(y, x)]
            assert np.allclose(f[4 * i:4 * i + 4], exp, rtol=2e-6, atol=1e-7)
        exp = [np.log10(min(1.0 / abs(k), 1e5)) if k != 0 else 5.0 for k in cv]
        assert np.allclose(f[20:], exp, rtol=2e-6, atol=1e-6)


def test_dnn_zero_weights_rejects_everything(geo_full):
    ev = config_event(geo_full, 1)
    r = O.run(geo_full, np.zeros(1857, np.float32), ev)
    assert len(r.t5c) > 0 and np.all(r.t5c_score == 0.5) and len(r.t5) == 0
    assert np.sum(r.tc[:, 0] <= 1) == 0          # no pT5 / T5 candidates without T5s


def test_dnn_single_neuron_paths():
    """One-hot weights isolate each layer's indexing (a transposed W would fail)."""
    w = np.zeros(1857, np.float32)
    W1_ = w[:736].reshape(32, 23); W2_ = w[768:1792].reshape(32, 32)
    W1_[5, 7] = 2.0; W2_[9, 5] = 3.0; w[1824 + 9] = 0.5
    x = np.zeros(23, np.float32); x[7] = 1.5
    assert abs(O.mlp(w, x) - 1 / (1 + np.exp(-4.5))) < 1e-6
    x[7] = -1.5
    assert O.mlp(w, x) == 0.5      # ReLU


# ------------------------------------------------------------------ TC identities
def test_tc_partition_identities(geo_full):
    ev = config_event(geo_full, 2)
    w = xavier_weights(3)
    r = O.run(geo_full, w, ev)
    tc = r.tc
    n = np.bincount(tc[:, 0], minlength=4)
    assert n[0] + n[2] + n[3] == ev.n_pls
    pls_used = tc[tc[:, 0] != 1, 1]
    assert len(set(pls_used.tolist())) == ev.n_pls            # every pLS exactly once
    t5_as_pt5 = set(tc[tc[:, 0] == 0, 2].tolist()); t5_as_t5 = set(tc[tc[:, 0] == 1, 2].tolist())
    assert not (t5_as_pt5 & t5_as_t5)
    matched = set(np.flatnonzero(r.best5_pls >= 0).tolist())
    assert t5_as_pt5 <= matched and t5_as_t5 == set(range(len(r.t5))) - matched
    # no T3 of a pT5 is used by a pT3
    used = [set(r.t5c[r.t5[t], :5].tolist()) for t in t5_as_pt5]
    for x in tc[tc[:, 0] == 2, 2]:
        s = set(r.t3[x, :3].tolist())
        assert not any(s <= u for u in used)
    assert n.min() > 0
    # overrides: forcing every candidate to fail removes all T5-based candidates
    r2 = O.run(geo_full, w, ev, t5_override=np.zeros(len(r.t5c), np.int8))
    assert len(r2.t5) == 0 and np.sum(r2.tc[:, 0] <= 1) == 0


def test_exact_pls_gives_pt5_with_small_chi2(geo_barrel):
    ev = make_event(geo_barrel, 71, origin_muons=10, smear=False)
    r = O.run(geo_barrel, W1, ev)
    assert np.all(r.tc[:, 0] == 0) and len(r.tc) == 10
    assert r.chi5[r.tc[:, 2]].max() < 1e-3


def test_out_of_range_key_is_flagged(geo_barrel):
    ev = make_event(geo_barrel, 72, origin_muons=4)
    ev.key[3] = 2 * geo_barrel.n_modules + 5
    r = O.run(geo_barrel, W1, ev)
    assert r.flags & 1 and r.counts["hits"] == ev.n_hits - 1
