"""f2: truth-matched efficiency / fake rate / duplicate rate of the track candidates on the SYNTHETIC truth.

PAPER.md:41 / :99: "a TC is matched to a simulated track if more than 75 % of its hits belong to it"; efficiency = fraction of
simulated tracks with at least one matched TC, fake rate = fraction of TCs matched to no simulated track, shown against pT,
eta and the production radius (Figs. 2, 7-9).  The paper's plots need its CMS samples and trained weights; this module does
the same bookkeeping on the generator's truth (`lstgen.Event.hit_particle`, `.particles`), so that the frozen cut values of
SPEC.md can be judged physically and the effect of the duplicate cleaning (f1) and of a DNN cut can be tabulated.

Pure host-side bookkeeping on hit-index tuples: it takes the candidates' ORIGINAL hit indices (lst_get TCX / the e2e rows of
lst_read_tc_hits_batch_host, or the oracle's `tc_hits` in tests) and contains none of the method's arithmetic.

    python -m paper_2403_13166_b200.evaluate --events 8 [--pileup 200] [--displaced]      (needs a GPU)
"""
import argparse
import json
import sys

import numpy as np

MATCH_FRACTION = 0.75
PT_EDGES = np.array([0.9, 1.2, 1.5, 2.0, 3.0, 5.0, 10.0, 50.0])
ETA_EDGES = np.linspace(-2.4, 2.4, 13)
RVTX_EDGES = np.array([0.0, 1.0, 5.0, 10.0, 20.0, 30.0, 50.0])


def truth_match(ev, tc_types, tc_pls, tc_hits):
    """Particle index matched to every candidate, or -1.
    Candidates with outer-tracker hits (pT5, T5, pT3): the particle that owns more than 75 % of their hits.
    pLS candidates carry no outer-tracker hits here: they are matched to the particle their seed was made from."""
    hp = ev.hit_particle
    out = -np.ones(len(tc_types), dtype=np.int64)
    for i, ty in enumerate(tc_types):
        if ty == 3:
            out[i] = int(ev.pls_particle[tc_pls[i]])
            continue
        h = tc_hits[i][tc_hits[i] >= 0]
        owners = hp[h]
        owners = owners[owners >= 0]
        if owners.size == 0:
            continue
        vals, cnt = np.unique(owners, return_counts=True)
        k = int(np.argmax(cnt))
        if cnt[k] > MATCH_FRACTION * h.size:
            out[i] = int(vals[k])
    return out


def reconstructable(ev, pt_min=0.9, eta_max=2.4):
    """Denominator of the efficiency: generated particles with pT > pt_min and |eta| < eta_max that left at least three
    complete module crossings (both sensors hit) -- enough for a T3."""
    p = ev.particles
    n = p["pt"].size
    mod = (ev.key >> 1).astype(np.int64)
    pm = {}
    for h in np.flatnonzero(ev.hit_particle >= 0):
        pm.setdefault((int(ev.hit_particle[h]), int(mod[h])), set()).add(int(ev.key[h] & 1))
    crossings = np.zeros(n, dtype=np.int64)
    for (part, _), sides in pm.items():
        if len(sides) == 2:
            crossings[part] += 1
    return (p["pt"] > pt_min) & (np.abs(p["eta"]) < eta_max) & (crossings >= 3)


class Tally:
    """accumulates over events"""

    def __init__(self):
        self.den = {k: None for k in ("pt", "eta", "rvtx")}
        self.num = {k: None for k in ("pt", "eta", "rvtx")}
        self.n_tc = self.n_fake = self.n_dup = self.n_part = self.n_found = 0
        self.n_found_ot = 0                                   # found by a candidate WITH outer-tracker hits (pT5 / T5 / pT3)
        self.by_type = np.zeros((4, 2), dtype=np.int64)       # [type][all, fake]
        self.found_by_type = np.zeros(4, dtype=np.int64)      # reconstructable particles with >= 1 matched candidate of the type

    def add(self, ev, tc_types, tc_pls, tc_hits):
        tc_types = np.asarray(tc_types); tc_hits = np.asarray(tc_hits).reshape(len(tc_types), -1)[:, :10]
        m = truth_match(ev, tc_types, np.asarray(tc_pls), tc_hits)
        ok = reconstructable(ev)
        p = ev.particles
        found = np.zeros(p["pt"].size, dtype=np.int64)
        np.add.at(found, m[m >= 0], 1)
        rv = np.hypot(p["xv"], p["yv"])
        for name, val, edges in (("pt", p["pt"], PT_EDGES), ("eta", p["eta"], ETA_EDGES), ("rvtx", rv, RVTX_EDGES)):
            d, _ = np.histogram(val[ok], bins=edges)
            f, _ = np.histogram(val[ok & (found > 0)], bins=edges)
            self.den[name] = d if self.den[name] is None else self.den[name] + d
            self.num[name] = f if self.num[name] is None else self.num[name] + f
        self.n_part += int(ok.sum()); self.n_found += int((ok & (found > 0)).sum())
        # A pLS candidate is matched through its seed's label, and the generator gives every prompt particle a seed, so `found`
        # alone says little about the outer-tracker chain: count separately what the hit rule found, per candidate type.
        for t in range(4):
            ft = np.zeros(p["pt"].size, dtype=bool)
            ft[m[(m >= 0) & (tc_types == t)]] = True
            self.found_by_type[t] += int((ok & ft).sum())
        f_ot = np.zeros(p["pt"].size, dtype=bool)
        f_ot[m[(m >= 0) & (tc_types != 3)]] = True
        self.n_found_ot += int((ok & f_ot).sum())
        self.n_tc += len(m); self.n_fake += int((m < 0).sum())
        self.n_dup += int(sum(c - 1 for c in found[found > 1]))
        for t in range(4):
            self.by_type[t, 0] += int((tc_types == t).sum()); self.by_type[t, 1] += int(((tc_types == t) & (m < 0)).sum())

    def summary(self):
        frac = lambda a, b: None if b == 0 else round(a / b, 4)
        tab = {}
        for name, edges in (("pt", PT_EDGES), ("eta", ETA_EDGES), ("rvtx", RVTX_EDGES)):
            tab[name] = [dict(lo=round(float(edges[i]), 3), hi=round(float(edges[i + 1]), 3), n=int(self.den[name][i]),
                              eff=frac(int(self.num[name][i]), int(self.den[name][i]))) for i in range(len(edges) - 1)]
        names = ("pT5", "T5", "pT3", "pLS")
        n_ot, fake_ot = int(self.by_type[:3, 0].sum()), int(self.by_type[:3, 1].sum())
        return dict(efficiency=frac(self.n_found, self.n_part), fake_rate=frac(self.n_fake, self.n_tc), duplicate_rate=frac(self.n_dup, self.n_tc),
                    n_particles=self.n_part, n_tc=self.n_tc,
                    # headline for the outer-tracker chain: only pT5 / T5 / pT3, matched by the > 75 % hit rule
                    efficiency_outer_tracker=frac(self.n_found_ot, self.n_part), fake_rate_outer_tracker=frac(fake_ot, n_ot),
                    efficiency_by_type={n: frac(int(self.found_by_type[t]), self.n_part) for t, n in enumerate(names)},
                    caveat="`efficiency` counts pLS candidates, which are matched through their seed's label; the generator seeds every prompt "
                           "particle above 0.8 GeV and makes no fake seeds, so it is close to 1 by construction and the pLS fake rate is 0. "
                           "`efficiency_outer_tracker` / `fake_rate_outer_tracker` use only candidates with outer-tracker hits and the hit rule.",
                    fake_rate_by_type={n: frac(int(self.by_type[t, 1]), int(self.by_type[t, 0])) for t, n in enumerate(("pT5", "T5", "pT3", "pLS"))},
                    n_by_type={n: int(self.by_type[t, 0]) for t, n in enumerate(("pT5", "T5", "pT3", "pLS"))}, vs=tab)


def pass_all_weights(n_feat=23, n_hidden=2):
    """DNN weights that accept every T5 candidate (all zero, output bias +20): the 'no DNN cut' arm"""
    n = 32 * n_feat + 32 + (n_hidden - 1) * 1056 + 33
    w = np.zeros(n, dtype=np.float32)
    w[-1] = 20.0
    return w


def run_gpu(events, geo, weights, cleaned):
    """TC lists of `events` through the CUDA library; returns a Tally"""
    import paper_2403_13166_b200 as P
    lst = P.LST(geo, weights, P.Caps(n_slots=len(events), max_hits=196608, max_md=98304, max_ls=98304, max_t3=65536, max_t5c=32768, max_t5=32768, max_pls=8192))
    for i, ev in enumerate(events):
        lst.load_numpy_event(i, ev)
    lst.lst_run_batch(0, len(events))
    t = Tally()
    for i, ev in enumerate(events):
        out = lst.fetch(i)
        assert out["status"] == 0
        tc = out["tc"]["tc"].reshape(-1, 3)
        hits = out["tcx"]["hits"].reshape(-1, 12)[:, :10]
        keep = out["tcx"]["keep"].astype(bool) if cleaned else np.ones(len(tc), bool)
        t.add(ev, tc[keep, 0], tc[keep, 1], hits[keep])
    lst.close()
    return t


def main(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--events", type=int, default=8)
    ap.add_argument("--pileup", type=int, default=200)
    ap.add_argument("--displaced", action="store_true", help="configs[4] events (adds 500 displaced particles)")
    ap.add_argument("--seed", type=int, default=300)
    args = ap.parse_args(argv)
    import torch
    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device (no CPU fallback)")
    from lstgen import build_geometry, make_event, xavier_weights
    geo = build_geometry(True)
    evs = [make_event(geo, args.seed + i, n_particles=30 * args.pileup, n_noise=50 * args.pileup, n_displaced=500 if args.displaced else 0,
                      inefficiency=0.05) for i in range(args.events)]
    res = dict(workload=f"{args.events} synthetic events, pile-up {args.pileup}" + (" + 500 displaced" if args.displaced else ""),
               match=f"> {MATCH_FRACTION:.0%} of the candidate's outer-tracker hits from one particle (PAPER.md:41, :99)",
               denominator="pT > 0.9 GeV, |eta| < 2.4, at least three complete module crossings")
    for label, w in (("dnn_random_init", xavier_weights(3)), ("no_dnn_cut", pass_all_weights())):
        for cl in (False, True):
            res[f"{label}.{'cleaned' if cl else 'raw'}"] = run_gpu(evs, geo, w, cl).summary()
    print(json.dumps(res))


if __name__ == "__main__":
    sys.exit(main())
