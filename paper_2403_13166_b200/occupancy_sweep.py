"""configs[4] of BASELINE.json: displaced-track and occupancy stress.  Each event = the PU-scaled config-2 recipe
plus 500 displaced particles; pile-up 0 / 100 / 200 / 300, 8 events per point (seeds 200-231).  Prints events/s,
mean object counts and the status word (any overflow flag) per point as a markdown table.

    python -m paper_2403_13166_b200.occupancy_sweep
"""
import sys
import numpy as np


def main():
    import torch
    import paper_2403_13166_b200 as P
    from lstgen import build_geometry, config_event, xavier_weights
    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device (no CPU fallback)")
    geo, w = build_geometry(True), xavier_weights(3)
    caps = P.Caps(n_slots=8, max_hits=196608, max_md=98304, max_ls=98304, max_t3=65536, max_t5c=32768, max_t5=32768, max_pls=8192)
    lst = P.LST(geo, w, caps)
    print("| pile-up | events/s | us/event | hits | MD | LS | T3 | T5 cand | T5 | pLS | TC | status |")
    print("|---|---|---|---|---|---|---|---|---|---|---|---|")
    seed = 200
    for pu in (0, 100, 200, 300):
        evs = [config_event(geo, 4, seed=seed + i, pileup=pu) for i in range(8)]
        seed += 8
        for i, ev in enumerate(evs):
            lst.load_numpy_event(i, ev)
        for _ in range(3):
            lst.lst_run_batch(0, 8)
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        reps = 20
        a.record()
        for _ in range(reps):
            lst.lst_run_batch(0, 8)
        b.record()
        torch.cuda.synchronize()
        ms = a.elapsed_time(b) / reps
        st, cs = zip(*[lst.lst_status(i) for i in range(8)])
        mean = lambda k: np.mean([c[k] for c in cs])
        print(f"| {pu} | {8 / ms * 1e3:.0f} | {ms * 1e3 / 8:.1f} | {mean('hit'):.0f} | {mean('md'):.0f} | {mean('ls'):.0f} | {mean('t3'):.0f} | "
              f"{mean('t5c'):.0f} | {mean('t5'):.0f} | {np.mean([ev.n_pls for ev in evs]):.0f} | {mean('tc'):.0f} | {max(st):#x} |")
    lst.close()


if __name__ == "__main__":
    sys.exit(main())
