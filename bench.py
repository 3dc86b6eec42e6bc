#!/usr/bin/env python
"""bench.py -- events/s of the whole LST hot path (a0 ingest -> MD -> LS -> T3 -> T5 + DNN -> TC) at PU200.

Contract (one JSON line on stdout from rank 0):
  python bench.py --gpus N --steps K --warmup W            our CUDA path through the C ABI
  python bench.py --impl reference ...                     the CPU oracle, as it stands, on host cores

A "step" = one pass of the whole hot path over one batch of `--events` synthetic PU200 events
(BASELINE.json configs[2] recipe, the seeds of configs[3]); `value` = events/s with the inputs resident
in HBM; `e2e` = the same through lst_load_batch_host16 / lst_read_tc_hits_batch_host with pinned HOST buffers, copies
inside the timed region; `single_event` = configs[2] exactly (one event, seed 3); `--config 4` = the occupancy sweep.  Events are independent, so N GPUs run N replicas on different seeds (weak
scaling, no collective on the data path -- DESIGN.md "Multi-GPU").
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "events/s at PU200 (MD->LS->T3->T5+DNN->TC)"
UNIT = "events/s"
WORKLOAD = "configs[2] HL-LHC PU200 events (6000 particles, 5% inefficiency, 10000 noise hits), seeds 100.. as in configs[3]"

# ---- per-unit algorithmic work: un-fused fp32 operations per pair test and
# compulsory bytes per object; FP32 non-fused peak = 148 SM x 128 lanes x sm_max_mhz.
FLOPS = dict(md_pair=34, ls_pair=60, t3_pair=86, t5_pair=80, dnn_cand=3584 + 140, match_pair=10, match_full=45)   # ls_pair: SURVEY.md 8.d
SM_COUNT, LANES = 148, 128
TC_ROWS = 4096          # TC rows per event read back by the e2e leg (a PU200 event has ~3.3 k)


def shard_seeds(rank: int, world: int, n_events: int, base: int = 100):
    """Event seeds of one rank: every rank gets its own `n_events` (weak scaling)."""
    return [base + rank * n_events + i for i in range(n_events)]


def aggregate(local_ms_per_step: float, local_events_per_step: int, world: int, reduce_max=None, reduce_sum=None):
    """Whole-job throughput = all ranks' events / the slowest rank's time."""
    t = local_ms_per_step if reduce_max is None else reduce_max(local_ms_per_step)
    n = local_events_per_step * world if reduce_sum is None else reduce_sum(local_events_per_step)
    return n / (t * 1e-3), t


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([c.strip() for c in line.split(",")])

    def stop(self):
        if self.proc is None:
            return dict(sm_mhz=None, sm_max_mhz=None, reasons=["nvidia-smi unavailable"])
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except (ValueError, IndexError):
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return dict(sm_mhz=float(np.median(sm)) if sm else None, sm_max_mhz=max(mx) if mx else None,
                    reasons=sorted(reasons), samples=len(sm))


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=float(d["hbm_gbs"]), sm_max_mhz=float(d.get("sm_max_mhz", 1965.0)), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def make_events(geo, seeds):
    from lstgen import config_event
    return [config_event(geo, 2, seed=s) for s in seeds]


# ------------------------------------------------------------------------------------------------
def algorithmic_work(lst, geo, slots):
    """Pair-test counts, bytes and flops per stage, summed over `slots`, from the device-side range
    tables of a finished run (pure bookkeeping, never the oracle)."""
    import torch
    M = geo.n_modules
    rowptr = torch.from_numpy(geo.conn_rowptr.astype(np.int64)).to(lst.device)
    col = torch.from_numpy(geo.conn_col.astype(np.int64)).to(lst.device)
    tot = dict(hits=0, md_pairs=0, md=0, ls_pairs=0, ls=0, t3_pairs=0, t3=0, t5_pairs=0, t5c=0, t5=0, pls=0, tc=0, match5=0, match3=0, match_tests=0)
    for s in slots:
        _, c = lst.lst_status(s)
        rg = lst.ranges(s, c)
        ss = rg["sensor_start"].long()
        n_lo, n_up = ss[1:2 * M:2] - ss[0:2 * M:2], ss[2:2 * M + 1:2] - ss[1:2 * M:2]
        nmd = (rg["md_start"][1:] - rg["md_start"][:-1]).long()
        cs = torch.cat([torch.zeros(1, dtype=torch.long, device=lst.device), torch.cumsum(nmd[col], 0)])
        cand = cs[rowptr[1:]] - cs[rowptr[:-1]]
        nls_in = (rg["ls_start"][1:] - rg["ls_start"][:-1]).long()
        nt3_in = (rg["t3_start"][1:] - rg["t3_start"][:-1]).long()
        ls_b = lst.lst_get(s, "ls", c["ls"])["ab"].view(-1, 2)[:, 1].long()
        t3_c = lst.lst_get(s, "t3", c["t3"])["abc"].view(-1, 4)[:, 2].long()
        n_pls = lst.n_pls[s]
        tot["hits"] += c["hit"]; tot["md"] += c["md"]; tot["ls"] += c["ls"]; tot["t3"] += c["t3"]; tot["t5c"] += c["t5c"]
        tot["t5"] += c["t5"]; tot["tc"] += c["tc"]; tot["pls"] += n_pls
        tot["md_pairs"] += int((n_lo * n_up).sum()); tot["ls_pairs"] += int((nmd * cand).sum())
        tot["t3_pairs"] += int(nls_in[ls_b].sum()) if c["ls"] else 0
        tot["t5_pairs"] += int(nt3_in[t3_c].sum()) if c["t3"] else 0
        tot["match5"] += c["m5_cand"]; tot["match3"] += c["m3_cand"]; tot["match_tests"] += c["m5_tests"] + c["m3_tests"]
    nnz, nslot = int(geo.conn_col.size), len(slots)
    stages = {
        # compulsory bytes: each input once, each output once
        "a0": dict(bytes=tot["hits"] * (16 + 16 + 4 + 4) + nslot * 2 * M * 4 * 2, flops=0),
        "a1": dict(bytes=tot["hits"] * 20 + nslot * M * 8 + tot["md"] * 36, flops=FLOPS["md_pair"] * tot["md_pairs"]),
        "a2": dict(bytes=tot["md"] * 28 + nslot * (nnz + M) * 4 + tot["ls"] * 12, flops=FLOPS["ls_pair"] * tot["ls_pairs"]),
        "a3": dict(bytes=tot["ls"] * 12 + tot["md"] * 20 + tot["t3"] * 24, flops=FLOPS["t3_pair"] * tot["t3_pairs"]),
        "a4": dict(bytes=tot["t3"] * 24 + tot["md"] * 20 + tot["t5c"] * 40, flops=FLOPS["t5_pair"] * tot["t5_pairs"]),
        "a5": dict(bytes=tot["t5c"] * (32 + 80 + 92 + 12) + nslot * 7428, flops=FLOPS["dnn_cand"] * tot["t5c"]),
        # a6: the (pLS, object) pairs whose first anchor passes the transverse test must be tested by any exact
        # method; the bucket walk's failed first-anchor tests are overhead, reported as per_event.match_tests
        "a6": dict(bytes=tot["pls"] * (17 + 28) + tot["t5"] * (20 + 80 + 8) + tot["t3"] * (12 + 48 + 8) + tot["tc"] * 12,
                   flops=FLOPS["match_full"] * (tot["match5"] + tot["match3"]) + FLOPS["match_pair"] * (tot["t5"] + tot["t3"])),
        # f1 duplicate cleaning: per TC row the row itself, its hit tuple (written and read), its list links, keep flag, cleaned row
        "f1": dict(bytes=tot["tc"] * (12 + 2 * 40 + 40 + 4 + 4 + 12), flops=0),
    }
    return tot, stages


def stage_of(name):
    return name.split(".")[0]


_CPU_EVENTS = None


def _cpu_worker(args):
    """one oracle process: runs its share of the events, returns (events, seconds)"""
    idx, reps = args
    from oracle import lst_oracle as O
    geo, w, events = _CPU_EVENTS
    O.run(geo, w, events[idx[0]], counts_only=True)
    t0 = time.perf_counter()
    n = 0
    for _ in range(reps):
        for i in idx:
            O.run(geo, w, events[i], counts_only=True)
            n += 1
    return n, time.perf_counter() - t0


def cpu_baseline(geo, w, events, n_single, budget_s=8.0):
    """The oracle as it stands on the host cores: one core, all cores (one process per core, different events), and the
    per-stage split of one event.  Runs BEFORE CUDA is initialised (the workers are forked)."""
    import multiprocessing as mp
    from oracle import lst_oracle as O
    global _CPU_EVENTS
    O.build()
    O.run(geo, w, events[0], counts_only=True)
    t0 = time.perf_counter()
    for ev in events[:n_single]:
        O.run(geo, w, ev, counts_only=True)
    dt1 = time.perf_counter() - t0
    per_core = n_single / dt1
    # per-stage: cumulative runs that stop after each stage
    names = ["sort", "md", "ls", "t3", "t5", "tc"]
    cum = []
    for st in names:
        t0 = time.perf_counter()
        for ev in events[:2]:
            O.run(geo, w, ev, last_stage=st, counts_only=True)
        cum.append((time.perf_counter() - t0) / 2 * 1e3)
    stage_ms = {"a0": cum[0], "a1": cum[1] - cum[0], "a2": cum[2] - cum[1], "a3": cum[3] - cum[2], "a4+a5": cum[4] - cum[3], "a6": cum[5] - cum[4]}
    ncpu = os.cpu_count() or 1
    per_proc = max(1, int(round(budget_s * per_core)))
    _CPU_EVENTS = (geo, w, events)
    jobs = [([(p * per_proc + k) % len(events) for k in range(per_proc)], 1) for p in range(ncpu)]
    try:
        with mp.get_context("fork").Pool(ncpu) as pool:
            res = pool.map(_cpu_worker, jobs)
        all_cores = sum(n for n, _ in res) / max(t for _, t in res)
    except Exception as e:      # a box that cannot fork: report the single-core number only
        all_cores, ncpu = None, 1
    model = "?"
    try:
        for line in open("/proc/cpuinfo"):
            if line.startswith("model name"):
                model = line.split(":", 1)[1].strip(); break
    except OSError:
        pass
    return dict(value=round(per_core, 3), unit=UNIT, cores=1, kind="oracle",
                sample=f"first {n_single} of the PU200 events of one step, single thread, {dt1:.1f} s",
                all_cores=dict(value=None if all_cores is None else round(all_cores, 2), cores=ncpu,
                               sample=f"{ncpu} oracle processes x {per_proc} events each, events / slowest process"),
                cpu_model=model, nproc=os.cpu_count(),
                stage_ms_per_event={k: round(v, 2) for k, v in stage_ms.items()})


def stage_table(prof, stages, n_events, pk, alu_peak, fma_peak):
    """per-stage us / event, bound and achieved fraction of the stage's own roofline"""
    stage_ms = {}
    for k, v in prof.items():
        st_name = "a0" if k == "memset" else stage_of(k)
        stage_ms[st_name] = stage_ms.get(st_name, 0.0) + v
    rows = {}
    for st_name, wk in stages.items():
        t_s = stage_ms[st_name] * 1e-3
        peak_f = fma_peak if st_name == "a5" else alu_peak
        t_hbm, t_alu = wk["bytes"] / (pk["hbm_gbs"] * 1e9), wk["flops"] / (peak_f * 1e12)
        rows[st_name] = dict(us_per_event=round(stage_ms[st_name] * 1e3 / n_events, 3), bound="hbm" if t_hbm >= t_alu else "alu",
                             roofline_us_per_event=round(max(t_hbm, t_alu) * 1e6 / n_events, 4),
                             frac=round(max(t_hbm, t_alu) / t_s, 4) if t_s > 0 else None,
                             gbs=round(wk["bytes"] / t_s / 1e9, 1), tflops=round(wk["flops"] / t_s / 1e12, 3))
    return rows


def run_ours(args):
    rank, world, local = int(os.environ.get("RANK", 0)), int(os.environ.get("WORLD_SIZE", 1)), int(os.environ.get("LOCAL_RANK", 0))
    assert world == args.gpus or world == 1, (world, args.gpus)
    from lstgen import build_geometry, xavier_weights, config_event
    geo = build_geometry(True)
    w = xavier_weights(3)
    E, S = args.events, args.streams
    assert E % S == 0
    events = make_events(geo, shard_seeds(rank, world, E))
    ev_c2 = config_event(geo, 2)                    # configs[2] exactly: seed 3, the single-event headline
    # ---- oracle on the host cores (rank 0, N = 1), before CUDA is initialised: the workers are forked
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        cpu = cpu_baseline(geo, w, events, min(E, args.cpu_sample))

    import torch
    import paper_2403_13166_b200 as P
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback (use --impl reference for the oracle)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    P.load_library()
    caps = P.Caps(n_slots=E, max_hits=114688, max_md=49152, max_ls=49152, max_t3=32768, max_t5c=16384, max_t5=16384, max_pls=4096)
    lst = P.LST(geo, w, caps, device=dev)
    lst.n_pls = [ev.n_pls for ev in events]
    streams = [torch.cuda.Stream(device=dev) for _ in range(S)]
    main = torch.cuda.current_stream(dev)
    for i, ev in enumerate(events):
        lst.load_numpy_event(i, ev)
    torch.cuda.synchronize()
    per = E // S
    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)

    def step():
        if S == 1:
            lst.lst_run_batch(0, E, main)
            return
        ev0 = torch.cuda.Event(); ev0.record(main)
        for si, st in enumerate(streams):
            st.wait_event(ev0)
            lst.lst_run_batch(si * per, per, st)
            e = torch.cuda.Event(); e.record(st); main.wait_event(e)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    for i in range(E):     # a run with any status bit set is a failed run
        bits, c = lst.lst_status(i)
        assert bits == 0 and c["md"] > 0 and c["tc"] > 0, (i, bits, c)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- timed region: K steps, per-step CUDA events, L2 flushed (256 MiB write) between steps ----
    sampler = ClockSampler(local); sampler.start()
    barrier()
    t_wall = time.perf_counter()
    evs = []
    for _ in range(args.steps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(main); step(); b.record(main)
        evs.append((a, b))
    barrier()
    t_wall = time.perf_counter() - t_wall
    clocks = sampler.stop()
    step_ms = [a.elapsed_time(b) for a, b in evs]
    ms_local = float(np.mean(step_ms))

    # ---- e2e: per stream ONE pinned blob in (all its events, lst_load_batch_host) and ONE pinned buffer out (counters + TC
    # rows WITH their original hit indices, lst_read_tc_hits_batch_host): 1 H2D + 1 D2H copy per 16-event batch, every step
    e2e_streams = streams if S > 1 else [main]
    nb = E // len(e2e_streams)
    blobs = [P.pack_batch(events[si * nb:(si + 1) * nb], key16=True) for si in range(len(e2e_streams))]      # 14 bytes per hit
    h_outs = [torch.zeros((nb, 32 + 13 * TC_ROWS), dtype=torch.int32).pin_memory() for _ in e2e_streams]
    h2d = sum(int(b.numel()) for b in blobs)
    d2h = E * (32 * 4 + TC_ROWS * 13 * 4)

    def e2e_step():
        for si, st in enumerate(e2e_streams):
            lst.lst_load_batch_host16(si * nb, nb, blobs[si], stream=st)
            lst.lst_run_batch(si * nb, nb, st)
            lst.lst_read_tc_hits_batch_host(si * nb, nb, h_outs[si], stream=st)

    for _ in range(3):
        e2e_step()
    barrier()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        e2e_step()
    barrier()
    e2e_ms_local = (time.perf_counter() - t0) * 1e3 / args.steps
    for h in h_outs:
        for i in range(nb):
            ntc = int(h[i, P.CNT["tc"]])
            assert int(h[i, 31]) == 0 and 0 < ntc <= TC_ROWS, "e2e run failed or TC rows truncated"
            rows = h[i, 32:32 + 13 * ntc].view(ntc, 13)
            t5 = rows[rows[:, 0] <= 1]
            assert bool((t5[:, 3:] >= 0).all()), "a T5-based candidate came back without its ten hits"
    # rebind the resident inputs for the profile pass
    for i, ev in enumerate(events):
        lst.load_numpy_event(i, ev)
    torch.cuda.synchronize()

    # ---- per-kernel device times (same launch configuration as the timed region) ------------------
    def profile(first, n, reps=5):
        acc = {}
        for r in range(reps + 1):
            flush.zero_()
            torch.cuda.synchronize()
            d = lst.lst_run_batch_profile(first, n, main)
            if r:       # first one is warm-up
                for k, v in d.items():
                    acc[k] = acc.get(k, 0.0) + v / reps
        return acc

    n_prof = E if S == 1 else per       # one stream's share of the batch; the S streams run the same sequence concurrently
    prof = profile(0, n_prof)
    tot, stages = algorithmic_work(lst, geo, range(n_prof))

    # ---- f4: MD / LS graph export of one stream's batch (PAPER.md:127 quotes "1 to 2 ms" for graph building per event)
    torch.cuda.synchronize()
    ga, gb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    for _ in range(3):
        lst.lst_export_graph(0, n_prof, main)
    ga.record(main)
    for _ in range(20):
        lst.lst_export_graph(0, n_prof, main)
    gb.record(main)
    torch.cuda.synchronize()
    graph_ms = ga.elapsed_time(gb) / 20

    # ---- single event: configs[2] exactly (seed 3), one event, one stream ---------------------------------------------
    lst.load_numpy_event(0, ev_c2)
    torch.cuda.synchronize()
    one = streams[0]
    for _ in range(5):
        lst.lst_run_batch(0, 1, one)
    torch.cuda.synchronize()
    bits1, c1 = lst.lst_status(0)
    assert bits1 == 0
    lat = []
    for _ in range(args.single_reps):
        flush.zero_()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        one.wait_stream(main)
        a.record(one); lst.lst_run_batch(0, 1, one); b.record(one)
        main.wait_stream(one)
        lat.append((a, b))
    torch.cuda.synchronize()
    lat_ms = float(np.median([a.elapsed_time(b) for a, b in lat]))
    # back to back, L2 warm (no flush): the steady-state rate of a stream that keeps feeding single events
    a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    a.record(one)
    for _ in range(args.single_reps):
        lst.lst_run_batch(0, 1, one)
    b.record(one)
    torch.cuda.synchronize()
    warm_ms = a.elapsed_time(b) / args.single_reps
    prof1 = profile(0, 1)
    lst.n_pls[0] = ev_c2.n_pls
    tot1, stages1 = algorithmic_work(lst, geo, [0])
    lst.n_pls[0] = events[0].n_pls

    # launch floor: the smallest kernel of the library (a 1-thread bind), back to back on one stream -- the time
    # below which no stage of a small batch can go (report it beside the per-stage fractions)
    torch.cuda.synchronize()
    fa, fb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    fa.record(main)
    for _ in range(200):
        lst.lib.lst_load_event(lst.ctx, 0, 0, None, None, None, None, 0, None, None, None, None, None, lst._st(main))
    fb.record(main)
    torch.cuda.synchronize()
    launch_floor_us = fa.elapsed_time(fb) * 1e3 / 200
    lst.load_numpy_event(0, events[0])
    # fp32 throughput of this GPU, measured with the library's probe kernels
    alu_meas, fma_meas = lst.lst_measure_fp32(False, main), lst.lst_measure_fp32(True, main)

    # ---- configs[3] "per-stage overlap": the same E events split over 1 / 2 / 4 / 8 streams (1, 2, 4, 8 CUDA streams)
    def sweep_point(n_st):
        sts = [torch.cuda.Stream(device=dev) for _ in range(n_st)]
        per_s = E // n_st
        def stp():
            ev0 = torch.cuda.Event(); ev0.record(main)
            for si, st in enumerate(sts):
                st.wait_event(ev0)
                lst.lst_run_batch(si * per_s, per_s, st)
                e = torch.cuda.Event(); e.record(st); main.wait_event(e)
        for _ in range(3):
            stp()
        torch.cuda.synchronize()
        tt = []
        for _ in range(max(5, min(args.steps, 20))):
            flush.zero_()
            a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            a.record(main); stp(); b.record(main)
            tt.append((a, b))
        torch.cuda.synchronize()
        t_ms = float(np.median([a.elapsed_time(b) for a, b in tt]))
        return dict(streams=n_st, events_per_launch=per_s, ms_per_step=round(t_ms, 4), events_per_s=round(E / t_ms * 1e3, 1))
    streams_sweep = [sweep_point(n_st) for n_st in (1, 2, 4, 8) if E % n_st == 0]

    def red_max(v):
        if dist is None:
            return v
        t = torch.tensor([v], dtype=torch.float64, device=dev); dist.all_reduce(t, op=dist.ReduceOp.MAX); return float(t.item())

    value, ms = aggregate(ms_local, E, world, red_max)
    e2e_value, e2e_ms = aggregate(e2e_ms_local, E, world, red_max)
    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    pk = peaks()
    alu_nominal = SM_COUNT * LANES * pk["sm_max_mhz"] * 1e6 / 1e12        # one op per lane per clock
    alu_peak = alu_meas if alu_meas > 0 else alu_nominal
    fma_peak = fma_meas if fma_meas > 0 else 2 * alu_nominal
    stage_rows = stage_table(prof, stages, n_prof, pk, alu_peak, fma_peak)
    roof_stages = {k: dict(us_per_event=v["us_per_event"], bound=v["bound"], frac=v["frac"]) for k, v in stage_rows.items()}
    # overlap: what one stream's launch sequence takes alone (sum of its kernels, measured with events between them) x S streams,
    # against the measured step in which the S sequences run concurrently; per stage = the share of the step during which that stage
    # is busy on some stream (the shares add up to `factor`; > 1 means the streams really overlap)
    chain_ms = sum(prof.values())
    stage_busy = {}
    for k, v in prof.items():
        sn = "a0" if k == "memset" else stage_of(k)
        stage_busy[sn] = stage_busy.get(sn, 0.0) + v
    overlap = dict(streams=S, chain_alone_ms=round(chain_ms, 4), serial_ms=round(S * chain_ms, 4), step_ms=round(ms, 4),
                   factor=round(S * chain_ms / ms, 3),
                   busy_share_of_step={k: round(S * v / ms, 3) for k, v in stage_busy.items()},
                   streams_sweep=streams_sweep,
                   note="chain_alone_ms: one stream's 16-event sequence timed alone with an event after every kernel (adds launch gaps); "
                        "factor = S x chain_alone / step; streams_sweep: the same 64 events over 1 / 2 / 4 / 8 streams, median step")
    # dominant kernel
    kname = max((k for k in prof if k != "memset"), key=lambda k: prof[k])
    kst = stage_of(kname)
    wk = stages[kst]
    k_s = prof[kname] * 1e-3
    if kst == "a0" or wk["bytes"] / (pk["hbm_gbs"] * 1e9) >= wk["flops"] / (alu_peak * 1e12):
        roof = dict(bound="hbm", achieved=round(wk["bytes"] / k_s / 1e9, 2), peak=pk["hbm_gbs"], unit="GB/s", peak_source=f"MEASURED_PEAKS.json ({pk['source']})")
    else:
        peak_f = fma_peak if kst == "a5" else alu_peak
        roof = dict(bound="alu", achieved=round(wk["flops"] / k_s / 1e12, 3), peak=round(peak_f, 2), unit="TFLOP/s",
                    peak_source="measured in this run by lst_measure_fp32 (separately rounded multiply + add)")
    traffic, tsrc = None, None       # DRAM bytes per launch of this kernel from the committed ncu --set full capture
    for tname in ("r03_traffic.csv", "r02_traffic.csv"):
        tpath = os.path.join(ROOT, "profiles", tname)
        if traffic is None and os.path.exists(tpath):
            for line in open(tpath).read().splitlines()[1:]:
                f = line.split(",")
                if f and f[0] == kname:
                    traffic, tsrc = round((float(f[3]) + float(f[4])) * n_prof / float(f[2])), "profiles/" + tname
    roof.update(frac=round(roof["achieved"] / roof["peak"], 4), traffic=traffic, traffic_source=tsrc, kernel=kname, kernel_ms=round(prof[kname], 4),
                kernel_share_of_step=round(prof[kname] / sum(prof.values()), 3), algorithmic_per_unit="60 flop per LS pair test (SURVEY.md 8.d)" if kst == "a2" else None,
                fp32_tflops=dict(unfused_measured=round(alu_meas, 2), fma_measured=round(fma_meas, 2), unfused_nominal=round(alu_nominal, 2),
                                 note="nominal = 148 SM x 128 lanes x sm_max_mhz, one op per lane per clock; the cut kernels may not fuse (north_star)"))
    roof["stages"] = roof_stages      # every stage of the 16-event launch: us / event, bound, fraction of its own roofline
    single = dict(workload="configs[2] exactly: one HL-LHC PU200 event, seed 3, one stream, one lst_run (CUDA-graph replay)",
                  value=round(1e3 / lat_ms, 1), unit=UNIT, us_per_event=round(lat_ms * 1e3, 1),
                  timing=f"median of {args.single_reps} runs, CUDA events on the launching stream, L2 flushed before every run",
                  back_to_back=dict(value=round(1e3 / warm_ms, 1), us_per_event=round(warm_ms * 1e3, 1), note="same event resubmitted without flush (L2 warm)"),
                  launches=lst.launches_per_run(), launch_floor_us=round(launch_floor_us, 2),
                  launch_floor_total_us=round(launch_floor_us * lst.launches_per_run(), 1),
                  stages=stage_table(prof1, stages1, 1, pk, alu_peak, fma_peak),
                  kernels_us={k: round(v * 1e3, 2) for k, v in prof1.items()},
                  objects={k: v for k, v in tot1.items()})

    out = dict(metric=METRIC, value=round(value, 1), unit=UNIT, n_gpus=world, steps=args.steps, warmup=max(args.warmup, 3),
               ms_per_step=round(ms, 4), higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f32", data="synthetic",
               config=dict(workload=WORKLOAD, events_per_step_per_gpu=E, streams=S, events_per_launch=per,
                           l2="flushed between steps (256 MiB write outside the per-step CUDA-event brackets)",
                           timing="mean of per-step CUDA-event durations on the launching stream, max over ranks",
                           parallelism=f"replicas x{world}" if world > 1 else "single GPU"),
               e2e=dict(value=round(e2e_value, 1), unit=UNIT, h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h, ms_per_step=round(e2e_ms, 4),
                        timing="wall clock around K steps incl. pinned H2D of every input and D2H of counters + TC rows with their hit indices",
                        host_link_gbs=round((h2d + d2h) / (e2e_ms * 1e-3) / 1e9, 1)),
               gpu_launches=args.steps * S * lst.launches_per_run(), launch_floor_us=round(launch_floor_us, 2),
               step_ms=dict(min=round(float(np.min(step_ms)), 4), median=round(float(np.median(step_ms)), 4), max=round(float(np.max(step_ms)), 4)),
               clocks=clocks, roofline=roof, cpu_baseline=cpu, stages=stage_rows, overlap=overlap, single_event=single,
               graph_export=dict(us_per_event=round(graph_ms * 1e3 / n_prof, 3), us_per_launch=round(graph_ms * 1e3, 2), events_per_launch=n_prof,
                                 nodes_per_event=round(tot["md"] / n_prof, 1), edges_per_event=round(tot["ls"] / n_prof, 1),
                                 note="lst_export_graph after lst_run: packs node features + CSR columns (SPEC.md 4.8); the paper quotes 1 to 2 ms per event for graph building (PAPER.md:127, other hardware)"),
               kernels_ms={k: round(v, 4) for k, v in prof.items()},
               per_event=dict(us=round(ms * 1e3 / E, 2), objects={k: round(v / n_prof, 1) for k, v in tot.items()}),
               wall_ms_per_step_incl_flush=round(t_wall * 1e3 / args.steps, 3))
    print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def run_sweep(args):
    """configs[4]: displaced-track and occupancy stress.  config 2 recipe scaled to pile-up 0 / 100 / 200 / 300 plus 500
    displaced particles, 8 events per point (seeds 200-231): events/s, object counts and the overflow status per point."""
    import torch
    import paper_2403_13166_b200 as P
    from lstgen import build_geometry, config_event, xavier_weights
    if not torch.cuda.is_available():
        raise SystemExit("needs a CUDA device (no CPU fallback)")
    geo, w = build_geometry(True), xavier_weights(3)
    caps = P.Caps(n_slots=8, max_hits=196608, max_md=98304, max_ls=98304, max_t3=65536, max_t5c=32768, max_t5=32768, max_pls=8192)
    lst = P.LST(geo, w, caps)
    st = torch.cuda.Stream()
    points, seed = [], 200
    for pu in (0, 100, 200, 300):
        evs = [config_event(geo, 4, seed=seed + i, pileup=pu) for i in range(8)]
        seed += 8
        for i, ev in enumerate(evs):
            lst.load_numpy_event(i, ev)
        torch.cuda.synchronize()
        for _ in range(3):
            lst.lst_run_batch(0, 8, st)
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(st)
        for _ in range(args.steps):
            lst.lst_run_batch(0, 8, st)
        b.record(st)
        torch.cuda.synchronize()
        ms = a.elapsed_time(b) / args.steps
        stat, cs = zip(*[lst.lst_status(i) for i in range(8)])
        mean = lambda k: round(float(np.mean([c[k] for c in cs])), 1)
        points.append(dict(pileup=pu, events_per_s=round(8 / ms * 1e3, 1), us_per_event=round(ms * 1e3 / 8, 1), status_or=int(np.bitwise_or.reduce(stat)),
                           hits=mean("hit"), md=mean("md"), ls=mean("ls"), t3=mean("t3"), t5c=mean("t5c"), t5=mean("t5"),
                           pls=round(float(np.mean([ev.n_pls for ev in evs])), 1), tc=mean("tc")))
    lst.close()
    print(json.dumps(dict(metric="events/s vs occupancy (configs[4]: PU-scaled config 2 + 500 displaced, 8 events per point, seeds 200-231)",
                          unit=UNIT, n_gpus=1, steps=args.steps, data="synthetic", dtype="f32", points=points,
                          timing="8-event batched launches back to back on one stream (CUDA-graph replay), CUDA events, L2 warm")))


def run_reference(args):
    """The CPU oracle as it stands, on the host cores, on the same config / metric / unit."""
    rank = int(os.environ.get("RANK", 0))
    if rank != 0:
        return
    from lstgen import build_geometry, xavier_weights
    from oracle import lst_oracle as O
    O.build()
    geo = build_geometry(True)
    w = xavier_weights(3)
    n_s = args.ref_events
    events = make_events(geo, shard_seeds(0, 1, n_s))
    for _ in range(max(1, min(args.warmup, 2))):
        O.run(geo, w, events[0], counts_only=True)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        for ev in events:
            O.run(geo, w, ev, counts_only=True)
    dt = time.perf_counter() - t0
    v = args.steps * n_s / dt
    sample = f"each step = the first {n_s} of the {args.events} PU200 events of our arm's step, single thread"
    print(json.dumps(dict(impl="reference", metric=METRIC, value=round(v, 3), unit=UNIT, n_gpus=args.gpus, steps=args.steps,
                          warmup=args.warmup, ms_per_step=round(dt * 1e3 / args.steps, 3), higher_is_better=True, scaling="weak",
                          vs_baseline=None, dtype="f32", data="synthetic",
                          config=dict(workload=WORKLOAD, events_per_step=n_s, sample=sample),
                          cpu_baseline=dict(value=round(v, 3), unit=UNIT, cores=1, kind="oracle", sample=sample),
                          e2e=dict(value=round(v, 3), unit=UNIT, h2d_bytes_per_step=0, d2h_bytes_per_step=0),
                          gpu_launches=0)))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--events", type=int, default=64, help="PU200 events per step per GPU (configs[3]: 64)")
    ap.add_argument("--streams", type=int, default=4, help="CUDA streams the batch is split over (configs[3]: 4 x 16 events)")
    ap.add_argument("--cpu-sample", type=int, default=48)
    ap.add_argument("--ref-events", type=int, default=8)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--single-reps", type=int, default=50, help="timed runs of the single-event (configs[2]) block")
    ap.add_argument("--config", type=int, default=3, choices=[3, 4], help="3: the batched PU200 throughput line; 4: the occupancy sweep")
    args = ap.parse_args()
    if args.impl == "reference":
        run_reference(args)
    elif args.config == 4:
        run_sweep(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
