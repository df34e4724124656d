"""bench.py -- throughput of the JUMP hot path on B200 (one JSON line on stdout).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--mode respa] [--impl reference]

Workload (default): BASELINE.json configs[4], the largest single-GPU configuration -- 999 999-atom flexible water
box, 215.2 A, cutoffs 6 / 12 A, JUMP-RESPA with inner step 1 fs (bonded + short-range pair force) and outer step
4 fs (jump half-phases C'J' / J'C' in place of the 6-12 A pair force), equilibrated by BAOAB steps (untimed).
A "step" is one inner MD step of 1 fs, i.e. a quarter of one jump_respa_step(1): the whole hot path -- outer jump
phases, A-O-A, list rebuild at its natural period, F0 = bonded + short-range pairs -- over the box.  Metric: ns/day
(higher is better); atom-steps/s, the same box under plain JUMP and under same-GPU BAOAB / BAOAB-RESPA with the
unsplit 12 A force, the per-kernel rooflines, the end-to-end figure through host buffers and the fp64 oracle on the
host cores ride along in the same line; `secondary` repeats JUMP vs BAOAB on configs[1] (12 000 atoms).
N > 1: the path does not shard on one GPU's box sizes (replicas only), so every rank
runs an independent replica with its own seed; value = sum over ranks / max-over-ranks time.
"""
import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np

BLOCK = 20                 # steps per timed API call: a multiple of n_inner and of the rebuild period
FLOPS_PER_PAIR = 2 * 50    # ~50 FP32-pipe instructions per in-range half pair, counted as FMAs
PROPOSAL_INSTR = 250       # ~150 FP32-pipe + ~100 INT-pipe (one Philox block) instructions per proposal
CHAIN_INSTR = 60           # chain set-up + expiry per half-phase chain
L2_FLUSH_BYTES = 256 << 20


def ns_per_day(steps_per_s, dt_fs):
    return 86400.0 * steps_per_s * dt_fs * 1e-6


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md, clocks line)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], [], set()
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm_gbs=d.get("hbm_gbs", 6650.0), sm_max_mhz=d.get("sm_max_mhz", 1965.0), source="measured")
    return dict(hbm_gbs=6650.0, sm_max_mhz=1965.0, source="fallback")


def oracle_sample(sysd, run, mode, budget_s, state=None):
    """The fp64 oracle as it stands on the host cores: whole-box steps of the same workload in the same mode until
    ~budget_s of CPU time (at least one API unit).  state = (pos, vel) to start from, else the generator's lattice
    state after two oracle BAOAB steps.  Returns (steps, seconds, cores, description)."""
    from oracle import jump_oracle as jo
    s2 = sysd if state is None else dict(sysd, pos=state[0], vel=state[1])
    o = jo.Oracle(s2, **run)
    if state is None:
        o.baoab_step(2)
    unit = run["n_inner"] if mode == "respa" else 1
    call = (lambda: o.jump_respa_step(1)) if mode == "respa" else (lambda: o.jump_step(1))
    t0 = time.perf_counter()
    n = 0
    while True:
        call()
        n += unit
        dt = time.perf_counter() - t0
        if dt > budget_s or n >= 400:
            break
    o.close()
    what = "%d whole-box %s steps of 1 fs of the same %d-atom box (%.1f s), started from %s" % (
        n, "JUMP-RESPA" if mode == "respa" else "JUMP", sysd["n_atoms"], dt,
        "the state the timed GPU run started from" if state is not None else "the lattice state (2 oracle BAOAB steps)")
    return n, dt, jo.num_threads(), what


def run_reference(args):
    """--impl reference: the fp64 oracle, as it stands, on the host cores (same config, mode, metric and unit).  The
    GPU arm equilibrates the box with its own BAOAB steps before timing; the oracle cannot do that for 10^6 atoms within
    minutes, so its bounded sample starts from the generator's lattice state (said in config.workload)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_2412_15073_b200 import workloads as wl
    sysd, run = wl.make_config(args.config)
    n, dt, cores, what = oracle_sample(sysd, run, args.mode, budget_s=max(10.0, 0.02 * args.steps))
    sps = n / dt
    val = ns_per_day(sps, run["dt_fs"])
    line = {"impl": "reference", "metric": "ns_per_day_jump" if args.mode == "jump" else "ns_per_day_jump_respa", "value": val,
            "unit": "ns/day", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / n,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE configs[%d]: %d-atom flexible water box, %s; oracle sample: %s"
                                   % (args.config, sysd["n_atoms"], "JUMP-RESPA n_inner %d" % run["n_inner"] if args.mode == "respa" else "JUMP", what)},
            "atom_steps_per_s": sps * sysd["n_atoms"],
            "cpu_baseline": {"value": val, "unit": "ns/day", "cores": cores, "kind": "oracle", "sample": what},
            "e2e": {"value": val, "unit": "ns/day", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def _dist_setup(n_gpus):
    """One process per GPU (torchrun env).  Returns (rank, world, dist or None)."""
    rank, world = int(os.environ.get("RANK", "0")), int(os.environ.get("WORLD_SIZE", "1"))
    if world == 1:
        return 0, 1, None
    import torch.distributed as dist
    os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
    dist.init_process_group("nccl")
    return rank, world, dist


def run_cpu_baseline(sysd, run, mode, state, budget_s=15.0):
    """cpu_baseline leg: the oracle on the same workload, same mode, from the state the timed GPU run started from."""
    n, dt, cores, what = oracle_sample(sysd, run, mode, budget_s, state=state)
    sps = n / dt
    return {"value": ns_per_day(sps, run["dt_fs"]), "unit": "ns/day", "cores": cores, "kind": "oracle", "sample": what,
            "atom_steps_per_s": sps * sysd["n_atoms"]}


def timed_blocks(torch, sim, stream, call, n_steps, block, flush):
    """Time n_steps as ceil(n_steps/block) API calls; CUDA events on the context's stream bracket each call, the L2
    flush (a 256 MiB write) sits between the brackets.  Returns total milliseconds of the bracketed regions."""
    evs = []
    left = n_steps
    with torch.cuda.stream(stream):
        while left > 0:
            b = min(block, left)
            flush.zero_()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record(stream)
            call(b)
            e1.record(stream)
            evs.append((e0, e1))
            left -= b
    stream.synchronize()
    return sum(a.elapsed_time(b) for a, b in evs)


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the `ncu --set full` captures of
# `python bench.py --steps 40 --warmup 8 --equil 60 --no-cpu-baseline --secondary-config -1` on the default workload
# (profiles/r2_cfg4_README.md, profiles/r2_cfg4_dram_bytes.csv); other workloads have no capture: null
NCU_TRAFFIC_CFG4 = {"pair": 653.1e6, "update": 870.1e6, "build": 2584.0e6, "bonded": 41.8e6}   # build: k_build_rows + k_sort
BONDED_BYTES_PER_ATOM = 56    # per water: 16 B record + 3 x (16 + 16 B read, 16 B written)


def kernel_rooflines(torch, sim, stream, step_call, K, block, flush, run, n, props, peaks, traffic=None):
    """Per-kernel device times of K more steps (CUDA events on the streams the kernels are launched on, recorded by
    the library around each kernel group) against each kernel's roofline.  Returns (dominant line, other lines).
    The bonded kernels run on a side stream beside k_pair, so their bracket inside a step is stretched by the overlap:
    their own time is taken from five stand-alone evaluations (jump_get_forces(3): bonded kernels + one 13 us copy)."""
    with torch.cuda.stream(stream):
        sim.reset_stats()
        r0 = sim.stats()["rebuilds"]
        sim.set_profiling(True)
        timed_blocks(torch, sim, stream, step_call, K, block, flush)
        prof = sim.profile()
        sim.set_profiling(False)
        pstats = sim.stats()
        n_pairs_ordered = sim.count_pairs(0, run["r_short"])           # ordered in-range entries of the short row
        row_entries = sum(sim.count_pairs(k, 1e3) for k in (0, 1, 2) if pstats["cap_row"][k])
        sim.forces(3)
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        for _ in range(5):
            sim.forces(3)
        e1.record(stream)
        stream.synchronize()
        bonded_ms = e0.elapsed_time(e1) / 5
    rebuilds = max(pstats["rebuilds"] - r0, 1)
    tot = {k: v[0] for k, v in prof.items()}
    tot["bonded"] = bonded_ms * prof["bonded"][1]
    tot_prof = sum(tot.values())
    share = {k: (v / tot_prof if tot_prof else 0.0) for k, v in tot.items()}
    peak_tflops = props.multi_processor_count * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    alu_src = "%d SMs x 128 FP32 lanes x 2 x %.0f MHz (%s sm_max_mhz)" % (props.multi_processor_count, peaks["sm_max_mhz"],
                                                                      peaks["source"])
    hbm_src = "%s HBM copy bandwidth (MEASURED_PEAKS.json)" % peaks["source"]

    def avg_ms(cat):
        return prof[cat][0] / max(prof[cat][1], 1)

    def alu_line(kernel, flops, what, cat):
        ach = flops / (avg_ms(cat) * 1e-3) / 1e12 if avg_ms(cat) > 0 else 0.0
        return {"kernel": kernel, "bound": "alu", "achieved": ach, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": ach / peak_tflops, "traffic": None, "peak_source": alu_src, "algorithmic": what,
                "avg_launch_us": 1e3 * avg_ms(cat), "share_of_step": share[cat]}

    def hbm_line(kernel, nbytes, what, ms, cat):
        ach = nbytes / (ms * 1e-3) / 1e9 if ms > 0 else 0.0
        return {"kernel": kernel, "bound": "hbm", "achieved": ach, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": ach / peaks["hbm_gbs"], "traffic": None, "peak_source": hbm_src, "algorithmic": what,
                "avg_launch_us": 1e3 * ms, "share_of_step": share[cat]}

    half_pairs = n_pairs_ordered / 2.0
    n_upd = max(prof["update"][1], 1)
    chains = 2.0 * n * (2 if run["flags"] & 2 else 1)                  # half-phases x (C' [+ J']) per jump update launch
    upd_instr = pstats["proposals"] / n_upd * PROPOSAL_INSTR + chains * CHAIN_INSTR
    build_ms = prof["build"][0] / rebuilds                             # k_sort + k_build_rows (and their idle launches), per rebuild
    lines = {
        "pair": alu_line("k_pair (short-range switched pair gradient, a5)", half_pairs * FLOPS_PER_PAIR,
                         "%.0f in-range half pairs x %d flop" % (half_pairs, FLOPS_PER_PAIR), "pair"),
        "update": alu_line("k_update (jump chains of the phases it carries + A-O-A, a6-a8), average over its launches",
                           2.0 * upd_instr,
                           "%.0f proposals x %d + %.0f chains x %d FP32/INT-pipe instructions, x 2 flop, per launch"
                           % (pstats["proposals"] / n_upd, PROPOSAL_INSTR, chains, CHAIN_INSTR), "update"),
        "build": hbm_line("k_sort + k_build_rows (a1-a3), per rebuild", row_entries * 4.0 + n * 48.0,
                          "%.0f row entries x 4 B + %d atoms x 48 B" % (row_entries, n), build_ms, "build"),
        "bonded": hbm_line("k_bonded_mol (+ k_bonded_csr) (a4), stand-alone", n * float(BONDED_BYTES_PER_ATOM),
                           "%d atoms x %d B" % (n, BONDED_BYTES_PER_ATOM), bonded_ms, "bonded"),
    }
    for k, line in lines.items():
        if traffic and k in traffic:
            line["traffic"] = traffic[k]
            line["traffic_source"] = "ncu --set full capture of the %s kernel, profiles/r2_cfg4_dram_bytes.csv (bytes per launch)" % k
    share_note = ("device time per kernel group / sum over groups (bonded: stand-alone time x launches; inside a step it "
                  "runs on a side stream beside k_pair)")
    dominant = max(lines, key=lambda k: share[k])
    roofline = dict(lines[dominant], kernel_ms_share=share, share_note=share_note)
    return roofline, {k: v for k, v in lines.items() if k != dominant}


def comparators(torch, sim, stream, flush, run, n, steps):
    """Same box, same state, other schemes (reported baselines): plain JUMP, BAOAB with the unsplit force to r_long,
    and -- for the RESPA headline -- nothing else: BAOAB-RESPA needs its own context (a flag fixed at init)."""
    out = {}
    with torch.cuda.stream(stream):
        for name, call in (("jump", sim.jump_step), ("baoab", sim.baoab_step)):
            call(2 * BLOCK)   # 40 untimed steps: the rows only the other scheme reads leave the active set (36 steps)
            sim.sync()
            ms = timed_blocks(torch, sim, stream, call, steps, BLOCK, flush)
            out[name] = {"ms_per_step": ms / steps, "ns_per_day": ns_per_day(steps / (ms * 1e-3), run["dt_fs"]),
                         "atom_steps_per_s": n * steps / (ms * 1e-3), "steps": steps}
    out["baoab"]["force"] = "unsplit pair force to r_long = %.0f A" % run["r_long"]
    return out


def secondary_config(torch, jb, wl, dev, stream, flush, config, equil, steps):
    """JUMP vs same-GPU BAOAB on a small box (BASELINE configs[1]: 'JUMP vs BAOAB'), where every kernel is bound by
    latency rather than throughput."""
    sysd, run = wl.make_config(config)
    n = sysd["n_atoms"]
    with torch.cuda.stream(stream):
        sim = jb.JumpSim(sysd, device=dev, stream=stream, **run)
        sim.set_lax_skin(True)
        sim.baoab_step(equil)
        sim.set_lax_skin(False)
        sim.sync()
        sim.reset_stats()
        cmp_ = comparators(torch, sim, stream, flush, run, n, steps)
        st = sim.stats()
    sim.close()
    return {"workload": "BASELINE configs[%d]: %d-atom flexible water box %.1f A, equilibrated by %d BAOAB steps + 40 steps of the timed scheme"
                        % (config, n, sysd["box"], equil),
            "jump": cmp_["jump"], "baoab_same_gpu": cmp_["baoab"],
            "jump_vs_baoab": cmp_["baoab"]["ms_per_step"] / cmp_["jump"]["ms_per_step"], "error": st["error"],
            "max_disp_A": st["max_disp"]}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=1000)
    ap.add_argument("--warmup", type=int, default=100)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--equil", type=int, default=600, help="untimed BAOAB equilibration steps from the lattice start")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--secondary-config", type=int, default=1,
                    help="also report JUMP vs BAOAB on this small config, N=1 only; -1: skip")
    ap.add_argument("--mode", default="respa", choices=["jump", "respa"])
    ap.add_argument("--r-mid", type=float, default=None, help="outer ring edge r_M (default: the config's)")
    ap.add_argument("--r-mid-in", type=float, default=None, help="inner ring edge r_A (default: the config's)")
    ap.add_argument("--skin", type=float, default=None)
    ap.add_argument("--nlist-every", type=int, default=None)
    ap.add_argument("--eps-jump", type=float, default=None)
    ap.add_argument("--cell-edge", type=float, default=None, help="edge of the contract grid's cells, A (default: the library's)")
    ap.add_argument("--lanes", type=int, default=0, help="lanes per jump chain in k_update: 1, 4, 8, 16 (default 0: the library's choice)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    from paper_2412_15073_b200 import binding as jb, workloads as wl, replicas
    rank, world, dist = _dist_setup(args.gpus)
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)
    props = torch.cuda.get_device_properties(dev)
    peaks = measured_peaks()

    sysd, run = wl.make_config(args.config)
    run = dict(run, seed=replicas.rank_seed(run["seed"], rank))       # independent replicas
    for key, val in (("r_mid", args.r_mid), ("r_mid_in", args.r_mid_in), ("skin", args.skin), ("nlist_every", args.nlist_every),
                     ("eps_jump", args.eps_jump), ("cell_edge", args.cell_edge)):
        if val is not None:
            run[key] = val
    n, dt_fs = sysd["n_atoms"], run["dt_fs"]
    respa = args.mode == "respa"
    per_call = run["n_inner"] if respa else 1                          # MD steps of length dt per API unit
    block = BLOCK
    stream = torch.cuda.Stream(dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    with torch.cuda.stream(stream):
        sim = jb.JumpSim(sysd, device=dev, stream=stream, **run)
        if args.lanes:
            sim.set_lanes(args.lanes)
        sim.set_lax_skin(True)                                         # the lattice start is hot: no skin check while it relaxes
        sim.baoab_step(args.equil)
        sim.set_lax_skin(False)                                        # from here on a displacement beyond skin/2 is an error
        sim.sync()
        step_call = (lambda b: sim.jump_respa_step(b // per_call)) if respa else sim.jump_step
        # still equilibration: 40 steps of the timed scheme, after which the rows only BAOAB reads (the full 12 A list) have
        # left the library's active set -- they would otherwise be rebuilt during the first 36 steps of a short timed run
        step_call(2 * block)
        sim.sync()
        sim.reset_stats()
        rebuilds0 = sim.stats()["rebuilds"]                             # the sort counter runs on through reset_stats
        K = max(args.steps // block * block, block)
        W = max(args.warmup, 3)
        W_steps = max((W + block - 1) // block * block, block)
        step_call(W_steps)
        sim.sync()
        state0 = (sim.pos.detach().cpu().numpy().astype(np.float64), sim.vel.detach().cpu().numpy().astype(np.float64))

    # ---- timed region: K steps, device time, max over ranks --------------------------------------------------
    sampler = ClockSampler(local)
    sampler.start()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize(dev)
    l0 = sim.launches
    wall0 = time.perf_counter()
    ms = timed_blocks(torch, sim, stream, step_call, K, block, flush)
    torch.cuda.synchronize(dev)
    wall = time.perf_counter() - wall0
    if dist is not None:
        dist.barrier()
    launches = sim.launches - l0
    clocks = sampler.stop()
    timed_error = None
    try:
        sim.sync()                                                     # any device error flag (skin, bound, overflow) is reported
    except jb.JumpError as e:
        timed_error = str(e)
    ms_max = replicas.max_over_ranks(ms, dist, dev)
    stats = sim.stats()

    # ---- per-kernel times of K more steps (CUDA events on the launch streams, separate pass) -------------------
    Kp = min(K, 200)
    roofline, roofline_other = kernel_rooflines(torch, sim, stream, step_call, Kp, block, flush, run, n, props, peaks,
                                                traffic=NCU_TRAFFIC_CFG4 if args.config == 4 else None)

    # ---- the same box under plain JUMP and under same-GPU BAOAB with the unsplit r_long force -------------------
    same_box = comparators(torch, sim, stream, flush, run, n, min(K, 200))

    # ---- end to end through the public API with HOST buffers -------------------------------------------------
    with torch.cuda.stream(stream):
        Ke = min(K, 200)
        hp = sim.pos.detach().cpu().pin_memory()
        hv = sim.vel.detach().cpu().pin_memory()
        sim.run_host(hp, hv, block, mode=args.mode)                      # warm-up
        stream.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(stream)
        calls = 0
        for _ in range(max(Ke // block, 1)):
            sim.run_host(hp, hv, block, mode=args.mode)
            calls += 1
        e1.record(stream)
        stream.synchronize()
        ms_e = e0.elapsed_time(e1)
    ms_e_max = replicas.max_over_ranks(ms_e, dist, dev)
    e2e_steps = calls * block
    bytes_each_way = 2 * n * 3 * 4
    e2e = {"value": world * ns_per_day(e2e_steps / (ms_e_max * 1e-3), dt_fs), "unit": "ns/day",
           "h2d_bytes_per_step": bytes_each_way / block, "d2h_bytes_per_step": bytes_each_way / block,
           "l2": "not flushed between calls (the host round trip itself evicts the state: %d MB each way)" % (bytes_each_way >> 20),
           "call": "JumpSim.run_host: pinned host (x, v) -> device, jump_refresh_lazy (rows rebuilt only if an atom left its "
                   "skin/2 ball), %d steps, device -> host, per call" % block}
    err_end = sim.stats()["error"]
    sim.close()

    second = None
    if rank == 0 and world == 1 and args.secondary_config >= 0:
        second = secondary_config(torch, jb, wl, dev, stream, flush, args.secondary_config, 2000, 1000)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = run_cpu_baseline(sysd, run, args.mode, state0)

    if rank == 0:
        sps = K / (ms_max * 1e-3)
        value = world * ns_per_day(sps, dt_fs)
        line = {"metric": "ns_per_day_jump" if not respa else "ns_per_day_jump_respa", "value": value, "unit": "ns/day",
                "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_max / K, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "BASELINE configs[%d]: %d-atom flexible water box %.1f A, r_c %.0f / r_long %.0f A, "
                                       "dt %.0f fs, %s, equilibrated by %d BAOAB steps + 40 steps of the timed scheme"
                                       % (args.config, n, sysd["box"], run["r_short"], run["r_long"], dt_fs,
                                          "JUMP-RESPA n_inner %d (outer step %.0f fs; one step = one inner step)" % (run["n_inner"], run["n_inner"] * dt_fs)
                                          if respa else "JUMP (C'J'AOAJ'C')", args.equil),
                           "eps_jump": run["eps_jump"], "r_mid_in": run["r_mid_in"], "r_mid": run["r_mid"], "skin": run["skin"],
                           "nlist_every": run["nlist_every"], "cell_edge": run.get("cell_edge", 0.0), "steps_per_api_call": block,
                           "l2": "value: flushed by a 256 MiB write between timed API calls (outside the event brackets); e2e: not flushed",
                           "baseline_note": "there is no reference implementation (the paper's lives in Tinker-HP): --impl reference and "
                                            "cpu_baseline time this repo's own fp64 oracle; absolute ns/day and roofline fractions are the figures of merit",
                           "parallelism": "independent replicas x%d" % world},
                "atom_steps_per_s": world * sps * n,
                "clocks": clocks, "gpu_launches": launches, "wall_s": wall,
                "e2e": e2e, "roofline": roofline, "roofline_other": roofline_other,
                "same_box": {"jump": same_box["jump"], "baoab_same_gpu": same_box["baoab"],
                             "jump_vs_baoab": same_box["baoab"]["ms_per_step"] / same_box["jump"]["ms_per_step"],
                             "jump_respa_vs_baoab": same_box["baoab"]["ms_per_step"] / (ms_max / K) if respa else None},
                "events": {"proposals_per_atom_step": stats["proposals"] / (n * (K + W_steps)),
                           "accepts_per_atom_step": stats["accepts"] / (n * (K + W_steps)), "max_p": stats["max_p"],
                           "timed_region_error": timed_error,
                           "max_disp_A": stats["max_disp"], "rebuilds": stats["rebuilds"] - rebuilds0,
                           "steps_per_rebuild": (K + W_steps) / max(stats["rebuilds"] - rebuilds0, 1), "error": err_end}}
        if second is not None:
            line["secondary"] = second
        if cpu is not None:
            line["cpu_baseline"] = cpu
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
