"""bench.py -- throughput of the JUMP hot path on B200 (one JSON line on stdout).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 1] [--impl reference]

A "step" is one jump_step(1): the whole hot path (jump half-phases C'J', A-O-A, list rebuild at its natural
period, F0 = bonded + short-range pairs, jump half-phases J'C') over one synthetic water box.  Workload:
BASELINE.json configs[1] (12 000 atoms, 49.3 A, cutoffs 6 / 12 A, dt 1 fs), equilibrated by 2 000 BAOAB steps
(untimed).  Metric: ns/day (higher is better); atom-steps/s, same-GPU BAOAB with the unsplit 12 A force,
the kernel roofline and the fp64 oracle on the host cores ride along in the same line.
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

BLOCK = 10                 # steps per timed block = nlist_every, so every block holds exactly one rebuild
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


def run_reference(args):
    """--impl reference: the fp64 oracle, as it stands, on the host cores (same config, metric and unit)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from oracle import jump_oracle as jo
    from paper_2412_15073_b200 import workloads as wl
    sysd, run = wl.make_config(args.config)
    o = jo.Oracle(sysd, **run)
    o.jump_step(max(args.warmup, 1))
    t0 = time.perf_counter()
    o.jump_step(args.steps)
    dt = time.perf_counter() - t0
    sps = args.steps / dt
    val = ns_per_day(sps, run["dt_fs"])
    cores = jo.num_threads()
    line = {"impl": "reference", "metric": "ns_per_day_jump", "value": val, "unit": "ns/day", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BASELINE configs[%d]: %d-atom flexible water box, lattice start (not equilibrated)"
                                   % (args.config, sysd["n_atoms"])},
            "atom_steps_per_s": sps * sysd["n_atoms"],
            "cpu_baseline": {"value": val, "unit": "ns/day", "cores": cores, "kind": "oracle",
                             "sample": "%d whole-box JUMP steps" % args.steps},
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


def run_cpu_baseline(sysd, run, budget_s=15.0):
    """The fp64 oracle as it stands on the host cores: whole-box JUMP steps of the same workload until ~budget_s."""
    from oracle import jump_oracle as jo
    o = jo.Oracle(sysd, **run)
    o.jump_step(1)
    t0 = time.perf_counter()
    n = 0
    while True:
        o.jump_step(1)
        n += 1
        dt = time.perf_counter() - t0
        if dt > budget_s or n >= 200:
            break
    o.close()
    sps = n / dt
    return {"value": ns_per_day(sps, run["dt_fs"]), "unit": "ns/day", "cores": jo.num_threads(), "kind": "oracle",
            "sample": "%d whole-box JUMP steps of the same %d-atom box (%.1f s)" % (n, sysd["n_atoms"], dt),
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


# dram__bytes_read.sum + dram__bytes_write.sum per launch from the `ncu --set full` captures of this command on the
# configs[1] workload (profiles/r1_final_README.md); other workloads have no capture: null
NCU_TRAFFIC_CFG1 = {"update": 9.67e6, "pair": 7.99e6, "build": 6.16e6}


def kernel_rooflines(torch, sim, stream, step_call, K, block, flush, run, n, props, peaks, traffic=None):
    """Per-kernel device times of K more steps (CUDA events on the streams the kernels are launched on, recorded by
    the library around each kernel group) against each kernel's roofline.  Returns (dominant line, other lines)."""
    with torch.cuda.stream(stream):
        sim.reset_stats()
        r0 = sim.stats()["rebuilds"]
        sim.set_profiling(True)
        timed_blocks(torch, sim, stream, step_call, K, block, flush)
        prof = sim.profile()
        sim.set_profiling(False)
        pstats = sim.stats()
        n_pairs_ordered = sim.count_pairs(0, run["r_short"])           # ordered in-range entries of the short row
        row_entries = sum(sim.count_pairs(k, 1e3) for k in (0, 1, 2, 3) if pstats["cap_row"][k])
    rebuilds = max(pstats["rebuilds"] - r0, 1)
    tot_prof = sum(v[0] for v in prof.values())
    share = {k: (v[0] / tot_prof if tot_prof else 0.0) for k, v in prof.items()}
    peak_tflops = props.multi_processor_count * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
    alu_src = "%d SMs x 128 FP32 lanes x 2 x %.0f MHz (%s sm_max_mhz)" % (props.multi_processor_count, peaks["sm_max_mhz"],
                                                                      peaks["source"])

    def avg_ms(cat):
        return prof[cat][0] / max(prof[cat][1], 1)

    def alu_line(kernel, flops, what, cat):
        ach = flops / (avg_ms(cat) * 1e-3) / 1e12 if avg_ms(cat) > 0 else 0.0
        return {"kernel": kernel, "bound": "alu", "achieved": ach, "peak": peak_tflops, "unit": "TFLOP/s",
                "frac": ach / peak_tflops, "traffic": None, "peak_source": alu_src, "algorithmic": what,
                "avg_launch_us": 1e3 * avg_ms(cat), "share_of_step": share[cat]}

    half_pairs = n_pairs_ordered / 2.0
    n_upd = max(prof["update"][1], 1)
    chains = 2.0 * n * (2 if run["flags"] & 2 else 1)                  # half-phases x (C' [+ J']) per update launch
    upd_instr = pstats["proposals"] / n_upd * PROPOSAL_INSTR + chains * CHAIN_INSTR
    build_ms = prof["build"][0] / rebuilds                             # sort (5 kernels) + k_build_rows, per rebuild
    build_bytes = row_entries * 4.0 + n * 48.0
    build_ach = build_bytes / (build_ms * 1e-3) / 1e9 if build_ms > 0 else 0.0
    lines = {
        "pair": alu_line("k_pair (short-range switched pair gradient, a5)", half_pairs * FLOPS_PER_PAIR,
                         "%.0f in-range half pairs x %d flop" % (half_pairs, FLOPS_PER_PAIR), "pair"),
        "update": alu_line("k_update (jump chains C'J' of two half-phases + A-O-A, a6-a8)", 2.0 * upd_instr,
                           "%.0f proposals x %d + %.0f chains x %d FP32/INT-pipe instructions, x 2 flop"
                           % (pstats["proposals"] / n_upd, PROPOSAL_INSTR, chains, CHAIN_INSTR), "update"),
        "build": {"kernel": "sort + k_build_rows (a1-a3), one group per rebuild", "bound": "hbm", "achieved": build_ach,
                  "peak": peaks["hbm_gbs"], "unit": "GB/s", "frac": build_ach / peaks["hbm_gbs"], "traffic": None,
                  "peak_source": "%s HBM copy bandwidth" % peaks["source"],
                  "algorithmic": "%.0f row entries x 4 B + %d atoms x 48 B" % (row_entries, n),
                  "avg_launch_us": 1e3 * build_ms, "share_of_step": share["build"]},
    }
    for k, line in lines.items():
        if traffic and k in traffic:
            line["traffic"] = traffic[k]
            line["traffic_source"] = "ncu --set full capture of k_%s, profiles/r1_final_dram_bytes.csv (bytes per launch)" % k
    share_note = "device time per kernel group / sum over groups; k_bonded runs on a side stream beside k_pair, so the groups overlap"
    dominant = max(("pair", "update", "build"), key=lambda k: share[k])
    roofline = dict(lines[dominant], kernel_ms_share=share, share_note=share_note)
    return roofline, {k: v for k, v in lines.items() if k != dominant}


def large_box_rooflines(torch, jb, wl, dev, stream, flush, props, peaks, config, steps):
    """The same kernel lines on a box large enough to fill the GPU (BASELINE configs[4], ~1e6 atoms: 'throughput and
    roofline at 1 B200'); the configs[1] box of the headline metric leaves every kernel latency-bound."""
    sysd, run = wl.make_config(config)
    n = sysd["n_atoms"]
    with torch.cuda.stream(stream):
        sim = jb.JumpSim(sysd, device=dev, stream=stream, **run)
        sim.baoab_step(300)
        sim.jump_step(30)
        sim.sync()
        ms = timed_blocks(torch, sim, stream, sim.jump_step, steps, BLOCK, flush)
        line, other = kernel_rooflines(torch, sim, stream, sim.jump_step, steps, BLOCK, flush, run, n, props, peaks)
        n_in = run["n_inner"]
        sim.jump_respa_step(5)
        sim.sync()
        ms_r = timed_blocks(torch, sim, stream, lambda b: sim.jump_respa_step(b // n_in), (steps // 20) * 20, 20, flush)
        sim.baoab_step(20)
        sim.sync()
        ms_b = timed_blocks(torch, sim, stream, sim.baoab_step, steps, BLOCK, flush)
        err = sim.stats()["error"]
    sim.close()
    lines = dict(other)
    lines["dominant"] = line
    return {"workload": "BASELINE configs[%d]: %d-atom flexible water box %.1f A, JUMP, equilibrated by 300 BAOAB steps"
                        % (config, n, sysd["box"]),
            "steps": steps, "ms_per_step": ms / steps, "ns_per_day": ns_per_day(steps / (ms * 1e-3), run["dt_fs"]),
            "atom_steps_per_s": n * steps / (ms * 1e-3), "baoab_ms_per_step": ms_b / steps,
            "jump_respa": {"n_inner": n_in, "ms_per_inner_step": ms_r / ((steps // 20) * 20),
                           "ns_per_day": ns_per_day(((steps // 20) * 20) / (ms_r * 1e-3), run["dt_fs"]),
                           "what": "JUMP-RESPA, inner %g fs (bonded + short-range), outer %g fs (jumps), configs[4]'s mode"
                                   % (run["dt_fs"], n_in * run["dt_fs"])},
            "jump_vs_baoab": ms_b / ms, "error": err, "kernels": lines}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2000)
    ap.add_argument("--warmup", type=int, default=200)
    ap.add_argument("--config", type=int, default=1)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--equil", type=int, default=2000, help="untimed BAOAB equilibration steps from the lattice start")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--large-config", type=int, default=4,
                    help="also report the kernel rooflines on this (GPU-filling) config, N=1 only; -1: skip")
    ap.add_argument("--mode", default="jump", choices=["jump", "respa"])
    ap.add_argument("--r-mid", type=float, default=None, help="ring split r_M (default: the config's)")
    ap.add_argument("--skin", type=float, default=None)
    ap.add_argument("--nlist-every", type=int, default=None)
    ap.add_argument("--eps-jump", type=float, default=None)
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
    for key, val in (("r_mid", args.r_mid), ("skin", args.skin), ("nlist_every", args.nlist_every), ("eps_jump", args.eps_jump)):
        if val is not None:
            run[key] = val
    n, dt_fs = sysd["n_atoms"], run["dt_fs"]
    stream = torch.cuda.Stream(dev)
    flush = torch.empty(L2_FLUSH_BYTES, dtype=torch.uint8, device=dev)
    with torch.cuda.stream(stream):
        sim = jb.JumpSim(sysd, device=dev, stream=stream, **run)
        sim.baoab_step(args.equil)
        sim.sync()
        sim.reset_stats()
        respa = args.mode == "respa"
        per_call = run["n_inner"] if respa else 1                      # MD steps of length dt per API unit
        step_call = (lambda b: sim.jump_respa_step(b // per_call)) if respa else sim.jump_step
        block = BLOCK
        K = max(args.steps // per_call * per_call, per_call)
        W = max(args.warmup, 3)
        step_call(max(W // per_call * per_call, per_call))
        sim.sync()

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
    sim.sync()
    ms_max = replicas.max_over_ranks(ms, dist, dev)
    stats = sim.stats()

    # ---- per-kernel times of the same K steps (CUDA events on the launch stream, separate pass) --------------
    roofline, roofline_other = kernel_rooflines(torch, sim, stream, step_call, K, block, flush, run, n, props, peaks,
                                                traffic=NCU_TRAFFIC_CFG1 if (args.config == 1 and not respa) else None)

    # ---- same-GPU BAOAB with the unsplit r_long force (reported baseline) -------------------------------------
    with torch.cuda.stream(stream):
        sim.baoab_step(50)
        sim.sync()
        Kb = min(K, 500)
        ms_b = timed_blocks(torch, sim, stream, sim.baoab_step, Kb, block, flush)
    baoab = {"ns_per_day": ns_per_day(Kb / (ms_b * 1e-3), dt_fs), "ms_per_step": ms_b / Kb, "steps": Kb,
             "force": "unsplit pair force to r_long = %.0f A" % run["r_long"]}

    # ---- the paper's preferred setting, adaptive eps(x) = eps0 |F_ij(x)| (NEXT-1, R-19), same box ------
    adaptive = None
    if not respa:
        with torch.cuda.stream(stream):
            run_a = dict(run, eps_mode=1, eps_jump=2.0)
            sim_a = jb.JumpSim(sysd, device=dev, stream=stream, **run_a)
            sim_a.baoab_step(args.equil)
            sim_a.jump_step(max(W, 50))
            sim_a.sync()
            sim_a.reset_stats()
            Ka = min(K, 1000)
            ms_a = timed_blocks(torch, sim_a, stream, sim_a.jump_step, Ka, block, flush)
            st_a = sim_a.stats()
            sim_a.close()
        adaptive = {"eps0_A_mol_per_kcal": 2.0, "steps": Ka, "ms_per_step": ms_a / Ka,
                    "ns_per_day": ns_per_day(Ka / (ms_a * 1e-3), dt_fs),
                    "proposals_per_atom_step": st_a["proposals"] / (n * Ka), "accepts_per_atom_step": st_a["accepts"] / (n * Ka),
                    "max_p": st_a["max_p"], "error": st_a["error"]}

    # ---- NEXT-2: three-level JUMP-RESPA1 1:2:6 fs (the paper's Table 2 setting) against BAOAB-RESPA1 1:2:6, the
    # reciprocal Ewald sum as the slow force (R-21), same box --------------------------------------------
    respa1 = None
    if not respa and rank == 0:
        respa1 = {"levels_fs": [dt_fs, 2 * dt_fs, 6 * dt_fs],
                  "what": "delta: bonded; kappa = 2 delta: short non-bonded + jumps (JUMP) or kick (BAOAB); Delta = 3 kappa: "
                          "reciprocal Ewald sum + exclusion correction (+ long pair gradient for BAOAB-RESPA1, P:L511)"}
        for name, fl in (("jump_respa1", 3 | 8), ("baoab_respa1", 3 | 8 | 16)):
            with torch.cuda.stream(stream):
                sim_r = jb.JumpSim(sysd, device=dev, stream=stream, **dict(run, flags=fl, n_inner=2))
                sim_r.baoab_step(args.equil)
                nk = sim_r.ewald_setup()
                sim_r.jump_respa1_step(10, 3)
                sim_r.sync()
                Kr = max(min(K, 600) // 6, 1)
                ms_r = timed_blocks(torch, sim_r, stream, lambda b: sim_r.jump_respa1_step(b, 3), Kr, 2, flush)
                if name == "jump_respa1":   # the slow force alone (three kernels), per evaluation
                    sim_r.forces(5)
                    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    e0.record(stream)
                    for _ in range(10):
                        sim_r.forces(5)
                    e1.record(stream)
                    stream.synchronize()
                    ms_s = e0.elapsed_time(e1) / 10
                    # algorithmic work per (atom, k-vector) pair in the factorised form: structure
                    # factor 5 fp64 multiply-adds (one complex multiply-accumulate + the amortised Ex Ey product), force 9
                    # fp32 ones (phase product 4, term 2, sums 2, amortised 1); an fp64 multiply-add takes two slots of
                    # the FP32-pipe peak it is reported against (the fp64 pipe runs at half rate): 19 slots x 2 flop
                    peak_tf = props.multi_processor_count * 128 * 2 * peaks["sm_max_mhz"] * 1e6 / 1e12
                    ach_tf = 1.0 * nk * n * 19 * 2 / (ms_s * 1e-3) / 1e12
                    respa1["slow_force"] = {"n_k": nk, "ms_per_evaluation": ms_s,
                                            "terms_per_s": 2.0 * nk * n / (ms_s * 1e-3),
                                            "what": "S(k) pass + force pass, n_k half-space vectors x n atoms x 2 terms",
                                            "roofline": {"bound": "alu", "achieved": ach_tf, "peak": peak_tf, "unit": "TFLOP/s",
                                                         "frac": ach_tf / peak_tf, "traffic": None,
                                                         "algorithmic": "%d (atom, k) pairs x (5 fp64 x 2 + 9 fp32) multiply-add slots x 2 flop" % (nk * n),
                                                         "peak_source": "%d SMs x 128 FP32 lanes x 2 x %.0f MHz (sm_max_mhz)" % (props.multi_processor_count, peaks["sm_max_mhz"])}}
                err_r = sim_r.stats()["error"]
                sim_r.close()
            respa1[name] = {"ms_per_outer_step": ms_r / Kr, "ns_per_day": ns_per_day(Kr / (ms_r * 1e-3), 6 * dt_fs),
                            "outer_steps": Kr, "error": err_r}
        respa1["jump_vs_baoab"] = respa1["baoab_respa1"]["ms_per_outer_step"] / respa1["jump_respa1"]["ms_per_outer_step"]

    # ---- end to end through the public API with HOST buffers -------------------------------------------------
    with torch.cuda.stream(stream):
        Ke = min(K, 500)
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
           "call": "JumpSim.run_host: pinned host (x, v) -> device, jump_refresh_lazy (rows rebuilt only if an atom left its "
                   "skin/2 ball), %d steps, device -> host, per call" % block}

    large = None
    if rank == 0 and world == 1 and args.large_config >= 0:
        large = large_box_rooflines(torch, jb, wl, dev, stream, flush, props, peaks, args.large_config, 100)

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = run_cpu_baseline(sysd, run)

    if rank == 0:
        sps = K / (ms_max * 1e-3)
        value = world * ns_per_day(sps, dt_fs)
        line = {"metric": "ns_per_day_jump" if not respa else "ns_per_day_jump_respa", "value": value, "unit": "ns/day",
                "n_gpus": world, "steps": K, "warmup": W, "ms_per_step": ms_max / K, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": "BASELINE configs[%d]: %d-atom flexible water box %.1f A, r_c %.0f / r_long %.0f A, "
                                       "dt %.0f fs, %s, equilibrated by %d BAOAB steps"
                                       % (args.config, n, sysd["box"], run["r_short"], run["r_long"], dt_fs,
                                          "JUMP-RESPA n_inner %d" % run["n_inner"] if respa else "JUMP (C'J'AOAJ'C')", args.equil),
                           "eps_jump": run["eps_jump"], "r_mid": run["r_mid"], "skin": run["skin"],
                           "nlist_every": run["nlist_every"], "steps_per_api_call": block,
                           "l2": "flushed by a 256 MiB write between timed API calls (outside the event brackets)",
                           "parallelism": "independent replicas x%d" % world},
                "atom_steps_per_s": world * sps * n,
                "clocks": clocks, "gpu_launches": launches, "wall_s": wall,
                "e2e": e2e, "roofline": roofline, "roofline_other": roofline_other, "baoab_same_gpu": baoab,
                "jump_vs_baoab": (K / ms_max) / (Kb / ms_b),
                "events": {"proposals_per_atom_step": stats["proposals"] / (n * (K + W)) if K + W else None,
                           "accepts_per_atom_step": stats["accepts"] / (n * (K + W)), "max_p": stats["max_p"],
                           "error": stats["error"]}}
        if adaptive is not None:
            line["jump_adaptive_eps"] = adaptive
        if respa1 is not None:
            line["jump_respa1"] = respa1
        if large is not None:
            line["roofline_large_box"] = large
        if cpu is not None:
            line["cpu_baseline"] = cpu
        print(json.dumps(line))
    sim.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
