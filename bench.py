#!/usr/bin/env python
"""bench.py -- individual-generations/s of the sPEGG per-time-step update on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config 3]

One "step" is one pass of the whole hot path (Fig. 1 A-F: fecundity + scan + parents, gametes,
phenotype, survival, compaction, reductions) over the whole population.  Workload at N=1:
BASELINE.json's metric configuration, config 3 (N0 = K = 1,000,000 diploids, L = 1,024 bit-packed
loci), synthetic seeded input.  Prints ONE JSON line (see the contract in the task statement):
`value` is device-timed with inputs resident in HBM, `e2e` goes through the C ABI with host
buffers, `roofline` is the dominant kernel against the measured HBM copy bandwidth, `cpu_baseline`
is the oracle timed on the host cores on a bounded sample.

N > 1 (torchrun): a single panmictic population does not shard (every father row may live on any
GPU), so ranks run independent replicas with different seeds -- "replicas only", weak scaling, no
data-path collective; NCCL is used for the barrier and the max-over-ranks time only.
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

METRIC = "individual-generations/sec"
UNIT = "individual-generations/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            return float(json.load(open(p))["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """Samples SM clocks and throttle reasons with nvidia-smi while the timed region runs."""

    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": []}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0]))
                mx = float(r[1])
                for nm, v in zip(names, r[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(nm)
            except Exception:
                continue
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm)}


VARIANTS = {
    # the widenings of SURVEY.md 8(f) on top of a configuration (R17-R21); context lines, not the metric
    "none": {},
    "noise": {"resid_sd": 0.5},                        # R17
    "overlap": {"adult_survival": 0.6},                # R18 (capacity x 4)
    "mating": {"mate_skew": 1.0},                      # R19
    "sexes": {"separate_sexes": 1},                    # R21 (fecundity parameter x 2: half the adults lay eggs)
    "encounters": {},                                  # R20 (configuration 4 only: 3 meetings, attack 0.1)
    "cost": {"fec_cost": 0.05},                        # R22
    "mothers": {"mother_skew": 1.0},                   # R24
    "monogamy": {"monogamy": 1},                       # R25
}


def apply_variant(cfg, variant):
    sp = cfg["species"][0]
    sp.update(VARIANTS[variant])
    if variant == "overlap":
        sp["capacity"] = 4 * sp["capacity"]
    if variant == "sexes":
        sp["fec_a"] = 2.0 * sp["fec_a"]
    if variant == "encounters":
        sp["predation"].update(encounters=3, attack=0.1)
    if variant != "none":
        cfg["name"] = "%s+%s" % (cfg["name"], variant)
    return cfg


SWEEP = {"patches": 16, "per_patch": 50_000, "k_scale": 1.0}   # --patches / --per-patch (configuration 6), --k-scale


def workload(which, seed_offset=0, world=1, variant="none"):
    """Rank `seed_offset`'s workload.  Configs 1-5: an independent replica (own seed).  Config 6 (the
    sweep of unlinked patches): the rank's block of --patches patches out of a patches x world sweep."""
    from paper_1603_09255_b200 import replicas, workloads
    if which == 6:
        return apply_variant(replicas.sweep_shard(SWEEP["patches"] * world, seed_offset, world, per_patch=SWEEP["per_patch"]), variant)
    cfg = apply_variant(replicas.replica_config(workloads.config(which), seed_offset), variant)
    if SWEEP["k_scale"] != 1.0:
        cfg["species"][0]["K"] = cfg["species"][0]["K"] * SWEEP["k_scale"]
        cfg["name"] = "%s(K x %g)" % (cfg["name"], SWEEP["k_scale"])
    return cfg


def describe(cfg):
    sp = cfg["species"][0]
    if len(cfg["species"]) == 2:
        what = "two species (resource N0=%d, K=%d + consumer N0=%d), each one panmictic population" % (
            cfg["n0"][0], int(sp["K"]), cfg["n0"][1])
    elif cfg["grid"] != (1, 1):
        what = "N0=%d diploids in patches %dx%d" % ((cfg["n0"][0],) + tuple(cfg["grid"]))
    else:
        what = "N0=K=%d diploids, one panmictic population" % cfg["n0"][0]
    return "%s: %s, L=%d %s loci, %d chromosomes" % (
        cfg["name"], what, sp["n_loci"], "bit-packed" if sp["kind"] == "bit" else "2^-10-quantised", len(sp["chrom_len"]))


L2_BYTES = 126 * 2 ** 20


def l2_note(cfg):
    """Timing rule: inputs larger than L2, or say that they are not."""
    pop = sum(int(sp["capacity"]) * row_bytes(sp) for sp in cfg["species"])
    live = sum(n * row_bytes(sp) for n, sp in zip(cfg["n0"], cfg["species"]))
    if 2 * live > L2_BYTES:
        return "inputs larger than L2 (two population buffers of %d MB, about %d MB of live rows read and written per step, vs 126 MB L2)" % (
            pop // 2 ** 20, 2 * live // 2 ** 20)
    return ("L2-RESIDENT workload (about %.1f MB of live rows per buffer vs 126 MB L2; no flush between steps: a step's "
            "input IS the previous step's output, so this is the workload's own steady state)") % (live / 2 ** 20)


def row_bytes(sp):
    return 2 * (sp["n_loci"] // 32) * 4 if sp["kind"] == "bit" else 4 * sp["n_loci"]


def alg_bytes(cfg, log, kernel_only):
    """Algorithmic bytes: G*(N_t + M_t + N_{t+1}) + 8*M_t for the gamete kernel
    (+ 4*N_t for the scan when the whole step is counted), summed over the given log entries."""
    G = row_bytes(cfg["species"][0])
    tot = 0
    for e in log:
        tot += G * (e["n_t"] + e["m_t"] + e["n_next"]) + 8 * e["m_t"]
        if not kernel_only:
            tot += 4 * e["n_t"]
    return tot


def host_info():
    """CPU model and core count of the box the oracle is timed on."""
    model = "unknown"
    try:
        for ln in open("/proc/cpuinfo"):
            if ln.startswith("model name"):
                model = ln.split(":", 1)[1].strip()
                break
    except OSError:
        pass
    return {"cpu_model": model, "nproc": os.cpu_count()}


class pinned_to_one_core:
    """The oracle is single-threaded: pin the process to ONE core while it is timed (the `taskset` of
    SURVEY.md 8(d)), so that the scheduler cannot move it, and give the mask back afterwards."""
    def __enter__(self):
        self.old, self.core = None, None
        try:
            self.old = os.sched_getaffinity(0)
            self.core = max(self.old)          # the last allowed core: away from core 0's interrupts
            os.sched_setaffinity(0, {self.core})
        except (AttributeError, OSError):
            self.old = None
        return self

    def __exit__(self, *exc):
        if self.old is not None:
            os.sched_setaffinity(0, self.old)
        return False


def oracle_run(cfg, n_steps, warm=0):
    """Times the oracle as it stands on the host cores (one thread; the caller pins it)."""
    import oracle
    from paper_1603_09255_b200 import workloads
    o = oracle.Oracle(cfg)
    for s in range(len(cfg["species"])):
        o.write_state(s, workloads.initial_rows(cfg, s), workloads.initial_patch_start(cfg, s), 0)
        if cfg["species"][s].get("separate_sexes"):
            o.write_sex(s, workloads.initial_sex(cfg, s))
    if warm:
        o.step(warm)
    k0 = len(o.log(0))
    t0 = time.perf_counter()
    o.step(n_steps)
    dt = time.perf_counter() - t0
    units = sum(sum(e["n_t"] for e in o.log(s)[k0:]) for s in range(len(cfg["species"])))
    return units, dt


def run_reference(args):
    """--impl reference: the oracle is this tier's reference arm (rank 0 only)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1603_09255_b200 import workloads
    full = workload(args.config, variant=args.variant)
    # bounded sample: shrink the population so that K+W oracle steps end within ~2 minutes
    per_step_s = args.ref_budget_s / max(1, args.steps + args.warmup)
    scale = min(1.0, max(0.001, per_step_s * 7.0e4 / full["n0"][0]))
    cfg = apply_variant(workloads.config(args.config, scale=scale), args.variant)
    with pinned_to_one_core() as pin:
        units, dt = oracle_run(cfg, args.steps, warm=args.warmup)
    val = units / dt
    host = dict(host_info(), pinned_core=pin.core)
    what = "1 core, plain single-threaded oracle (-O2), population scaled down: context, not a target"
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "u32", "data": "synthetic",
        "config": {"workload": describe(full), "sample": "population scaled by %.4g (N0=%d) per step" % (scale, cfg["n0"][0]),
                   "same_config": scale == 1.0,
                   "why": ("the plain oracle needs about 6 s per full-size step: K+W steps are bounded to ~%d s by shrinking "
                           "N0, K and capacity together; the metric is a per-individual rate and the full-size "
                           "cpu_baseline leg of the other arm agrees with it" % int(args.ref_budget_s)) if scale != 1.0 else "full size",
                   "ratio_is": what},
        "cpu_baseline": dict({"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "what": what,
                              "sample": "%d steps of the workload at N0=%d (scale %.4g)" % (args.steps, cfg["n0"][0], scale)}, **host),
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_ours(args):
    import numpy as np
    import torch
    from paper_1603_09255_b200 import binding, replicas, workloads

    rank, local, world = replicas.env_rank()
    dist = None
    if world > 1:
        import torch.distributed as dist
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        torch.cuda.set_device(local)
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    dev = torch.device("cuda", local)
    torch.cuda.set_device(dev)
    binding.load()  # fails loudly if the CUDA extension is missing

    cfg = workload(args.config, seed_offset=rank, world=world, variant=args.variant)
    n_sp = len(cfg["species"])
    sim = binding.Sim(cfg, debug=False, log_capacity=max(4096, args.steps * 4 + args.warmup + 256), device=str(dev))
    rows0 = [workloads.initial_rows(cfg, s) for s in range(n_sp)]
    ps0 = [workloads.initial_patch_start(cfg, s) for s in range(n_sp)]
    sex0 = [workloads.initial_sex(cfg, s) if cfg["species"][s].get("separate_sexes") else None for s in range(n_sp)]
    for s in range(n_sp):
        sim.write_state(s, rows0[s], ps0[s], 0)
        if sex0[s] is not None:
            sim.write_sex(s, sex0[s])

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    # ---- clock warm: the GPU leaves its idle clocks only after some milliseconds of work, far more than
    # W = 5 steps of 0.15 ms.  Untimed steps on the same handle, then the initial state is written again,
    # so the W warm-up and K timed steps below start from exactly the state of a fresh run.
    if args.clock_warm_steps > 0:
        sim.step(args.clock_warm_steps)
        sim.synchronize()
        for s in range(n_sp):
            sim.write_state(s, rows0[s], ps0[s], 0)
            if sex0[s] is not None:
                sim.write_sex(s, sex0[s])

    # ---- device-timed run: inputs resident in HBM, K graph replays, no host sync inside
    sim.step(args.warmup)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    k0 = len(sim.read_log(0))
    barrier()
    with torch.cuda.stream(sim.stream):
        ev0.record(sim.stream)
        sim.step(args.steps)
        ev1.record(sim.stream)
    barrier()
    ms = ev0.elapsed_time(ev1)
    clocks = sampler.stop() if rank == 0 else None
    flags = sim.status()
    # two more timed sections of K steps ("run the timed section 3x, report the median and the
    # spread"): `value` / `ms_per_step` are those of the MEDIAN section, with that section's own counts
    section_ms = [ms]
    for _ in range(2):
        r0, r1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        barrier()
        with torch.cuda.stream(sim.stream):
            r0.record(sim.stream)
            sim.step(args.steps)
            r1.record(sim.stream)
        barrier()
        section_ms.append(r0.elapsed_time(r1))
    repeats = [x / args.steps for x in section_ms]
    med = sorted(range(3), key=lambda i: section_ms[i])[1]
    ms = section_ms[med]
    all_logs = [sim.read_log(s) for s in range(n_sp)]
    logs = [lg[k0 + med * args.steps:k0 + (med + 1) * args.steps] for lg in all_logs]
    units = sum(sum(e["n_t"] for e in lg) for lg in logs)
    offspring = sum(sum(e["m_t"] for e in lg) for lg in logs)

    # ---- dominant kernel timed alone with CUDA events on its own stream (direct launches)
    kt_steps = min(args.steps, 100)
    sim.kernel_timing(True)
    kl0 = len(sim.read_log(0))
    sim.step(kt_steps)
    k_ms, k_n = sim.kernel_timing(False)
    klog = sim.read_log(0)[kl0:kl0 + kt_steps]
    # a one-launch step does the scan too: the kernel is charged the whole step's bytes
    k_bytes = alg_bytes(cfg, klog, kernel_only=sim.launches_per_step() > 1) / max(1, len(klog))

    # ---- end to end through the C ABI with HOST buffers: upload, K x (step + read of the step's
    # result), download -- all inside the timed region
    e2e_steps = min(args.steps, 50)
    pinned = [torch.from_numpy(r.view(np.int32).reshape(-1) if r.dtype == np.uint32 else r.view(np.int16).reshape(-1)).pin_memory() for r in rows0]
    host_rows = [p.numpy().view(rows0[s].dtype).reshape(rows0[s].shape) for s, p in enumerate(pinned)]
    outs = [torch.empty(int(cfg["species"][s]["capacity"]) * sim.row_shape[s], dtype=torch.int32 if rows0[s].dtype == np.uint32 else torch.int16).pin_memory() for s in range(n_sp)]
    out_np = [o.numpy().view(rows0[s].dtype).reshape(-1, sim.row_shape[s]) for s, o in enumerate(outs)]
    barrier()
    t0 = time.perf_counter()
    for s in range(n_sp):
        sim.write_state(s, host_rows[s], ps0[s], 0)
        if sex0[s] is not None:
            sim.write_sex(s, sex0[s])
    h2d = sum(r.nbytes for r in host_rows) + sum(x.nbytes for x in sex0 if x is not None)
    e_units, d2h = 0, 0
    for _ in range(e2e_steps):
        sim.step(1)
        for s in range(n_sp):
            e = sim.read_log(s, last=1)[-1]      # device -> host read of the step's result (64-byte entry)
            e_units += e["n_t"]
            d2h += 64
    for s in range(n_sp):
        r, _, _ = sim.read_state(s, want_zi=False, out=out_np[s])
        d2h += r.nbytes
    torch.cuda.synchronize()
    e2e_s = time.perf_counter() - t0

    # ---- reduce over ranks: max time, summed units
    (ms, e2e_s), (units, e_units, offspring) = replicas.reduce_over_ranks(
        dist, [ms, e2e_s], [units, e_units, offspring], device=dev)
    launches = sim.launches_per_step() * args.steps

    if rank == 0:
        peak, peak_src = load_peaks()
        achieved = k_bytes / (k_ms * 1e-3) / 1e9 if k_ms > 0 else 0.0
        step_bytes = alg_bytes(cfg, logs[0], kernel_only=False) / max(1, len(logs[0]))
        traffic, traffic_src = measured_traffic(cfg["name"])
        # oracle on a bounded sample of the same workload: ~10-30 s of CPU work
        cb_cfg = workload(args.config, variant=args.variant)
        cb_steps = 1 if cb_cfg["n0"][0] >= 500_000 else max(1, int(1.0e6 / cb_cfg["n0"][0]))
        with pinned_to_one_core() as pin:
            cb_units, cb_dt = oracle_run(cb_cfg, cb_steps)
        cb_host = dict(host_info(), pinned_core=pin.core)
        line = {
            "metric": METRIC, "value": units / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "u32", "data": "synthetic",
            "config": {"workload": describe(cfg), "parallelism": ("patches sharded x%d, no collective" if args.config == 6 else "replicas only x%d") % world,
                       "l2": l2_note(cfg),
                       "clock_warm": "%d untimed steps, then the initial state written again, before the W warm-up steps" % args.clock_warm_steps,
                       "ms_per_step_repeats": [round(x, 6) for x in repeats], "reported_section": "median of 3 (section %d)" % (med + 1),
                       "spread": (max(repeats) - min(repeats)) / sorted(repeats)[1],
                       "mean_N_t": units / args.steps / world, "mean_M_t": offspring / args.steps / world,
                       "flags": flags, "offspring_per_s": offspring / (ms * 1e-3),
                       "step_alg_bytes": step_bytes,
                       "step_frac_of_peak": step_bytes / (ms / args.steps * 1e-3) / 1e9 / peak},
            "clocks": clocks,
            "e2e": {"value": e_units / e2e_s, "unit": UNIT, "h2d_bytes_per_step": h2d / e2e_steps,
                    "d2h_bytes_per_step": d2h / e2e_steps, "steps": e2e_steps,
                    "what": "spegg_write_state(host) + K x (spegg_step(1) + spegg_read_log) + spegg_read_state(host)"},
            "gpu_launches": launches,
            "roofline": {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s",
                         "frac": achieved / peak, "traffic": traffic, "traffic_source": traffic_src,
                         "frac_is": "ALGORITHMIC bytes per launch / kernel time / peak (DRAM traffic is below the algorithmic bytes: L2 hits)",
                         "traffic_frac": (traffic / (k_ms * 1e-3) / 1e9 / peak) if (traffic and k_ms > 0) else None,
                         "kernel": ("fused step kernel: scan+parents+gametes+phenotype+survival+compaction" if sim.launches_per_step() == 1 else "gamete kernel") if k_n else "none",
                         "kernel_ms": k_ms, "kernel_launches_timed": k_n, "alg_bytes_per_launch": k_bytes,
                         "peak_source": peak_src},
            "cpu_baseline": dict({"value": cb_units / cb_dt, "unit": UNIT, "cores": 1, "kind": "oracle",
                                  "what": "1 core, plain single-threaded oracle (-O2) as it stands: context, not a target",
                                  "sample": "%d step(s) of the full workload (N0=%d), %.1f s" % (cb_steps, cb_cfg["n0"][0], cb_dt)}, **cb_host),
        }
        sp0 = cfg["species"][0]
        if sp0["kind"] == "q10" and k_ms > 0:
            # quantised-effect genomes draw one Philox word per locus per gamete (R7): the second ceiling of the
            # gamete kernel is integer issue ('ALU roofline'), reported beside the HBM one
            ops = alu_ops_per_offspring(sp0["n_loci"]) * sum(e["m_t"] for e in klog) / max(1, len(klog))
            a_alu = ops / (k_ms * 1e-3) / 1e12
            line["roofline"]["alu"] = {"achieved": a_alu, "peak": ALU_PEAK_TINST, "unit": "Tinst/s",
                                       "frac": a_alu / ALU_PEAK_TINST, "alg_inst_per_launch": ops,
                                       "peak_source": "148 SMs x 4 schedulers x 32 lanes x 1.965 GHz (DESIGN.md 5)"}
        if args.others and world == 1 and args.config == 3 and args.variant == "none":
            # the other BASELINE.json configurations, driver-visible: short timed passes after the metric's own
            sim.close()
            line["config"]["other_workloads"] = [measure_other(w, 30, 5, dev) for w in (1, 2, 4, 5)]
        print(json.dumps(line))
    sim.close()
    if dist is not None:
        dist.destroy_process_group()


# ALU roofline of the q10 gamete kernel: algorithmic thread-instructions per offspring =
# Philox blocks x 44 (ten rounds of two 32x32->64 multiplies and two three-input XORs, plus the
# counter set-up) + 4 per locus per gamete (threshold compare, phase parity, select, allele sum);
# blocks = 2L/4 RECOMB + 1 SCALAR + 2 MUT.  Peak = one warp instruction per scheduler per clock.
ALU_PEAK_TINST = 148 * 4 * 32 * 1.965e9 / 1e12


def alu_ops_per_offspring(n_loci):
    return (2 * n_loci // 4 + 3) * 44 + 2 * n_loci * 4


def measured_traffic(name):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, from the
    `ncu --set full` capture recorded in profiles/dominant_kernel_traffic.csv -- but only while the
    kernel's source file still has the SHA-256 the capture was taken with; else None (a constant
    that silently outlives the kernel it was measured on is worse than no number)."""
    import csv
    import hashlib
    path = os.path.join(ROOT, "profiles", "dominant_kernel_traffic.csv")
    if not os.path.exists(path):
        return None, "no capture recorded"
    for row in csv.DictReader(open(path)):
        if row["workload"] != name:
            continue
        src = os.path.join(ROOT, "paper_1603_09255_b200", "csrc", row["source_file"])
        sha = hashlib.sha256(open(src, "rb").read()).hexdigest()
        if sha != row["source_sha256"]:
            return None, "capture %s predates the current %s" % (row["capture"], row["source_file"])
        return float(row["dram_read_bytes"]) + float(row["dram_write_bytes"]), row["capture"]
    return None, "no capture recorded for %s" % name


def measure_other(which, steps, warmup, dev):
    """A short device-timed pass of another BASELINE.json configuration (context lines under
    config.other_workloads; `value` stays the metric's configuration)."""
    import torch
    from paper_1603_09255_b200 import binding, workloads
    cfg = workloads.config(which)
    n_sp = len(cfg["species"])
    sim = binding.Sim(cfg, debug=False, log_capacity=4096, device=str(dev))
    for s in range(n_sp):
        sim.write_state(s, workloads.initial_rows(cfg, s), workloads.initial_patch_start(cfg, s), 0)
    sim.step(warmup)
    sim.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(sim.stream):
        e0.record(sim.stream)
        sim.step(steps)
        e1.record(sim.stream)
    sim.synchronize()
    ms = e0.elapsed_time(e1) / steps
    logs = [sim.read_log(s)[warmup:warmup + steps] for s in range(n_sp)]
    units = sum(sum(e["n_t"] for e in lg) for lg in logs)
    peak, _ = load_peaks()
    step_bytes = sum(alg_bytes(dict(species=[cfg["species"][s]]), logs[s], kernel_only=False) for s in range(n_sp)) / steps
    out = {"workload": describe(cfg), "steps": steps, "warmup": warmup, "ms_per_step": ms,
           "value": units / (ms * steps * 1e-3), "unit": UNIT, "launches_per_step": sim.launches_per_step(),
           "mean_N_t": units / steps, "flags": sim.status(), "step_alg_bytes": step_bytes,
           "step_frac_of_hbm_peak": step_bytes / (ms * 1e-3) / 1e9 / peak, "l2": l2_note(cfg)}
    sp0 = cfg["species"][0]
    if sp0["kind"] == "q10":
        kt = min(steps, 10)
        sim.kernel_timing(True)
        kl0 = len(sim.read_log(0))
        sim.step(kt)
        k_ms, k_n = sim.kernel_timing(False)
        klog = sim.read_log(0)[kl0:kl0 + kt]
        if k_ms > 0:
            ops = alu_ops_per_offspring(sp0["n_loci"]) * sum(e["m_t"] for e in klog) / max(1, len(klog))
            out["gamete_kernel_ms"] = k_ms
            out["gamete_kernel_alu_frac"] = ops / (k_ms * 1e-3) / 1e12 / ALU_PEAK_TINST
    sim.close()
    del sim
    torch.cuda.empty_cache()
    return out


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--variant", default="none", choices=sorted(VARIANTS),
                    help="a widening of SURVEY.md 8(f) on top of --config (context lines; the metric is --variant none)")
    ap.add_argument("--clock-warm-steps", type=int, default=300,
                    help="untimed steps before the W warm-up steps (the initial state is written again after them)")
    ap.add_argument("--patches", type=int, default=16, help="configuration 6: patches per rank (PAPER.md:64 runs 1-100)")
    ap.add_argument("--per-patch", type=int, default=50_000, help="configuration 6: individuals per patch at the start")
    ap.add_argument("--k-scale", type=float, default=1.0,
                    help="multiply the carrying capacity K of species 0 (fixed / variable cost of the step; profiles/r02_fused_full.md)")
    ap.add_argument("--no-others", dest="others", action="store_false",
                    help="skip the short timed passes of configurations 1, 2, 4, 5 (config.other_workloads)")
    ap.add_argument("--ref-budget-s", type=float, default=120.0,
                    help="--impl reference: CPU seconds the K+W oracle steps are sized for")
    args = ap.parse_args()
    SWEEP.update(patches=args.patches, per_patch=args.per_patch, k_scale=args.k_scale)
    if args.warmup < 3:
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
