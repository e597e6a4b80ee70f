#!/usr/bin/env python
"""bench.py -- spin flips/ns of the checkerboard Metropolis hot path on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl graft|reference] [--workload NAME]

One STEP = `--sweeps-per-step` full sweeps (colour 0 then colour 1) of the workload followed by
one energy / magnetisation measurement -- every row of SURVEY.md section 8(a).  Default workload:
BASELINE.json configs[1], the 2D Ising lattice L = 16384 with int8 spins (the configuration the
">= 70 % of the HBM roofline" target is quoted on).  Prints ONE JSON line.

  value         attempted spin updates per ns, whole job, state resident in HBM, CUDA-event timed
  e2e           the same through the C ABI with HOST buffers: every step uploads the spin configuration
                (spin_set_spins from pinned host memory), sweeps, and reads E, M back (spin_measure)
  roofline      dominant kernel (the half-sweep): algorithmic bytes per launch / mean launch duration
  cpu_baseline  the oracle (oracle/, plain single-threaded C++) on this box's host cores, bounded sample
  per_model     flips/ns and roofline fraction of the other BASELINE.json workloads (short runs)

--impl reference times the oracle itself (the CPU arm of the driver's ratio).
N > 1 (torchrun): every rank runs its own independent lattice (weak scaling, no data-path collective).
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

METRIC = "spin flips/ns (device-timed) and achieved HBM GB/s vs B200 peak, per model"
UNIT = "flips/ns"
DEFAULT_WORKLOAD = "ising2d_L16384_int8"
# per-model legs of the default run: (workload, sweeps timed)
PER_MODEL = [("ising2d_L64_int8", 1000), ("ising2d_L16384_bitpack", 40), ("ising3d_L512_bitpack", 40),
             ("ea3d_L256_R16_bitpack", 40), ("ea3d_L256_R16_bitpack_ownstreams", 20), ("ea2d_L64_R4096_bitpack", 200),
             ("ea2d_L32_R131072_msc", 100), ("heisenberg3d_L256_fp32", 20), ("heisenberg2d_L4096_fp32", 20), ("xy3d_L256_fp32", 20)]
RECORDED = ("ising2d_L16384_bitpack", "ea3d_L256_R16_bitpack", "heisenberg3d_L256_fp32", "xy3d_L256_fp32")
DTYPE = {"int8": "u8", "bitpack": "u32 (bit-packed, 32 spins per word)", "fp32": "f32",
         "msc": "u32 (bit-packed, 32 realisations of one site per word)"}


def measured_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    try:
        with open(path) as f:
            p = json.load(f)
        return float(p["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md: 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks and throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    QUERY = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
             "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
             "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.rows, self.proc, self.thread = [], None, None
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(index), "--query-gpu=" + self.QUERY,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, mx, reasons, power = [], None, set(), []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [r for (t, r) in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for (_, r) in self.rows]
        for r in rows:
            f = [x.strip() for x in r.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx = float(f[1]); power.append(float(f[2]))
            except ValueError:
                continue
            for name, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        sm.sort()
        return {"sm_mhz": sm[len(sm) // 2] if sm else None, "sm_max_mhz": mx, "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(power) if power else None}


def time_sweeps(S, beta, sweeps, warm=4, record=False):
    """ms per half-sweep (time / 2 sweeps, whatever the number of launches), flips/ns and launches of `sweeps` sweeps of
    system S (state resident, CUDA events on the launching stream)."""
    import torch

    run = S.sweep_record if record else S.sweep
    if S.N * S.R < 5e7:
        warm = max(warm, 48)    # launch-bound lattices replay a CUDA graph of 16 sweeps: build it outside the timed region
    run(beta, warm)
    torch.cuda.synchronize()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = S.launch_count
    e0.record()
    run(beta, sweeps)
    e1.record()
    torch.cuda.synchronize()
    ms = e0.elapsed_time(e1)
    return ms / (2 * sweeps), S.N * S.R * sweeps / (ms * 1e6), S.launch_count - l0


def run_per_model(P, peak):
    import torch

    out = {}
    for name, sweeps in PER_MODEL:
        # "<workload>_ownstreams": the same lattice with the replica index in the Philox counter (replica_streams = 1)
        base = name
        w = P.workloads.WORKLOADS[name]
        S = P.from_workload(w, P.workloads.SEED)
        if w["record"]:
            # config 1: E and M after every sweep (spin_sweep_record)
            S.sweep_record(w["beta"], 3)
            torch.cuda.synchronize()
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            S.sweep_record(w["beta"], sweeps)
            e1.record()
            torch.cuda.synchronize()
            ms = e0.elapsed_time(e1)
            out[name] = {"flips_per_ns": S.N * S.R * sweeps / (ms * 1e6), "us_per_sweep_recorded": 1e3 * ms / sweeps,
                         "note": "one launch of the shared-memory-resident kernel for all sweeps; E and M recorded "
                                 "every sweep; latency-bound (64 words per colour)"}
        else:
            ms_half, fpn, launches = time_sweeps(S, w["beta"], sweeps)
            bpu = P.workloads.BYTES_PER_UPDATE[base]
            cnt = COUNTERS.get(name, {})
            out[name] = {"flips_per_ns": fpn, "ms_per_halfsweep": ms_half, "launches_per_sweep": launches / sweeps,
                         "algorithmic_GBps": fpn * bpu, "hbm_frac": fpn * bpu / peak, "bytes_per_update": bpu,
                         "kernel": cnt.get("kernel")}
            if name.endswith("_ownstreams"):
                out[name]["note"] = "16 replicas with their OWN update streams (replica_streams = 1): no mask reuse across replicas"
            elif w["replicas"] > 1 and not w["replica_streams"]:
                out[name]["note"] = "shared update stream (DESIGN.md R-17): the acceptance masks of a word serve every replica"
            if cnt.get("bound") == "alu":
                # executed warp-instructions per launch (committed ncu capture) / launch time, against the issue rate; the
                # pipe that binds is the ALU pipe (LOP3 / IADD3 / SHF / ISETP at one warp-instruction per 2 clocks)
                ms_launch = 2 * sweeps * ms_half / launches
                # the capture's instruction count, scaled if a launch here serves more updates (resident kernels: a launch per call)
                scale = (S.N * S.R * sweeps / launches) / cnt["updates_per_launch"] if cnt.get("updates_per_launch") else 1.0
                gwips = cnt["warp_instr_per_launch"] * scale / (ms_launch * 1e6)
                out[name]["roofline"] = {"bound": "alu", "achieved": gwips, "peak": ISSUE_PEAK_GWIPS, "unit": "Gwarp-instr/s",
                                         "frac": gwips / ISSUE_PEAK_GWIPS, "traffic": cnt.get("dram_bytes_per_launch"),
                                         "alu_pipe_busy_pct_in_capture": cnt.get("alu_pipe_pct"),
                                         "note": "instructions per launch from the committed ncu capture (%s); peak = issue "
                                                 "rate; state L2-resident" % cnt.get("capture")}
            else:
                out[name]["roofline"] = {"bound": "hbm", "achieved": fpn * bpu, "peak": peak, "unit": "GB/s",
                                         "frac": fpn * bpu / peak, "frac_of_nominal_8000": fpn * bpu / 8000.0,
                                         "traffic": cnt.get("dram_bytes_per_launch"), "capture": cnt.get("capture")}
            if name in RECORDED:
                # E and M after every sweep, fused into the colour-1 half-sweep
                ms_rec, fpn_rec, l_rec = time_sweeps(S, w["beta"], max(4, sweeps // 2), record=True)
                out[name]["recorded"] = {"flips_per_ns": fpn_rec, "ms_per_halfsweep": ms_rec, "launches_per_sweep": l_rec / max(4, sweeps // 2),
                                         "cost_vs_unrecorded": ms_rec / ms_half}
        S.close()
        del S
        torch.cuda.empty_cache()
    # heat-bath rule ("very similar speed-ups"): the same lattices, update_rule = heat bath
    for name, sweeps in (("ising2d_L16384_int8", 20), ("ising3d_L512_bitpack", 20), ("heisenberg3d_L256_fp32", 10)):
        w = P.workloads.WORKLOADS[name]
        S = P.from_workload(w, P.workloads.SEED, rule="heatbath")
        ms_launch, fpn, _ = time_sweeps(S, w["beta"], sweeps)
        bpu = P.workloads.BYTES_PER_UPDATE[name]
        cnt = COUNTERS.get(name + "#heatbath", {})
        out[name + "_heatbath"] = {"flips_per_ns": fpn, "ms_per_halfsweep": ms_launch, "algorithmic_GBps": fpn * bpu,
                                   "hbm_frac": fpn * bpu / peak, "bytes_per_update": bpu, "update_rule": "heat bath",
                                   "kernel": cnt.get("kernel"), "traffic": cnt.get("dram_bytes_per_launch"),
                                   "capture": cnt.get("capture")}
        S.close()
        del S
        torch.cuda.empty_cache()
    return out


def oracle_sample(w):
    """The bounded sample of workload w the oracle is timed on: the same recipe on a strip of the lattice."""
    dims = list(w["dims"])
    if dims[2] == 1:
        dims[1] = min(dims[1], 1024)
        what = "%d x %d strip of the %d x %d lattice" % (dims[0], dims[1], w["dims"][0], w["dims"][1])
    else:
        dims[2] = min(dims[2], 16)
        what = "%d x %d x %d slab of the %d^3 lattice" % (dims[0], dims[1], dims[2], w["dims"][0])
    return tuple(dims), what


def make_oracle_system(w, dims, seed):
    import oracle

    kinds = {"uniform": oracle.J_UNIFORM, "per_direction": oracle.J_PER_DIRECTION, "bond_pm1": oracle.J_BOND_PM1}
    return oracle.System(dims, n=w["n"], coupling_kind=kinds[w["coupling"]], J=w["J"], n_replicas=w["replicas"],
                         replica_streams=w["replica_streams"], seed=seed)


def cpu_baseline(P, name, budget_s=15.0):
    """The oracle as it stands, single thread, on a bounded sample (about `budget_s` seconds of CPU work)."""
    w = P.workloads.WORKLOADS[name]
    dims, what = oracle_sample(w)
    O = make_oracle_system(w, dims, P.workloads.SEED)
    updates_per_sweep = dims[0] * dims[1] * dims[2] * w["replicas"]
    t0 = time.perf_counter()
    sweeps = 0
    while True:
        O.sweep(w["beta"], 1)
        sweeps += 1
        el = time.perf_counter() - t0
        if el > budget_s or sweeps >= 1000:
            break
    O.measure()
    el = time.perf_counter() - t0
    return {"value": updates_per_sweep * sweeps / (el * 1e9), "unit": UNIT, "cores": 1, "kind": "oracle",
            "sample": "%d sweeps + 1 E/M measurement of a %s, %.1f s" % (sweeps, what, el),
            "ns_per_update": el * 1e9 / (updates_per_sweep * sweeps), "host_cores_present": os.cpu_count()}


def run_reference(args):
    """--impl reference: the oracle on the host cores, same metric and config; rank 0 only."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    from paper_1107_5463_b200 import workloads as WL

    w = WL.WORKLOADS[args.workload]
    dims, what = oracle_sample(w)
    O = make_oracle_system(w, dims, WL.SEED)
    updates = dims[0] * dims[1] * dims[2] * w["replicas"]
    for _ in range(args.warmup):
        O.sweep(w["beta"], 1)
        O.measure()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        O.sweep(w["beta"], 1)
        O.measure()
    el = time.perf_counter() - t0
    value = updates * args.steps / (el * 1e9)
    sample = "each step: 1 sweep + 1 E/M measurement of a %s" % what
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * el / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": DTYPE[w["storage"]], "data": "synthetic",
            "config": {"workload": args.workload, "dims": list(w["dims"]), "beta": w["beta"], "sample": sample},
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_slab(args):
    """--mode slab: ONE lattice cut into N slabs along its slowest axis, one per rank (strong scaling): per
    half-sweep each rank updates its boundary planes, exchanges them with its two ring neighbours (point-to-point over
    NCCL, on a side stream) while it updates the interior.  Prints the whole-lattice metric plus per-rank times and bytes."""
    import torch
    import torch.distributed as dist

    from paper_1107_5463_b200 import ranks, slab

    rank, local_rank, world = ranks.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = "cuda:%d" % local_rank
    os.environ.setdefault("NCCL_DEBUG", "INFO")      # the ranks and their transports show in the log
    if "RANK" in os.environ and "MASTER_ADDR" in os.environ:
        # under torchrun (any world size, 1 included): its rendezvous -- an explicit tcp:// address would be taken for the
        # agent's store and wait for a server that is not there
        dist.init_process_group("nccl", device_id=torch.device(dev))
    else:
        dist.init_process_group("nccl", init_method="tcp://127.0.0.1:29541", rank=0, world_size=1, device_id=torch.device(dev))
    import paper_1107_5463_b200 as P

    P.lib()
    w = P.workloads.WORKLOADS[args.workload]
    ring = slab.DistRing(P.SpinSystem, w["dims"], dist, dev, n=w["n"], storage=w["storage"], coupling=w["coupling"], J=w["J"],
                         replicas=w["replicas"], replica_streams=w["replica_streams"], seed=P.workloads.SEED)
    beta, SPS = w["beta"], args.sweeps_per_step
    N = w["dims"][0] * w["dims"][1] * w["dims"][2] * w["replicas"]
    for _ in range(args.warmup):
        ring.sweep(beta, SPS)
        ring.measure()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    bytes0 = ring.comm_bytes
    sampler = ClockSampler(local_rank) if rank == 0 else None
    dist.barrier()
    torch.cuda.synchronize()
    t0 = time.time()
    e0.record()
    for _ in range(args.steps):
        ring.sweep(beta, SPS)
        E, M = ring.measure()
    e1.record()
    dist.barrier()
    torch.cuda.synchronize()
    t1 = time.time()
    clocks = sampler.stop(t0, t1) if sampler else None
    ms = e0.elapsed_time(e1)
    per_rank = torch.tensor([ms, float(ring.comm_bytes - bytes0)], dtype=torch.float64, device=dev)
    allr = [torch.zeros_like(per_rank) for _ in range(world)]
    dist.all_gather(allr, per_rank)
    ms_max = max(float(t[0]) for t in allr)
    if rank == 0:
        halfsweeps = 2 * SPS * args.steps
        line = {"metric": METRIC, "value": N * SPS * args.steps / (ms_max * 1e6), "unit": UNIT, "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms_max / args.steps, "higher_is_better": True, "scaling": "strong",
                "vs_baseline": None, "dtype": DTYPE[w["storage"]], "data": "synthetic", "mode": "slab",
                "config": {"workload": args.workload, "dims": list(w["dims"]), "beta": beta, "sweeps_per_step": SPS,
                           "parallelism": "%d slabs of %d planes along the slowest axis, ring halo exchange per half-sweep" % (world, ring.own),
                           "overlap": ring.overlap},
                "per_rank": [{"rank": r, "us_per_halfsweep": 1e3 * float(t[0]) / halfsweeps,
                              "comm_bytes_per_halfsweep": float(t[1]) / halfsweeps} for r, t in enumerate(allr)],
                "comm": {"kind": "point-to-point ring (torch.distributed batch_isend_irecv over NCCL)", "halo_bytes_per_face": ring.hb},
                "E": float(E[0]), "clocks": clocks, "gpu_launches": int(ring.system.launch_count)}
        print(json.dumps(line), flush=True)
    dist.barrier()
    dist.destroy_process_group()


def run_graft(args):
    import numpy as np
    import torch

    from paper_1107_5463_b200 import ranks

    rank, local_rank, world = ranks.env_rank()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local_rank)
    dev = "cuda:%d" % local_rank
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device(dev))
    import paper_1107_5463_b200 as P

    P.lib()
    peak, peak_src = measured_peaks()
    w = P.workloads.WORKLOADS[args.workload]
    rule_kw = {"rule": "heatbath"} if args.rule == "heatbath" else {}
    S = P.from_workload(w, ranks.rank_seed(P.workloads.SEED, rank), device=dev, **rule_kw)  # every rank: its own independent lattice
    for kv in args.opt:
        k, v = kv.split("=")
        S.set_option(int(k), int(v))
    beta, SPS = w["beta"], args.sweeps_per_step
    updates_per_step = S.N * S.R * SPS

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        return ranks.max_over_ranks(x, dist, dev)

    # ---- device-resident arm -------------------------------------------------------------------
    for _ in range(args.warmup):
        S.sweep(beta, SPS)
        S.measure()
    sweep_ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches0 = S.launch_count
    sampler = ClockSampler(local_rank) if rank == 0 else None
    barrier()
    t_wall0 = time.time()
    e0.record()
    for k in range(args.steps):
        sweep_ev[k][0].record()
        S.sweep(beta, SPS)
        sweep_ev[k][1].record()
        E, M = S.measure()
    e1.record()
    barrier()
    t_wall1 = time.time()
    clocks = sampler.stop(t_wall0, t_wall1) if sampler else None
    launches = S.launch_count - launches0
    # counters of the kernel that ran: with --opt another kernel may serve the workload -- its capture if there is one
    # (profiles/counters.json "<workload>#<variant>"), else none (null traffic rather than another kernel's numbers)
    variant = {("4=0",): "#strip", ("1=1",): "#tma"}.get(tuple(args.opt)) if args.opt else ""
    if args.rule == "heatbath":
        variant = "#heatbath" if not args.opt else None
    cnt = COUNTERS.get(args.workload + variant, {}) if variant is not None else {}
    ms_total = max_over_ranks(e0.elapsed_time(e1))
    ms_sweeps = sum(a.elapsed_time(b) for a, b in sweep_ev)
    value = world * updates_per_step * args.steps / (ms_total * 1e6)
    sweep_launches = launches - 2 * args.steps                  # spin_measure: one pass + one finalize per step
    ms_launch = ms_sweeps / sweep_launches
    bpu = P.workloads.BYTES_PER_UPDATE[args.workload]
    updates_per_launch = S.N * S.R * SPS * args.steps / sweep_launches   # N R / 2 per half-sweep launch, 2 N R per two-sweep pass
    bytes_per_launch = bpu * updates_per_launch
    achieved = bytes_per_launch / (ms_launch * 1e6)  # GB/s

    # ---- end-to-end arm: host buffers through the C ABI ------------------------------------------
    # Ising: the configuration travels as the canonical BIT array (one bit per spin; spin_set_spins_bits_async), continuous
    # spins as the canonical fp32 array (spin_set_spins_async); both from pinned host memory on the timed stream
    use_bits = S.n == 1 and w["storage"] in ("int8", "bitpack")
    host = torch.from_numpy(S.get_spins_bits() if use_bits else S.get_spins()).pin_memory()
    host_np = host.numpy()
    upload = S.set_spins_bits_async if use_bits else S.set_spins_async
    for _ in range(2):
        upload(host_np)
        S.sweep(beta, SPS)
        S.measure()
    S.set_spins_status()
    f0, f1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    f0.record()
    for k in range(args.steps):
        upload(host_np)                  # pinned host array -> device on this stream, then the conversion kernel
        S.sweep(beta, SPS)
        E, M = S.measure()               # blocking: host doubles
    f1.record()
    barrier()
    S.set_spins_status()                 # the +-1 check of the last upload (raises if it failed)
    ms_e2e = max_over_ranks(f0.elapsed_time(f1))
    e2e = {"value": world * updates_per_step * args.steps / (ms_e2e * 1e6), "unit": UNIT,
           "h2d_bytes_per_step": int(host_np.nbytes), "d2h_bytes_per_step": int(8 * S.R * (1 + S.n)),
           "ms_per_step": ms_e2e / args.steps,
           "what": ("spin_set_spins_bits_async(pinned host bit array, one bit per spin" if use_bits else "spin_set_spins_async(pinned host fp32 array")
                   + ", same stream) + spin_sweep + spin_measure(host E, M) per step"}
    S_N_R = S.N * S.R
    S.close()
    del S, host, host_np
    torch.cuda.empty_cache()

    if rank != 0:
        if dist is not None:
            dist.barrier()
            dist.destroy_process_group()
        return
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": DTYPE[w["storage"]], "data": "synthetic",
        "config": {"workload": args.workload, "dims": list(w["dims"]), "n": w["n"], "beta": beta,
                   "storage": w["storage"], "replicas": w["replicas"], "sweeps_per_step": SPS,
                   "step": "%d sweeps + 1 E/M measurement" % SPS, "seed": P.workloads.SEED,
                   "l2": "state (%.0f MB) larger than L2 (126 MB); no flush needed" % (w["dims"][0] * w["dims"][1] * w["dims"][2] * w["replicas"] / 1e6)
                   if w["storage"] != "bitpack" else "bit-packed state is L2-resident by design (33.5 MB); not flushed",
                   "parallelism": "independent lattice per GPU (weak scaling, no collective)" if world > 1 else "1 GPU",
                   "options": args.opt, "update_rule": args.rule},
        "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        "roofline": {"bound": "hbm", "kernel": cnt.get("kernel", "half-sweep of %s" % args.workload), "achieved": achieved,
                     "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": cnt.get("dram_bytes_per_launch"),
                     "peak_source": peak_src, "bytes_per_launch": bytes_per_launch, "ms_per_launch": ms_launch,
                     "updates_per_launch": updates_per_launch, "bytes_per_update": bpu,
                     "frac_of_nominal_8000": achieved / 8000.0, "capture": cnt.get("capture")},
    }
    if cnt.get("dram_bytes_per_launch") and cnt.get("updates_per_launch"):
        # what the kernel really moves: DRAM bytes of the committed ncu capture, per update and as a bandwidth at this run's time
        tr = cnt["dram_bytes_per_launch"] * (updates_per_launch / cnt["updates_per_launch"])
        line["roofline"].update({"dram_bytes_per_update": tr / updates_per_launch, "dram_GBps": tr / (ms_launch * 1e6),
                                 "dram_frac": tr / (ms_launch * 1e6) / peak})
    if cnt.get("warp_instr_per_launch") and cnt.get("updates_per_launch"):
        wi = cnt["warp_instr_per_launch"] * (updates_per_launch / cnt["updates_per_launch"])
        line["roofline"].update({"issue_frac": wi / (ms_launch * 1e6) / ISSUE_PEAK_GWIPS,
                                 "alu_pipe_busy_pct_in_capture": cnt.get("alu_pipe_pct")})
    if updates_per_launch > S_N_R and "tblock" not in str(cnt.get("kernel", "tblock")):
        line["roofline"]["note"] = ("one launch = all sweeps of the call with the state resident in shared memory: the HBM fraction on "
                                    "algorithmic bytes is nominal (frac > 1 is possible); the kernel is bound by instruction issue")
    elif updates_per_launch > S_N_R:
        line["roofline"]["note"] = ("exact temporal blocking (SURVEY f3): one launch = two full sweeps, each row read once and written "
                                    "once, so the DRAM traffic is a third of the algorithmic 3 B per update the fraction is quoted on "
                                    "(frac > 1 is that saving, not idle work); the kernel is bound by the integer ALU pipe")
    if not args.no_per_model and world == 1:
        line["per_model"] = run_per_model(P, peak)
    if not args.no_cpu_baseline:
        line["cpu_baseline"] = cpu_baseline(P, args.workload)
    print(json.dumps(line), flush=True)
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


# Counters of the dominant kernel of each workload, from the committed `ncu --set full` captures: profiles/counters.json is
# written from the ncu exports (each entry names its kernel and its capture), so a replaced kernel cannot keep the numbers of
# its predecessor -- an entry whose kernel no longer runs is dropped there and the fields here become null.
#   dram_bytes_per_launch = dram__bytes_read.sum + dram__bytes_write.sum, warp_instr_per_launch = smsp__inst_executed.sum
def load_counters():
    try:
        with open(os.path.join(ROOT, "profiles", "counters.json")) as f:
            return json.load(f)
    except Exception:
        return {}


COUNTERS = load_counters()
# issue rate: 148 SMs x 4 sub-cores x 1 warp-instruction per clock x 1.965 GHz
ISSUE_PEAK_GWIPS = 148 * 4 * 1.965


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="graft", choices=["graft", "reference"])
    ap.add_argument("--workload", default=DEFAULT_WORKLOAD)
    ap.add_argument("--sweeps-per-step", type=int, default=100)
    ap.add_argument("--mode", default="replicas", choices=["replicas", "slab"],
                    help="replicas: one independent lattice per GPU (weak scaling, the default and the driver's contract); "
                         "slab: ONE lattice cut into one slab per GPU with a halo exchange per half-sweep (strong scaling)")
    ap.add_argument("--opt", action="append", default=[], metavar="ID=VALUE",
                    help="spin_set_option(ID, VALUE) on the timed handle (A/B of kernel variants, e.g. 1=1: TMA-staged kernel, "
                         "4=0: no temporal blocking); repeatable")
    ap.add_argument("--rule", default="metropolis", choices=["metropolis", "heatbath"],
                    help="update rule of the timed handle (heat bath: SURVEY f1; the per-model legs time it on three lattices)")
    ap.add_argument("--no-per-model", action="store_true")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.warmup < 3 and args.impl == "graft":
        args.warmup = 3
    if args.impl == "reference":
        run_reference(args)
    elif args.mode == "slab":
        run_slab(args)
    else:
        run_graft(args)


if __name__ == "__main__":
    main()
