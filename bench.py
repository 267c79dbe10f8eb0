#!/usr/bin/env python
"""bench.py -- throughput of the batched TB-SMA MD step on B200 (one JSON line on stdout).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 3] [--impl tbsma|reference]

A "step" is one MD step of EVERY replica of the workload: integrate (B A O A + grips), per-replica
neighbour rebuild when due, density pass, force pass (+ closing half kick).  Default workload =
BASELINE.json configs[2] ("config3": 256 replicas x 3 nm x 24 nm Au wire, 2 673 408 atoms, 10 K and
298 K halves, Langevin + pulling) -- the headline batched configuration; configs 1-2 are latency
cases and parity tests, configs 4, 5a, 5b can be selected with --config.
metric = atom-timesteps/s (whole job).  N > 1 (torchrun): every rank runs its own batch of replicas
(weak scaling, replicas only, no collective on the data path).
--impl reference times the fp64 CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import json
import os
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

from paper_1311_3890_b200 import workloads as W  # noqa: E402

METRIC = "atom_timesteps_per_s"
UNIT = "atom-steps/s"


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, burst copy)"
    return 6650.0, "fallback (B200_PROFILING.md)"


def make_workload(cfg, rank=0, replicas=None):
    seed_shift = 1000 * rank
    if cfg == "1":
        return W.config1(1 + seed_shift)
    if cfg == "2":
        return W.config2(2 + seed_shift)
    if cfg == "3":
        return W.config3(replicas or 256, 3 + seed_shift)
    if cfg == "4":
        return W.config4(replicas or 2048, 4 + seed_shift)
    if cfg == "5a":
        return W.config5a(64, 5 + seed_shift)
    if cfg == "5b":
        return W.config5b(6 + seed_shift)
    if cfg.startswith("paper"):       # paper:k:T[:replicas], e.g. paper:12:10 = the largest row of the paper's Table 2
        f = cfg.split(":")
        k = int(f[1]) if len(f) > 1 else 1
        T = float(f[2]) if len(f) > 2 else 10.0
        return W.paper_wire(k, T, replicas or (int(f[3]) if len(f) > 3 else 1), 7 + seed_shift)
    raise SystemExit(f"unknown --config {cfg}")


def force_kernel_name(ctx):
    """the kernel the force pass of this batch is launched as (what roofline.kernel names)"""
    n_tiles, box, persistent = ctx.get_tiling()
    if not n_tiles:
        return "k_force (thread per atom, int32 list)"
    if persistent:
        return "k_gather_persist<1,...> (persistent force/energy pass + closing half kick)"
    if "cooperative" in ctx.describe_gather():
        return "k_step_small (whole step in one cooperative kernel; force pass = its third phase)"
    return "k_force_tile (one CTA per %s tile)" % ("box" if box else "layer")


def measure_workload(cfg, args, B, torch, dev, local_rank, peak):
    """One of the other BASELINE workloads, measured like the headline (same --steps / --warmup / --preroll, CUDA events on
    the launching stream, per-kernel pass, clocks sampled during the timed region): a compact record for the `workloads`
    block of the JSON line."""
    w = make_workload(cfg, 0, None)
    ctx = B.make_context(w)
    st = B.DeviceState(w, dev)
    stream = torch.cuda.Stream(device=dev)
    K, Wm, P0 = args.steps, args.warmup, max(args.preroll, 0)

    def run(step0, n):
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, step0, n, st.slab_rate * float(step0),
                   st.slab_rate, w.rebuild_every, st.e_rep, None, st.ekin)

    with torch.cuda.stream(stream):
        ctx.build_cells(st.pos, st.vel, st.tag)
        ctx.build_neighbors(st.pos, st.vel, st.tag)
        ctx.compute(st.pos, st.force, st.e_rep, None)
        if P0:
            run(0, P0)
        run(P0, Wm)
    sampler = ClockSampler(local_rank)
    sampler.start()
    torch.cuda.synchronize()
    stats0 = ctx.get_stats()
    launches0 = ctx.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t0 = time.perf_counter()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        run(P0 + Wm, K)
        ev1.record(stream)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    sampler.stop_flag = True
    ms = ev0.elapsed_time(ev1)
    launches = ctx.launch_count() - launches0
    stats1 = ctx.get_stats()
    entries, pairs = ctx.count_pairs(st.pos, stream)
    n_l = entries / w.n_atoms
    k_eff = K * w.n_replicas / max(stats1["n_replica_builds"] - stats0["n_replica_builds"], 1)
    ctx.set_timing(True)
    with torch.cuda.stream(stream):
        run(P0 + Wm + K, min(args.kernel_steps, 512))
    tms, tsteps = ctx.get_timing()
    ctx.set_timing(False)
    pk = {k: v / max(tsteps, 1) for k, v in tms.items()}
    status = ctx.status()
    step_bytes = (8.0 * n_l + 160.0 + (4.0 * n_l + 120.0) / k_eff) * w.n_atoms
    out = {"workload": w.name, "atoms": w.n_atoms, "replicas": w.n_replicas, "value": w.n_atoms * K / (ms * 1e-3),
           "unit": UNIT, "ms_per_step": ms / K, "pair_interactions_per_s": 0.5 * pairs * K / (ms * 1e-3),
           "variant": {1: "global gather (int32 list)", 2: "shared-memory tiles (u16 lists)"}.get(ctx.get_variant()),
           "gather_kernels": ctx.describe_gather(), "force_kernel": force_kernel_name(ctx),
           "mean_list_length": n_l, "mean_steps_between_rebuilds": k_eff,
           "whole_step_frac": step_bytes / (ms / K * 1e-3) / 1e9 / peak,
           "force_frac": ((4.0 * n_l + 40.0) * w.n_atoms / (pk["force"] * 1e-3) / 1e9 / peak) if pk["force"] > 0 else None,
           "density_frac": ((4.0 * n_l + 24.0) * w.n_atoms / (pk["density"] * 1e-3) / 1e9 / peak) if pk["density"] > 0 else None,
           "per_kernel_ms": pk, "gpu_launches": int(launches), "status_flags": status,
           "clocks": sampler.summary(t0, t1)}
    ctx.destroy()
    del st
    torch.cuda.empty_cache()
    return out


class ClockSampler(threading.Thread):
    """SM clock / throttle reasons sampled with NVML while the timed region runs."""

    def __init__(self, index, period=0.002):
        super().__init__(daemon=True)
        self.index, self.period = index, period
        self.samples, self.stop_flag, self.ok = [], False, False
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
            self.ok = True
        except Exception as e:  # pragma: no cover
            self.err = repr(e)

    def run(self):
        if not self.ok:
            return
        nv = self.nv
        while not self.stop_flag:
            try:
                mhz = nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)
                reasons = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                self.samples.append((time.perf_counter(), mhz, int(reasons)))
            except Exception:
                pass
            time.sleep(self.period)

    def summary(self, t0, t1):
        if not self.ok:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvml unavailable"]}
        nv = self.nv
        sel = [s for s in self.samples if t0 <= s[0] <= t1] or self.samples[-3:]
        names = {
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwPowerBrakeSlowdown", 0x80): "hw_power_brake_slowdown",
        }
        seen = set()
        for _, _, r in sel:
            for bit, nm in names.items():
                if r & bit:
                    seen.add(nm)
        mhz = sorted(s[1] for s in sel)
        return {"sm_mhz": mhz[len(mhz) // 2] if mhz else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(seen), "samples": len(sel)}


def cpu_oracle_rate(w, n_rep, n_steps, cells=True):
    """The oracle as it stands (fp64, OpenMP), timed on a bounded sample: the first n_rep replicas for n_steps MD steps.
    cells=True: its linked-cell path (SURVEY 8(d) "Oracle-CL", the fair CPU baseline); cells=False: the brute-force
    O(N^2) path the parity tests use (SURVEY 8(d) "Oracle-BF").  Returns (atom-steps/s, cores, text)."""
    import oracle
    sub = w.take(0, min(n_rep, w.n_replicas))
    md = oracle.MD(sub.x64(), sub.v64(), sub.flags, sub.r_cut, offsets=sub.offsets, lo=sub.box_lo, hi=sub.box_hi,
                   periodic=sub.periodic, fp32_pred=False, cells=cells, zref=sub.vel4[:, 3].astype(np.float64))
    t0 = time.perf_counter()
    for s in range(n_steps):
        md.step(sub.dt, sub.T.astype(np.float64), sub.gamma, sub.seed, s, slab_disp=sub.slab_rate * (s + 1))
    dt = time.perf_counter() - t0
    how = "linked-cell fp64 OpenMP oracle (Oracle-CL)" if cells else "brute-force O(N^2) fp64 OpenMP oracle (Oracle-BF)"
    return sub.n_atoms * n_steps / dt, oracle.num_threads(), \
        f"first {sub.n_replicas} replica(s) of {w.name} ({sub.n_atoms} atoms) x {n_steps} steps, {how}"


def run_reference(args, rank):
    """--impl reference: the CPU oracle on the box's host cores, same metric / config."""
    if rank != 0:
        return
    w = make_workload(args.config, 0, replicas=2 if args.config in ("3", "4") else None)
    if args.config == "5a":
        w = W.config5a(16, 5)    # 16 384-atom periodic block of the same lattice: a bounded sample of the 10^6-atom box
    sub = w.take(0, 1)
    import oracle
    md = oracle.MD(sub.x64(), sub.v64(), sub.flags, sub.r_cut, offsets=sub.offsets, lo=sub.box_lo, hi=sub.box_hi,
                   periodic=sub.periodic, fp32_pred=False, cells=True, zref=sub.vel4[:, 3].astype(np.float64))
    s = 0
    for _ in range(args.warmup):
        md.step(sub.dt, sub.T.astype(np.float64), sub.gamma, sub.seed, s, slab_disp=sub.slab_rate * (s + 1))
        s += 1
    t0 = time.perf_counter()
    for _ in range(args.steps):
        md.step(sub.dt, sub.T.astype(np.float64), sub.gamma, sub.seed, s, slab_disp=sub.slab_rate * (s + 1))
        s += 1
    dt = time.perf_counter() - t0
    value = sub.n_atoms * args.steps / dt
    sample = f"each step = 1 replica of {w.name} ({sub.n_atoms} atoms), linked-cell fp64 OpenMP oracle (Oracle-CL)"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w.name, "sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=300)
    ap.add_argument("--warmup", type=int, default=60)
    ap.add_argument("--config", default="3",
                    help="1, 2, 3, 4, 5a, 5b (BASELINE.json configs) or paper:k:T[:replicas] (shapes of the paper's Table 2)")
    ap.add_argument("--replicas", type=int, default=None, help="override the replica count of config 3/4")
    ap.add_argument("--impl", default="tbsma", choices=["tbsma", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--workloads", default=None,
                    help="comma-separated configs measured after the headline and reported under `workloads` in the same "
                         "JSON line (default with --config 3 on one GPU: 4,5a,5b,1,2; 'none' to skip)")
    ap.add_argument("--kernel-steps", type=int, default=60, help="steps of the per-kernel CUDA-event timing pass")
    ap.add_argument("--preroll", type=int, default=300,
                    help="declared, untimed steps before the warm-up: replicas built together rebuild together at first; "
                         "the timed region should see the steady rebuild cadence, not that transient")
    ap.add_argument("--outer-skin", type=float, default=None,
                    help="buffer radius S of the candidate lists of the tile variant (tbsma_set_outer_skin; library default if omitted)")
    ap.add_argument("--variant", type=int, default=None,
                    help="tbsma_set_variant: 0 = automatic (library default), 1 = global gather, 2 = shared-memory tiles")
    ap.add_argument("--gather", type=int, default=None,
                    help="tbsma_set_gather: 1 = persistent gather kernels (library default), 0 = one CTA per tile")
    ap.add_argument("--plain-graph", action="store_true",
                    help="capture the step without the conditional node (Nsight Compute cannot profile kernel nodes "
                         "of graphs that hold conditional nodes): for the ncu passes under profiles/")
    args = ap.parse_args()
    if args.warmup < 3:
        args.warmup = 3
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return
    if args.gpus != world:
        if world == 1 and args.gpus > 1:
            raise SystemExit("for --gpus N > 1 launch with: python -m torch.distributed.run --nnodes=1 "
                             "--nproc-per-node N --master-addr 127.0.0.1 --master-port P bench.py --gpus N ...")
    import torch
    import torch.distributed as dist
    from paper_1311_3890_b200 import binding as B

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = f"cuda:{local_rank}"
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(dev))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    def max_over_ranks(x):
        if world > 1:
            t = torch.tensor([x], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
            return float(t.item())
        return float(x)

    def sum_over_ranks(x):
        if world > 1:
            t = torch.tensor([x], dtype=torch.float64, device=dev)
            dist.all_reduce(t, op=dist.ReduceOp.SUM)
            return float(t.item())
        return float(x)

    # Multi-GPU = replicas only: the job is one batch of world x R replicas, partitioned contiguously
    # by sharding.replica_range; rank k owns replicas [r0, r1) and builds just those (seeds are a function of the global
    # replica index through the per-rank seed shift), no data-path collective.
    from paper_1311_3890_b200 import sharding
    w = make_workload(args.config, rank, args.replicas)
    r0, r1 = sharding.replica_range(w.n_replicas * world, rank, world)
    assert r1 - r0 == w.n_replicas
    ctx = B.make_context(w)
    if args.plain_graph:
        ctx.set_graph(True, conditional=False)
    if args.outer_skin is not None:
        ctx.set_outer_skin(args.outer_skin)
    if args.gather is not None:
        ctx.set_gather(args.gather)
    if args.variant is not None:
        ctx.set_variant(args.variant)
    st = B.DeviceState(w, dev)
    stream = torch.cuda.Stream(device=dev)
    K, Wm, P0 = args.steps, args.warmup, max(args.preroll, 0)

    def run(step0, n):
        """steps step0 .. step0 + n - 1; the pulled slab continues where the previous call left it"""
        ctx.md_run(st.pos, st.vel, st.force, st.tag, w.dt, st.T, w.gamma, st.seed, step0, n, st.slab_rate * float(step0),
                   st.slab_rate, w.rebuild_every, st.e_rep, None, st.ekin)

    with torch.cuda.stream(stream):
        ctx.build_cells(st.pos, st.vel, st.tag)
        ctx.build_neighbors(st.pos, st.vel, st.tag)
        ctx.compute(st.pos, st.force, st.e_rep, None)
        if P0:
            run(0, P0)
        run(P0, Wm)
    sampler = ClockSampler(local_rank)
    sampler.start()
    barrier()
    stats0 = ctx.get_stats()
    launches0 = ctx.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_host0 = time.perf_counter()
    with torch.cuda.stream(stream):
        ev0.record(stream)
        run(P0 + Wm, K)
        ev1.record(stream)
    barrier()
    t_host1 = time.perf_counter()
    sampler.stop_flag = True
    ms = max_over_ranks(ev0.elapsed_time(ev1))
    launches = ctx.launch_count() - launches0
    stats1 = ctx.get_stats()
    status = ctx.status()
    # the only traffic of the job: per-replica observables of the last step onto every rank (a few doubles per replica)
    obs = sharding.gather_replica_values(np.stack([st.e_rep.cpu().numpy(), st.ekin.cpu().numpy()], axis=1),
                                         w.n_replicas * world, rank, world, dist if world > 1 else None, dev if world > 1 else None)
    n_total = sum_over_ranks(w.n_atoms)
    value = n_total * K / (ms * 1e-3)
    entries, pairs = ctx.count_pairs(st.pos, stream)
    n_l = entries / w.n_atoms
    builds = stats1["n_replica_builds"] - stats0["n_replica_builds"]
    k_eff = K * w.n_replicas / max(builds, 1)          # mean steps between rebuilds of a replica
    pair_rate = sum_over_ranks(0.5 * pairs) * K / (ms * 1e-3)

    # per-kernel pass: CUDA events on the launching stream around every kernel class
    ctx.set_timing(True)
    ks = min(args.kernel_steps, 512)
    with torch.cuda.stream(stream):
        run(P0 + Wm + K, ks)
    tms, tsteps = ctx.get_timing()
    ctx.set_timing(False)
    peak, peak_src = load_peaks()
    per_kernel_ms = {k: v / max(tsteps, 1) for k, v in tms.items()}
    # algorithmic bytes per launch: force pass 4 n_L + 40 B/atom,
    # density pass 4 n_L + 24 B/atom, whole step 8 n_L + 160 + (4 n_L + 120)/K_eff B/atom.  That budget is the survey's:
    # an int32 list.  The tile variant streams 16-bit entries, so what it must move is less ("as_built" below, 2 B per
    # entry): both are reported, and so is the DRAM traffic ncu measured.
    force_bytes = (4.0 * n_l + 40.0) * w.n_atoms
    dens_bytes = (4.0 * n_l + 24.0) * w.n_atoms
    step_bytes = (8.0 * n_l + 160.0 + (4.0 * n_l + 120.0) / k_eff) * w.n_atoms
    eb = 2.0 if ctx.get_variant() == 2 else 4.0          # bytes per list entry of the variant that ran
    force_bytes_built = (eb * n_l + 40.0) * w.n_atoms
    dens_bytes_built = (eb * n_l + 24.0) * w.n_atoms
    step_bytes_built = (2 * eb * n_l + 160.0 + (eb * n_l + 120.0) / k_eff) * w.n_atoms
    ach_force = force_bytes / (per_kernel_ms["force"] * 1e-3) / 1e9 if per_kernel_ms["force"] > 0 else 0.0
    ach_dens = dens_bytes / (per_kernel_ms["density"] * 1e-3) / 1e9 if per_kernel_ms["density"] > 0 else 0.0
    ach_step = step_bytes / (ms / K * 1e-3) / 1e9
    roofline = {"bound": "hbm", "kernel": force_kernel_name(ctx),
                "achieved": ach_force, "peak": peak, "unit": "GB/s", "frac": ach_force / peak, "traffic": None,
                "peak_source": peak_src, "algorithmic_bytes_per_launch": force_bytes,
                "avg_launch_ms": per_kernel_ms["force"],
                "density_pass": {"achieved": ach_dens, "frac": ach_dens / peak, "avg_launch_ms": per_kernel_ms["density"]},
                "whole_step": {"achieved": ach_step, "frac": ach_step / peak, "bytes_per_atom_step": step_bytes / w.n_atoms},
                "bytes_model": "SURVEY 8(d): int32 list, 4 B per entry (the designated budget; the tile variant stores 2 B entries)",
                "as_built": {
                    "bytes_per_list_entry": eb,
                    "force_pass": {"bytes_per_launch": force_bytes_built,
                                   "achieved": force_bytes_built / (per_kernel_ms["force"] * 1e-3) / 1e9 if per_kernel_ms["force"] > 0 else 0.0},
                    "density_pass": {"bytes_per_launch": dens_bytes_built,
                                     "achieved": dens_bytes_built / (per_kernel_ms["density"] * 1e-3) / 1e9 if per_kernel_ms["density"] > 0 else 0.0},
                    "whole_step": {"bytes_per_atom_step": step_bytes_built / w.n_atoms,
                                   "achieved": step_bytes_built / (ms / K * 1e-3) / 1e9}},
                "per_kernel_ms": per_kernel_ms, "timed_steps": tsteps,
                "per_kernel_note": "CUDA events between the kernel classes with graph replay and overlap OFF (kernels one "
                                   "after the other); in the timed step the list renewal runs beside the gather passes, so "
                                   "per_kernel_ms.rebuild is not what the step pays"}
    for k in ("force_pass", "density_pass", "whole_step"):
        roofline["as_built"][k]["frac"] = roofline["as_built"][k]["achieved"] / peak
    # dram__bytes_read.sum + dram__bytes_write.sum of one launch of the dominant kernel, from the committed ncu capture
    # (a number from a committed capture, NOT measured in this run: it names the capture it comes from and is refreshed
    # with every change of the kernel; null for workloads that have no capture)
    traffic_file = next((f for f in (os.path.join(ROOT, "profiles", "r%d_force_kernel_traffic.csv" % r) for r in (3, 2))
                         if os.path.exists(f)), "")
    if os.path.exists(traffic_file):
        try:
            import csv
            for row in csv.DictReader(open(traffic_file)):
                if row["workload"] == w.name and row["kernel"].startswith(("k_force", "k_gather_persist<1")):
                    roofline["traffic"] = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
                    roofline["traffic_from"] = "committed ncu capture: " + row["source"]
        except Exception:
            pass
    roofline["note"] = ("HBM is the designated roofline (BASELINE.json); with 16-bit lists the gather passes move less than "
                        "the algorithmic bytes and are bound on chip: MUFU, shared-memory data pipe and issue slots at "
                        "55-75 % each (profiles/r2_ncu_full_summary.md)")

    # end to end through the C ABI with HOST buffers (pinned), copies inside the timed region
    e2e = None
    if not args.no_e2e:
        ctx2 = B.make_context(w)
        hp = torch.from_numpy(w.pos4.copy()).pin_memory()
        hv = torch.from_numpy(w.vel4.copy()).pin_memory()
        hf = torch.zeros_like(hp).pin_memory()
        ht = torch.arange(w.n_atoms, dtype=torch.int32).pin_memory()
        he, hk = np.zeros(w.n_replicas), np.zeros(w.n_replicas)
        k2 = max(10, K)              # one call of the end-to-end entry point integrates as many steps as the timed region
        # warm-up call (allocates the staging buffers, instantiates the graph)
        ctx2.md_run_host(hp.numpy(), hv.numpy(), hf.numpy(), ht.numpy(), w.dt, w.T, w.gamma, w.seed, 0, 8, None,
                         w.slab_rate, w.rebuild_every, he, None, hk)
        hp.copy_(torch.from_numpy(w.pos4)); hv.copy_(torch.from_numpy(w.vel4))
        ht.copy_(torch.arange(w.n_atoms, dtype=torch.int32))
        barrier()
        t0 = time.perf_counter()
        ctx2.md_run_host(hp.numpy(), hv.numpy(), hf.numpy(), ht.numpy(), w.dt, w.T, w.gamma, w.seed, 0, k2, None,
                         w.slab_rate, w.rebuild_every, he, None, hk)
        dt_e2e = max_over_ranks(time.perf_counter() - t0)
        h2d = w.n_atoms * 36 + w.n_replicas * 28
        d2h = w.n_atoms * 52 + w.n_replicas * 16
        e2e = {"value": n_total * k2 / dt_e2e, "unit": UNIT, "h2d_bytes_per_step": h2d / k2,
               "d2h_bytes_per_step": d2h / k2, "steps": k2,
               "call": "tbsma_md_run_host (H2D pos/vel/tag, cell+list build, initial forces, steps, D2H pos/vel/force/tag)"}
        ctx2.destroy()

    # the other workloads of BASELINE.json, same binary, same call, same --steps / --warmup (one GPU, headline config only)
    others = None
    variant_ran, gather_desc = ctx.get_variant(), ctx.describe_gather()
    wl = args.workloads if args.workloads is not None else ("4,5a,5b,1,2" if args.config == "3" and world == 1 else "none")
    if rank == 0 and world == 1 and wl != "none":
        ctx.destroy()
        del st
        torch.cuda.empty_cache()
        others = {}
        for cfg in wl.split(","):
            others[cfg] = measure_workload(cfg, args, B, torch, dev, local_rank, peak)

    cpu = cpu_bf = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        # bounded samples (about 10-20 s of CPU work together): the linked-cell oracle is the CPU baseline, the brute-force
        # one (what the parity tests run) is reported beside it
        nrep, nst = (8, 20) if args.config in ("3",) else (16, 40) if args.config == "4" else (1, 40)
        if args.config == "5a":
            wc = W.config5a(24, 5)
            rate, cores, sample = cpu_oracle_rate(wc, 1, 10, cells=True)
            rbf, _, sbf = cpu_oracle_rate(W.config5a(8, 5), 1, 10, cells=False)
        elif args.config == "5b":
            rate, cores, sample = cpu_oracle_rate(w, 1, 10, cells=True)
            rbf, _, sbf = cpu_oracle_rate(W.config2(), 1, 10, cells=False)
        else:
            rate, cores, sample = cpu_oracle_rate(w, nrep, nst, cells=True)
            rbf, _, sbf = cpu_oracle_rate(w, 2 if args.config in ("3", "4") else 1, 4, cells=False)
        cpu = {"value": rate, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample}
        cpu_bf = {"value": rbf, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sbf}

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "atoms_per_gpu": w.n_atoms, "replicas_per_gpu": w.n_replicas,
                       "r_cut": w.r_cut, "skin": w.skin, "dt_fs": w.dt, "gamma_per_fs": w.gamma,
                       "rebuild": "displacement > skin/2 per replica" if not w.rebuild_every else f"every {w.rebuild_every} steps",
                       "mean_list_length": n_l, "mean_steps_between_rebuilds": k_eff,
                       "l2": "inputs larger than L2 (index list %.0f MB per pass)" % (entries * 4 / 1e6),
                       "variant": {1: "global gather (int32 list)", 2: "shared-memory tiles (u16 lists)"}.get(variant_ran),
                       "gather_kernels": gather_desc,
                       "list_renewal": "asynchronous, margin 0.03 A, beside the gather passes (density pass = programmatic dependent of the filter kernel)" if variant_ran == 2 and not w.rebuild_every else "ahead of the gather passes",
                       "graph": "plain" if args.plain_graph else "conditional node around the cells+candidates chain",
                       "preroll_steps": P0,
                       "parallelism": "replicas only" if world > 1 else "1 gpu"},
            "pair_interactions_per_s": pair_rate,
            "observables": {"replicas": int(obs.shape[0]), "e_pot_eV_per_atom": float(obs[:, 0].sum() / n_total),
                            "e_kin_eV_per_atom": float(obs[:, 1].sum() / n_total)},
            "clocks": sampler.summary(t_host0, t_host1),
            "e2e": e2e, "gpu_launches": int(launches), "status_flags": status,
            "roofline": roofline, "cpu_baseline": cpu, "cpu_baseline_cl": cpu, "cpu_baseline_bf": cpu_bf,
            "workloads": others,
        }
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
