#!/usr/bin/env python
"""bench.py -- whole-generation throughput of the LIETS growth path on B200 (one JSON line).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--storage 0|1|2]

A "step" is one pass of the whole hot path over one synthetic workload: liets_seed (keyed seeding +
L1 seed spacing) followed by liets_generate (device-resident growth loop to the target fraction)
on BASELINE.json's 400^3 timing configuration (workloads.BENCH).  `value` = voxel nodes/s =
N_voxels * n_gpus / device time, timed with CUDA events on the launching stream; `e2e` = the same
through the C ABI with a HOST output buffer (device->host copy of the phase array inside the
timed region).  Multi-GPU = independent replicas (one realisation per rank, no collective on the
data path), timing = max over ranks.
"""
import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import workloads  # noqa: E402


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            return json.load(f), "measured"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler(threading.Thread):
    """Samples SM clock and throttle reasons with NVML while the timed regions run."""

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.samples, self.reasons, self.max_mhz = index, [], set(), None
        self._stop_evt = threading.Event()
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.max_mhz = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception:
            self.nv = None

    def run(self):
        if self.nv is None:
            return
        nv = self.nv
        names = {
            getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8): "hw_slowdown",
            getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40): "hw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20): "sw_thermal_slowdown",
            getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4): "sw_power_cap",
        }
        while not self._stop_evt.is_set():
            try:
                self.samples.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                try:
                    r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h)
                except Exception:
                    r = nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in names.items():
                    if r & bit:
                        self.reasons.add(name)
            except Exception:
                pass
            time.sleep(0.01)

    def stop(self):
        self._stop_evt.set()
        self.join(timeout=2)
        s = sorted(self.samples)
        return {"sm_mhz": s[len(s) // 2] if s else None, "sm_max_mhz": self.max_mhz,
                "reasons": sorted(self.reasons), "samples": len(s)}


def algorithmic_bytes(storage, N, front, solid_after, n_seeds, on_tiles=None, front_voxels=None):
    """bytes the list-indexed step itself must move, per step.

    Voxel list (STORAGE_U8, b = w = 1 byte; or the small-front steps of STORAGE_TILE on the bit grid, b = 1/8, w = 8:
    one 64-bit word per claim and grid copy):  4|A_t| + b min(27|A_t|, N) + w c_t + 4|A_{t+1}|
    Tile list (STORAGE_TILE, 128x8x8 tiles of 1 KiB): 4|L_t| + min(1625|L_t|, N/8) + 1024|L_t| + 4|L_{t+1}|
      (read the tile list; each needed grid byte once -- a tile plus its one-voxel halo is 130x10x10
      bits = 1625 B; write the tile's rows into the next buffer; write the next list).
    on_tiles[t]: step t of STORAGE_TILE ran on the tile list (default: all); front_voxels[t]: its front voxels."""
    out, prev = [], n_seeds
    for t in range(len(front)):
        a_t = int(front[t])
        a_n = int(front[t + 1]) if t + 1 < len(front) else a_t
        c_t = int(solid_after[t]) - prev
        prev = int(solid_after[t])
        if storage == 0:
            out.append(4 * a_t + min(27 * a_t, N) + c_t + 4 * a_n)
        elif storage == 2:                            # full-field sweep: read g_t once, write g_{t+1} once
            out.append(2 * ((N + 7) // 8))
        elif on_tiles is None or on_tiles[t]:
            out.append(4 * a_t + min(1625 * a_t, N // 8) + 1024 * a_t + 4 * a_n)
        else:
            v_t = int(front_voxels[t]) if front_voxels is not None else a_t
            out.append(4 * v_t + min(27 * v_t, N) // 8 + 2 * 8 * c_t + 4 * a_n)
    return out


def max_over_ranks(values, dist, device):
    """Replicas only: the one exchange of a multi-GPU run is the max of the device times."""
    if dist is None:
        return [float(v) for v in values]
    import torch
    tt = torch.tensor(values, dtype=torch.float64, device=device)
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return [float(v) for v in tt]


def whole_job_throughput(n_voxels, world, steps, total_ms):
    """nodes/s of the whole job: every rank generates `steps` grids of n_voxels in total_ms (max over ranks)."""
    return n_voxels * world * steps / (total_ms * 1e-3)


def run_reference(args):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the same workload."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import oracle
    oracle.build()
    w = workloads.BENCH_CPU_SAMPLE
    nx, ny, nz = w["dims"]
    N = nx * ny * nz

    def one():
        return time_oracle(w, False)
    for _ in range(args.warmup):
        one()
    total = sum(one() for _ in range(args.steps))
    value = N * args.steps / total
    sample = "%s: %dx%dx%d sub-volume of %s, same parameters, serial C oracle" % (w["name"], nx, ny, nz, workloads.BENCH["name"])
    print(json.dumps({
        "impl": "reference", "metric": "voxel nodes/s (whole generation: seeding + growth to target)",
        "value": value, "unit": "nodes/s", "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": 1e3 * total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "u32", "data": "synthetic",
        "config": {"workload": workloads.BENCH["name"], "sample": sample},
        "cpu_baseline": {"value": value, "unit": "nodes/s", "cores": 1, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "nodes/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
    }))


def bench_workload(args):
    """workloads.BENCH (BASELINE.json's timing configuration) unless --workload names another config (its first
    spacing, rng seed and target): the other configs are parity cases, timed for information only."""
    if not args.workload:
        return workloads.BENCH
    c = workloads.CONFIGS[args.workload]
    s = c["s"] if isinstance(c["s"], int) else c["s"][0]
    return dict(name=args.workload, dims=c["dims"], periodic=c["periodic"], core=c["core"], s=s, seed=c["seeds"][0],
                g=c["g"], target=c["targets"][0])


def run_ours(args):
    import numpy as np
    import torch
    import paper_2602_11734_b200 as liets

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    w = bench_workload(args)
    nx, ny, nz = w["dims"]
    N = nx * ny * nz
    storage = args.storage if args.storage is not None else DEFAULT_STORAGE
    gen = liets.Liets(nx, ny, nz, int(w["periodic"]), storage, device="cuda:%d" % local)
    gen.set_growth(*w["g"], liets.LAW_EQ1)
    rng_seed = w["seed"] + rank                      # replicas: one realisation per rank
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")     # > 126 MB L2
    host_out = torch.empty(N, dtype=torch.uint8, pin_memory=True)        # e2e destination (pinned host)

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    host_bits = torch.empty((N + 7) // 8, dtype=torch.uint8, pin_memory=True)

    def one(e2e):
        flush.zero_()                                # L2 flush between iterations (outside the events)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        n_seeds = gen.seed(w["core"], w["s"], rng_seed)
        rc, steps, n_solid = gen.generate(w["target"])
        if e2e == "bits":
            gen.grid_into(host_bits.data_ptr(), (N + 7) // 8, liets.FORMAT_BITS)
        elif e2e:
            gen.grid_into(host_out.data_ptr(), N, liets.FORMAT_U8)
        ev1.record()
        ev1.synchronize()
        assert rc == liets.OK
        return ev0.elapsed_time(ev1), n_seeds, steps, n_solid

    for _ in range(args.warmup):
        one(False)
    sampler = ClockSampler(local)
    sampler.start()
    # --- device-resident leg -------------------------------------------------------------------
    barrier()
    launches0 = gen.launch_count
    t_dev, seed_ms, gen_ms = 0.0, [], []
    for _ in range(args.steps):
        ms, n_seeds, n_steps, n_solid = one(False)
        t_dev += ms
        a, b = gen.timings()
        seed_ms.append(a)
        gen_ms.append(b)
    launches = gen.launch_count - launches0
    barrier()
    # --- end-to-end leg: host output buffer, D2H copy inside the timed region ---------------------
    one(True)
    barrier()
    t_e2e = 0.0
    for _ in range(args.steps):
        t_e2e += one(True)[0]
    barrier()
    t_bits = 0.0                                     # the same with the bit-packed output format (N/8 bytes to the host)
    for _ in range(args.steps):
        t_bits += one("bits")[0]
    barrier()
    clocks = sampler.stop()
    t_dev, t_e2e, t_bits = max_over_ranks([t_dev, t_e2e, t_bits], dist, "cuda")

    # --- roofline of the dominant kernel (the tile growth kernel), timed live with CUDA events ------------
    gen.set_profiling(True)
    gen.seed(w["core"], w["s"], rng_seed)
    gen.generate(w["target"])
    step_ms = gen.step_times()[:n_steps]
    gen.set_profiling(False)
    front, solid_after, philox_blocks = gen.step_log()
    on_tiles = gen.step_on_tiles[:n_steps] if storage == 1 else np.ones(n_steps, dtype=bool)
    handover = gen.step_handover[:n_steps] if storage == 1 else np.zeros(n_steps, dtype=bool)
    front = front[:n_steps].astype(np.int64)
    for t in np.flatnonzero(handover):                # the hand-over step's tile count: that of the step after it
        front[t] = front[t + 1] if t + 1 < n_steps else front[t]
    b_alg = np.array(algorithmic_bytes(storage, N, front, solid_after[:n_steps], n_seeds, on_tiles, gen.front_voxels[:n_steps]), dtype=np.float64)
    dom = on_tiles                                    # launches of the dominant kernel that did a step
    peaks, peaks_kind = load_peaks()
    grow_ms = float(np.sum(step_ms[dom]))
    n_dom = int(dom.sum())
    n_blocks = float(np.sum(philox_blocks[:n_steps][dom]))
    n_fvox = float(np.sum(gen.front_voxels[:n_steps][dom]))
    sm_count = torch.cuda.get_device_properties(local).multi_processor_count
    # measured roofs of this box (liets_probe, csrc/probe.cu), taken after the timed legs
    scratch = torch.empty(1 << 30, dtype=torch.uint8, device="cuda")
    probes = {}
    for kind, name in ((liets.liets.PROBE_PHILOX, "philox_blocks_per_s"), (liets.liets.PROBE_LOP3, "lop3_per_s"),
                       (liets.liets.PROBE_IMAD, "imad_per_s"), (liets.liets.PROBE_MIX, "mix_per_s"),
                       (liets.liets.PROBE_L2_READ, "l2_read_bytes_per_s"), (liets.liets.PROBE_HBM_READ, "hbm_read_bytes_per_s")):
        probes[name] = liets.liets.probe(kind, scratch, reps=5)[0]
    del scratch
    # the path is bound by integer issue, not by bytes.  Algorithmic work of a launch =
    #   40 integer instructions per Philox4x32-10 block the keyed draws need (20 32x32->64 multiplies + 20
    #   three-input XORs), plus 2 per (front voxel, direction): the void test of the target and the compare of the
    #   draw with the threshold (Algorithm 3 lines 6 and 8), 52 per front voxel that makes attempts.
    # Peak = the MEASURED rate of an even multiply-add / logic-op mix on this box (liets_probe MIX); the figure derived
    # from unit counts (SMs x 4 schedulers x 32 lanes x max clock) is quoted beside it.
    derived_peak = sm_count * 4 * 32 * float(peaks.get("sm_max_mhz", 1965.0)) * 1e6 / 1e12
    alu_peak = probes["mix_per_s"] / 1e12
    alg_ops = n_blocks * PHILOX_INT_OPS + n_fvox * PER_FRONT_VOXEL_OPS
    sec = grow_ms * 1e-3 if grow_ms > 0 else float("inf")
    alu_achieved = alg_ops / sec / 1e12
    bytes_dom = float(np.sum(b_alg[dom]))
    traffic, traffic_src = traffic_from_profile(w["name"], storage)
    roofline = {"bound": "alu", "achieved": alu_achieved, "peak": alu_peak, "unit": "Tiop/s (thread-level integer instructions)",
                "frac": alu_achieved / alu_peak, "traffic": traffic, "traffic_source": traffic_src,
                "kernel": KERNEL_NAMES[storage],
                "peak_kind": "measured: liets_probe MIX (one 32-bit multiply-add per three-input logic op, 8 independent chains per "
                             "thread, every warp slot) on this GPU, best of 5",
                "peak_derived": derived_peak, "measured_over_derived": alu_peak / derived_peak,
                "peak_derived_kind": "%d SMs x 4 schedulers x 32 lanes x %.0f MHz (sm_max_mhz, %s)" % (
                    sm_count, float(peaks.get("sm_max_mhz", 1965.0)), peaks_kind),
                "launches": n_dom, "launches_on_voxel_list": int(n_steps - n_dom),
                "philox_blocks_per_launch": n_blocks / max(n_dom, 1), "front_voxels_per_launch": n_fvox / max(n_dom, 1),
                "int_ops_per_philox_block": PHILOX_INT_OPS, "int_ops_per_front_voxel": PER_FRONT_VOXEL_OPS,
                "avg_launch_ms": grow_ms / max(n_dom, 1),
                "growth_kernel_share_of_generate": grow_ms / max(float(np.median(gen_ms)), 1e-9),
                "philox": {"bound": "alu", "achieved": n_blocks / sec, "peak": probes["philox_blocks_per_s"], "unit": "Philox4x32-10 blocks/s",
                           "frac": n_blocks / sec / probes["philox_blocks_per_s"],
                           "peak_kind": "measured: liets_probe PHILOX (blocks back to back, nothing else) on this GPU"},
                "hbm": {"bound": "hbm", "achieved": bytes_dom / sec / 1e9, "peak": peaks["hbm_gbs"], "unit": "GB/s",
                        "frac": bytes_dom / sec / 1e9 / peaks["hbm_gbs"],
                        "peak_kind": "%s (MEASURED_PEAKS.json hbm_gbs, burst copy); liets_probe HBM read: %.0f GB/s" % (
                            peaks_kind, probes["hbm_read_bytes_per_s"] / 1e9),
                        "algorithmic_bytes_per_launch": bytes_dom / max(n_dom, 1),
                        "note": "SURVEY.md 8(d) byte model; the grid (2 x %.1f MB) is L2 resident" % (N / 8e6)},
                "l2": {"bound": "l2", "achieved": bytes_dom / sec / 1e9, "peak": probes["l2_read_bytes_per_s"] / 1e9, "unit": "GB/s",
                       "frac": bytes_dom / sec / probes["l2_read_bytes_per_s"],
                       "peak_kind": "measured: liets_probe L2_READ (ld.cg of a 32 MiB window, 16 passes) on this GPU"},
                "probes": probes}

    out = None
    if rank == 0:
        value = whole_job_throughput(N, world, args.steps, t_dev)
        e2e_value = whole_job_throughput(N, world, args.steps, t_e2e)
        out = {
            "metric": "voxel nodes/s (whole generation: seeding + growth to target)",
            "value": value, "unit": "nodes/s", "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": t_dev / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "u32", "data": "synthetic",
            "config": {"workload": w["name"], "grid": [nx, ny, nz], "core_prob": w["core"], "spacing_s": w["s"],
                       "g_face_edge_corner": list(w["g"]), "target_solid_fraction": w["target"], "rng_seed": w["seed"],
                       "storage": ["u8+voxel-list", "bit-rows+voxel-list/tile-list", "bit-rows+full-field sweep (Algorithm 2)"][storage], "parallelism": "replicas" if world > 1 else "1gpu",
                       "l2": "flushed between iterations (256 MiB memset outside the timed events)",
                       "growth_steps": int(n_steps), "seeds": int(n_seeds), "final_solid": int(n_solid)},
            "seconds_per_generation": t_dev / args.steps * 1e-3,
            "seed_ms": float(np.median(seed_ms)), "generate_ms": float(np.median(gen_ms)),
            "e2e": {"value": e2e_value, "unit": "nodes/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": N,
                    "ms_per_step": t_e2e / args.steps, "note": "inputs are parameters only; output = uint8 phase array to pinned host",
                    "bit_packed_output": {"value": whole_job_throughput(N, world, args.steps, t_bits), "ms_per_step": t_bits / args.steps,
                                          "d2h_bytes_per_step": (N + 7) // 8}},
            "gpu_launches": int(launches), "clocks": clocks, "roofline": roofline,
        }
    if rank == 0 and world == 1 and args.workload in BATCH_WORKLOADS:
        out["batch"] = batch_leg(liets, w, BATCH_WORKLOADS[args.workload], args.steps, t_dev / args.steps)
    if rank == 0 and world == 1 and not args.no_cpu_baseline and not args.workload:
        out["cpu_baseline"] = cpu_baseline()
    if rank == 0:
        print(json.dumps(out))
    if dist is not None:
        dist.destroy_process_group()


def time_oracle(w, omp):
    """One run (seeding + growth to the target) of the CPU oracle on workload w; seconds."""
    import oracle
    nx, ny, nz = w["dims"]
    o = oracle.Oracle(nx, ny, nz, w["periodic"], omp=omp)
    o.set_growth(*w["g"], 1)
    t0 = time.perf_counter()
    o.seed(w["core"], w["s"], w["seed"])
    o.generate(w["target"], 10**6, True)
    dt = time.perf_counter() - t0
    o.close()
    return dt


def batch_leg(liets, w, seeds, reps, one_ms):
    """the realisations of a sweep (rng seeds `seeds` of workload w) in ONE batched device loop
    (liets_generate_batch) against the same grids generated one after the other (one_ms each, device time)."""
    import torch
    nx, ny, nz = w["dims"]
    B = liets.LietsBatch(len(seeds), nx, ny, nz, int(w["periodic"]))
    for i in range(len(seeds)):
        B[i].set_growth(*w["g"], liets.LAW_EQ1)
    total = 0.0
    for rep in range(reps + 1):                        # first round = warm-up (graph build)
        ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ev0.record()
        for i, sd in enumerate(seeds):
            B[i].seed(w["core"], w["s"], sd)
        res = B.generate(w["target"])
        ev1.record()
        ev1.synchronize()
        if rep:
            total += ev0.elapsed_time(ev1)
    ms = total / reps
    B.close()
    return {"realisations": len(seeds), "rng_seeds": list(seeds), "ms_per_batch": ms,
            "value": nx * ny * nz * len(seeds) / (ms * 1e-3), "unit": "nodes/s",
            "one_by_one_ms": one_ms * len(seeds), "speedup_over_one_by_one": one_ms * len(seeds) / ms,
            "note": "seeding of every grid + one batched growth loop (one tile-kernel launch per step over all grids), device time; "
                    "one_by_one = the device-resident leg of this run times the number of grids",
            "statuses": [r[0] for r in res], "steps": [r[1] for r in res]}


def cpu_baseline():
    """The oracle as it stands, on the box's host cores, on a bounded sample: one serial run (the checker of record)
    and one run of the same source built with OpenMP over the front (liboracle_omp.so) on all host cores."""
    import oracle
    oracle.build()
    oracle.build_omp()
    w = workloads.BENCH_CPU_SAMPLE
    nx, ny, nz = w["dims"]
    n = nx * ny * nz
    dt1 = time_oracle(w, False)
    dtn = time_oracle(w, True)
    cores = oracle.threads(True)
    return {"value": n / dtn, "unit": "nodes/s", "cores": cores, "kind": "oracle", "seconds": dtn,
            "value_1core": n / dt1, "seconds_1core": dt1, "value_allcores": n / dtn, "seconds_allcores": dtn,
            "host_cpu_count": os.cpu_count(),
            "sample": "%s: %dx%dx%d sub-volume of %s with the same parameters (densities, spacing, target); one serial run of "
                      "oracle/liets_oracle.c (gcc -O2) and one run of the same source with OpenMP over the front on %d threads; "
                      "seeding (brute-force greedy) is serial in both" % (w["name"], nx, ny, nz, workloads.BENCH["name"], cores)}


def traffic_from_profile(workload, storage):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of the dominant kernel, averaged over all launches of one
    generation, from the committed ncu capture of this round (profiles/*_dram.csv: launch, read bytes, write bytes).
    Only for the workload and storage the capture was made on; None otherwise."""
    import glob
    if workload != workloads.BENCH["name"] or storage != 1:
        return None, None
    files = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_k_grow_tile_dram.csv")))
    if not files:
        return None, None
    rows = [l.split(",") for l in open(files[-1]) if l.strip() and not l.startswith("#") and l[0].isdigit()]
    if not rows:
        return None, None
    return sum(float(r[1]) + float(r[2]) for r in rows) / len(rows), os.path.relpath(files[-1], ROOT)


# workloads whose sweep of realisations is also timed as one batch (rng seeds)
BATCH_WORKLOADS = {"cfg1_64": (1, 2, 3, 4, 5, 6, 7, 8), "cfg2_200": (1, 2, 3, 4)}
DEFAULT_STORAGE = 1
PHILOX_INT_OPS = 40
PER_FRONT_VOXEL_OPS = 52
KERNEL_NAMES = {0: "k_grow_u8", 1: "k_grow_tile", 2: "k_grow_full"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=None)
    ap.add_argument("--warmup", type=int, default=None)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--storage", type=int, default=None)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--workload", default=None, choices=sorted(workloads.CONFIGS), help="time another config (information only)")
    args = ap.parse_args()
    if args.impl == "reference":
        args.steps = args.steps or 2
        args.warmup = 0 if args.warmup is None else min(args.warmup, 1)
        return run_reference(args)
    args.steps = args.steps or 20
    args.warmup = 3 if args.warmup is None else max(args.warmup, 3)
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and "RANK" not in os.environ:
        # not under torchrun: spawn one rank per GPU ourselves, exactly as the driver would
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        os.execv(sys.executable, [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", "--nproc-per-node", str(args.gpus),
                                  "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:])
    if args.gpus != world:
        raise SystemExit("bench.py: --gpus %d but WORLD_SIZE is %d" % (args.gpus, world))
    run_ours(args)


if __name__ == "__main__":
    main()
