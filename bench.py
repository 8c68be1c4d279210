#!/usr/bin/env python
"""bench.py -- BSSN RHS+RK4 grid-point updates/sec, fp64 4th-order 256^3 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--size 256]

A "step" is one pass of the whole hot path over the grid: 4 x (ghost fill + fused derivative/RHS/RK4-stage
kernel) = one chemora_rk4_step.  Workload: BASELINE.json configs[3] (BSSN, 256^3, g=3, O4 + upwind + KO,
Minkowski + 1e-4 Gaussians), synthetic, seeded.  One process per GPU; the path does not shard without a
halo exchange (north_star: one GPU), so N>1 runs N independent replicas ("replicas only", weak scaling).
--impl reference times the CPU oracle (oracle/) on a bounded sample of the same workload.
Prints ONE JSON line on rank 0.
"""
import argparse
import json
import os
import statistics
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "BSSN RHS+RK4 grid-point updates/sec, fp64 4th-order 256^3; % HBM/FP64 roofline"   # BASELINE.json, byte for byte
UNIT = "grid-point updates/s"
# algorithmic HBM traffic of the fused 4-buffer RK4 scheme (reading S9), V = 25:
# stage 1 reads U, writes S,Yb (75 doubles); stages 2-3 read Y,U,S write S,Y' (125 each); stage 4 reads
# Y,S,U writes U (100): 425 doubles = 3400 B per grid-point update, i.e. 850 B per RHS-kernel launch and point.
BYTES_PER_UPDATE = 3400.0
BYTES_PER_POINT_PER_LAUNCH = BYTES_PER_UPDATE / 4.0
# CONSTANTS from earlier captures, printed as such (never measured by this script):
# FP64 work the fused kernel executes per point and RHS evaluation: 1365 DADD + 671 DMUL + 2 x 1026 DFMA thread
# instructions (SASS of the middle-stage 16x4x4 instance, static count + 5 more trips of the At_ij loop;
# tests/test_abi.py::test_flop_counts_of_the_fused_kernels re-counts it from the built library).  An upper bound on the
# paper's convention.
FLOPS_PER_RHS_POINT = 4088.0
FLOPS_SOURCE = "constant: SASS count of bssn_tma_kernel<16,4,4,MODE_MID,4>, DESIGN.md section 6 / tests/test_abi.py"
# dram__bytes_read.sum + dram__bytes_write.sum of the fused kernel at 256^3, mean over the 4 launches of an RK4 step,
# from the one ncu --set full capture named here; reported under "traffic_constant", "traffic" itself stays null
# because this script does not run under ncu.
NCU_TRAFFIC_BYTES_256 = 19.60e9
NCU_TRAFFIC_SOURCE = "profiles/r01_j_fused_ncu_full.md"


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        return json.load(open(p)), "measured (MEASURED_PEAKS.json)"
    return {"hbm_gbs": 6650.0, "sm_max_mhz": 1965.0}, "fallback (B200_PROFILING.md)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.lines, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            threading.Thread(target=lambda: self.lines.extend(self.proc.stdout), daemon=True).start()
        except Exception:
            self.proc = None

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
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); mx.append(float(f[1]))
            except ValueError:
                continue
            for n, v in zip(names, f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": statistics.median(sm) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def time_oracle(sample_n, steps, warmup):
    """The oracle as it stands, on the host cores, on a bounded sample: configs[3] recipe at sample_n^3."""
    from oracle import oracle
    from paper_1307_6488_b200 import inputs
    c = inputs.config(3, scale=sample_n)
    cores = len(os.sched_getaffinity(0))
    oracle.set_threads(cores)
    st = oracle.with_ghosts(c["state"](), c["ghost"])
    prm = oracle.params(eps_diss=c["eps_diss"])
    dt = 0.25 * c["dx"]
    if warmup:
        oracle.rk4(oracle.SYS_BSSN, st, c["ghost"], c["order"], c["dx"], dt, prm, warmup)
    t0 = time.perf_counter()
    oracle.rk4(oracle.SYS_BSSN, st, c["ghost"], c["order"], c["dx"], dt, prm, steps)
    el = time.perf_counter() - t0
    return sample_n ** 3 * steps / el, el, cores


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    n = args.ref_sample
    steps, warmup = max(1, args.steps), args.warmup
    # keep the whole run within a few minutes whatever K is: cap the oracle work at ~6e6 point updates
    while n > 16 and n ** 3 * (steps + warmup) > 6e6:
        n -= 8
    val, el, cores = time_oracle(n, steps, warmup)
    sample = "%d RK4 steps (+%d warm-up) of the configs[3] recipe on a %d^3 periodic block, %d OpenMP threads" % (
        steps, warmup, n, cores)
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
            "warmup": warmup, "ms_per_step": el / steps * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": "BSSN O4 fp64, configs[3] recipe, bounded sample %d^3 (CPU oracle)" % n},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def headline_handle(binding, inputs, replicas, n, rank, local):
    """the headline workload (configs[3] recipe at n^3): its config, this rank's replica (host array) and a handle"""
    c = inputs.config(3, scale=n)
    u0 = inputs.bssn_gaussians(n, n, n, seed=replicas.replica_seed(inputs.SEED_BASE + 3, rank))   # one replica per rank
    h = binding.Chemora(n, n, n, c["ghost"], c["order"], binding.SYS_BSSN, c["dx"], device="cuda:%d" % local)
    h.set_param("eps_diss", c["eps_diss"])
    return c, u0, h


def run_probe(args):
    """Child of isolated_sweep: the runtime sweep (chemora_autotune) on the headline workload in a process of its own.
    Prints {"probe": {...}} and exits 0.  Nothing here is timed for the bench line."""
    import torch
    from paper_1307_6488_b200 import binding, inputs, replicas
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback")
    local = int(os.environ.get("LOCAL_RANK", "0"))
    torch.cuda.set_device(local)
    _, u0, h = headline_handle(binding, inputs, replicas, args.size, int(os.environ.get("RANK", "0")), local)
    h.set_state(u0)
    if args.probe_ids:
        h.set_param("autotune_fused_ids", args.probe_ids)
    fused, tile, ms = h.autotune()
    col_rows = int(h.get_param("col_rows"))
    h.destroy()
    print(json.dumps({"probe": {"fused": fused, "tile": tile, "col_rows": col_rows, "sweep_ms": ms}}))


ROUND1_FUSED_IDS = 5      # fused tile ids 0..4: the kernels that ran on hardware in round 1


def isolated_sweep(size, fused_ids=0, timeout_s=900):
    """The runtime sweep in a child process (python bench.py --probe): its candidates include kernels no GPU has run
    yet (fused ids 5..7), and a device fault is sticky for the CUDA context that saw it -- in a child it
    costs the sweep, in this process it would cost the headline measurement.  fused_ids > 0 bounds the candidates to
    the fused tile ids below it ("autotune_fused_ids").  Returns (pick or None, error or None)."""
    cmd = [sys.executable, os.path.abspath(__file__), "--probe", "--size", str(size)]
    if fused_ids:
        cmd += ["--probe-ids", str(fused_ids)]
    try:
        r = subprocess.run(cmd, capture_output=True, text=True, timeout=timeout_s)
    except subprocess.TimeoutExpired:
        return None, "isolated sweep: no result within %d s" % timeout_s
    for ln in reversed(r.stdout.strip().splitlines()):
        if ln.startswith('{"probe"'):
            try:
                p = json.loads(ln)["probe"]
                return (int(p["fused"]), int(p["tile"]), int(p["col_rows"]), list(p["sweep_ms"])), None
            except (ValueError, KeyError, TypeError):
                break
    tail = " | ".join((r.stderr or r.stdout).strip().splitlines()[-3:])
    return None, "isolated sweep failed (exit %s): %s" % (r.returncode, tail[-400:])


def run_ours(args):
    import numpy as np
    import torch
    from paper_1307_6488_b200 import binding, inputs, replicas

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    n = args.size
    sweep_error, pick = None, None
    isolated = args.variant == "auto" and not args.sweep_in_process
    if isolated:      # before this process touches the device: the child has the GPU (and its memory) to itself
        pick, sweep_error = isolated_sweep(n)
        if pick is None:                      # once more over the tiles that have run on hardware before
            pick, again = isolated_sweep(n, ROUND1_FUSED_IDS)
            sweep_error += "; sweep bounded to fused ids 0..%d: %s" % (ROUND1_FUSED_IDS - 1, again or "done")
    c, u0, h = headline_handle(binding, inputs, replicas, n, rank, local)
    g, dx = c["ghost"], c["dx"]
    dt = 0.25 * dx
    host = torch.from_numpy(u0).pin_memory()
    h.set_state(host.numpy())
    if isolated:
        fused, tile, rows, sweep_ms = pick if pick else (1, 0, None, None)   # failed sweeps: the default tile, said so
        h.set_variant(fused, tile)
        if rows:
            h.set_param("col_rows", rows)
    elif args.variant == "auto":
        try:
            fused, tile, sweep_ms = h.autotune()
        except binding.ChemoraError as e:     # the sweep must not cost the headline run: fall back to the default tile
            sweep_error, sweep_ms = str(e), None
            h.synchronize_quietly()
            fused, tile = 1, 0
            h.set_variant(fused, tile)
    else:
        fused, tile = [int(x) for x in args.variant.split(",")]
        h.set_variant(fused, tile)
        sweep_ms = None
    info = h.kernel_info()
    col_rows = int(h.get_param("col_rows"))

    # ---- device-resident timing: W warm-up, then exactly K steps ------------------------------------------
    for _ in range(args.warmup):
        h.rk4_step(dt)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    h.timing(1)
    l0 = h.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    e0.record()
    for _ in range(args.steps):
        h.rk4_step(dt)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    launches = h.launch_count() - l0
    kt = h.timing_read()
    h.timing(0)
    clocks = sampler.stop() if rank == 0 else None
    value, worst = replicas.aggregate_throughput(ms * 1e-3, n ** 3 * args.steps, dist, "cuda")   # max over ranks
    ms = worst * 1e3

    # ---- end to end through the C ABI with HOST buffers: H2D + K' steps... per step: set_state, rk4_step, get_state
    # Two handles on two streams, the public asynchronous calls: one handle's copies run under the other's kernels,
    # and the two copy directions under each other; every step still moves its own input in and its result out.
    e2e_steps = max(2, min(args.e2e_steps, args.steps))
    pipe = [h]
    side = torch.cuda.Stream()
    with torch.cuda.stream(side):
        h2 = binding.Chemora(n, n, n, g, c["order"], binding.SYS_BSSN, dx, device="cuda:%d" % local)
    h2.set_param("eps_diss", c["eps_diss"])
    h2.set_variant(*h.get_variant())
    h2.set_param("col_rows", col_rows)
    pipe.append(h2)
    outs = [torch.empty_like(host).pin_memory() for _ in pipe]
    for hh, o in zip(pipe, outs):   # warm-up (staging allocation)
        hh.set_state_async(host); hh.rk4_step(dt); hh.get_state_async(o); hh.synchronize()
    barrier()
    t0 = time.perf_counter()
    for s in range(e2e_steps):
        hh, o = pipe[s % 2], outs[s % 2]
        hh.synchronize()            # the handle's previous step (its staging buffer and its output) is done
        hh.set_state_async(host)
        hh.rk4_step(dt)
        hh.get_state_async(o)
    for hh in pipe:
        hh.synchronize()
    barrier()
    e2e_s = time.perf_counter() - t0
    h2.destroy()
    e2e_val, _ = replicas.aggregate_throughput(e2e_s, n ** 3 * e2e_steps, dist, "cuda")
    nbytes = host.numel() * 8

    fp64_gf = h.measure_fp64_peak() if rank == 0 else None
    h.destroy()
    if dist is not None:
        dist.destroy_process_group()
    if rank != 0:
        return

    pk, pk_src = peaks()
    rhs_launch_ms = kt["rhs_ms"] / max(kt["rhs_launches"], 1) * (1 if fused else 2)   # per RHS evaluation
    achieved = BYTES_PER_POINT_PER_LAUNCH * n ** 3 / (rhs_launch_ms * 1e-3) / 1e9
    hbm_peak = pk["hbm_gbs"]
    gf = FLOPS_PER_RHS_POINT * n ** 3 / (rhs_launch_ms * 1e-3) / 1e9
    cpu_val, cpu_el, cores = time_oracle(args.cpu_sample, 3, 0)
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": {"workload": "BSSN (25 vars) O4 centred FD + upwind advection + KO5, fp64, %d^3 interior, g=3, "
                               "RK4 4-buffer, configs[3] recipe (Minkowski + 1e-4 Gaussians)" % n,
                   "variant": {"fused": fused, "tile_id": tile, "tile": list(binding.tile_shape(tile, binding.SYS_BSSN, fused)),
                               "col_rows": col_rows, "sweep_ms": sweep_ms, "sweep_error": sweep_error,
                               "sweep_process": None if args.variant != "auto" else "this" if args.sweep_in_process else "child"},
                   "kernel": info, "multi_gpu": "replicas only",
                   "l2": "inputs larger than L2 (%.2f GB per state buffer vs 126 MB)" % (h.nvars * h.var_stride * 8 / 1e9)},
        "roofline": {"bound": "hbm", "kernel": ("bssn_tma_il_kernel" if tile >= 5 else "bssn_tma_kernel") if fused else "bssn_derivs+from_derivs",
                     "achieved": achieved, "peak": hbm_peak, "unit": "GB/s", "frac": achieved / hbm_peak,
                     "traffic": None,
                     "traffic_constant": {"bytes_per_launch": NCU_TRAFFIC_BYTES_256, "source": NCU_TRAFFIC_SOURCE}
                                         if (fused and tile < 5 and n == 256) else None,
                     "algorithmic_bytes_per_launch": BYTES_PER_POINT_PER_LAUNCH * n ** 3, "peak_source": pk_src, "ms_per_launch": rhs_launch_ms,
                     # the whole step (4 fills + 4 launches, the driver-timed number) against the same roof
                     "step_frac": BYTES_PER_UPDATE * n ** 3 / (ms / args.steps * 1e-3) / 1e9 / hbm_peak,
                     "share_of_step": kt["rhs_ms"] / ms, "fill_share_of_step": kt["fill_ms"] / ms},
        "roofline_fp64": {"bound": "alu", "achieved": gf, "peak": fp64_gf, "unit": "GFLOP/s",
                          "frac": gf / fp64_gf if fp64_gf else None, "flops_per_rhs_point": FLOPS_PER_RHS_POINT,
                          "flops_source": FLOPS_SOURCE,
                          "peak_source": "measured in this run: DFMA chains on all SMs (chemora_measure_fp64_peak)"},
        "cpu_baseline": {"value": cpu_val, "unit": UNIT, "cores": cores, "kind": "oracle",
                         "sample": "3 RK4 steps of the configs[3] recipe on a %d^3 periodic block (%.1f s)" % (
                             args.cpu_sample, cpu_el)},
        "e2e": {"value": e2e_val, "unit": UNIT, "h2d_bytes_per_step": nbytes, "d2h_bytes_per_step": nbytes,
                "steps": e2e_steps, "pipeline": "2 handles on 2 streams, chemora_set_state_async / rk4_step / "
                                                "get_state_async; every step copies its input in and its result out"},
        "gpu_launches": launches, "clocks": clocks,
    }
    print(json.dumps(line))


def run_sweep(args):
    """configs[4]: fused vs split x tile ids on 96^3, 160^3, 200x200x400 (Minkowski + 1e-10 noise): ms per RHS
    evaluation (one middle RK4 stage, timed by chemora_autotune), updates/s, registers, algorithmic HBM GB/s."""
    import torch
    from paper_1307_6488_b200 import binding, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback")
    table, picks = [], []
    for (nx, ny, nz) in inputs.SWEEP_GRIDS:
        h = binding.Chemora(nx, ny, nz, 3, 4, binding.SYS_BSSN, 0.05)
        h.set_param("eps_diss", 0.1)
        h.set_state(inputs.bssn_noise(nx, ny, nz))
        h.set_param("autotune_split", 1)        # configs[4] asks for both variants
        fused, tile, ms = h.autotune()
        for f in (1, 0):
            for t in binding.variants(binding.SYS_BSSN, 4, f):
                m = ms[f * binding.NUM_TILES + t]
                if m <= 0:
                    continue
                h.set_variant(f, t)
                info = h.kernel_info()
                npts = nx * ny * nz
                bytes_pt = BYTES_PER_POINT_PER_LAUNCH + (0 if f else 2176.0)   # split: 136 arrays written + read
                table.append({"grid": [nx, ny, nz], "fused": f, "tile_id": t,
                              "tile": list(binding.tile_shape(t, binding.SYS_BSSN, f)), "ms_per_rhs": round(m, 4),
                              "updates_per_s": npts / (4 * m * 1e-3), "regs": info["regs"],
                              "spill_bytes": info["local_bytes"], "hbm_gbs_algorithmic": bytes_pt * npts / (m * 1e-3) / 1e9,
                              "best": (f, t) == (fused, tile)})
                if f == 1 and t < 5:     # the paper's tile cost model covers the five tile shapes of the plain layout next to the measurement
                    table[-1]["sigma_model"] = binding.tile_cost(4, 3, t)[0]
        h.destroy()
        rows = [r for r in table if r["grid"] == [nx, ny, nz] and "sigma_model" in r]
        picks.append({"grid": [nx, ny, nz], "model_pick": min(rows, key=lambda r: r["sigma_model"])["tile"],
                      "sweep_pick_among_modelled": min(rows, key=lambda r: r["ms_per_rhs"])["tile"],
                      "ms_of_model_pick_over_best": min(rows, key=lambda r: r["sigma_model"])["ms_per_rhs"]
                                                    / min(r["ms_per_rhs"] for r in rows)})
    print(json.dumps({"metric": "BSSN RHS variant sweep (configs[4])", "unit": "ms per RHS evaluation", "rows": table,
                      "tile_cost_model": picks}))


def run_fill_floor(args):
    """DESIGN.md 6.5's box-fill floor through the library (chemora_measure_box_fill): for every fused 4th-order BSSN
    tile id at the headline size, ms of a fill-only launch (all TMA traffic of a middle RK4 stage, no arithmetic, no
    stores) next to ms of the full middle-stage launch as the runtime sweep times it."""
    import torch
    from paper_1307_6488_b200 import binding, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback")
    n = args.size
    h = binding.Chemora(n, n, n, 3, 4, binding.SYS_BSSN, 0.05)
    h.set_param("eps_diss", 0.1)
    h.set_state(inputs.bssn_gaussians(n, n, n))
    _, _, ms = h.autotune()
    rows = []
    for t in binding.variants(binding.SYS_BSSN, 4):
        fill_ms = h.measure_box_fill(t)
        full_ms = ms[binding.NUM_TILES + t]
        rows.append({"tile_id": t, "tile": list(binding.tile_shape(t, binding.SYS_BSSN, 1)), "fill_only_ms": fill_ms,
                     "full_mid_stage_ms": full_ms if full_ms > 0 else None,
                     "fill_share": fill_ms / full_ms if full_ms > 0 else None})
    h.destroy()
    print(json.dumps({"metric": "fused BSSN kernel: fill-only vs full middle-stage launch, %d^3" % n, "unit": "ms per launch",
                      "rows": rows}))


def run_wave(args):
    """configs[1]: wave (phi, pi) 256^3, O8 + KO eps=0.1, 8 plane waves; RK4 steps; HBM roofline at 272 B per update."""
    import torch
    from paper_1307_6488_b200 import binding, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback")
    c = inputs.config(1, scale=args.size)
    n = args.size
    # --wave1: the paper's Sample-1 system (u, rho, v_i) on the same grid, order and dissipation, Gaussian pulse of
    # width n/16 cells; 5 variables: 17 x 5 doubles = 680 B per update, 170 B per launch
    sysid = binding.SYS_WAVE1 if args.wave1 else binding.SYS_WAVE
    bpl = 170.0 if args.wave1 else 68.0
    h = binding.Chemora(n, n, n, c["ghost"], c["order"], sysid, c["dx"])
    h.set_param("eps_diss", c["eps_diss"])
    h.set_state(inputs.wave1_gaussian(n, n, n, width_cells=n / 16.0) if args.wave1 else c["state"]())
    fused, tile, sweep_ms = h.autotune()
    dt = 0.25 * c["dx"]
    for _ in range(max(args.warmup, 3)):
        h.rk4_step(dt)
    torch.cuda.synchronize()
    h.timing(1)
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for _ in range(args.steps):
        h.rk4_step(dt)
    e1.record(); torch.cuda.synchronize()
    kt = h.timing_read(); h.timing(0)
    ms = e0.elapsed_time(e1) / args.steps
    pk, pk_src = peaks()
    rhs_ms = kt["rhs_ms"] / max(kt["rhs_launches"], 1)
    ach = bpl * n ** 3 / (rhs_ms * 1e-3) / 1e9
    print(json.dumps({"metric": "wave %s RHS+RK4 grid-point updates/sec, fp64 8th-order + KO, %d^3" % (
                          "(u, rho, v_i)" if args.wave1 else "(phi, pi)", n),
                      "value": n ** 3 / (ms * 1e-3), "unit": UNIT, "ms_per_step": ms,
                      "config": {"workload": "Sample-1 system on the configs[1] grid" if args.wave1 else "configs[1]",
                                 "tile_id": tile, "tile": list(binding.tile_shape(tile, sysid, 1)),
                                 "sweep_ms": sweep_ms[binding.NUM_TILES:]},
                      "roofline": {"bound": "hbm", "kernel": "wave_tma_kernel" if 6 <= tile < 9 else (
                                       "wave1_kernel" if args.wave1 else "wave_kernel"),
                                   "achieved": ach, "peak": pk["hbm_gbs"], "unit": "GB/s", "frac": ach / pk["hbm_gbs"],
                                   "ms_per_launch": rhs_ms, "algorithmic_bytes_per_point_per_launch": bpl,
                                   "peak_source": pk_src, "fill_share_of_step": kt["fill_ms"] / (ms * args.steps)}}))
    h.destroy()


def run_paper_shape(args):
    """The shape of the paper's own single-GPU benchmark: BSSN, 8th-order FD, 5 ghost zones,
    RK3 (+ constraint enforcement), 9th-order KO (reading S6b), 100^3 evolved points; synthetic Minkowski +
    1e-4 Gaussians.  Context line, not the headline; variant picked by the runtime sweep (fused 8th-order kernel or
    the derivative-split variant)."""
    import torch
    from paper_1307_6488_b200 import binding, inputs
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device and no CPU fallback")
    rows = []
    for n in (100, args.size):
        h = binding.Chemora(n, n, n, 5, 8, binding.SYS_BSSN, 0.05)
        h.set_param("eps_diss", 0.1)
        h.set_param("ko_order", args.ko_order)
        h.set_state(inputs.bssn_gaussians(n, n, n, width_cells=n / 16.0))
        fused, tile, _ = h.autotune()
        dt = 0.0125
        for _ in range(max(args.warmup, 3)):
            h.rk3_step(dt); h.enforce_constraints()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for _ in range(args.steps):
            h.rk3_step(dt); h.enforce_constraints()
        e1.record(); torch.cuda.synchronize()
        ms = e0.elapsed_time(e1) / args.steps
        rows.append({"grid": n, "ms_per_rk3_step": ms, "updates_per_s": n ** 3 / (ms * 1e-3),
                     "variant": {"fused": fused, "tile": list(binding.tile_shape(tile, binding.SYS_BSSN, fused))}})
        h.destroy()
    print(json.dumps({"metric": "BSSN O8 (5 ghosts) RK3 + enforcement grid-point updates/sec, fp64", "unit": UNIT,
                      "ko_order": args.ko_order, "rows": rows, "paper_context": {"value": 1.05e6, "hardware": "NVIDIA M2050, 100^3, derived from "
                                                      "25 GFlop/s / 7900 flop / 3 substeps (PAPER.md:55, :338, :388)"}}))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--size", type=int, default=256)
    ap.add_argument("--variant", default="auto", help="'auto' (runtime sweep) or 'fused,tile' e.g. 1,3")
    ap.add_argument("--sweep-in-process", action="store_true",
                    help="--variant auto: run the sweep in this process instead of a child (see isolated_sweep)")
    ap.add_argument("--probe", action="store_true", help=argparse.SUPPRESS)   # the child of isolated_sweep
    ap.add_argument("--probe-ids", type=int, default=0, help=argparse.SUPPRESS)
    ap.add_argument("--e2e-steps", type=int, default=8)
    ap.add_argument("--cpu-sample", type=int, default=128)
    ap.add_argument("--ref-sample", type=int, default=64)
    ap.add_argument("--sweep", action="store_true", help="configs[4] variant/tile sweep instead of the headline run")
    ap.add_argument("--fill-floor", action="store_true", help="fill-only vs full launch per fused id (DESIGN.md 6.5)")
    ap.add_argument("--wave", action="store_true", help="configs[1]: the (phi, pi) wave system at 256^3, O8 + KO")
    ap.add_argument("--wave1", action="store_true", help="the paper's Sample-1 wave system (u, rho, v_i) at 256^3, O8 + KO")
    ap.add_argument("--paper-shape", action="store_true", help="BSSN O8 + RK3 at 100^3 (the paper's own benchmark shape)")
    ap.add_argument("--ko-order", type=int, default=9, choices=[5, 9], help="--paper-shape: dissipation order")
    args = ap.parse_args()
    if args.probe:
        run_probe(args)
    elif args.sweep:
        run_sweep(args)
    elif args.fill_floor:
        run_fill_floor(args)
    elif args.wave or args.wave1:
        run_wave(args)
    elif args.paper_shape:
        run_paper_shape(args)
    elif args.impl == "reference":
        run_reference(args)
    else:
        run_ours(args)


if __name__ == "__main__":
    main()
