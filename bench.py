#!/usr/bin/env python
"""bench.py -- headline benchmark of the PIMD hot path (BASELINE.json metric).

A "step" is one pass of the whole hot path (neighbour list -> GFN forces -> normal-mode
propagation + PILE-L) over all beads of the workload, i.e. one `pimd_step(1)`.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload ice512] [--impl ours|reference]

Prints ONE JSON line (rank 0).  N > 1 runs N independent replicas of the workload, one per GPU
("replicas only": the path has no data-path collective), value = all ranks' units / max-over-ranks time.
`--impl reference` times the fp64 CPU oracle as it stands on a bounded sample of the same workload.
"""
from __future__ import annotations

import os

os.environ.setdefault("OMP_WAIT_POLICY", "passive")

import argparse
import json
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import pimd_inputs as pi  # noqa: E402

METRIC = "pimd_atom_bead_steps_per_s"
UNIT = "atom*bead*steps/s"
FP32_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12  # 74.4: SMs x FP32 lanes x 2 (FMA) x clocks.max.sm; the roofline uses the MEASURED rate


def measured_peaks():
    try:
        return json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
    except Exception:
        return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.index, self.proc, self.lines = index, None, []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append(line.strip())

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, smax, reasons = [], [], set()
        for ln in self.lines:
            f = [x.strip() for x in ln.split(",")]
            if len(f) < 7:
                continue
            try:
                sm.append(float(f[0])); smax.append(float(f[1]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), f[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smax) if smax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def flops_per_pair_pass(K, H):
    """Algorithmic flops of one directed pair in one pair pass: 2KH + 2H^2 + ~8H."""
    return 2 * K * H + 2 * H * H + 8 * H


def flops_per_pair_launch_as_built(K, H, L, tensor_path):
    """Mean flops per directed pair per pair-kernel launch of the kernels AS BUILT.

    fp32 path: every one of the L+1 launches evaluates the whole filter.  tcgen05 path: the first launch of a force
    evaluation evaluates both filter layers, the other L launches reload h1 and evaluate the second layer only.
    """
    full = 2 * K * H + 2 * H * H + 8 * H
    if not tensor_path or L == 0:
        return float(full)
    later = 2 * H * H + 8 * H
    return (full + L * later) / (L + 1.0)


def max_over_ranks(times, dist, device):
    """Device times of this rank -> the slowest rank's times (a multi-GPU number is the max over ranks, never a mean).

    `dist` is torch.distributed (initialised; NCCL on the GPU box, gloo in the CPU test) or None for a single process."""
    import torch
    t = torch.tensor(list(times), dtype=torch.float64, device=device)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return [float(x) for x in t]


def whole_job_value(rows_per_rank, steps, world, seconds):
    """atom*bead*steps/s of the whole job: every rank steps its own replica of the workload ("replicas only", weak scaling)."""
    return rows_per_rank * steps * world / seconds


def rank_seed(base_seed, rank):
    """Philox key of rank r: independent thermostat streams, same workload shape."""
    return base_seed + rank


# ------------------------------------------------------------------------------------------------
def run_reference(args):
    """The oracle, as it stands, on the host cores; each step = one PIMD step of a bounded sample."""
    import oracle
    w = pi.make_workload(args.workload)
    P_s = min(w.P, args.ref_beads)
    ref = oracle.RefPIMD(w.species, w.masses_amu, w.positions[:1], w.box, P_s, w.T, w.dt, w.gamma, w.seed,
                         oracle.RefNet.from_spec(w.net))
    ref.forces()
    for _ in range(args.warmup):
        ref.step(1)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        ref.step(1)
    dt = time.perf_counter() - t0
    units = w.n_atoms * P_s * args.steps
    v = units / dt
    sample = f"{args.workload}: first {P_s} of {w.P} bead-systems of replica 0 (a P={P_s} ring at the same T), all {w.n_atoms} atoms"
    out = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
           "warmup": args.warmup, "ms_per_step": 1e3 * dt / args.steps, "higher_is_better": True, "scaling": "weak",
           "vs_baseline": None, "dtype": "f64", "data": "synthetic",
           "config": {"workload": args.workload, "sample": sample},
           "cpu_baseline": {"value": v, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle", "sample": sample},
           "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(out))


def cpu_baseline(w, budget_beads):
    import oracle
    P_s = min(w.P, budget_beads)
    ref = oracle.RefPIMD(w.species, w.masses_amu, w.positions[:1], w.box, P_s, w.T, w.dt, w.gamma, w.seed,
                         oracle.RefNet.from_spec(w.net))
    ref.forces()
    t0 = time.perf_counter()
    n = 0
    while True:
        ref.step(1)
        n += 1
        if time.perf_counter() - t0 > 10.0 or n >= 200:
            break
    dt = time.perf_counter() - t0
    out = {"value": w.n_atoms * P_s * n / dt, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
           "sample": f"{n} oracle step(s) of {w.name} restricted to the first {P_s} of {w.P} bead-systems "
                     f"({w.n_atoms} atoms each), {dt:.1f} s"}
    # the same oracle on ONE thread (OMP_NUM_THREADS = 1 and = all cores), a shorter sample
    threads = oracle.num_threads()
    oracle.set_num_threads(1)
    t0 = time.perf_counter()
    n1 = 0
    while True:
        ref.step(1)
        n1 += 1
        if time.perf_counter() - t0 > 5.0 or n1 >= 200:
            break
    dt1 = time.perf_counter() - t0
    oracle.set_num_threads(threads)
    out["single_thread"] = {"value": w.n_atoms * P_s * n1 / dt1, "cores": 1, "sample": f"{n1} step(s), {dt1:.1f} s"}
    return out


# ------------------------------------------------------------------------------------------------
def run_ours(args):
    import torch
    import paper_2503_23728_b200 as pb

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local}"))
    dev = torch.device(f"cuda:{local}")
    torch.cuda.set_device(dev)

    w = pi.make_workload(args.workload)
    if world > 1:  # independent replica per rank: different thermostat stream, same workload shape
        w.seed = rank_seed(w.seed, rank)
    sim = pb.PIMD.from_workload(w, device=str(dev))
    stream = torch.cuda.current_stream(dev)
    flush = torch.empty(512 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)  # 512 MB > 126 MB L2

    def barrier():
        torch.cuda.synchronize(dev)
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize(dev)

    # ---- device-resident timing: K steps, CUDA events around each step, L2 flushed between steps
    sim.step(args.warmup)
    sim.sync()
    rp0, _ = sim.nlist()
    pairs_first = int(rp0[-1].item())
    sampler = ClockSampler(local)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    barrier()
    if rank == 0:
        sampler.start()
    l0 = sim.launch_count()
    wall0 = time.perf_counter()
    for a, b in ev:                      # the timed region: the library replays its captured step (CUDA graph)
        flush.add_(1.0)
        a.record(stream)
        sim.step(1)
        b.record(stream)
    barrier()
    wall = time.perf_counter() - wall0
    launches = sim.launch_count() - l0
    clocks = sampler.stop() if rank == 0 else None
    t_dev = sum(a.elapsed_time(b) for a, b in ev) * 1e-3
    # the same K steps again with the library's per-class CUDA events (plain launches: events cannot be timed inside a graph):
    # kernel_ms_per_step and the roofline's launch durations come from this pass
    ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    sim.profile(True)
    for a, b in ev2:
        flush.add_(1.0)
        a.record(stream)
        sim.step(1)
        b.record(stream)
    barrier()
    prof = sim.profile_read()
    sim.profile(False)
    t_prof = sum(a.elapsed_time(b) for a, b in ev2) * 1e-3
    sim.sync()
    rp1, _ = sim.nlist()
    pairs_last = int(rp1[-1].item())

    # ---- end to end: the full dynamical state (q, p and the forces at q) of EVERY step comes from pinned host memory and
    # goes back to it through the C-ABI with HOST pointers: pimd_set_state + pimd_set_forces_cached (H2D on the library's
    # stream) -> pimd_step(1) -> pimd_get_forces_cached + pimd_get_state (D2H; pimd_get_state synchronises: the host owns the
    # result before the next step starts)
    q, p, st = sim.get_state()
    F = sim.get_forces_cached()
    hq, hp, hF = q.cpu().pin_memory(), p.cpu().pin_memory(), F.cpu().pin_memory()
    hq2, hp2, hF2 = torch.empty_like(hq).pin_memory(), torch.empty_like(hp).pin_memory(), torch.empty_like(hF).pin_memory()
    e2e_steps = max(3, min(args.steps, 10))
    lib = pb.load_library()
    import ctypes as C
    h = sim._h
    sim.sync()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    for i in range(e2e_steps):
        rc = lib.pimd_set_state(h, C.c_void_p(hq.data_ptr()), C.c_void_p(hp.data_ptr()), C.c_int64(st + i))
        rc = rc or lib.pimd_set_forces_cached(h, C.c_void_p(hF.data_ptr()))
        rc = rc or lib.pimd_step(h, 1)
        rc = rc or lib.pimd_get_forces_cached(h, C.c_void_p(hF2.data_ptr()))
        stc = C.c_int64()
        rc = rc or lib.pimd_get_state(h, C.c_void_p(hq2.data_ptr()), C.c_void_p(hp2.data_ptr()), C.byref(stc))
        assert rc == 0, lib.pimd_last_error()
        hq, hq2 = hq2, hq; hp, hp2 = hp2, hp; hF, hF2 = hF2, hF   # the step's output is the next step's input
    e1.record(stream)
    barrier()
    t_e2e = e0.elapsed_time(e1) * 1e-3
    state_bytes = int(q.numel() * 8 * 3)

    t_dev, t_e2e = max_over_ranks([t_dev, t_e2e], dist, dev)

    if rank == 0:
        value = whole_job_value(w.rows, args.steps, world, t_dev)
        K, H, L = w.net.n_rbf, w.net.hidden, w.net.n_layers
        pairs = 0.5 * (pairs_first + pairs_last)
        pair_ms, pair_n = prof["gfn.pair"]
        head_ms, head_n = prof["gfn.head"]
        # dominant kernel: the pair kernel (message passes + force head share one code path)
        n_launch = pair_n + head_n
        avg_s = (pair_ms + head_ms) * 1e-3 / max(n_launch, 1)
        tensor_path = bool(w.net.gemm_dtype == 1 and K == 64 and H == 128)
        fl_launch = pairs * flops_per_pair_launch_as_built(K, H, L, tensor_path)
        achieved = fl_launch / avg_s / 1e12 if n_launch else 0.0
        mp = measured_peaks()
        if tensor_path:   # kernel timed inside a long step -> the sustained figure (B200_PROFILING.md)
            bound = "tensor"
            peak = float(mp["bf16_tflops_sustained"]) if mp and "bf16_tflops_sustained" in mp else 1400.0
            peak_source = ("MEASURED_PEAKS.json bf16_tflops_sustained (of measured)" if mp and "bf16_tflops_sustained" in mp
                           else "B200_PROFILING.md sustained fallback 1.4 PFLOP/s (of fallback)")
            kname = "gfn_pipe::pair_pipe_kernel (message + head passes, tcgen05)"
        else:
            bound, peak = "alu", pb.measure_fp32_fma_tflops(stream)
            peak_source = (f"measured in this run: FMA-chain micro-kernel (pimd_measure_fp32_fma_tflops; nominal 148 SM x 128 lanes x 2 x "
                           f"1.965 GHz = {FP32_NOMINAL_TFLOPS:.1f})")
            kname = "gfn::pair_kernel (message + head passes, fp32 FFMA)"
        hbm = float(mp["hbm_gbs"]) if mp and "hbm_gbs" in mp else 6650.0
        # HBM-bound kernel classes: algorithmic bytes per step / measured ms per step
        steps = args.steps
        alg_bytes = {"pimd_nm": 108.0 * w.rows, "nlist": 8.0 * pairs + 48.0 * w.rows,
                     "gfn.node": 3072.0 * w.rows * L}
        hbm_kernels = {}
        for kcls, b in alg_bytes.items():
            ms = prof[kcls][0] / steps
            if ms > 0 and b > 0:
                gbs = b / (ms * 1e-3) / 1e9
                hbm_kernels[kcls] = {"bound": "hbm", "ms_per_step": ms, "achieved": gbs, "peak": hbm, "unit": "GB/s",
                                     "frac": gbs / hbm}
        traffic = None
        try:
            traffic = json.load(open(os.path.join(ROOT, "profiles", "traffic.json"))).get(args.workload)
        except Exception:
            pass
        out = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": 1e3 * t_dev / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "bf16" if tensor_path else "f32", "data": "synthetic",
            "config": {"workload": args.workload, "atoms": w.n_atoms, "beads": w.P, "replicas_per_gpu": w.n_replicas,
                       "rows_per_gpu": w.rows, "n_rbf": K, "hidden": H, "layers": L, "r_cut": w.net.r_cut,
                       "pairs_per_row_first": pairs_first / w.rows, "pairs_per_row_last": pairs_last / w.rows,
                       "l2": "512 MB buffer rewritten between timed steps (flush)", "parallelism": f"replicas x{world}",
                       "timing": "sum of per-step CUDA-event intervals on the launch stream; the library replays one captured step (CUDA graph); "
                                 "kernel_ms_per_step and the roofline durations come from a second pass of the same K steps with the library's "
                                 "per-class events (plain launches)"},
            "ms_per_step_profiled_pass": 1e3 * t_prof / args.steps,
            "ns_per_day": args.steps / t_dev * w.dt * 86400e-6,
            "wall_ms_per_step_incl_flush": 1e3 * wall / args.steps,
            "e2e": {"value": whole_job_value(w.rows, e2e_steps, world, t_e2e), "unit": UNIT, "h2d_bytes_per_step": state_bytes,
                    "d2h_bytes_per_step": state_bytes, "steps": e2e_steps,
                    "path": "pinned host q,p,F -> pimd_set_state + pimd_set_forces_cached (host pointers: the H2D copies are inside the C-ABI calls) -> pimd_step(1) -> pimd_get_forces_cached + pimd_get_state (host pointers: D2H inside the calls; pimd_get_state synchronises), every step"},
            "gpu_launches": int(launches),
            "clocks": clocks,
            "kernel_ms_per_step": {k: v[0] / args.steps for k, v in prof.items()},
            "roofline": {"kernel": kname, "bound": bound, "achieved": achieved,
                         "peak": peak, "unit": "TFLOP/s", "frac": achieved / peak,
                         "peak_source": peak_source,
                         "launches_timed": n_launch, "avg_launch_ms": avg_s * 1e3,
                         "flops_per_launch": fl_launch,
                         "flops_note": "as built: mean over the L+1 pair launches of one force evaluation (DESIGN.md section 6); "
                                       f"definition-level (every pass evaluates the whole filter) would be {flops_per_pair_pass(K, H)} per pair",
                         "traffic": traffic},
            "roofline_hbm_kernels": hbm_kernels,
        }
        if world == 1 and not args.no_cpu_baseline:
            out["cpu_baseline"] = cpu_baseline(w, args.ref_beads)
        print(json.dumps(out))
    if dist is not None:
        dist.barrier()
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=20, help="untimed steps before the timed window (SURVEY D5: the beads start collapsed)")
    ap.add_argument("--workload", default="ice512", choices=pi.workload_names())
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--ref-beads", type=int, default=2, help="bead-systems in the oracle's bounded sample")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    args = ap.parse_args()
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # started as a plain `python bench.py --gpus N`: start the N ranks ourselves (one process per GPU; torch.distributed.run)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) == 0:
            run_reference(args)
        return
    run_ours(args)


if __name__ == "__main__":
    main()
