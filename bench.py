#!/usr/bin/env python
"""bench.py -- atom-steps/s of the full qNEP+PPPM force evaluation (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 4] [--impl ours|reference]

A "step" is one pass of the whole hot path (neighbour build amortised at the
configured interval, descriptors, NN, PPPM, folded back-prop, force/virial assembly) inside the library's
velocity-Verlet driver (qnep_md_run), i.e. BASELINE.json configs[4]: 1,029,000-atom water-like box,
PPPM 256^3, neighbour rebuild every 10 steps, timed per force evaluation.

Prints ONE JSON line (see the keys below).  N > 1 runs N independent replicas (the path is single-GPU by
the north_star: "replicas only"), one process per GPU, timed as the max over ranks.

The contract value is the step that produces the FULL output set of the north_star call (energy, forces, virial,
charges); the cheaper energy + forces step an NVE run needs is timed in a second leg and reported beside it.

--impl reference times the fp64 CPU oracle (oracle/) on the same workload (the whole config 4: ~11 s per evaluation on
16 cores, at most 3 evaluations; --cpu-sample-side bounds it further).
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import qnep_inputs as I  # noqa: E402

METRIC = "atom-steps/s for full qNEP+PPPM force eval"
FS = 1.0 / 10.180505          # 1 fs in natural units (Angstrom * sqrt(amu/eV))

# ---- algorithmic work model, frozen before optimisation --------
FLOPS_ANG_BWD_PER_NEIGHBOUR = 1500.0   # angular backward, per angular neighbour inside r_c^A
FLOPS_ANG_FWD_PER_NEIGHBOUR = 450.0
FLOPS_RAD_FWD_PER_NEIGHBOUR = 150.0
FLOPS_RAD_BWD_PER_NEIGHBOUR = 250.0
FLOPS_NN_FWD_H80 = 5100.0               # per atom, H = 80 (scaled linearly with H)
FLOPS_NN_BWD_H80 = 4400.0
FP32_PEAK_NOMINAL_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12     # 74.4: 148 SMs x 128 lanes x 2 x 1.965 GHz


def max_over_ranks(x, dist=None, device="cpu"):
    """Job time of a multi-rank run: every rank contributes its own device time, the job took the longest."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_value(n_atoms, steps, world, ms_total):
    """Replicas only: every rank evaluates its own copy of the workload, so the whole job processed
    world * n_atoms * steps atom-steps in the time of the slowest rank."""
    return world * n_atoms * steps / (ms_total * 1e-3)


# ncu counters per launch on config 4 in the launch configuration timed here (all outputs), from the ncu --set full capture
# summarised in NCU_COUNTERS["source"]: DRAM traffic (dram__bytes_read.sum + dram__bytes_write.sum) and EXECUTED FP32 flops
# (predicated-on thread executions per SASS opcode from the source page: FFMA 2, packed FFMA2 4, FMUL / FADD / MUFU 1,
# FMUL2 / FADD2 2; the op_ffma counter does not see the packed instructions).  Reported only for that workload.  They are the
# north_star's evidence ("ncu-counted achieved FP32 FLOP/s"), so `roofline.frac` is the EXECUTED fraction whenever they apply;
# the frozen algorithmic work model above stays beside it as `frac_model`.  The capture belongs to one state of the kernel
# sources: "csrc_sha256" is the digest of csrc/ at capture time (csrc_digest() below), and the JSON line says
# "counters_stale": true when the sources have changed since (re-capture, then update both).
NCU_COUNTERS = {
    "source": "profiles/r03_ncu_full.txt",
    "captured_at_commit": "5825272",
    "csrc_sha256": "f53fb14d5da0a24d1288e2b1c662d037407f3b4180d42560ee695bb416a014cc",
    "kernels": {
        "k_pairs": {"dram_bytes": 1.596e9, "executed_flops": 7.975e9},
        "k_desc_angular": {"dram_bytes": 1.032e9, "executed_flops": 1.151e10},
        # k_nn_umma: the contraction runs on the tensor cores (42 tcgen05.mma per 128-atom tile, 3xTF32: 4.74e10 tensor flops
        # per launch); executed_flops is its FP32 part (activation, splits)
        "k_nn": {"dram_bytes": 0.2644e9, "executed_flops": 1.188e9, "tensor_flops": 4.74e10},
        "k_force_angular": {"dram_bytes": 1.451e9, "executed_flops": 2.590e10},
        "k_force_radial": {"dram_bytes": 0.6782e9, "executed_flops": 1.349e10},
    },
    "pppm_dram_bytes": 1.915e9,          # spread + five FFT kernels + gather, same capture
}
TF32_OVER_BF16_NOMINAL = 0.5             # dense tensor peak of kind::tf32 relative to bf16 (B200_PROFILING.md nominal ratio)


def csrc_digest() -> str:
    """sha256 over the CUDA sources of the library, in name order: the state of the kernels the ncu counters belong to."""
    import hashlib
    d = os.path.join(ROOT, "paper_2601_19034_b200", "csrc")
    h = hashlib.sha256()
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh")):
            h.update(name.encode())
            with open(os.path.join(d, name), "rb") as f:
                h.update(f.read())
    return h.hexdigest()


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return dict(hbm_gbs=float(p["hbm_gbs"]), bf16_tflops=float(p.get("bf16_tflops_sustained", p.get("bf16_tflops", 1400.0))),
                    source="measured (MEASURED_PEAKS.json)")
    return dict(hbm_gbs=6650.0, bf16_tflops=1400.0, source="fallback (B200_PROFILING.md)")


def make_workload(cfg: int, args):
    if cfg == 4:
        return I.config4(n_side=args.n_side) if args.n_side else I.config4()
    if cfg == 3:
        return I.config3()
    return I.CONFIGS[cfg]()


class ClockSampler:
    """nvidia-smi clocks / throttle reasons DURING the timed region (B200_PROFILING.md recipe)."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index: int):
        self.gpu = gpu_index
        self.proc = None
        self.lines = []

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.gpu}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.lines.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=2)
        except Exception:
            self.proc.kill()
        sm, smmax, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        rows = [l for (t, l) in self.lines if t0 - 0.05 <= t <= t1 + 0.2] or [l for (_, l) in self.lines]
        for l in rows:
            f = [x.strip() for x in l.split(",")]
            if len(f) < 9:
                continue
            try:
                sm.append(float(f[1]))
                smmax.append(float(f[2]))
            except ValueError:
                continue
            for name, val in zip(names, f[5:9]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(smmax) if smmax else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def time_oracle(sample_side: int, steps: int, warmup: int, workload=None):
    """The fp64 oracle as it stands, on the host cores.  sample_side = 70 is the full config 4 (1,029,000 atoms,
    PPPM 256^3: about 10 s per evaluation on 16 cores); smaller values give a bounded sample of the same construction."""
    from oracle import oracle as O
    O.build()
    grid = 32 if sample_side <= 10 else (64 if sample_side <= 20 else (128 if sample_side <= 40 else 256))
    w = workload if workload is not None else I.config4(n_side=sample_side, grid=grid)
    grid = int(w.es.grid[0])
    for _ in range(warmup):
        O.compute_workload(w)
    t0 = time.perf_counter()
    for _ in range(steps):
        O.compute_workload(w)
    dt = (time.perf_counter() - t0) / max(steps, 1)
    sample = (f"fp64 oracle, one force evaluation of {w.name} = "
              f"{w.n_atoms} atoms, PPPM {grid}^3, wall clock")
    return w.n_atoms / dt, dt, O.num_threads(), sample, w.n_atoms


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    steps, warmup = max(args.steps, 1), args.warmup
    # bounded: keep the whole run within a few minutes (one evaluation of the full config 4 takes ~10 s on 16 cores)
    steps = min(steps, 3)
    warmup = min(warmup, 1)
    v, dt, cores, sample, n = time_oracle(args.cpu_sample_side, steps, warmup)
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": "atom-steps/s", "n_gpus": args.gpus,
            "steps": steps, "warmup": warmup, "ms_per_step": dt * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": f"config4 water-like box ({n} atoms), one oracle evaluation per step", "sample": sample},
            "cpu_baseline": {"value": v, "unit": "atom-steps/s", "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": v, "unit": "atom-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--impl", default="ours")
    ap.add_argument("--n-side", type=int, default=0, help="override molecules per side of config 4 (debug)")
    ap.add_argument("--skin", type=float, default=1.0)
    ap.add_argument("--rebuild-every", type=int, default=10)
    ap.add_argument("--dt-fs", type=float, default=0.5)
    ap.add_argument("--cpu-sample-side", type=int, default=70, help="molecules per side of the oracle's sample (70 = full config 4)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=10)
    ap.add_argument("--zbl", type=float, nargs=2, default=None, metavar=("R_INNER", "R_OUTER"),
                    help="switch the ZBL core on (water: Z = 8, 1); off by default: BASELINE.json's config has none")
    ap.add_argument("--nn-kernel", type=int, default=-1, help="qnep_set_nn_kernel: 0 packed FP32, 1 mma.sync 3xTF32, 2 tcgen05 3xTF32 (-1: the library's default)")
    ap.add_argument("--pppm-kernels", type=int, default=0, help="qnep_set_pppm_kernels: 0 automatic, 1 per-atom spread, 2 sweep spread")
    ap.add_argument("--optional-legs", action="store_true",
                    help="also time the optional terms of SURVEY 8(f) on this workload (per-atom virial, ZBL core, triclinic cell, "
                         "NEP4 4-/5-body terms): untimed by default, reported under \"optional_legs\"")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2601_19034_b200 as Q

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=dev)
    K, Wm = max(args.steps, 1), max(args.warmup, 3)

    w = make_workload(args.config, args)
    if args.zbl:
        assert w.model.n_types == 2, "--zbl names the atomic numbers of the water-like configs only"
        w.zbl = (args.zbl[0], args.zbl[1], (8.0, 1.0))
    n = w.n_atoms
    h = Q.from_workload(w)
    h.set_neighbor_policy(args.skin, args.rebuild_every)
    h.set_pppm_kernels(args.pppm_kernels)
    if args.nn_kernel >= 0:
        h.set_nn_kernel(args.nn_kernel)
    masses = w.masses if w.masses is not None else np.ones(w.model.n_types)
    pos0 = torch.tensor(w.pos, dtype=torch.float64, device=dev)
    types = torch.tensor(w.types, dtype=torch.int32, device=dev)
    vel0 = torch.tensor(I.maxwell_boltzmann(replace_masses(w, masses)), dtype=torch.float64, device=dev)

    def md(pos, vel, nsteps, dt_fs):
        return h.md_run(pos, vel, types, w.box, masses, dt_fs * FS, nsteps)

    def restart():
        h.md_reset()                      # a new trajectory from the initial state: no kept forces, fresh lists
        return pos0.clone(), vel0.clone()

    # dt search, untimed: a random-init model has no repulsive core and can be violent; the library reports an atom that
    # moved more than skin/2 between rebuilds (QNEP_ERR_SKIN_VIOLATED) and the run is repeated with half the time step
    # until warm-up + timed steps go through (the metric is per force evaluation, so dt does not change it).  The same
    # loop lets the library grow its neighbour capacity (QNEP_ERR_NEIGHBOR_OVERFLOW).
    dt_fs = args.dt_fs
    for attempt in range(12):
        pos, vel = restart()
        try:
            md(pos, vel, Wm + K, dt_fs)
            break
        except Q.QnepError as err:
            if err.code == Q.QNEP_ERR_SKIN_VIOLATED:
                dt_fs *= 0.5
            elif err.code != Q.QNEP_ERR_NEIGHBOR_OVERFLOW:
                raise
    else:
        raise RuntimeError("no stable time step found")
    # safety margin: the order of fp32 atomics makes trajectories differ in the last bits from run to run, so the real
    # run uses half the first time step that went through
    dt_fs *= 0.5
    # ---- secondary leg: energy + forces only (what an NVE run needs), exactly K steps after Wm warm-up steps ---------
    def timed_leg():
        pos, vel = restart()
        e_a = md(pos, vel, Wm, dt_fs).cpu().numpy()
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()
        h.profile_reset()
        la = h.kernel_launches()
        ea, eb = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        ta = time.time()
        ea.record()
        e_b = md(pos, vel, K, dt_fs)             # synchronises at the end (device-side error check: skin, capacity)
        eb.record()
        torch.cuda.synchronize()
        tb = time.time()
        if dist is not None:
            dist.barrier()
        return e_a, e_b, ea.elapsed_time(eb), h.kernel_launches() - la, ta, tb

    h.md_set_outputs()
    _, _, ms_ef, _, _, _ = timed_leg()
    ms_ef = max_over_ranks(ms_ef, dist, dev)

    # ---- timed region (contract): the full output set -- energy, forces, virial, charges -- every step ---------------
    vir_t = torch.zeros(9, dtype=torch.float64, device=dev)
    chg_t = torch.zeros(n, dtype=torch.float64, device=dev)
    h.md_set_outputs(virial=vir_t, charges=chg_t)
    sampler = ClockSampler(local)
    sampler.start()
    time.sleep(0.25)
    e_start, e_end, ms_total, launches, tw0, tw1 = timed_leg()
    stage_ms, n_evals = h.profile_sum()
    md_graphs = n_evals == 0
    if md_graphs:
        # launch-bound sizes replay CUDA graphs, which carry no stage events: the per-stage breakdown below comes from a
        # short untimed re-run of the first steps with plain launches
        h.set_md_graphs(0)
        h.profile_reset()
        md(*restart(), min(Wm + K, 20), dt_fs)                      # inside the validated part of the trajectory
        stage_ms, n_evals = h.profile_sum()
        h.set_md_graphs(1)
    clocks = sampler.stop(tw0, tw1)
    ms_total = max_over_ranks(ms_total, dist, dev)
    ms_per_step = ms_total / K
    # the MD must have stayed an MD: (E_pot + E_kin) conserved between the end of the warm-up and the end of the
    # timed run, no skin violation (md_run raises), kinetic temperature reported
    e_end = e_end.cpu().numpy()
    kB = 8.617333262e-5
    md_sanity = {"etot_start_eV": float(e_start[0] + e_start[1]), "etot_end_eV": float(e_end[0] + e_end[1]),
                 "drift_eV_per_atom": float((e_end[0] + e_end[1] - e_start[0] - e_start[1]) / n),
                 "T_start_K": float(e_start[1] / (1.5 * n * kB)), "T_end_K": float(e_end[1] / (1.5 * n * kB))}
    value = whole_job_value(n, K, world, ms_total)
    value_ef = whole_job_value(n, K, world, ms_ef)
    outputs_sanity = {"sum_charges_e": float(chg_t.sum().item()), "virial_trace_eV": float((vir_t[0] + vir_t[4] + vir_t[8]).item())}
    stats = h.neighbor_stats()

    # ---- roofline of the dominant kernel ------------------------------------------------------------------
    per_eval = {k: v / max(n_evals, 1) for k, v in stage_ms.items()}
    # neighbours inside the cutoffs at the last step (the exact per-step lists)
    live_a, live_r = stats["mean_angular"], stats["mean_radial"]
    fma_measured = Q.fma_peak()
    H = w.model.n_neurons
    kernels = {   # stage time (the kernel is bracketed alone, or with O(N) helpers), algorithmic flops per launch
        "k_pairs": (per_eval["desc_radial"], FLOPS_RAD_FWD_PER_NEIGHBOUR * live_r * n),
        "k_desc_angular": (per_eval["desc_angular"], FLOPS_ANG_FWD_PER_NEIGHBOUR * live_a * n),
        # k_nn_umma by default: the contraction runs on the tensor cores (3xTF32), still counted by the FP32 work model
        "k_nn": (per_eval["nn"], (FLOPS_NN_FWD_H80 + FLOPS_NN_BWD_H80) * (H / 80.0) * n),
        "k_force_angular": (per_eval["force_angular"], FLOPS_ANG_BWD_PER_NEIGHBOUR * live_a * n),
        "k_force_radial": (per_eval["force_radial"], FLOPS_RAD_BWD_PER_NEIGHBOUR * live_r * n),
    }
    dom = max(kernels, key=lambda k: kernels[k][0])
    dom_ms, dom_flops = kernels[dom]
    # the workload and kernel selection the ncu counters were taken on
    full4 = args.config == 4 and not args.n_side and args.nn_kernel in (-1, 2) and not args.zbl
    ctr = NCU_COUNTERS["kernels"] if full4 else {}
    digest = csrc_digest()
    peaks = load_peaks()
    nn_on_tensor = args.nn_kernel != 0                 # library default (-1) and modes 1, 2: the contraction is not FP32 work
    fp32_kernels = [k for k in kernels if not (k == "k_nn" and nn_on_tensor)]

    def frac_of_peak(flops, ms):
        return flops / (ms * 1e-3) / 1e12 / FP32_PEAK_NOMINAL_TFLOPS if ms > 0 else 0.0

    def tflops(flops, ms):
        return flops / (ms * 1e-3) / 1e12 if ms > 0 else 0.0

    fp32_ms = sum(kernels[k][0] for k in fp32_kernels)
    fp32_flops = sum(kernels[k][1] for k in fp32_kernels)
    exe_flops = sum(ctr[k]["executed_flops"] for k in fp32_kernels) if ctr else None
    achieved_model = tflops(dom_flops, dom_ms)
    achieved = tflops(ctr[dom]["executed_flops"], dom_ms) if ctr else achieved_model
    tf32_peak = peaks["bf16_tflops"] * TF32_OVER_BF16_NOMINAL
    nn_ms = kernels["k_nn"][0]
    nn_tensor = None
    if nn_on_tensor and ctr:
        nn_tensor = {"kernel": "k_nn_umma (tcgen05 kind::tf32, 3xTF32)" if args.nn_kernel in (-1, 2) else "k_nn_mma (mma.sync TF32, 3xTF32)",
                     "bound": "tensor", "ms": nn_ms, "tensor_flops_per_launch": ctr["k_nn"]["tensor_flops"],
                     "achieved": tflops(ctr["k_nn"]["tensor_flops"], nn_ms), "unit": "TFLOP/s", "peak": tf32_peak,
                     "peak_source": "%s bf16 sustained x %.1f (nominal TF32 : bf16 ratio)" % (peaks["source"], TF32_OVER_BF16_NOMINAL),
                     "frac": tflops(ctr["k_nn"]["tensor_flops"], nn_ms) / tf32_peak,
                     "note": "three TF32 products per term (3xTF32) are counted as executed; latency-bound at 128-atom tiles, "
                             "not part of the FP32 aggregate"}
    roofline = {"kernel": dom, "bound": "alu", "achieved": achieved, "peak": FP32_PEAK_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                "frac": achieved / FP32_PEAK_NOMINAL_TFLOPS,
                "frac_is": ("executed: ncu-counted FP32 flops per launch / live launch time / nominal peak (the north_star's "
                            "evidence); frac_model beside it is the frozen algorithmic work model of SURVEY 8(d)") if ctr else
                           "frac_model: algorithmic flops of the frozen work model / live time / nominal peak (no ncu counters "
                           "for this workload)",
                "achieved_model": achieved_model, "frac_model": achieved_model / FP32_PEAK_NOMINAL_TFLOPS,
                "executed_flops_per_launch": ctr[dom]["executed_flops"] if ctr else None,
                "executed_frac": frac_of_peak(ctr[dom]["executed_flops"], dom_ms) if ctr else None,
                "traffic": ctr[dom]["dram_bytes"] if ctr else None,
                "traffic_source": "ncu dram__bytes_read.sum + dram__bytes_write.sum per launch, " + NCU_COUNTERS["source"],
                "counters_source": NCU_COUNTERS["source"], "counters_commit": NCU_COUNTERS["captured_at_commit"],
                "counters_stale": bool(ctr) and NCU_COUNTERS["csrc_sha256"] != digest, "csrc_sha256": digest,
                "peak_source": "nominal FP32 FMA: 148 SMs x 128 lanes x 2 x 1.965 GHz (DESIGN.md)",
                "fma_loop_measured_tflops": fma_measured, "frac_of_measured_fma_loop": achieved / fma_measured if fma_measured else None,
                "ms_per_launch": dom_ms, "algorithmic_flops_per_launch": dom_flops,
                "per_kernel": {k: {"ms": v[0], "tflops_model": tflops(v[1], v[0]),
                                   "frac": frac_of_peak(ctr[k]["executed_flops"], v[0]) if ctr else frac_of_peak(v[1], v[0]),
                                   "frac_model": frac_of_peak(v[1], v[0]),
                                   "executed_flops_per_launch": ctr[k]["executed_flops"] if ctr else None,
                                   "executed_frac": frac_of_peak(ctr[k]["executed_flops"], v[0]) if ctr else None,
                                   "tensor_flops_per_launch": ctr[k].get("tensor_flops") if ctr else None,
                                   "in_fp32_aggregate": k in fp32_kernels,
                                   "dram_bytes_per_launch": ctr[k]["dram_bytes"] if ctr else None}
                               for k, v in kernels.items()},
                "all_fp32_stages": {"kernels": fp32_kernels, "ms": fp32_ms, "algorithmic_flops": fp32_flops,
                                    "tflops_model": tflops(fp32_flops, fp32_ms),
                                    "frac": frac_of_peak(exe_flops, fp32_ms) if exe_flops else frac_of_peak(fp32_flops, fp32_ms),
                                    "frac_model": frac_of_peak(fp32_flops, fp32_ms),
                                    "executed_flops": exe_flops,
                                    "executed_frac": frac_of_peak(exe_flops, fp32_ms) if exe_flops else None},
                "nn_tensor": nn_tensor}
    mesh_bytes = float(np.prod(w.es.grid)) * 8.0
    fft_bytes = 3 * 3 * 2 * mesh_bytes - float(np.prod(w.es.grid)) * 4.0   # 3 transforms x 3 passes x (read + write)
    pppm = {"stage": "reciprocal (spread + 3 FFTs + influence + gather)", "bound": "hbm", "ms": per_eval["reciprocal"],
            "algorithmic_bytes": 2.4e9 * float(np.prod(w.es.grid)) / 256 ** 3,
            "peak": peaks["hbm_gbs"], "unit": "GB/s", "peak_source": peaks["source"]}
    pppm["achieved"] = pppm["algorithmic_bytes"] / (pppm["ms"] * 1e-3) / 1e9 if pppm["ms"] > 0 else 0.0
    pppm["frac"] = pppm["achieved"] / pppm["peak"]
    pppm["frac_is"] = "frac_model: the survey's 3-pass byte model (2.4 GB at 256^3) / live stage time / measured copy peak"
    pppm["frac_model"] = pppm["frac"]
    pppm["dram_bytes_measured"] = NCU_COUNTERS["pppm_dram_bytes"] if full4 else None
    pppm["frac_measured_bytes"] = (NCU_COUNTERS["pppm_dram_bytes"] / (pppm["ms"] * 1e-3) / 1e9 / pppm["peak"]
                                   if (full4 and pppm["ms"] > 0) else None)
    pppm["traffic"] = pppm["dram_bytes_measured"]
    pppm["traffic_source"] = "ncu dram__bytes_read.sum + dram__bytes_write.sum over the stage's kernels, " + NCU_COUNTERS["source"]

    # ---- end to end through the C ABI with HOST buffers (pinned), copies inside the timed region ----------
    # Every call gets its own positions: the start structure displaced along the initial velocities (0.5 fs per call), so
    # lists are reused on atoms that did move; all four outputs come back to the host.
    Ke = max(1, min(args.e2e_steps, K))
    n_frames = min(Ke + 3, args.rebuild_every if args.rebuild_every > 1 else 2)
    vel_host = vel0.cpu().numpy()
    frames = []
    for k in range(n_frames):
        hp = torch.empty((3, n), dtype=torch.float64).pin_memory()
        hp.copy_(torch.from_numpy(np.ascontiguousarray(w.pos + k * 0.5 * FS * vel_host)))
        frames.append(hp)
    ht = torch.from_numpy(np.ascontiguousarray(w.types)).pin_memory()
    he = torch.empty(1, dtype=torch.float64).pin_memory()
    hf = torch.empty((3, n), dtype=torch.float64).pin_memory()
    hw = torch.empty(9, dtype=torch.float64).pin_memory()
    hq = torch.empty(n, dtype=torch.float64).pin_memory()
    want = Q.WANT_ALL
    box9 = Q._box(w.box)
    h2 = Q.from_workload(w)
    h2.set_neighbor_policy(args.skin, n_frames)      # the frames repeat after n_frames calls: rebuild there
    h2.set_pppm_kernels(args.pppm_kernels)
    if args.nn_kernel >= 0:
        h2.set_nn_kernel(args.nn_kernel)

    def e2e_step(k):
        h2.compute_host_raw(n, frames[k % n_frames].data_ptr(), ht.data_ptr(), box9, want, he.data_ptr(), hf.data_ptr(),
                            hw.data_ptr(), hq.data_ptr(), 0)

    for k in range(n_frames):                        # warm-up: one full cycle of frames (ends before a rebuild call)
        try:
            e2e_step(k)
        except Q.QnepError as err:
            if err.code != Q.QNEP_ERR_NEIGHBOR_OVERFLOW:
                raise
            e2e_step(k)
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for k in range(Ke):
        e2e_step(k)
    torch.cuda.synchronize()
    t_e2e = time.perf_counter() - t0
    t_e2e = max_over_ranks(t_e2e, dist, dev)
    e2e = {"value": whole_job_value(n, Ke, world, t_e2e * 1e3), "unit": "atom-steps/s", "steps": Ke,
           # positions every call; the species travel only with the calls that rebuild the neighbour list (one in n_frames)
           "h2d_bytes_per_step": int(frames[0].numel() * 8 + ht.numel() * 4 // n_frames),
           "d2h_bytes_per_step": int(hf.numel() * 8 + hq.numel() * 8 + 9 * 8 + 8),
           "outputs": "energy, forces, virial, charges",
           "api": "qnep_compute_host (pinned host buffers, a different frame per call; neighbour rebuild every %d calls)" % n_frames}

    # ---- CPU baseline: the oracle as it stands, on rank 0 at N = 1 only -----------------------------------
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        same = args.config == 4 and args.cpu_sample_side == (args.n_side or 70)
        v, dt, cores, sample, _ = time_oracle(args.cpu_sample_side, 1, 0, workload=w if same else None)
        cpu = {"value": v, "unit": "atom-steps/s", "cores": cores, "kind": "oracle", "sample": sample, "seconds": dt}

    extra_legs = None
    if args.optional_legs and rank == 0:
        h.destroy(); h2.destroy()
        del vir_t, chg_t
        torch.cuda.empty_cache()
        extra_legs = optional_legs(Q, torch, w, args, dev)

    if rank == 0:
        line = {
            "metric": METRIC, "value": value, "unit": "atom-steps/s", "n_gpus": world, "steps": K, "warmup": Wm,
            "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": "f32", "data": "synthetic",
            "config": {"workload": w.name, "n_atoms": n, "species": w.model.n_types, "pppm_grid": list(w.es.grid),
                       "mode": w.model.mode, "n_neurons": w.model.n_neurons, "md": "velocity-Verlet via qnep_md_run" + (", steps replayed as CUDA graphs (stage times from plain launches)" if md_graphs else ""),
                       "nn_kernel": {-1: "library default (tcgen05 3xTF32)", 0: "packed FP32", 1: "mma.sync 3xTF32", 2: "tcgen05 3xTF32"}[args.nn_kernel],
                       "dt_fs": dt_fs, "zbl": list(w.zbl[:2]) if w.zbl else None, "skin_A": args.skin, "rebuild_every": args.rebuild_every,
                       "parallelism": "replicas only" if world > 1 else "single GPU",
                       "l2_policy": "inputs larger than L2 (neighbour lists + meshes >> 126 MB); no flush needed",
                       "mean_skin_list": stats["mean_list"], "mean_neighbours_radial": stats["mean_radial"],
                       "mean_neighbours_angular": stats["mean_angular"]},
            "outputs_per_step": "energy, forces, virial, charges (qnep_md_set_outputs)",
            "value_energy_forces_only": value_ef, "ms_per_step_energy_forces_only": ms_ef / K,
            "outputs_sanity": outputs_sanity,
            "roofline": roofline, "roofline_pppm": pppm,
            "stage_ms_per_eval": per_eval, "evals_profiled": n_evals,
            "md_sanity": md_sanity,
            "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches), "clocks": clocks,
        }
        if extra_legs is not None:
            line["optional_legs"] = extra_legs
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()


def optional_legs(Q, torch, w, args, dev, evals=20, warm=5):
    """ms per evaluation (CUDA events around `evals` qnep_compute calls at fixed positions, lists rebuilt every
    args.rebuild_every calls, all four outputs) of the workload as it is and with each optional term of SURVEY 8(f):
    per-atom virial (qnep_compute_atom_virial), ZBL core, the same fractional coordinates in a tilted cell, NEP4's 4-/5-body
    descriptors (35-descriptor model on the scalar network kernel).  One handle at a time."""
    from dataclasses import replace

    def leg(wl, atom_virial=False):
        h = Q.from_workload(wl)
        h.set_neighbor_policy(args.skin, args.rebuild_every)
        h.set_pppm_kernels(args.pppm_kernels)
        pos = torch.tensor(wl.pos, dtype=torch.float64, device=dev)
        types = torch.tensor(wl.types, dtype=torch.int32, device=dev)
        out = {}

        def one():
            if atom_virial:
                h.compute_atom_virial(pos, types, wl.box)
            else:
                h.compute(pos, types, wl.box, want=Q.WANT_ALL, out=out, check=False)

        for k in range(warm + 1):
            try:
                one()
                h.check()
            except Q.QnepError as err:
                if err.code != Q.QNEP_ERR_NEIGHBOR_OVERFLOW:
                    raise
        h.set_neighbor_policy(args.skin, args.rebuild_every)          # the timed calls start with a rebuild
        torch.cuda.synchronize()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record()
        for k in range(evals):
            one()
        b.record()
        torch.cuda.synchronize()
        h.check()
        h.destroy()
        return a.elapsed_time(b) / evals

    legs = {"as_configured": leg(w), "atom_virial": leg(w, atom_virial=True), "triclinic_cell": leg(I.triclinic_variant(w))}
    if w.model.n_types == 2:
        legs["zbl_core"] = leg(replace(w, zbl=(0.35, 0.7, (8.0, 1.0))))
    key = {2: "config1_45body", 4: "config2_45body"}.get(w.model.n_types)
    if key:
        legs["higher_body_terms"] = leg(I.with_higher_body_terms(w, key))
    return {"ms_per_eval": legs, "evals": evals, "unit": "ms",
            "note": "qnep_compute at fixed positions, all four outputs, neighbour rebuild every %d calls; atom_virial through "
                    "qnep_compute_atom_virial (synchronises per call)" % args.rebuild_every}


def replace_masses(w, masses):
    if w.masses is None:
        from dataclasses import replace
        return replace(w, masses=np.asarray(masses, dtype=np.float64))
    return w


if __name__ == "__main__":
    main()
