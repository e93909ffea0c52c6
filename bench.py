#!/usr/bin/env python
"""bench.py -- atom-steps/s of the graph-captured MD step (energy + forces + velocity-Verlet)
on seeded synthetic gas-phase workloads (BASELINE.json:configs), one B200 per rank.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--impl reference]

A "step" is one MD step = one pass of the whole hot path (K1 neighbour build, K2 AEV,
K3 MLP fwd+bwd, K4 force chain rule + gather, energy sum, K5 velocity-Verlet) over the
whole batch, replayed from one CUDA graph.  Prints ONE JSON line (rank 0).
Multi-GPU: replicas only -- every rank runs the same workload on its own
GPU, no data-path collective; value = atoms * steps * N / max-over-ranks time ("weak").
`--impl reference` times the fp64 CPU oracle (oracle/) on a bounded sample of the same
workload; it is a deliberately slow baseline, not the target.
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

from paper_2412_18271_b200 import workloads as W  # noqa: E402

METRIC = "atom_steps_per_s"
UNIT = "atom-steps/s"
DT_FS = 0.5
MLP_FLOPS_PER_ATOM = 4.0 * 94304                     # fwd + bwd, 94,304 MAC each, 2 flop per MAC = 377,216
FP32_PEAK_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12     # 74.5: SMs x FP32 lanes x 2 x max SM clock
SFU_PEAK_TOPS = 148 * 16 * 1.965e9 / 1e12            # 4.65: SMs x 16 SFU lanes x max SM clock
KERNEL_SOURCES = {"K1": ["k1_neighbors.cuh"], "K2": ["k2_aev.cuh", "aev_common.cuh"], "K3_tc": ["k3_mlp_tc.cuh", "tc_ptx.cuh"],
                  "K3_fp32": ["k3_mlp_fp32.cuh"], "K4a": ["k4_forces.cuh", "aev_common.cuh"], "K4b": ["k4_forces.cuh"]}


def _source_hash(kernel):
    """sha256 (first 16 hex digits) of the kernel's source files: profiles/traffic.csv rows carry the hash of
    the sources they were captured from, so a stale capture is never printed as this binary's traffic."""
    import hashlib
    h = hashlib.sha256()
    for f in KERNEL_SOURCES[kernel]:
        path = os.path.join(ROOT, "paper_2412_18271_b200", "csrc", f)
        if os.path.exists(path):
            h.update(open(path, "rb").read())
    return h.hexdigest()[:16]


def _traffic(kernel, config):
    """dram__bytes_read.sum + dram__bytes_write.sum of one launch of `kernel` on `config`, from the committed
    `ncu --set full` capture listed in profiles/traffic.csv -- or None when no row matches the present sources."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    if not os.path.exists(path):
        return None, None
    want = _source_hash(kernel)
    for line in open(path):
        if line.startswith("#") or not line.strip():
            continue
        k, cfg, rd, wr, sha, src = [c.strip() for c in line.split(",")][:6]
        if k == kernel and int(cfg) == config and sha == want:
            return float(rd) + float(wr), src
    return None, None


def _peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return json.load(f), "measured"
    except Exception:
        return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0}, "fallback"


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        super().__init__(daemon=True)
        self.index, self.rows, self._stop_evt, self.proc = index, [], threading.Event(), None

    def run(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            for line in self.proc.stdout:
                self.rows.append([c.strip() for c in line.split(",")])
                if self._stop_evt.is_set():
                    break
        except Exception:
            pass

    def stop(self):
        self._stop_evt.set()
        if self.proc:
            self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
                for n, v in zip(names, r[2:6]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                continue
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


def _oracle_steps_per_s(wl, weights, n_steps):
    import oracle
    t = time.perf_counter()
    oracle.step(wl.pos, wl.vel, wl.species, wl.sys_offsets, weights, DT_FS, n_steps, cell=wl.n_atoms > 4096)
    dt = time.perf_counter() - t
    # oracle.step evaluates forces n_steps + 1 times (once at step 0)
    return wl.n_atoms * (n_steps + 1) / dt, dt


WORKLOAD_NAMES = ("cfg0_molecule22", "cfg1_256x22", "cfg2_water1500", "cfg3_droplet20000", "cfg4_ragged4096")


def _sample_workload(k, budget_atoms):
    """A bounded sample of config k for the CPU legs: whole replicas / a smaller droplet."""
    if k == 0:
        return W.config0(), "config 0 whole (22 atoms)"
    if k == 1:
        n = max(1, min(256, budget_atoms // 22))
        return W.config1(n_replicas=n), f"first {n} of 256 replicas of config 1"
    if k == 2:
        n = max(10, min(500, budget_atoms // 3))
        return W.config2(n_mol=n), f"{n}-molecule droplet built by config 2's recipe"
    if k == 3:
        n = max(100, min(20000, budget_atoms))
        return W.config3(n_atoms=n), f"{n}-atom droplet built by config 3's recipe"
    n = max(1, min(4096, budget_atoms // 56))
    return W.config4(n_replicas=n), f"first {n} of 4096 replicas of config 4"


def run_reference(args):
    """The oracle as it stands on the host cores; each step = one oracle MD step on a bounded sample."""
    import oracle
    weights = W.make_weights()
    cores = oracle.num_threads()
    probe, _ = _sample_workload(args.config, 2000)
    rate, _ = _oracle_steps_per_s(probe, weights, 2)               # atom-evals/s, calibration
    budget_s = 90.0
    atoms = int(rate * budget_s / max(1, args.steps + args.warmup + 1))
    wl, what = _sample_workload(args.config, max(22, atoms))
    if args.warmup:
        _oracle_steps_per_s(wl, weights, args.warmup)
    value, dt = _oracle_steps_per_s(wl, weights, args.steps)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / (args.steps + 1) * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": _config_dict(args, W.make_config(args.config)),
        "sample": {"what": what, "atoms_in_sample": wl.n_atoms},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": what},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def _config_dict(args, wl):
    """The `config` object of the JSON line: the workload only, identical in both arms (the pfc arm's
    kernel path is reported under `path`, the reference arm's bounded sample under `sample`)."""
    world = int(os.environ.get("WORLD_SIZE", "1"))
    return {"workload": wl.name, "config_index": args.config, "atoms": wl.n_atoms, "systems": wl.n_systems,
            "dt_fs": DT_FS, "integrator": args.integrator,
            "parallelism": "replicas only" if world > 1 else "1 gpu",
            "l2": "per-step working set (aev + g + lists + edge) exceeds the 126 MB L2"
                  if wl.n_atoms * 3072 > 126e6 else "working set fits L2: neighbour/AEV/MLP buffers are "
                  "rewritten every step, no flush"}


def per_kernel_roofline(stage_ms, counts, n_atoms, n_systems, mlp_is_tensor, peaks, tensor_peak, step_ms=None):
    """Every kernel's achieved rate against the roof that bounds it (SURVEY.md 8(d) "Which roof bounds which
    kernel"), from the stage times measured in THIS run (CUDA events on the launching stream) and the
    run's own list sizes (pfc_work_counts).  Algorithmic counts, DESIGN.md section 4:
      K1  distance tests x 8 flop (3 sub, 3 mul, 2 add; plain ALU)         ; 16 B pos read + 4 B per entry written
      K2  90 flop per radial entry + 150 per triple                         ; 1,536 B aev row written + 4 B per entry
      K3  377,216 flop per atom                                             ; aev row read + g row written
      K4a 2 x K2's flops (value + derivative chains)                        ; 1,536 B g row read + 16 B per entry
      K4b streaming: 16 B per entry gathered + 4 B index + 32 B per atom
      K5  64 B read + 48 B written per atom
    HBM fractions are quoted against the measured copy bandwidth (and ~8 TB/s nominal in `hbm_frac_nominal`)."""
    hbm = peaks["hbm_gbs"]
    R, T, tests = counts["radial"], counts["triples"], counts["brute_tests"]
    aev_flops = 90.0 * R + 150.0 * T
    rows = {
        "K1_neighbors": ("alu", 8.0 * tests, 32.0 * n_atoms + 4.0 * R + 32.0 * n_atoms),
        "K2_aev_fwd": ("alu", aev_flops, 1536.0 * n_atoms + 4.0 * R + 32.0 * n_atoms),
        "K3_mlp": ("tensor" if mlp_is_tensor else "alu", MLP_FLOPS_PER_ATOM * n_atoms, 3072.0 * n_atoms),
        "K4a_aev_bwd": ("alu", 2.0 * aev_flops, 1536.0 * n_atoms + 20.0 * R + 32.0 * n_atoms),
        "K4b_gather": ("hbm", 0.0, 20.0 * R + 48.0 * n_atoms),
        "energy_sum": ("hbm", 0.0, 16.0 * n_atoms + 4.0 * n_systems),
    }
    out = {}
    for (name, (bound, flops, nbytes)), ms in zip(rows.items(), stage_ms):
        if not ms > 0.0:                                         # small systems: the energy sum is part of the K4b kernel
            out[name] = {"bound": bound, "ms": 0.0, "fused_into": "K4b_gather"}
            continue
        sec = ms * 1e-3
        e = {"bound": bound, "ms": float(ms), "algorithmic_bytes": nbytes, "gbs": nbytes / sec / 1e9,
             "hbm_frac": nbytes / sec / 1e9 / hbm, "hbm_frac_nominal": nbytes / sec / 1e9 / 8000.0}
        if flops:
            peak = tensor_peak if bound == "tensor" else FP32_PEAK_TFLOPS
            e.update({"algorithmic_flops": flops, "tflops": flops / sec / 1e12, "peak_tflops": peak,
                      "frac": flops / sec / 1e12 / peak})
        else:
            e["frac"] = e["hbm_frac"]
        out[name] = e
    if len(stage_ms) > 6:                                        # the fused integrator kernel (stage 6 of pfc_profile_stages)
        ms = max(float(stage_ms[6]), 1e-6)
        nbytes = 112.0 * n_atoms
        out["K5_integrate"] = {"bound": "hbm", "ms": ms, "algorithmic_bytes": nbytes, "gbs": nbytes / ms / 1e6,
                               "hbm_frac": nbytes / ms / 1e6 / hbm, "hbm_frac_nominal": nbytes / ms / 1e6 / 8000.0,
                               "frac": nbytes / ms / 1e6 / hbm}
    return out


def max_over_ranks(seconds, device=None):
    """Whole-job time = the slowest rank's device time (no data-path collective: replicas only)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(seconds)
    tt = torch.tensor([seconds], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return float(tt.item())


def job_value(atoms_per_rank, steps, world, seconds):
    """atom-steps/s of the whole job: every rank advances its own copy of the batch (weak scaling)."""
    return world * atoms_per_rank * steps / seconds


INTEGRATOR = {"kind": "verlet"}                       # set by --integrator (paper protocol: langevin)


def _advance(p, n_steps):
    if INTEGRATOR["kind"] == "langevin":
        p.step_langevin(n_steps, DT_FS, 1e-4, 300.0, seed=2412)      # friction 0.1 ps^-1, 300 K
    else:
        p.step(n_steps, DT_FS)


def _time_steps(torch, p, stream, n_steps):
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    with torch.cuda.stream(stream):
        e0.record(stream)
        _advance(p, n_steps)
        e1.record(stream)
    stream.synchronize()
    return e0.elapsed_time(e1) * 1e-3


def run_pfc(args):
    import torch
    import torch.distributed as dist
    from paper_2412_18271_b200 import pfc

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device; there is no CPU fallback (use --impl reference)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    pfc.load_library()
    weights = W.make_weights()
    wl = W.make_config(args.config)
    if args.replicas and args.config in (1, 4):
        import dataclasses
        wl = (W.config1 if args.config == 1 else W.config4)(n_replicas=args.replicas)
        wl = dataclasses.replace(wl, name=f"{wl.name}_first{args.replicas}")
    N = wl.n_atoms
    stream = torch.cuda.Stream(device=dev)
    tuning = pfc.Tuning(skin_list=1) if args.skin else None
    p = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=args.mlp, device=dev, tuning=tuning)
    mlp = p.mlp_path()                                            # MLP_AUTO resolved by pfc_create
    pos0, vel0 = pfc.pack4(wl.pos), pfc.pack4(wl.vel)
    pos, vel = torch.from_numpy(pos0).to(dev), torch.from_numpy(vel0).to(dev)
    with torch.cuda.stream(stream):
        E, F = p.set_state(pos, vel, stream=stream)
        frames = None
        if args.integrator == "langevin":                        # the paper's protocol also writes 10 frames
            frames = torch.empty(10, N, 4, dtype=torch.float32, device=dev)
            p.set_frames(frames, max(1, (args.warmup + args.steps) // 10))
        _advance(p, args.warmup)                                 # W untimed steps (includes graph capture)
    stream.synchronize()

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
        time.sleep(0.3)
    barrier()
    t = _time_steps(torch, p, stream, args.steps)                # EXACTLY K steps, device time
    barrier()
    clocks = sampler.stop() if sampler else None
    t = max_over_ranks(t, dev)
    status = p.status()
    _, launches_step = p.launch_counts()
    value = job_value(N, args.steps, world, t)

    line = None
    if rank == 0:
        peaks, peak_src = _peaks()
        # ---- per-stage device times (CUDA events on the launching stream), averaged ----
        stage_ms = np.zeros(pfc.N_STAGES)
        reps = 10
        with torch.cuda.stream(stream):
            for _ in range(3):
                p.profile_stages(pos, E, F, stream=stream)
            for _ in range(reps):
                stage_ms += np.array(p.profile_stages(pos, E, F, stream=stream))
        stage_ms /= reps
        k3_s = stage_ms[2] * 1e-3
        flops = MLP_FLOPS_PER_ATOM * N
        # the burst bf16 peak when the clock record shows the run was never power-capped, else the sustained one
        capped = bool(clocks and "sw_power_cap" in (clocks.get("reasons") or []))
        bf16 = peaks["bf16_tflops_sustained"] if capped else peaks["bf16_tflops"]
        tensor_peak = bf16                                       # kind::f16 operands: the bf16 / fp16 dense rate
        if mlp == pfc.MLP_FP32:
            roof = {"bound": "alu", "achieved": flops / k3_s / 1e12, "peak": FP32_PEAK_TFLOPS, "unit": "TFLOP/s",
                    "peak_source": "148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz (guide unit counts and max SM clock)"}
        else:
            roof = {"bound": "tensor", "achieved": flops / k3_s / 1e12, "peak": tensor_peak, "unit": "TFLOP/s",
                    "peak_source": f"{peak_src} bf16 {'sustained (sw_power_cap seen)' if capped else 'burst (no power cap seen)'} "
                                   "(kind::f16 runs at the bf16 rate); achieved counts algorithmic flops once, the "
                                   "3-term split issues 3x"}
        k3_name = "K3_fp32" if mlp == pfc.MLP_FP32 else "K3_tc"
        traffic, traffic_src = _traffic(k3_name, args.config)
        counts = p.work_counts()
        per_kernel = per_kernel_roofline(stage_ms, counts, N, wl.n_systems, mlp != pfc.MLP_FP32, peaks, tensor_peak,
                                         step_ms=t / args.steps * 1e3)
        for kname, src in (("K1", "K1_neighbors"), ("K2", "K2_aev_fwd"), ("K4a", "K4a_aev_bwd"), ("K4b", "K4b_gather")):
            tr, tr_src = _traffic(kname, args.config)
            per_kernel[src]["traffic"], per_kernel[src]["traffic_source"] = tr, tr_src
        roof.update({"frac": roof["achieved"] / roof["peak"], "traffic": traffic, "traffic_source": traffic_src,
                     "algorithmic_bytes": 2 * 1536 * N,   # aev row read + g row written per atom
                     "kernel": "K3 MLP fwd+bwd",
                     "kernel_ms": float(stage_ms[2]),
                     "work_counts": counts,
                     "stage_ms": {n: float(v) for n, v in zip(pfc.STAGE_NAMES, stage_ms)},
                     "stage_share": {n: float(v / stage_ms.sum()) for n, v in zip(pfc.STAGE_NAMES, stage_ms)},
                     "step_ms_graph": t / args.steps * 1e3,
                     "per_kernel": per_kernel})

        # ---- end to end through the C ABI with HOST buffers: H2D + 1 step + D2H per step ----
        ph, vh = torch.from_numpy(pos0.copy()).pin_memory(), torch.from_numpy(vel0.copy()).pin_memory()
        Eh = torch.empty(wl.n_systems, dtype=torch.float32).pin_memory()
        Fh = torch.empty(N, 4, dtype=torch.float32).pin_memory()
        p2 = pfc.Pfc(wl.species, wl.sys_offsets, weights, mlp_path=args.mlp, device=dev)
        e2e_steps = max(3, min(args.steps, 50))
        with torch.cuda.stream(stream):
            p2.run_host(ph, vh, 0, DT_FS, Eh, Fh, stream=stream)            # forces at the start
            for _ in range(3):
                p2.run_host_resume(ph, vh, Fh, 1, DT_FS, Eh, stream=stream)
            t0 = time.perf_counter()
            for _ in range(e2e_steps):
                p2.run_host_resume(ph, vh, Fh, 1, DT_FS, Eh, stream=stream)     # synchronises inside
            t_e2e = time.perf_counter() - t0
        p2.close()
        e2e = {"value": N * e2e_steps / t_e2e, "unit": UNIT, "ranks_measured": 1, "h2d_bytes_per_step": 3 * N * 16,
               "d2h_bytes_per_step": 3 * N * 16 + 4 * wl.n_systems, "steps": e2e_steps,
               "call": "pfc_run_host_resume(n_steps=1) per step: pinned host pos/vel/F in, one MD step "
                       "(one force evaluation), pos/vel/F/E out"}

        # ---- the oracle on the host cores, bounded sample ----
        import oracle
        swl, what = _sample_workload(args.config, 14000)
        rate, _ = _oracle_steps_per_s(swl, weights, 1)               # calibration: atom-evaluations / s
        n_cpu_steps = int(min(400, max(3, 12.0 * rate / swl.n_atoms)))   # about 12 s of CPU work
        cpu_v, cpu_t = _oracle_steps_per_s(swl, weights, n_cpu_steps)
        cores = oracle.num_threads()
        oracle.set_num_threads(1)                                    # and on one core: ~3 s
        one_wl, one_what = _sample_workload(args.config, 1400)
        one_v, one_t = _oracle_steps_per_s(one_wl, weights, int(min(200, max(2, 3.0 * rate / cores / one_wl.n_atoms))))
        oracle.set_num_threads(cores)
        cpu = {"value": cpu_v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"{what}, {n_cpu_steps} steps ({cpu_t:.1f} s)",
               "single_thread": {"value": one_v, "sample": f"{one_what} ({one_t:.1f} s)"}}

        steps_per_s = args.steps / t
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None,
            "dtype": "f32" if mlp == 0 else "f16x3",     # MLP contractions as a 3-term fp16 hi|lo split, fp32 accumulate; all else f32
            "data": "synthetic",
            "config": _config_dict(args, wl),
            "path": {"mlp_path": "fp32_ffma" if mlp == 0 else "f16x3_tcgen05",
                     "mlp_path_requested": {0: "fp32", 1: "tensor", 2: "tensor_1term", 3: "auto"}[args.mlp],
                     "steps_per_graph": p.steps_per_graph(), "skin_list": bool(args.skin)},
            "ns_per_day_per_replica": steps_per_s * DT_FS * 1e-6 * 86400,
            "ns_per_day_aggregate": steps_per_s * DT_FS * 1e-6 * 86400 * wl.n_systems * world,
            "clocks": clocks, "e2e": e2e, "gpu_launches": launches_step * args.steps,
            "launches_per_step": launches_step, "device_status": status,
            "roofline": roof, "cpu_baseline": cpu,
        }
        if args.all_configs:
            others = {}
            for k in range(5):
                if k == args.config:
                    continue
                w2 = W.make_config(k)
                q = pfc.Pfc(w2.species, w2.sys_offsets, weights, mlp_path=args.mlp, device=dev)
                x2, v2 = torch.from_numpy(pfc.pack4(w2.pos)).to(dev), torch.from_numpy(pfc.pack4(w2.vel)).to(dev)
                with torch.cuda.stream(stream):
                    q.set_state(x2, v2, stream=stream)
                    q.step(2 * q.steps_per_graph() + 2, DT_FS)    # warm-up: calibration, and every graph captured
                stream.synchronize()
                n2 = 100
                t2 = _time_steps(torch, q, stream, n2)
                others[w2.name] = {"atoms": w2.n_atoms, "ms_per_step": t2 / n2 * 1e3,
                                   "atom_steps_per_s": w2.n_atoms * n2 / t2,
                                   "ns_per_day_per_replica": n2 / t2 * DT_FS * 1e-6 * 86400,
                                   "device_status": q.status()}
                q.close()
            line["other_configs"] = others
    p.close()
    if world > 1:
        dist.barrier()
        dist.destroy_process_group()
    if line is not None:
        print(json.dumps(line))


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--config", type=int, default=4, choices=range(5))
    ap.add_argument("--impl", default="pfc", choices=["pfc", "reference"])
    ap.add_argument("--integrator", default="verlet", choices=["verlet", "langevin"],
                    help="langevin = the paper's timing protocol (friction 0.1 ps^-1, 10 frames), PAPER.md:94")
    ap.add_argument("--mlp", type=int, default=3, choices=[0, 1, 3],
                    help="3 = auto (library default: tensor-core MLP from 1024 atoms on), 0 = FP32 FFMA, 1 = tcgen05 fp16 split")
    ap.add_argument("--all-configs", action="store_true", help="also time the other four configs (100 steps each)")
    ap.add_argument("--skin", action="store_true",
                    help="cell-list systems (config 3): neighbour candidates with a 0.5 A skin, reused between rebuilds "
                         "(pfc_tuning_t.skin_list; off by default)")
    ap.add_argument("--replicas", type=int, default=0,
                    help="configs 1 and 4 only: the first N replicas instead of all (profiling / sanitizer runs; "
                         "the workload name in the JSON line says so)")
    args = ap.parse_args()
    INTEGRATOR["kind"] = args.integrator
    if args.warmup < 3 and args.impl == "pfc":
        args.warmup = 3
    if args.impl == "reference":
        if int(os.environ.get("RANK", "0")) == 0:
            run_reference(args)
        return
    run_pfc(args)


if __name__ == "__main__":
    main()
