#!/usr/bin/env python
"""bench.py — throughput of one DP energy / force / virial evaluation (the whole hot path, S1..S9) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload W24k|Cu32k|W192|Cu864k] [--variant 0|1]
                    [--precision fp64|tf32]      # tf32 = BASELINE.json configs[3] (mixed precision, tcgen05 kernels)
    python bench.py --impl reference ...     # times the CPU oracle (the baseline arm) on a bounded sample

A "step" is one dpb_eval over one freshly perturbed copy of the workload's box (BASELINE.json config: positions
perturbed by sigma = 0.01 A between calls, neighbour build included every call).  Inputs are resident in HBM for
`value`; `e2e` goes through dpb_eval_host with pinned host buffers (H2D of coordinates and types, D2H of E, E_i, F and
the virial inside the timed region).  Prints ONE JSON line on rank 0.

Multi-GPU: the path is fixed to one GPU by BASELINE.json (north_star: "no sharding, no collectives") — "replicas
only": under torchrun every rank evaluates its own replica (own seed) on its own GPU, no data-path collective;
value = total atoms evaluated by all ranks / max-over-ranks device time.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import threading
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import gen  # noqa: E402
from gen.weights import MODELS  # noqa: E402

METRIC = "atom-steps/s"
FP64_PEAK_TFLOPS = 37.2   # 148 SMs x 64 DFMA/clk x 2 flop x 1.965 GHz; measured 37.0


def tf32_peak_tflops():
    """Dense TF32 tensor peak = the measured bf16 cuBLAS burst figure (MEASURED_PEAKS.json) x the nominal ratio 1/2
    (B200_PROFILING.md: 2.25 PF bf16, 1.1 PF tf32); fallback 1590 / 2."""
    try:
        return float(json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))["bf16_tflops"]) / 2.0, "measured bf16 x 1/2"
    except Exception:
        return 1590.0 / 2.0, "fallback bf16 x 1/2"


# ---- algorithmic work -------------------------------
def algorithmic_flops(spec, n_atoms, n_pairs):
    s1, M, Ma, w, D = spec.emb_s1, spec.m, spec.m_axis, spec.fit_width, spec.dim_descrpt
    gemm = 2 * (s1 + 2 * s1 * s1 + 8 * s1 * s1)                 # one direction, per neighbour
    emb_fwd = gemm + (s1 + 2 * s1 + 4 * s1) + (2 * s1 + 4 * s1) + 2 * 4 * M     # + bias, skip adds, T update
    emb_bwd = gemm + 2 * 4 * M + 2 * 4 * M + 2 * (7 * s1) + (2 * s1 + 4 * s1) + 60   # dg, dR~, (1-t^2), folds, chain
    fit = 2 * (D * w + 2 * w * w + w)                            # forward = backward, per atom
    contr = 3 * (2 * 4 * M * Ma)                                 # D, and the two dT terms
    return {
        "pass1": float(emb_fwd) * n_pairs,
        "fit": float(2 * fit + contr) * n_atoms,
        "pass2": float(emb_bwd) * n_pairs,
    }


# ---- clocks sampler ------------------------------------------------------------------------------------------
class ClockSampler:
    FIELDS = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
              "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
              "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.index = index
        self.proc = None
        self.path = None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.FIELDS}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=open(self.path, "w"), stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        sm, reasons, smax, pw = [], set(), None, []
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        try:
            for line in open(self.path):
                f = [x.strip() for x in line.split(",")]
                if len(f) < 7:
                    continue
                try:
                    sm.append(float(f[0])); smax = float(f[1]); pw.append(float(f[2]))
                except ValueError:
                    continue
                for nme, v in zip(names, f[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(nme)
            os.unlink(self.path)
        except Exception:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=smax, reasons=sorted(reasons), samples=len(sm),
                       power_w_max=max(pw) if pw else None)
        return out


# ---- the reference arm: the CPU oracle ------------------------------------------------------------------------
def oracle_step_sampler(name, seed, sample_atoms):
    """Returns (fn, n_atoms_per_step, description, threads).  One step = nlist rows + E_i + dE_i/dd for a fixed random
    sample of atoms of a perturbed copy of the box (the oracle as it stands; brute-force neighbour search per row)."""
    from oracle import Oracle
    spec = MODELS[name]
    coord, types, box = gen.make_system(name)
    emb, fit = gen.make_weights(spec)
    orc = Oracle.from_spec(spec, emb, fit)
    n = coord.shape[0]
    k = min(sample_atoms, n)
    rows = np.sort(np.random.default_rng(seed).choice(n, k, replace=False)).astype(np.int64)
    state = {"call": 0}

    def step():
        c = gen.perturbed(coord, box, 0.01, seed + 1000 + state["call"])
        state["call"] += 1
        nl, _ = orc.build_nlist(c, types, box, rows=rows)
        orc.atom_rows(c, types, box, rows, nl)
    desc = (f"{k} of {n} atoms per step (seeded sample): dpo_build_nlist_rows (brute force) + dpo_atom_rows "
            f"(E_i and dE_i/dd_ik), OpenMP over atoms")
    return step, k, desc, orc.num_threads()


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    name = args.workload
    step, k, desc, threads = oracle_step_sampler(name, gen.SEED_BASE, args.ref_sample)
    for _ in range(max(1, min(args.warmup, 2))):
        step()
    t0 = time.perf_counter()
    for _ in range(args.steps):
        step()
    dt = time.perf_counter() - t0
    value = k * args.steps / dt
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "atom-steps/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
        "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(name, args),
        "cpu_baseline": {"value": value, "unit": "atom-steps/s", "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": "atom-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))
    return 0


def workload_config(name, args):
    spec = MODELS[name]
    sysspec = gen.CONFIGS[name]
    return {"workload": f"{name} (BASELINE.json configs[{sysspec.config_id}])", "sel": list(spec.sel),
            "rcut": spec.rcut, "rcut_smth": spec.rcut_smth, "embedding": [1, spec.emb_s1, 2 * spec.emb_s1, 4 * spec.emb_s1],
            "m_axis": spec.m_axis, "fitting": [spec.dim_descrpt, spec.fit_width, spec.fit_width, spec.fit_width, 1],
            "weights": "random-init N(0,1/fan_in), biases N(0,1), seeded",
            "perturbation_sigma_A": 0.01, "neighbour_build": "every step",
            "parallelism": "replicas only (1 GPU per replica, no collectives)",
            "l2": "flushed between timed steps (256 MiB write)", "variant": getattr(args, "variant", 1),
            "precision": getattr(args, "precision", "fp64"),
            "pair_reuse": "pass 1, nets (a,a), single-chunk evaluations (library default; fp64 variant 1 only)"}


# ---- molecular dynamics: the paper's own unit, steps/s and ns/day ----------------------
def run_md(args, spec, name, coord, types, box, dev, emb, fit, mixed):
    """Random-init weights are not a physical potential: with the literal N(0, 1/fan_in) set the forces are ~4 eV/A rms
    and the box heats to 1e5 K within 500 steps.  The MD leg therefore uses the conditioned weight set (fitting W0 / Nm,
    DESIGN.md section 3: forces ~0.2 eV/A rms); the kernels and their cost are the same."""
    import torch
    from paper_2004_11658_b200 import DPModel
    model = DPModel.from_spec(spec, emb, gen.condition_fit_w0(spec, fit), precision=1 if mixed else 0)
    masses = gen.MASSES[name]
    dt_fs = 0.5 if spec.ntypes == 2 else 1.0                     # 0.5 fs water, 1.0 fs copper
    vel = gen.maxwell_boltzmann(types, masses, 330.0, seed=gen.SEED_BASE + 500)
    out = {}
    for label, kw in (("skin2A_rebuild50", dict(rebuild_every=50, skin=2.0)), ("search_every_step", dict())):
        if label.startswith("skin") and not (spec.rcut + 2.0 < 0.5 * min(box[0], box[4], box[8])):
            out[label] = "r_c + skin >= L/2 for this box"
            continue
        dc, dv = torch.tensor(coord, device=dev), torch.tensor(vel, device=dev)
        dt = torch.tensor(types, device=dev)
        wc, wv = dc.clone(), dv.clone()
        model.md_run(wc, wv, dt, masses, box, dt_fs, 10, thermo_every=10, **kw)          # warm-up on a copy
        torch.cuda.synchronize()
        t0 = time.perf_counter()
        thermo, info = model.md_run(dc, dv, dt, masses, box, dt_fs, args.md_steps, thermo_every=20, **kw)
        wall = time.perf_counter() - t0
        etot = thermo[:, 0] + thermo[:, 1]
        out[label] = {"steps": args.md_steps, "steps_per_s": args.md_steps / wall, "ms_per_step": wall / args.md_steps * 1e3,
                      "ns_per_day": args.md_steps / wall * dt_fs * 1e-6 * 86400.0, "dt_fs": dt_fs,
                      "atom_steps_per_s": coord.shape[0] * args.md_steps / wall,
                      "rebuilds": info["n_rebuilds"], "max_displacement_A": info["max_displacement"],
                      "skin_violated": info["skin_violated"],
                      "etot_drift_rel_to_ekin": float(np.abs(etot - etot[0]).max() / thermo[0, 1]),
                      "T_first_last_K": [float(thermo[0, 2]), float(thermo[-1, 2])],
                      "P_first_last_bar": [float(thermo[0, 3]), float(thermo[-1, 3])]}
    model.close()
    out["weights"] = "conditioned (fitting W0 / Nm)"
    return out


# ---- domain decomposition: weak scaling, one brick per rank ----------------------
def run_dd(args, spec, name, coord, types, box, dev, model, world, rank):
    """Every rank owns one copy of the workload's box as its brick of a px x py x pz times larger periodic box
    (weak scaling).  One step = forward ghost exchange, dpb_eval_local, reverse force exchange, all-reduce
    of E and the virial (paper_2004_11658_b200/dd.py).  With one rank the ghosts are the periodic images."""
    import torch
    import torch.distributed as dist
    from paper_2004_11658_b200.dd import BrickDecomposition, choose_grid
    grid = choose_grid(world, (1.0, 1.0, 1.0))
    L = np.array([box[0], box[4], box[8]])
    gbox = np.diag(L * np.array(grid)).reshape(-1)
    dd = BrickDecomposition(gbox, spec.rcut, grid=grid, rank=rank, world=world)
    w = coord - np.floor(coord / L) * L + dd.lo
    w = np.minimum(w, np.nextafter(dd.hi, dd.lo))                    # x + lo can round onto the upper face
    dc, dt = torch.tensor(w, device=dev), torch.tensor(types, device=dev)
    ev_local = lambda x, t, nloc, bounds: model.eval_local(x, t, nloc, bounds, want_info=False)
    steps, warm = max(3, min(args.steps, 20)), 3
    for _ in range(warm):
        out = dd.evaluate(ev_local, dc, dt)
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    marks = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(steps)]
    for k in range(steps):
        marks[k][0].record()
        x, t = dd.forward(dc, dt)
        marks[k][1].record()
        o = ev_local(x, t, dd.nloc, dd.bounds())
        marks[k][2].record()
        f = dd.reverse(o["force"])
        red = torch.cat([o["energy"].reshape(1), o["virial"].reshape(9)])
        if world > 1:
            dist.all_reduce(red)
        marks[k][3].record()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    seg = np.array([[m[i].elapsed_time(m[i + 1]) for i in range(3)] for m in marks]).sum(axis=0)
    tot = torch.tensor([sum(m[0].elapsed_time(m[3]) for m in marks)], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(tot, op=dist.ReduceOp.MAX)
    ms = float(tot[0]) / steps
    return {"grid": list(grid), "atoms_per_rank": int(coord.shape[0]), "atoms_with_ghosts": int(x.shape[0]),
            "steps": steps, "ms_per_step": ms, "atom_steps_per_s": world * coord.shape[0] / (ms * 1e-3),
            "ms_forward_exchange": seg[0] / steps, "ms_eval_local": seg[1] / steps,
            "ms_reverse_exchange_allreduce": seg[2] / steps, "energy_per_atom": float(red[0]) / (world * coord.shape[0]),
            "note": "times of rank 0 for the three parts, max over ranks for the step"}


# ---- the CUDA arm ---------------------------------------------------------------------------------------------
def run_cuda(args):
    import torch
    import torch.distributed as dist
    from paper_2004_11658_b200 import DPModel

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (this library has no CPU path)")
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)

    name = args.workload
    spec = MODELS[name]
    coord, types, box = gen.make_system(name, seed=gen.SEED_BASE + gen.CONFIGS[name].config_id + 7919 * rank)
    emb, fit = gen.make_weights(spec)
    n = coord.shape[0]
    mixed = args.precision == "tf32"
    model = DPModel.from_spec(spec, emb, fit, precision=1 if mixed else 0)
    model.set_variant(args.variant)
    model.set_timing(True)

    # pool of freshly perturbed copies (reading R24: fresh perturbation of the base positions per call)
    pool = min(args.steps + args.warmup, 16)
    host_coords = [gen.perturbed(coord, box, 0.01, gen.SEED_BASE + 1000 * (rank + 1) + k) for k in range(pool)]
    dcoords = [torch.tensor(c, device=dev) for c in host_coords]
    dtypes = torch.tensor(types, device=dev)
    out = None
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    # correctness guard + pair count (not timed)
    out = model.eval(dcoords[0], dtypes, box, want_info=True)
    info = out.pop("info")
    assert info.n_overflow == 0, "neighbour overflow in the benchmark workload"
    torch.cuda.synchronize()
    flops = algorithmic_flops(spec, n, info.n_real_pairs)

    for k in range(args.warmup):
        model.eval(dcoords[k % pool], dtypes, box, out=out)
    barrier()

    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    stage_sum = np.zeros(8)
    launches0 = model.kernel_launches()
    wall0 = time.perf_counter()
    for k in range(args.steps):
        flush.zero_()                                            # L2 flush, outside the timed events
        ev[k][0].record()
        model.eval(dcoords[(args.warmup + k) % pool], dtypes, box, out=out)
        ev[k][1].record()
        if args.stage_every and k % args.stage_every == 0:
            torch.cuda.synchronize()
            stage_sum += np.array(model.stage_us())
    barrier()
    wall = time.perf_counter() - wall0
    launches = model.kernel_launches() - launches0
    clocks = sampler.stop() if rank == 0 else {}
    dev_ms = sum(a.elapsed_time(b) for a, b in ev)
    n_stage = len(range(0, args.steps, args.stage_every)) if args.stage_every else 0

    # end to end through the host entry point (pinned host buffers, copies inside the timed region)
    pc = [torch.tensor(c).pin_memory() for c in host_coords[:4]]
    pt = torch.tensor(types).pin_memory()
    hout = {"energy": torch.empty(1, dtype=torch.float64).pin_memory(),
            "atom_energy": torch.empty(n, dtype=torch.float64).pin_memory(),
            "force": torch.empty((n, 3), dtype=torch.float64).pin_memory(),
            "virial": torch.empty((3, 3), dtype=torch.float64).pin_memory()}
    e2e_steps = max(3, min(args.steps, 20))
    for k in range(2):
        model.eval_host(pc[k % 4], pt, box, out=hout)
    barrier()
    t0 = time.perf_counter()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record()
    for k in range(e2e_steps):
        model.eval_host(pc[k % 4], pt, box, out=hout)
    e1.record()
    barrier()
    e2e_wall = time.perf_counter() - t0
    e2e_ms = max(e0.elapsed_time(e1), e2e_wall * 1e3)
    h2d = n * 3 * 8 + n * 4
    d2h = 8 + n * 8 + n * 24 + 72

    times = torch.tensor([dev_ms, e2e_ms], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(times, op=dist.ReduceOp.MAX)
    dev_ms, e2e_ms = float(times[0]), float(times[1])

    # optional extra leg, on every rank: the domain-decomposed step
    dd_leg = run_dd(args, spec, name, coord, types, box, dev, model, world, rank) if args.dd else None

    if rank == 0:
        ms_per_step = dev_ms / args.steps
        value = world * n * args.steps / (dev_ms * 1e-3)
        stage_us = (stage_sum / max(1, n_stage)).tolist()
        names = ["cell_sort", "nlist", "pass1_env_embed_T", "fit_fwd_bwd", "pass2_embed_bwd_force", "reduce"]
        stages = {nm: stage_us[i] for i, nm in enumerate(names)}
        dom = max(("pass1", 2), ("fit", 3), ("pass2", 4), key=lambda kv: stage_us[kv[1]])
        dom_t = stage_us[dom[1]] * 1e-6
        achieved = flops[dom[0]] / dom_t / 1e12 if dom_t > 0 else None
        total_flops = sum(flops.values())
        traffic = None
        tpath = os.path.join(ROOT, "profiles", "traffic.json")
        if os.path.exists(tpath):
            try:
                traffic = json.load(open(tpath)).get(f"{name}:{'tf32' if mixed else 'v' + str(args.variant)}:{dom[0]}")
            except Exception:
                traffic = None
        line = {
            "metric": METRIC, "value": value, "unit": "atom-steps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "tf32x3+f32acc (env/force/accumulations f64)" if mixed else "f64",
            "data": "synthetic", "config": workload_config(name, args),
            "natoms_per_gpu": n, "real_pairs": info.n_real_pairs, "wall_s": wall,
            "algorithmic_tflops": total_flops / (ms_per_step * 1e-3) / 1e12,
            "fp64_frac_of_peak": total_flops / (ms_per_step * 1e-3) / 1e12 / FP64_PEAK_TFLOPS,
            "stage_us": stages,
            "roofline": {"bound": "alu", "kernel": dom[0], "achieved": achieved, "peak": FP64_PEAK_TFLOPS,
                         "unit": "TFLOP/s", "frac": (achieved / FP64_PEAK_TFLOPS) if achieved else None,
                         "traffic": traffic,
                         "note": "fp64 pipe (DFMA/DMMA share one pipe, measured 37.0 TF/s; peak derived from 148 SM x 64 "
                                 "FMA/clk x 1.965 GHz); algorithmic flops of the stage / its CUDA-event time; the "
                                 "embedding passes execute 2.4-2.8x their algorithmic flops (pass 2 recomputes the "
                                 "forward chain and carries a tangent chain instead of reading stored activations; "
                                 "tanh; 25 -> 28 padding on water) and keep the fp64 pipe 74-81 % busy (ncu: "
                                 "profiles/r1_ncu_full_w24k.md, profiles/r1_ncu_full_cu32k.md)"},
            "e2e": {"value": world * n * e2e_steps / (e2e_ms * 1e-3), "unit": "atom-steps/s",
                    "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "steps": e2e_steps},
            "gpu_launches": int(launches),
            "clocks": {"sm_mhz": clocks.get("sm_mhz"), "sm_max_mhz": clocks.get("sm_max_mhz"),
                       "reasons": clocks.get("reasons", []), "samples": clocks.get("samples", 0),
                       "power_w_max": clocks.get("power_w_max")},
        }
        if mixed:
            # the GEMMs run on the tensor pipe: 3 TF32 MMAs per algorithmic product (3xTF32 split)
            peak, how = tf32_peak_tflops()
            line["roofline"] = {"bound": "tensor", "kernel": dom[0], "achieved": achieved, "peak": peak, "unit": "TFLOP/s",
                                "frac": (achieved / peak) if achieved else None, "traffic": traffic,
                                "note": f"algorithmic flops of the stage / its CUDA-event time against the dense TF32 peak "
                                        f"({how}); the tensor pipe executes 3x these flops (3xTF32 split); the stage is bound "
                                        f"by MUFU (fp32 tanh) and instruction issue, not by the tensor pipe (DESIGN.md)"}
            line.pop("fp64_frac_of_peak", None)
        if args.md_steps > 0:
            line["md"] = run_md(args, spec, name, coord, types, box, dev, emb, fit, mixed)
        if dd_leg is not None:
            line["dd"] = dd_leg
        if world == 1 and not args.no_cpu_baseline:
            step, k, desc, threads = oracle_step_sampler(name, gen.SEED_BASE, args.ref_sample)
            step()
            reps, t0 = 0, time.perf_counter()
            while reps < 3 or (time.perf_counter() - t0 < 10.0 and reps < 200):
                step(); reps += 1
            dt = time.perf_counter() - t0
            line["cpu_baseline"] = {"value": k * reps / dt, "unit": "atom-steps/s", "cores": threads, "kind": "oracle",
                                    "sample": f"{reps} steps x {desc}"}
        print(json.dumps(line))
    model.close()
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=100)
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", default="cuda", choices=["cuda", "reference"])
    ap.add_argument("--workload", default="W24k", choices=sorted(MODELS))
    ap.add_argument("--precision", default="fp64", choices=["fp64", "tf32"])
    ap.add_argument("--variant", type=int, default=int(os.environ.get("DPB_VARIANT", "1")))
    ap.add_argument("--ref-sample", type=int, default=2048, help="atoms per step of the CPU oracle arm")
    ap.add_argument("--stage-every", type=int, default=10, help="read the stage timers every n-th step (0: never)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--md-steps", type=int, default=0,
                    help="also run this many velocity-Verlet steps (dpb_md_run; PAPER.md:298: 330 K, 0.5 / 1.0 fs, 2 A skin "
                         "rebuilt every 50 steps) and report steps/s and ns/day in an extra 'md' object")
    ap.add_argument("--dd", action="store_true",
                    help="also time the domain-decomposed step (one brick per rank, ghost exchange + dpb_eval_local + "
                         "reverse force exchange + all-reduce) and report it in an extra 'dd' object")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
