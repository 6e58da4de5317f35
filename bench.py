#!/usr/bin/env python
"""bench.py — throughput of one DP energy / force / virial evaluation (the whole hot path, S1..S9) on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--workload W24k|Cu32k|W192|Cu864k] [--variant 0|1|2]
                    [--precision fp64|tf32|bf16]   # tf32 / bf16 = BASELINE.json configs[3] (mixed precision, tcgen05 kernels)
    python bench.py --impl reference ...     # times the CPU oracle (the baseline arm) on a bounded sample

The default run (W24k, fp64: the headline line) appends a `configs` object with short legs over every other
BASELINE.json config (W192, Cu32k, W24k tf32 / bf16, Cu864k); --no-configs skips them.  --variant 2 adds a `strawman`
object (the paper's own pipeline against the fused path).

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
FP64_FMA_PER_CLK = 148 * 64   # 148 SMs x 64 DFMA lanes per clock (measured 37.0 TF/s at 1965 MHz)


def fp64_peak_tflops(sm_mhz):
    """fp64 pipe peak at the SM clock sampled during the timed region (DFMA and DMMA share this pipe):
    148 x 64 FMA/clk x 2 flop x clock; 37.2 TFLOP/s at the 1965 MHz the B200 holds in these runs."""
    return FP64_FMA_PER_CLK * 2 * float(sm_mhz or 1965.0) * 1e6 / 1e12


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
    # dg = dT R~ and dR~ = dT^T g (2 x 2*4*M), 1 - t^2 and its product (3 x 7 s1), the two concat folds
    # (2 s1 + 4 s1), the chain to the displacement (36): 14,861 flop per neighbour for water, 23,492 for copper
    emb_bwd = gemm + 2 * (2 * 4 * M) + 3 * (7 * s1) + (2 * s1 + 4 * s1) + 36
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
            "pair_reuse": "nets (a,a): pass 2 always, pass 1 in single-chunk evaluations (library default; fp64 variant 1)",
            "stored_activations": ("library default (on when the records fit the workspace budget)" if STORED_ACT is None
                                   else bool(STORED_ACT)),
            "species_pipeline": "library default (on in the timed steps; the stage timers of stage_us separate the stages)"}


# ---- molecular dynamics: the paper's own unit, steps/s and ns/day ----------------------
def run_md(args, spec, name, coord, types, box, dev, emb, fit, mixed):
    """Random-init weights are not a physical potential: with the literal N(0, 1/fan_in) set the forces are ~4 eV/A rms
    and the box heats to 1e5 K within 500 steps.  The MD leg therefore uses the conditioned weight set (fitting W0 / Nm,
    DESIGN.md section 3: forces ~0.2 eV/A rms); the kernels and their cost are the same."""
    import torch
    from paper_2004_11658_b200 import DPModel
    model = DPModel.from_spec(spec, emb, gen.condition_fit_w0(spec, fit), precision={"fp64": 0, "tf32": 1, "bf16": 2, "bf16_plain": 3}[args.precision])
    if STORED_ACT is not None:
        model.set_stored_activations(STORED_ACT)
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
STAGES = ["cell_sort", "nlist", "pass1_env_embed_T", "fit_fwd_bwd", "pass2_embed_bwd_force", "reduce"]


STORED_ACT = None        # --stored-act: None = library default (on), 0 / 1 = dpb_model_set_stored_activations


def measure(name, precision, variant, steps, warmup, dev, rank=0, world=1, stage_every=10, want_e2e=False):
    """Time `steps` evaluations of workload `name` (each on a freshly perturbed copy of its box, L2 flushed in between,
    CUDA events on the launching stream, W untimed warm-up calls).  Returns a dict; times are this rank's."""
    import torch
    import torch.distributed as dist
    from paper_2004_11658_b200 import DPModel

    spec = MODELS[name]
    coord, types, box = gen.make_system(name, seed=gen.SEED_BASE + gen.CONFIGS[name].config_id + 7919 * rank)
    emb, fit = gen.make_weights(spec)
    n = coord.shape[0]
    mixed = precision != "fp64"
    model = DPModel.from_spec(spec, emb, fit, precision={"fp64": 0, "tf32": 1, "bf16": 2, "bf16_plain": 3}[precision])
    model.set_variant(variant)
    if STORED_ACT is not None:
        model.set_stored_activations(STORED_ACT)

    # pool of freshly perturbed copies (reading R24: fresh perturbation of the base positions per call)
    pool = min(steps + warmup, 16 if n < 200000 else 3)
    host_coords = [gen.perturbed(coord, box, 0.01, gen.SEED_BASE + 1000 * (rank + 1) + k) for k in range(pool)]
    dcoords = [torch.tensor(c, device=dev) for c in host_coords]
    dtypes = torch.tensor(types, device=dev)
    flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    out = model.eval(dcoords[0], dtypes, box, want_info=True)        # correctness guard + pair count (not timed)
    info = out.pop("info")
    assert info.n_overflow == 0, "neighbour overflow in the benchmark workload"
    torch.cuda.synchronize()
    torch.cuda.reset_peak_memory_stats(dev)
    flops = algorithmic_flops(spec, n, info.n_real_pairs)
    for k in range(warmup):
        model.eval(dcoords[k % pool], dtypes, box, out=out)
    barrier()

    sampler = ClockSampler(dev.index or 0)
    if rank == 0:
        sampler.start()
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    launches0 = model.kernel_launches()
    wall0 = time.perf_counter()
    for k in range(steps):
        flush.zero_()                                            # L2 flush, outside the timed events
        ev[k][0].record()
        model.eval(dcoords[(warmup + k) % pool], dtypes, box, out=out)
        ev[k][1].record()
    barrier()
    wall = time.perf_counter() - wall0
    launches = model.kernel_launches() - launches0
    clocks = sampler.stop() if rank == 0 else {}
    per_step = sorted(a.elapsed_time(b) for a, b in ev)
    dev_ms = float(sum(per_step))
    # per-stage device times from a few EXTRA steps with the library's stage timers on (events between the stages; they
    # switch the CUDA-graph replay off, so they are kept out of the timed region)
    stage_sum, n_stage = np.zeros(8), 0
    if stage_every:
        model.set_timing(True)
        for k in range(max(1, min(steps, 5))):
            flush.zero_()
            model.eval(dcoords[k % pool], dtypes, box, out=out)
            torch.cuda.synchronize()
            stage_sum += np.array(model.stage_us())
            n_stage += 1
        model.set_timing(False)
    stage_us = (stage_sum / max(1, n_stage)).tolist()
    res = {"name": name, "precision": precision, "variant": variant, "spec": spec, "n": n, "info": info, "flops": flops,
           "dev_ms": dev_ms, "ms_median": per_step[len(per_step) // 2], "ms_min": per_step[0], "wall": wall,
           "launches": int(launches), "clocks": clocks, "stage_us": stage_us,
           "coord": coord, "types": types, "box": box, "emb": emb, "fit": fit, "model": model}

    if want_e2e:
        # end to end through the host entry point (pinned host buffers, copies inside the timed region)
        pc = [torch.tensor(c).pin_memory() for c in host_coords[:4]]
        pt = torch.tensor(types).pin_memory()
        hout = {"energy": torch.empty(1, dtype=torch.float64).pin_memory(),
                "atom_energy": torch.empty(n, dtype=torch.float64).pin_memory(),
                "force": torch.empty((n, 3), dtype=torch.float64).pin_memory(),
                "virial": torch.empty((3, 3), dtype=torch.float64).pin_memory()}
        e2e_steps = max(3, min(steps, 20))
        for k in range(2):
            model.eval_host(pc[k % len(pc)], pt, box, out=hout)
        barrier()
        t0 = time.perf_counter()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record()
        for k in range(e2e_steps):
            model.eval_host(pc[k % len(pc)], pt, box, out=hout)
        e1.record()
        barrier()
        e2e_wall = time.perf_counter() - t0
        res.update(e2e_ms=max(e0.elapsed_time(e1), e2e_wall * 1e3), e2e_steps=e2e_steps,
                   h2d=n * 3 * 8 + n * 4, d2h=8 + n * 8 + n * 24 + 72)
    return res


def stage_roofline(res, sm_mhz):
    """Algorithmic roofline fraction of every fp64-pipe (or, in mixed precision, tensor-pipe) stage and of the whole step."""
    mixed = res["precision"] != "fp64"
    if mixed:
        peak, how = tf32_peak_tflops()
        if res["precision"].startswith("bf16"):
            peak, how = peak * 2.0, how.replace("x 1/2", "x 1")
    else:
        peak, how = fp64_peak_tflops(sm_mhz), f"148 SM x 64 FMA/clk x 2 x {sm_mhz or 1965.0:.0f} MHz (sampled)"
    idx = {"pass1": 2, "fit": 3, "pass2": 4}
    frac = {}
    for k, i in idx.items():
        t = res["stage_us"][i] * 1e-6
        frac[k] = (res["flops"][k] / t / 1e12 / peak) if t > 0 else None
    dom = max(idx, key=lambda k: res["stage_us"][idx[k]])
    return peak, how, frac, dom


def config_summary(res):
    """One entry of the `configs` object: a BASELINE.json config in the launch configuration of the headline run."""
    sm = res["clocks"].get("sm_mhz")
    peak, how, frac, dom = stage_roofline(res, sm)
    ms = res["ms_median"]
    total = sum(res["flops"].values())
    out = {"workload": f"{res['name']} (BASELINE.json configs[{gen.CONFIGS[res['name']].config_id}])",
           "precision": res["precision"], "natoms": res["n"], "real_pairs": res["info"].n_real_pairs,
           "n_overflow": res["info"].n_overflow, "n_chunks": res["info"].n_chunks,
           "ms_per_step": ms, "ms_min": res["ms_min"], "us_per_eval": ms * 1e3,
           "atom_steps_per_s": res["n"] / (ms * 1e-3),
           "stage_us": {nm: res["stage_us"][i] for i, nm in enumerate(STAGES)},
           "algorithmic_tflops": total / (ms * 1e-3) / 1e12,
           "frac_of_peak": total / (ms * 1e-3) / 1e12 / peak,
           "stage_frac_of_peak": frac, "dominant_stage": dom, "dominant_frac": frac[dom],
           "peak_tflops": peak, "peak_how": how, "sm_mhz": sm, "reasons": res["clocks"].get("reasons", []),
           "gpu_launches_per_step": res["launches"] / max(1, res["steps"])}
    return out


EXTRA_CONFIGS = [  # (workload, precision, steps, warmup): every BASELINE.json config beside the headline (W24k fp64)
    ("W192", "fp64", 200, 10), ("Cu32k", "fp64", 5, 3), ("W24k", "tf32", 20, 5), ("W24k", "bf16", 20, 5),
    ("W24k", "bf16_plain", 10, 3),   # measured for its cost only: it misses the tolerance (tests/test_gpu_mixed.py)
    ("Cu864k", "fp64", 3, 3),
]


def run_cuda(args):
    import torch
    import torch.distributed as dist

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
    mixed = args.precision != "fp64"
    res = measure(name, args.precision, args.variant, args.steps, args.warmup, dev, rank, world, args.stage_every,
                  want_e2e=True)
    res["steps"] = args.steps
    spec, n, info, flops, model = res["spec"], res["n"], res["info"], res["flops"], res["model"]
    coord, types, box, emb, fit = res["coord"], res["types"], res["box"], res["emb"], res["fit"]

    times = torch.tensor([res["dev_ms"], res["e2e_ms"]], dtype=torch.float64, device=dev)
    if world > 1:
        dist.all_reduce(times, op=dist.ReduceOp.MAX)
    dev_ms, e2e_ms = float(times[0]), float(times[1])

    # optional extra leg, on every rank: the domain-decomposed step
    dd_leg = run_dd(args, spec, name, coord, types, box, dev, model, world, rank) if args.dd else None

    if rank == 0:
        clocks = res["clocks"]
        ms_per_step = dev_ms / args.steps
        value = world * n * args.steps / (dev_ms * 1e-3)
        stage_us = res["stage_us"]
        stages = {nm: stage_us[i] for i, nm in enumerate(STAGES)}
        peak, how, frac, dom = stage_roofline(res, clocks.get("sm_mhz"))
        idx = {"pass1": 2, "fit": 3, "pass2": 4}
        dom_t = stage_us[idx[dom]] * 1e-6
        achieved = flops[dom] / dom_t / 1e12 if dom_t > 0 else None
        total_flops = sum(flops.values())
        traffic, traffic_src = None, None
        tpath = os.path.join(ROOT, "profiles", "r2_traffic.csv")
        if os.path.exists(tpath):
            try:
                want = f"{name}:{args.precision if mixed else 'v' + str(args.variant)}:{dom}"
                for ln in open(tpath).read().splitlines()[1:]:
                    key, val = ln.rsplit(",", 1)
                    if key == want:
                        traffic = int(val)
                traffic_src = "profiles/r2_traffic.md (dram__bytes_read.sum + dram__bytes_write.sum, one evaluation)"
            except Exception:
                traffic = None
        line = {
            "metric": METRIC, "value": value, "unit": "atom-steps/s", "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None,
            "dtype": {"fp64": "f64", "tf32": "tf32x3+f32acc (env/force/accumulations f64)",
                      "bf16": "bf16x6+f32acc (env/force/accumulations f64)",
                      "bf16_plain": "bf16+f32acc in the fitting GEMMs (fails the tolerance; measured only)"}[args.precision],
            "data": "synthetic", "config": workload_config(name, args),
            "natoms_per_gpu": n, "real_pairs": info.n_real_pairs, "wall_s": res["wall"],
            "algorithmic_tflops": total_flops / (ms_per_step * 1e-3) / 1e12,
            "stage_us": stages, "stage_frac_of_peak": frac,
            "roofline": {"bound": "tensor" if mixed else "alu", "kernel": dom, "achieved": achieved, "peak": peak,
                         "unit": "TFLOP/s", "frac": (achieved / peak) if achieved else None, "traffic": traffic,
                         "traffic_note": ("DRAM bytes summed over ALL launches of this stage in one evaluation (ncu --set "
                                          f"full, cold cache): {traffic_src}") if traffic else None,
                         "peak_how": how},
            "e2e": {"value": world * n * res["e2e_steps"] / (e2e_ms * 1e-3), "unit": "atom-steps/s",
                    "h2d_bytes_per_step": res["h2d"], "d2h_bytes_per_step": res["d2h"], "steps": res["e2e_steps"]},
            "gpu_launches": res["launches"],
            "clocks": {"sm_mhz": clocks.get("sm_mhz"), "sm_max_mhz": clocks.get("sm_max_mhz"),
                       "reasons": clocks.get("reasons", []), "samples": clocks.get("samples", 0),
                       "power_w_max": clocks.get("power_w_max")},
        }
        if not mixed:
            line["fp64_frac_of_peak"] = total_flops / (ms_per_step * 1e-3) / 1e12 / peak
            line["roofline"]["note"] = (
                "fp64 pipe: DFMA and DMMA share one pipe (measured 37.0 TF/s at 1965 MHz, profiles/r1_fp64_peaks.md); "
                "`achieved` = ALGORITHMIC flops of the stage (SURVEY.md 8(d): both directions of every pair, no recompute, "
                "no padding, tanh not counted) / its CUDA-event time.  What the kernels execute differs: tanh costs 19 pipe "
                "slots, 25 -> 28 padding on water; with the same-species pair reuse they execute fewer chains than the "
                "algorithmic count for the nets (a,a); pass 2 reads the activations pass 1 stored (value chain and tanh not "
                "re-run: its DRAM traffic is those records) unless --stored-act 0 or they do not fit — so this is a "
                "throughput figure, not a pipe-utilisation figure (that is ncu's, profiles/)")
        else:
            line["roofline"]["note"] = (
                f"algorithmic flops of the stage / its CUDA-event time against the dense tensor peak ({how}); the tensor "
                "pipe executes 3x (tf32) or 6x (bf16) these flops (error-compensated split); the stage is bound by MUFU "
                "(fp32 tanh) and instruction issue, not by the tensor pipe (DESIGN.md section 9)")
        if args.variant == 2 and not mixed:
            # what fusion and padding-skip buy = this run (the paper's pipeline) against variant 1
            free_b, total_b = torch.cuda.mem_get_info(dev)
            model.close()
            r1 = measure(name, "fp64", 1, max(3, min(args.steps, 10)), 3, dev, rank, world, args.stage_every)
            r1["model"].close()
            nm = sum(spec.sel)
            line["strawman"] = {
                "what": "variant 2 = PAPER.md section 3.2.3 on B200: GEMMs over all padded slots, bias and concat as GEMMs, "
                        "separate tanh / tanh-grad kernels, G and activations materialised, reverse-mode backward",
                "padded_slots": int(n * nm), "real_pairs": int(info.n_real_pairs),
                "device_memory_in_use_bytes": int(total_b - free_b),
                "variant1_ms_per_step": r1["ms_median"], "variant1_stage_us": {nm_: r1["stage_us"][i] for i, nm_ in enumerate(STAGES)},
                "ratio_variant2_over_variant1": ms_per_step / r1["ms_median"],
                "ratio_embedding_stages": (stage_us[2] + stage_us[4]) / max(1e-9, r1["stage_us"][2] + r1["stage_us"][4])}
        if args.md_steps > 0:
            line["md"] = run_md(args, spec, name, coord, types, box, dev, emb, fit, mixed)
        if dd_leg is not None:
            line["dd"] = dd_leg
    model.close()
    del res

    # every other BASELINE.json config, 1 GPU only, short: the driver's record then holds all of them
    if rank == 0 and world == 1 and args.configs and name == "W24k" and args.precision == "fp64":
        cfgs = {}
        for (wn, prec, st, wu) in EXTRA_CONFIGS:
            key = wn if prec == "fp64" else f"{wn}-{prec}"
            try:
                torch.cuda.empty_cache()
                r = measure(wn, prec, args.variant, st, wu, dev)
                r["steps"] = st
                cfgs[key] = config_summary(r)
                cfgs[key]["steps"] = st
                free_b, total_b = torch.cuda.mem_get_info(dev)      # the library's workspace is grow-only: in use = peak
                cfgs[key]["device_memory_in_use_bytes"] = int(total_b - free_b)
                r["model"].close()
                del r
            except Exception as exc:                              # a config that cannot run is reported, not hidden
                cfgs[key] = {"error": f"{type(exc).__name__}: {exc}"}
        line["configs"] = cfgs

    if rank == 0:
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
    ap.add_argument("--precision", default="fp64", choices=["fp64", "tf32", "bf16", "bf16_plain"])
    ap.add_argument("--variant", type=int, default=1)
    ap.add_argument("--stored-act", type=int, default=None, choices=[0, 1],
                    help="fp64 variant 1: pass 2 reads the activations pass 1 stored (default: the library's, on)")
    ap.add_argument("--no-configs", dest="configs", action="store_false",
                    help="skip the short legs over the other BASELINE.json configs (W192, Cu32k, W24k mixed, Cu864k) that the "
                         "default run appends as a `configs` object")
    ap.add_argument("--ref-sample", type=int, default=2048, help="atoms per step of the CPU oracle arm")
    ap.add_argument("--stage-every", type=int, default=1, help="0: do not run the extra stage-timer steps")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--md-steps", type=int, default=0,
                    help="also run this many velocity-Verlet steps (dpb_md_run; PAPER.md:298: 330 K, 0.5 / 1.0 fs, 2 A skin "
                         "rebuilt every 50 steps) and report steps/s and ns/day in an extra 'md' object")
    ap.add_argument("--dd", action="store_true",
                    help="also time the domain-decomposed step (one brick per rank, ghost exchange + dpb_eval_local + "
                         "reverse force exchange + all-reduce) and report it in an extra 'dd' object")
    args = ap.parse_args()
    global STORED_ACT
    STORED_ACT = args.stored_act
    if args.impl == "reference":
        return run_reference(args)
    return run_cuda(args)


if __name__ == "__main__":
    sys.exit(main())
