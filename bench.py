#!/usr/bin/env python
"""Benchmark of the DP energy/force/virial hot path (BASELINE.json metric: atom-steps/s on one B200).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--config 0..4] [--impl ours|reference]

The default run times config 4 (headline), then configs 0-3 (`configs_summary`, each with its own roofline and oracle
timing), measures the arithmetic-pipe peaks it quotes (`peaks`, dp_measure_peaks), runs the paper's MD protocol
(`md`) and the network-size study of PAPER.md:273-279 (`network_size_sweep`; alone: --config sweep).

One "step" = one dp_compute (all of SURVEY.md section 8(a): cell list, formatted neighbour list, environment
matrix, embedding net + contraction, fitting net forward/backward, embedding backward, ProdForce, ProdViral)
on one seeded synthetic configuration.  The path does not shard (BASELINE north_star: one GPU, no
collectives): with --gpus N every rank runs an independent replica ("replicas only") and the
value is the aggregate, scaling "weak".  Prints ONE JSON line on rank 0.
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
sys.path.insert(0, ROOT)

# algorithmic flops (FMA = 2, tanh not counted, no credit for padding or recomputation)
FLOP_ROW_FWD = 12550 + 800          # embedding GEMMs forward + contraction forward, per neighbour row   (widths 25, 50, 100)
FLOP_ROW_BWD = 12550 + 1600         # embedding GEMMs backward + contraction backward, per neighbour row
FLOP_ATOM_FIT = 2036160             # fitting fwd + bwd + descriptor fwd/bwd, per atom


def flops_of(model):
    """(per-row forward, per-row backward, per-atom fitting + descriptor, tanh per row) for the model's network widths."""
    m0, m1, m2 = model.embed_widths
    f0, f1, f2 = model.fit_widths
    gemm = 2 * (m0 + m0 * m1 + m1 * m2)
    fit = 2 * (m2 * model.axis * f0 + f0 * f1 + f1 * f2 + f2)
    return gemm + 2 * 4 * m2, gemm + 4 * 4 * m2, 2 * fit + 3 * 2 * 4 * m2 * model.axis, m0 + m1 + m2
# tensor-core flops the MIX-16 backward kernel actually executes per 128-row tile (M = 128, 2 flop per MAC):
# layer 2 (hi+lo) 2*32*64, layer 3 2*96*112, dR 2*208*16, dT3 32*112, dT2+dz3 W3^T (32+112)*64, dT1+dz3 W3f (32+112)*32, dz2 W2^T 64*32
EXEC_FLOP_ROW_BWD = 2 * (2 * 32 * 64 + 2 * 96 * 112 + 2 * 208 * 16 + 32 * 112 + 144 * 64 + 144 * 32 + 64 * 32)
# ncu --set full captures of the dominant kernel per config (dram__bytes_read.sum + dram__bytes_write.sum per launch are in
# these summaries; the bench line itself measures no DRAM traffic, so roofline.traffic is null and points here)
TRAFFIC_PROFILE = {"c4_cu1048576": "profiles/r02_c4_bwd_tc2_ncu.md", "c2_cu13500": "profiles/r02_c2_bwd_f64_ncu.md",
                   "c3_water110592": "profiles/r02_c3_bwd_mix_ncu.md"}


def peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return dict(hbm=d["hbm_gbs"], bf16=d["bf16_tflops"], bf16_sus=d.get("bf16_tflops_sustained", d["bf16_tflops"]),
                    src="measured (MEASURED_PEAKS.json)")
    return dict(hbm=6650.0, bf16=1590.0, bf16_sus=1400.0, src="fallback (B200_PROFILING.md)")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 200 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows = []
        self.proc = None
        self.index = index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200", "-i", str(self.index)], stdout=subprocess.PIPE, text=True)
            threading.Thread(target=self._read, daemon=True).start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([t.strip() for t in line.split(",")])

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.25)
        self.proc.terminate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx.append(float(r[1]))
            except Exception:
                continue
            for n, v in zip(names, r[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(n)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(s, ncen):
    """Time the oracle, as it stands, on ncen evenly spaced centres of the workload (host cores)."""
    from oracle import oracle
    cen = np.unique(np.linspace(0, s.natoms - 1, ncen).astype(np.int64))
    t0 = time.perf_counter()
    oracle.evaluate(s.coords, s.types, s.box, s.model, centers=cen)
    dt = time.perf_counter() - t0
    return len(cen), dt, oracle.num_threads()


def run_reference(args, s):
    """--impl reference: the CPU oracle on a bounded sample per step (a deliberately slow program)."""
    ncen = 256 if s.natoms > 2000 else min(s.natoms, 256)
    for _ in range(min(args.warmup, 1)):
        oracle_sample(s, ncen)
    tot = 0.0
    n = 0
    cores = 1
    for _ in range(args.steps):
        n, dt, cores = oracle_sample(s, ncen)
        tot += dt
    val = n * args.steps / tot
    line = {"impl": "reference", "metric": "atom_steps_per_s", "value": val, "unit": "atom-steps/s", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": s.name, "natoms": s.natoms, "precision": "fp64 oracle"},
            "cpu_baseline": {"value": val, "unit": "atom-steps/s", "cores": cores, "kind": "oracle",
                             "sample": f"{n} evenly spaced centre atoms of {s.name} per step (brute-force list + full E_i and slot gradients)"},
            "e2e": {"value": val, "unit": "atom-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}
    print(json.dumps(line))


def time_config(binding, torch, s, dev, steps, warmup, flush):
    """Device-resident timing of one config: per-step CUDA events, L2 flush between steps, per-phase events."""
    model = binding.DPModel(s.model, s.precision)
    coords = torch.from_numpy(s.coords).to(dev)
    types = torch.from_numpy(s.types).to(dev)
    out = model.compute(coords, types, s.box)
    rc, ntr = model.status()
    if rc != 0:
        raise SystemExit(f"dp_status = {rc} on {s.name}")
    nl = model.get_nlist()
    real_rows = int((nl >= 0).sum().item())
    rows_f, rows_b = model.last_row_counts()
    del nl
    st = torch.cuda.current_stream(dev)
    for _ in range(warmup):
        model.compute(coords, types, s.box, out=out)
    model.profile_enable(True)
    ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
    phases = np.zeros(6)
    torch.cuda.synchronize(dev)
    for k in range(steps):
        flush.fill_(k & 0xFF)                      # L2 flush, outside the timed events
        ev[k][0].record(st)
        model.compute(coords, types, s.box, out=out)
        ev[k][1].record(st)
        phases += model.profile_read()             # synchronises; the gap is outside the timed events
    torch.cuda.synchronize(dev)
    model.profile_enable(False)
    t_ms = sum(a.elapsed_time(b) for a, b in ev)
    return dict(model=model, coords=coords, types=types, out=out, t_ms=t_ms, phases=phases / steps, real_rows=real_rows,
                rows_f=rows_f, rows_b=rows_b, ntr=ntr)


def roofline_of(s, r, pk, mp):
    """Roofline record of the dominant kernel (the embedding backward in every precision mode) of one timed config.
    achieved = algorithmic flops of the kernel (14,150 per REAL neighbour row) / its CUDA-event duration;
    peak = the measured rate of the pipe its dtype runs on (pk: MEASURED_PEAKS.json, mp: dp_measure_peaks of this run)."""
    ph = r["phases"]
    _, frow_b, _, tanh_row = flops_of(s.model)
    dom_flops = r["real_rows"] * frow_b
    ach = dom_flops / (ph[5] * 1e-3) / 1e12
    if s.precision == "fp64":
        kname, peak = "k_embed_bwd_f64 (S7-S9 in one kernel)", mp["dmma_tflops"]
        peak_src = "measured in this run (dp_measure_peaks): fp64 tensor pipe, mma.sync m8n8k4 (DFMA shares the pipe: %.1f TF/s)" % mp["dfma_tflops"]
    elif s.precision == "mix32":
        kname, peak = "k_embed_bwd_mix (S7-S9 in one kernel)", mp["ffma_tflops"]
        peak_src = ("measured in this run (dp_measure_peaks): fp32 FMA pipe, the pipe of single-precision arithmetic; the kernel "
                    "forms its single-precision products as three fp16 mma.sync products (measured mma.sync rate %.0f TF/s)" % mp["hmma_sync_tflops"])
    else:
        kname, peak = "k_embed_bwd_tc2", pk["bf16_sus"]
        peak_src = f"{pk['src']}: dense bf16 sustained (fp16 has the same nominal rate)"
    rec = {"kernel": kname, "bound": "tensor", "achieved": ach, "peak": peak, "unit": "TFLOP/s", "frac": ach / peak,
           "traffic": None, "traffic_profile": TRAFFIC_PROFILE.get(s.name), "peak_source": peak_src,
           "flops_per_launch": dom_flops, "kernel_ms": ph[5]}
    if s.precision != "fp64":
        # the tanh of the recomputed forward, counted on the real rows only (175 per row), against the measured MUFU rate
        rec["mufu_tanh_frac"] = (r["real_rows"] * tanh_row / (ph[5] * 1e-3)) / (mp["tanh_tera_per_s"] * 1e12)
    if s.precision == "mix16":
        rec["executed_tflops"] = r["rows_b"] * EXEC_FLOP_ROW_BWD / (ph[5] * 1e-3) / 1e12
        rec["note"] = (f"algorithmic backward flops ({frow_b:,} per real neighbour row); the in-kernel forward recompute, the hi/lo operand "
                       "splitting and the K/N padding are executed (executed_tflops, widths 25-50-100 only) but not credited; "
                       "mufu_tanh_frac = tanh of the real rows / measured tanh.approx.f32 rate")
        if s.model.embed_widths[0] != 25:
            rec.pop("executed_tflops")
    return rec


def kernels_of(s, r, ms_step):
    ph, N, rr = r["phases"], s.natoms, r["real_rows"]
    FLOP_ROW_FWD, FLOP_ROW_BWD, FLOP_ATOM_FIT, _ = flops_of(s.model)
    return {"nlist_ms": ph[0], "embed_fwd_ms": ph[1], "fit_ms": ph[2], "embed_bwd_ms": ph[3], "finalize_ms": ph[4],
            "embed_bwd_kernel_ms": ph[5],
            "embed_fwd_tflops": rr * FLOP_ROW_FWD / (ph[1] * 1e-3) / 1e12,
            "fit_tflops": N * FLOP_ATOM_FIT / (ph[2] * 1e-3) / 1e12,
            "embed_bwd_tflops": rr * FLOP_ROW_BWD / (ph[5] * 1e-3) / 1e12,
            "fused_embed_fwd_bwd_tflops": rr * (FLOP_ROW_FWD + FLOP_ROW_BWD) / ((ph[1] + ph[3]) * 1e-3) / 1e12,
            "step_tflops": (rr * (FLOP_ROW_FWD + FLOP_ROW_BWD) + N * FLOP_ATOM_FIT) / (ms_step * 1e-3) / 1e12}


def sweep_leg(args, binding, torch, synth, dev, flush, pk, precision="mix16", ncell=None, mp=None):
    """Network-size study (Fig. 7): copper, embedding nets (W, 2 W, 4 W), last layer 2 W x 4 W from the
    paper's 64 x 128 to 1024 x 2048, in one precision.  Algorithmic flops of the whole evaluation / CUDA-event time of the
    evaluation, against the peak of the precision's arithmetic: MIX-16 the sustained dense bf16 rate (MEASURED_PEAKS.json), FP64
    the DMMA rate and MIX-32 the fp32 FFMA rate that dp_measure_peaks measures in this run (MIX-32 executes three TF32 tensor
    products per algorithmic product, so its fraction of the fp32 rate can exceed 1)."""
    rows = []
    ncell = ncell or args.sweep_ncell
    peak, peak_name = pk["bf16_sus"], "bf16_sustained"
    if precision != "mix16":
        mp = mp or binding.measure_peaks()
        peak, peak_name = (mp["dmma_tflops"], "dmma") if precision == "fp64" else (mp["ffma_tflops"], "ffma_fp32")
    for W in [int(x) for x in args.sweep_widths.split(",")]:
        s = (synth.paper_copper(ncell, synth.SEED0 + 20, shuffle=True, precision=precision) if W == 32
             else synth.wide_copper(ncell, W, synth.SEED0 + 20, shuffle=True, precision=precision))
        r = time_config(binding, torch, s, dev, args.steps, args.warmup, flush)
        ms = r["t_ms"] / args.steps
        ff, fb, fa, _ = flops_of(s.model)
        ph, rr = r["phases"], r["real_rows"]
        emb = rr * (ff + fb)
        rows.append({"W": W, "last_layer": f"{2 * W}x{4 * W}", "natoms": s.natoms, "real_neighbour_rows": rr, "ms_per_step": ms,
                     "atom_steps_per_s": s.natoms / (ms * 1e-3),
                     "step_tflops": (emb + s.natoms * fa) / (ms * 1e-3) / 1e12,
                     "embed_fwd_ms": ph[1], "fit_ms": ph[2], "embed_bwd_ms": ph[3], "nlist_ms": ph[0],
                     "embed_fwd_bwd_tflops": emb / ((ph[1] + ph[3]) * 1e-3) / 1e12,
                     "bwd_gemm_ms": ph[5] if W != 32 else None,
                     "bwd_gemm_tflops": (rr * 2 * (W * 2 * W + 2 * W * 4 * W) / (ph[5] * 1e-3) / 1e12) if W != 32 else None,
                     "precision": precision, "peak": peak_name, "peak_tflops": peak,
                     ("frac_of_bf16_sustained" if precision == "mix16" else "frac_of_" + peak_name): (emb + s.natoms * fa) / (ms * 1e-3) / 1e12 / peak})
        r["model"].close()
        del r
        torch.cuda.empty_cache()
    return rows


def max_over_ranks(times_ms, world, device):
    """Replicas only: every rank times the same number of steps of its own replica; the job time is the
    MAX over ranks (one all-reduce of the timings, no data-path collective)."""
    import torch
    tt = torch.tensor(list(times_ms), dtype=torch.float64, device=device)
    if world > 1:
        import torch.distributed as dist
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    return [float(x) for x in tt]


def whole_job_value(natoms, steps, world, t_ms):
    """Aggregate atom-steps/s of `world` independent replicas (weak scaling)."""
    return world * natoms * steps / (t_ms * 1e-3)


def spawn_replicas(ngpus: int, argv) -> int:
    """`python bench.py --gpus N` outside torchrun: launch the N replica ranks ourselves (one process per GPU, NCCL only for
    the max-over-ranks of the timings), exactly as the driver's torchrun line does."""
    import socket
    with socket.socket() as sk:
        sk.bind(("127.0.0.1", 0))
        port = sk.getsockname()[1]
    cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={ngpus}", "--master-addr", "127.0.0.1",
           "--master-port", str(port), os.path.abspath(__file__)] + list(argv)
    return subprocess.call(cmd)


def md_leg(args, torch, synth, s, model, coords, types, dev, st, barrier):
    """The paper's own time-to-solution: MD loop time / steps, one dp_md_run: velocity Verlet, 330 K,
    2 A buffered list searched every 50 evaluations, thermo record (E_pot, E_kin, T, P) of every evaluation."""
    N = s.natoms
    kind = "water" if s.model.ntypes == 2 else "cu"
    dt_fs = 0.5 if kind == "water" else 1.0
    vel = torch.from_numpy(synth.boltzmann_velocities(s.types, synth.MASS_AMU[kind], 330.0, 99)).to(dev)
    xmd = coords.clone()
    model.md_run(xmd, vel, types, synth.MASS_AMU[kind], s.box, dt_fs, 1, skin=2.0, rebuild_every=50)   # warm-up
    barrier()
    m0, m1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    m0.record(st)
    mo = model.md_run(xmd, vel, types, synth.MASS_AMU[kind], s.box, dt_fs, args.md_steps, skin=2.0, rebuild_every=50)
    m1.record(st)
    barrier()
    rc_md, _ = model.status()
    th = mo["thermo"].cpu().numpy()
    md_ms = m0.elapsed_time(m1)
    every = 20                                                     # recorded every 20 time-steps
    return {"steps": args.md_steps, "evaluations": args.md_steps + 1, "list_searches": args.md_steps // 50 + 1, "dt_fs": dt_fs,
            "temperature_K": 330.0, "loop_ms_per_step": md_ms / args.md_steps,
            "s_per_step_per_atom": md_ms * 1e-3 / args.md_steps / N, "status": rc_md,
            "e_total_first_last_eV": [float(th[0, :2].sum()), float(th[-1, :2].sum())], "e_kin_first_eV": float(th[0, 1]),
            "thermo_every_20_steps": {"step": list(range(0, args.md_steps + 1, every)),
                                      "e_pot_eV": [float(x) for x in th[::every, 0]], "e_kin_eV": [float(x) for x in th[::every, 1]],
                                      "temperature_K": [float(x) for x in th[::every, 2]],
                                      "pressure_bar": [float(x) for x in th[::every, 3]]},
            "skin_A": 2.0, "rebuild_every": 50,
            "note": "velocity Verlet, 2 A buffered list searched at evaluation 0 and every 50 (PAPER.md:153), no L2 flush between steps"}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="4",
                    help="BASELINE.json configs index 0..4 (default: 4 = copper 1,048,576 atoms MIX-16, the largest single-GPU "
                         "config), or paper_cu / paper_water: the paper's network shape (32, 64, 128), capacity 512 / 144 (PAPER.md:151), "
                         "or sweep: the network-size study of PAPER.md:273-279 (copper, last embedding layer 64 x 128 ... 1024 x 2048; MIX-16, or --precision)")
    ap.add_argument("--no-summary", action="store_true", help="skip the configs_summary leg (the other four configs)")
    ap.add_argument("--precision", default=None, choices=["fp64", "mix32", "mix16"],
                    help="override the config's precision (profiling aid; the default is the precision BASELINE.json names)")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--sweep-widths", default="32,64,128,256,512", help="--config sweep: first embedding widths W (nets W, 2 W, 4 W)")
    ap.add_argument("--sweep-ncell", type=int, default=16, help="--config sweep: FCC cells per edge (atoms = 4 n^3)")
    ap.add_argument("--md-steps", type=int, default=100,
                    help="also time an MD loop of this many velocity-Verlet steps (dp_md_run; 0 = skip; N = 1 only)")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup

    if args.impl == "ours" and args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        raise SystemExit(spawn_replicas(args.gpus, sys.argv[1:]))

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))

    from paper_2005_00223_b200 import synth

    def workload():
        if args.config in ("paper_cu", "paper_water"):
            return synth.paper_config(args.config, args.precision or "fp64")
        return synth.config(int(args.config))

    if args.impl == "reference":
        if rank == 0:
            run_reference(args, workload())
        return

    import torch
    import torch.distributed as dist
    from paper_2005_00223_b200 import binding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (there is no CPU fallback)")
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=dev)

    flush = torch.empty(256 << 20, dtype=torch.uint8, device=dev)     # > L2 (126 MB)
    if args.config == "sweep":
        if rank == 0:
            pk = peaks()
            sampler = ClockSampler(local_rank)
            sampler.start()
            prec = args.precision or "mix16"
            rows = sweep_leg(args, binding, torch, synth, dev, flush, pk, precision=prec)
            clocks = sampler.stop()
            print(json.dumps({"metric": "network_size_sweep_step_tflops", "value": max(x["step_tflops"] for x in rows),
                              "unit": "TFLOP/s", "n_gpus": 1, "steps": args.steps, "warmup": args.warmup, "higher_is_better": True,
                              "dtype": {"fp64": "f64", "mix32": "f32", "mix16": "f16"}[prec], "data": "synthetic", "vs_baseline": None,
                              "config": {"workload": "sweep_cu (PAPER.md:273-279, Fig. 7)", "precision": prec,
                                         "l2": "256 MB flush between timed steps"},
                              "peak": {"bf16_sustained_tflops": pk["bf16_sus"], "source": pk["src"]},
                              "sweep": rows, "clocks": clocks}))
        return
    s = workload()
    if args.precision:
        s.precision = args.precision
    N = s.natoms
    st = torch.cuda.current_stream(dev)
    coords_h = torch.from_numpy(s.coords).pin_memory()
    types_h = torch.from_numpy(s.types).pin_memory()

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()

    K = args.steps
    sampler = ClockSampler(local_rank)
    barrier()
    sampler.start()
    r = time_config(binding, torch, s, dev, K, args.warmup, flush)
    barrier()
    clocks = sampler.stop()
    model, coords, types, out = r["model"], r["coords"], r["types"], r["out"]
    t_ms = r["t_ms"]

    # end to end through the public API with HOST buffers: H2D of inputs, compute, D2H of results, every step
    res_h = dict(energy=torch.empty(1, dtype=torch.float64).pin_memory(),
                 forces=torch.empty((N, 3), dtype=torch.float64).pin_memory(),
                 virial=torch.empty(9, dtype=torch.float64).pin_memory(),
                 atom_energy=torch.empty(N, dtype=torch.float64).pin_memory())
    cdev = torch.empty_like(coords)
    tdev = torch.empty_like(types)

    def e2e_step():
        cdev.copy_(coords_h, non_blocking=True)
        tdev.copy_(types_h, non_blocking=True)
        model.compute(cdev, tdev, s.box, out=out)
        for k_, v in res_h.items():
            v.copy_(out[k_], non_blocking=True)

    e2e_step()
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(st)
    for k in range(K):
        e2e_step()
    e1.record(st)
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    h2d = N * 24 + N * 4
    d2h = 8 + N * 24 + 72 + N * 8

    t_ms, e2e_ms = max_over_ranks([t_ms, e2e_ms], world, dev)

    md = None
    if world == 1 and args.md_steps > 0:
        try:
            md = md_leg(args, torch, synth, s, model, coords, types, dev, st, barrier)
        except Exception as ex:      # the MD leg never takes the bench line down
            md = {"error": repr(ex)}

    if rank == 0:
        pk = peaks()
        mp = binding.measure_peaks()
        ms_step = t_ms / K
        value = whole_job_value(N, K, world, t_ms)
        line = {"metric": "atom_steps_per_s", "value": value, "unit": "atom-steps/s", "n_gpus": world, "steps": K,
                "warmup": args.warmup, "ms_per_step": ms_step, "s_per_step_per_atom": ms_step * 1e-3 / N,
                "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": {"fp64": "f64", "mix32": "f32", "mix16": "f16"}[s.precision], "data": "synthetic",
                "config": {"workload": s.name, "natoms": N, "precision": s.precision, "nm": s.model.nm,
                           "real_neighbour_rows": r["real_rows"], "rows_through_embedding_fwd": r["rows_f"],
                           "rows_through_embedding_bwd": r["rows_b"], "n_truncated_atoms": r["ntr"],
                           "parallelism": "replicas only" if world > 1 else "single GPU",
                           "l2": "256 MB flush between timed steps, per-step CUDA events"},
                "clocks": clocks,
                "e2e": {"value": world * N * K / (e2e_ms * 1e-3), "unit": "atom-steps/s", "h2d_bytes_per_step": h2d,
                        "d2h_bytes_per_step": d2h},
                "gpu_launches": model.launches_per_compute() * K,
                "roofline": roofline_of(s, r, pk, mp),
                "kernels": kernels_of(s, r, ms_step),
                "peaks": {"hbm_gbs": pk["hbm"], "bf16_tflops_burst": pk["bf16"], "bf16_tflops_sustained": pk["bf16_sus"],
                          "source_hbm_bf16": pk["src"], **mp,
                          "source_pipes": "dp_measure_peaks in this run: 8 independent chains per thread, 8 x 256 threads per SM, CUDA events"}}
        if md is not None:
            line["md"] = md
        if world == 1 and not args.no_cpu_baseline:
            ncen = min(N, 16384)
            n, dt, cores = oracle_sample(s, ncen)
            line["cpu_baseline"] = {"value": n / dt, "unit": "atom-steps/s", "cores": cores, "kind": "oracle",
                                    "sample": f"{n} evenly spaced centre atoms of {s.name}, one evaluation ({dt:.1f} s)"}
        if world == 1 and not args.no_summary and args.config == "4":
            # the other BASELINE configs: same timing method (warm-up, L2 flush, per-step events), own roofline and oracle timing
            summ = {s.name: {"precision": s.precision, "natoms": N, "ms_per_step": ms_step, "atom_steps_per_s": value,
                             "s_per_step_per_atom": ms_step * 1e-3 / N, "roofline_frac": line["roofline"]["frac"]}}
            model.close()
            del model, coords, types, out, cdev, tdev
            torch.cuda.empty_cache()
            for idx in range(5):
                if idx == 4:
                    continue
                s2 = synth.config(idx)
                k2 = max(10, K)
                r2 = time_config(binding, torch, s2, dev, k2, args.warmup, flush)
                ms2 = r2["t_ms"] / k2
                rec = {"precision": s2.precision, "natoms": s2.natoms, "steps": k2, "ms_per_step": ms2,
                       "atom_steps_per_s": s2.natoms / (ms2 * 1e-3), "s_per_step_per_atom": ms2 * 1e-3 / s2.natoms,
                       "real_neighbour_rows": r2["real_rows"], "n_truncated_atoms": r2["ntr"],
                       "roofline": roofline_of(s2, r2, pk, mp), "kernels": kernels_of(s2, r2, ms2)}
                r2["model"].close()
                if not args.no_cpu_baseline:
                    n2, dt2, cores2 = oracle_sample(s2, min(s2.natoms, 4096))
                    rec["cpu_baseline"] = {"value": n2 / dt2, "unit": "atom-steps/s", "cores": cores2, "kind": "oracle",
                                           "sample": f"{n2} evenly spaced centre atoms of {s2.name}, one evaluation ({dt2:.1f} s)"}
                summ[s2.name] = rec
            line["configs_summary"] = summ
            # network-size study (Fig. 7): copper, embedding nets up to 512-1024-2048, MIX-16.
            # The widest net keeps 77 GB of activations in its workspace: everything above is released first, and a failure
            # of this leg is recorded instead of losing the line.
            try:
                torch.cuda.empty_cache()
                args.steps_saved, args.steps = args.steps, 3
                rows = sweep_leg(args, binding, torch, synth, dev, flush, pk)
                args.steps = args.steps_saved
                line["network_size_sweep"] = {"workload": f"copper {4 * args.sweep_ncell ** 3} atoms, capacity 512, MIX-16, list build included",
                                              "unit": "TFLOP/s (algorithmic flops of the whole evaluation / CUDA-event time)",
                                              "peak_bf16_sustained_tflops": pk["bf16_sus"], "rows": rows}
            except (Exception, SystemExit) as e:      # noqa: BLE001
                line["network_size_sweep"] = {"error": repr(e)[:300]}
            # the double and MIX-32 curves of the same figure (csrc/wide_gen.cu): 4,000 atoms (the fp64 activations of the widest
            # net take 76 GB there), each against the peak of its own arithmetic
            for prec in ("fp64", "mix32"):
                try:
                    torch.cuda.empty_cache()
                    args.steps_saved, args.steps = args.steps, 2
                    rows = sweep_leg(args, binding, torch, synth, dev, flush, pk, precision=prec, ncell=10, mp=mp)
                    args.steps = args.steps_saved
                    line["network_size_sweep_" + prec] = {
                        "workload": "copper 4000 atoms, capacity 512, " + prec + ", list build included",
                        "unit": "TFLOP/s (algorithmic flops of the whole evaluation / CUDA-event time)", "rows": rows}
                except (Exception, SystemExit) as e:      # noqa: BLE001
                    args.steps = getattr(args, "steps_saved", args.steps)
                    line["network_size_sweep_" + prec] = {"error": repr(e)[:300]}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
