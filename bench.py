#!/usr/bin/env python
"""bench.py — PaiNN energy+force throughput of the B200 path (BASELINE.json metric) on synthetic input.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg3_fp32|cfg4|cfg5|...] [--impl reference]

One step = one pass of the whole hot path (graph build + forward + analytic adjoint) over
one batch.  Prints ONE JSON line (rank 0).  See DESIGN.md "Measurement" for every definition used here.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)
import gen  # noqa: E402

# workload name -> (config id, precision, forces, structures per step or None = the config's own count)
WORKLOADS = {
    "cfg1": (1, "fp64", True, None),
    "cfg2": (2, "fp32", True, None),
    "cfg2_fp64": (2, "fp64", True, None),
    # blended multi-head inference (Fig. 5): all 16 heads weighted per structure, branches below 0.01 skipped
    "cfg2_blended": (2, "fp32", True, None),
    "cfg3_fp32": (3, "fp32", True, None),
    "cfg3_bf16": (3, "bf16", True, None),
    "cfg4": (4, "bf16", False, 16384),
    "cfg4_fp32": (4, "fp32", False, 16384),
    "cfg5": (5, "fp64", True, None),
}
WORKLOAD_NAMES = {"cfg1": "cfg1_tiny_fp64", "cfg2": "cfg2_molecular_fp32", "cfg2_fp64": "cfg2_molecular_fp64",
                  "cfg2_blended": "cfg2_molecular_fp32_blended_heads",
                  "cfg3_fp32": "cfg3_crystals_fp32", "cfg3_bf16": "cfg3_crystals_bf16",
                  "cfg4": "cfg4_screening_bf16_batch16384", "cfg4_fp32": "cfg4_screening_fp32_batch16384",
                  "cfg5": "cfg5_large_fp64"}
DTYPE = {"fp64": "f64", "fp32": "f32", "bf16": "bf16"}
# plain-ALU peaks derived from the guide's unit counts and clocks:
# 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz; FP64 at half the FP32 lane count.
ALU_PEAK_TFLOPS = {"fp32": 148 * 128 * 2 * 1.965e9 / 1e12, "fp64": 148 * 64 * 2 * 1.965e9 / 1e12,
                   "bf16": 148 * 128 * 2 * 1.965e9 / 1e12}


def measured_peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as fh:
            p = json.load(fh)
        return dict(hbm=float(p["hbm_gbs"]), bf16=float(p["bf16_tflops"]), bf16_sust=float(p["bf16_tflops_sustained"]),
                    source="measured")
    except Exception:
        return dict(hbm=6650.0, bf16=1590.0, bf16_sust=1400.0, source="fallback")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 100 ms while the timed region runs."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.proc, self.path = index, None, None

    def start(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.fh = open(self.path, "w")
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"], stdout=self.fh,
                                         stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = dict(sm_mhz=None, sm_max_mhz=None, reasons=[], samples=0)
        if self.proc is None:
            return out
        try:
            time.sleep(0.15)
            self.proc.terminate()
            self.proc.wait(timeout=5)
            self.fh.close()
            rows = [l.strip().split(", ") for l in open(self.path) if l.strip()]
            os.unlink(self.path)
            sm = [float(r[0]) for r in rows if r[0].replace(".", "").isdigit()]
            if sm:
                out["sm_mhz"] = float(np.median(sm))
                out["sm_max_mhz"] = float(rows[0][1])
                out["power_w_max"] = max(float(r[2]) for r in rows)
                names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
                out["reasons"] = [n for q, n in enumerate(names) if any(r[3 + q].strip() == "Active" for r in rows)]
                out["samples"] = len(sm)
        except Exception:
            pass
        return out


def algorithmic_work(family: str, N: int, E: int, mc: gen.ModelCfg, prec: str, forces: bool):
    """(flops, bytes) per LAUNCH of one kernel family (per-atom and per-edge figures)."""
    F, K = mc.F, mc.K
    b = 8 if prec == "fp64" else 4
    eb = 4 + 4 * b                                    # col + (ux,uy,uz,d)
    if prec == "bf16":
        # BF16 model: phi, v gathered as BF16 copies (read once from HBM), FP32 residual rows read and written,
        # BF16 copies of the outputs written for the following GEMMs; 20 B per edge (sender index + geometry)
        if family == "edge_fwd":   # read phi16 6F, v16 6F, s 4F, v 12F; write s' 4F, v' 12F, s'16 2F, v'16 6F
            return E * (6 * K * F + 16 * F), N * 52 * F + E * 20
        if family == "edge_bwd":   # read phi16 6F, v16 6F, sb16 2F, vb16 6F, vb 12F; write phib16 6F, vb_in 12F
            return E * (12 * K * F + 60 * F), N * 50 * F + E * 20
        return None, None
    if prec == "fp32" and forces:
        # FP32 model with forces: the forward kernel also evaluates dw/dd and writes the edge tape (w, dw/dd: 24 F bytes
        # per edge); the reverse kernel reads the tape and does no filter arithmetic
        if family == "edge_fwd":
            return E * (12 * K * F + 16 * F), N * 11 * F * b + E * (eb + 24 * F)
        if family == "edge_bwd":
            return E * 60 * F, N * 16 * F * b + E * (eb + 24 * F)
    if family == "edge_fwd":
        return E * (6 * K * F + 16 * F), N * 11 * F * b + E * eb
    if family == "edge_bwd":
        return E * (12 * K * F + 60 * F), N * 16 * F * b + E * eb
    return None, None


def gemm_work(family: str, N: int, mc: gen.ModelCfg, prec: str, forces: bool):
    """(flops, bytes) per launch, averaged over the launches of one GEMM family in a step: 2 M N K flop; operands and
    result once (the SiLU GEMMs' stored pre-activation and the accumulating ones' read of C are not counted)."""
    F, T = mc.F, mc.T
    eb = 8 if prec == "fp64" else (2 if prec == "bf16" else 4)
    if family == "gemm_N":
        shapes = [(N, F, F), (N, 3 * F, F), (N, F, 2 * F), (N, 3 * F, F)] * T          # W1, W2, A1, A2
        if forces:
            shapes += [(N, F, 3 * F), (N, 2 * F, F)] * T + [(N, F, 3 * F), (N, F, F)] * (T - 1)
    elif family == "gemm_3N":
        shapes = [(3 * N, 2 * F, F)] * T + ([(3 * N, F, 2 * F)] * T if forces else [])  # U|V and its transpose
    else:
        return None, None, 0
    fl = sum(2.0 * m * n * k for m, n, k in shapes)
    by = sum(eb * (m * k + m * n + n * k) for m, n, k in shapes)
    return fl / len(shapes), by / len(shapes), len(shapes)


def measured_traffic(workload: str, family: str):
    """DRAM bytes per launch of the dominant kernel from the committed ncu capture (profiles/r01_traffic.csv), or None."""
    try:
        with open(os.path.join(ROOT, "profiles", "r01_traffic.csv")) as fh:
            for line in fh:
                q = line.strip().split(",")
                if len(q) >= 3 and q[0] == workload and q[1] == family:
                    return int(q[2])
    except Exception:
        pass
    return None


def run_reference(args, rank):
    """--impl reference: the CPU oracle, as it stands, on a bounded sample of the workload per step."""
    if rank != 0:
        return
    # torchrun exports OMP_NUM_THREADS=1 to every rank; the other ranks have exited, so the oracle gets the host's cores
    # here as it does in the N=1 launch (its OpenMP loops are unchanged: only the thread count is restored).
    if os.environ.get("TORCHELASTIC_RUN_ID") and os.environ.get("OMP_NUM_THREADS") == "1":
        try:
            import ctypes
            n_thr = len(os.sched_getaffinity(0))
            os.environ["OMP_NUM_THREADS"] = str(n_thr)
            ctypes.CDLL("libgomp.so.1").omp_set_num_threads(n_thr)
        except Exception:
            pass
    import oracle
    cfg_id, prec, forces, per_step = WORKLOADS[args.workload]
    mc = gen.model_cfg(cfg_id)
    n_sample = {1: 8, 2: 32, 3: 1, 4: 64, 5: 1}[cfg_id]
    b = gen.make_batch(cfg_id, 0, n_sample) if cfg_id != 5 else gen.make_batch(5, n_atoms=2000)
    w = gen.make_weights(mc, cfg_id)
    oracle.build()
    for _ in range(args.warmup):
        out = oracle.evaluate(mc, w, b, forces=forces)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        out = oracle.evaluate(mc, w, b, forces=forces)
    dt = time.perf_counter() - t0
    val = b.n_structs * args.steps / dt
    sample = (f"{b.n_structs} structures ({b.n_atoms} atoms, {out['n_edges']} directed edges) of "
              f"{WORKLOAD_NAMES[args.workload]} per step, FP64 oracle")
    line = dict(impl="reference", metric="painn_energy_force_structures_per_s", value=val, unit="structures/s",
                n_gpus=args.gpus, steps=args.steps, warmup=args.warmup, ms_per_step=1e3 * dt / args.steps,
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype="f64", data="synthetic",
                config=dict(workload=WORKLOAD_NAMES[args.workload], sample=sample),
                edges_per_s=out["n_edges"] * args.steps / dt,
                cpu_baseline=dict(value=val, unit="structures/s", cores=oracle.num_threads(), kind="oracle",
                                  sample=sample),
                e2e=dict(value=val, unit="structures/s", h2d_bytes_per_step=0, d2h_bytes_per_step=0))
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=50)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="cfg2", choices=sorted(WORKLOADS))
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-extra", action="store_true", help="skip the context timings of the other configs")
    args = ap.parse_args()
    args.warmup = max(args.warmup, 3) if args.impl == "b200" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.impl == "reference":
        run_reference(args, rank)
        return

    import torch
    import torch.distributed as dist
    import paper_2604_15380_b200 as pnn
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (there is no CPU fallback)"
    torch.cuda.set_device(local_rank)
    dev = torch.device("cuda", local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=dev)
    peaks = measured_peaks()

    def run_workload(name: str, steps: int, warmup: int, full: bool):
        cfg_id, prec, forces, per_step = WORKLOADS[name]
        c = gen.CONFIGS[cfg_id]
        mc = gen.model_cfg(cfg_id)
        S = per_step or c["S"]
        # weak scaling: rank r evaluates its own structures [r*S, (r+1)*S) of the same recipe
        b = gen.make_batch(cfg_id, rank * S, S)
        w = gen.make_weights(mc, cfg_id)
        deg_cap = 96 if cfg_id in (3, 5) else 40
        net = pnn.PaiNN(mc.F, mc.T, mc.K, mc.H, w, precision=prec, cutoff=mc.cutoff, Zmax=mc.Zmax,
                        norm_eps=mc.norm_eps, max_atoms=b.n_atoms, max_edges=b.n_atoms * deg_cap,
                        max_structs=b.n_structs, forces=forces)
        tt = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        d = dict(Z=tt(b.Z), pos=tt(b.pos), sp=tt(b.struct_ptr), head=tt(b.head), cell=tt(b.cell), pbc=tt(b.pbc))
        flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)  # 256 MB > 126 MB L2
        st = torch.cuda.current_stream()

        blended = name.endswith("_blended")
        if blended:
            # the composition -> softmax router runs on the device inside every step (Fig. 5)
            net.set_branch_mlp(gen.BRANCH_MLP_WIDTHS, gen.make_branch_mlp())

        def step():
            if blended:
                hw = net.branch_weights(d["Z"], d["sp"])
                return net.eval_blended(d["Z"], d["pos"], d["sp"], hw, d["cell"], d["pbc"], forces=forces,
                                        skip_below=0.01)
            return net.eval(d["Z"], d["pos"], d["sp"], d["head"], d["cell"], d["pbc"], forces=forces)

        for _ in range(warmup):
            flush.zero_()
            e, f = step()
        torch.cuda.synchronize()
        net.check()
        _, _, _, E = pnn.pnn_graph_view(net.ws)
        # ---- device-resident timing: L2 flushed (untimed) before every step, CUDA events on the launch stream
        ev = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
        sampler = ClockSampler(local_rank)
        if full:
            sampler.start()
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()
        l0 = net.launches
        t_wall0 = time.perf_counter()
        for a, z in ev:
            flush.zero_()
            a.record(st)
            e, f = step()
            z.record(st)
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
        t_wall = time.perf_counter() - t_wall0
        launches = net.launches - l0
        clocks = sampler.stop() if full else None
        ms = sum(a.elapsed_time(z) for a, z in ev)
        tmax = torch.tensor([ms], dtype=torch.float64, device=dev)
        tot = torch.tensor([float(b.n_structs), float(E), float(b.n_atoms)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
            dist.all_reduce(tot, op=dist.ReduceOp.SUM)
        ms = float(tmax.item())
        S_tot, E_tot, N_tot = (float(x) for x in tot.tolist())
        res = dict(name=name, prec=prec, forces=forces, mc=mc, batch=b, n_structs=S_tot, n_edges=E_tot, n_atoms=N_tot,
                   ms_per_step=ms / steps, structures_per_s=S_tot * steps / (ms * 1e-3),
                   edges_per_s=E_tot * steps / (ms * 1e-3), launches=launches, clocks=clocks, wall_s=t_wall,
                   ws_bytes=pnn.pnn_workspace_bytes(net.ws))
        if full:
            # ---- end to end through the host entry point: pinned host buffers, H2D + D2H inside the timed region
            pin = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
            hz, hp, hs, hh, hc, hb = pin(b.Z), pin(b.pos), pin(b.struct_ptr), pin(b.head), pin(b.cell), pin(b.pbc)
            eo = torch.empty(b.n_structs, dtype=net.out_dtype).pin_memory()
            fo = torch.empty((b.n_atoms, 3), dtype=net.out_dtype).pin_memory() if forces else None
            npv = lambda t_: None if t_ is None else t_.numpy()

            def step_host():
                net.eval_host(npv(hz), npv(hp), npv(hs), npv(hh), npv(hc), npv(hb), forces=forces,
                              energy_out=npv(eo), forces_out=npv(fo))

            for _ in range(warmup):
                step_host()
            ev2 = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(steps)]
            if world > 1:
                dist.barrier()
            torch.cuda.synchronize()
            for a, z in ev2:
                flush.zero_()
                a.record(st)
                step_host()
                z.record(st)
            torch.cuda.synchronize()
            ms2 = torch.tensor([sum(a.elapsed_time(z) for a, z in ev2)], dtype=torch.float64, device=dev)
            if world > 1:
                dist.all_reduce(ms2, op=dist.ReduceOp.MAX)
            h2d = sum(x.numel() * x.element_size() for x in (hz, hp, hs, hh, hc, hb) if x is not None)
            d2h = sum(x.numel() * x.element_size() for x in (eo, fo) if x is not None)
            res["e2e"] = dict(value=S_tot * steps / (float(ms2.item()) * 1e-3), unit="structures/s",
                              h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                              ms_per_step=float(ms2.item()) / steps)
            # ---- per-kernel-family CUDA-event timing (separate pass: the event pairs would perturb the step time)
            pnn.pnn_profile_enable(net.ws, True)
            for _ in range(steps):
                flush.zero_()
                step()
            prof = pnn.pnn_profile_read(net.ws)
            pnn.pnn_profile_enable(net.ws, False)
            res["profile"] = prof
        net.close()
        del flush
        torch.cuda.empty_cache()
        return res

    main_res = run_workload(args.workload, args.steps, args.warmup, full=True)
    mc, prec = main_res["mc"], main_res["prec"]
    N, E = int(main_res["n_atoms"] / world), int(main_res["n_edges"] / world)

    # roofline of the dominant kernel family
    kernels, tot_ms = {}, sum(v[0] for v in main_res["profile"].values())
    for fam, (ms, nl) in sorted(main_res["profile"].items(), key=lambda kv: -kv[1][0]):
        per = ms / max(nl, 1)
        kernels[fam] = dict(launches_per_step=nl / args.steps, ms_per_launch=per, share=ms / tot_ms)
    roof = None
    cand = [f for f in kernels if f.startswith("edge_") or f.startswith("gemm_")]
    if cand:
        fam = max(cand, key=lambda f: kernels[f]["share"])      # the dominant kernel family of the step
        per_s = kernels[fam]["ms_per_launch"] * 1e-3
        if fam.startswith("gemm_"):
            flops, byts, _ = gemm_work(fam, N, mc, prec, main_res["forces"])
        else:
            flops, byts = algorithmic_work(fam, N, E, mc, prec, main_res["forces"])
        if prec in ("fp32", "fp64"):
            ach, peak = flops / per_s / 1e12, ALU_PEAK_TFLOPS[prec]
            roof = dict(kernel=fam, bound="alu", achieved=ach, peak=peak, unit="TFLOP/s", frac=ach / peak,
                        traffic=measured_traffic(WORKLOAD_NAMES[args.workload], fam),
                        peak_source="derived: 148 SMs x lanes x 2 x 1.965 GHz (DESIGN.md)",
                        hbm_achieved_gbs=byts / per_s / 1e9, hbm_peak_gbs=peaks["hbm"], hbm_peak_source=peaks["source"])
            try:   # the nominal ALU peak is also measured on the box (FMA micro-benchmark)
                roof["alu_peak_measured"] = pnn.pnn_measure_alu_peak(pnn.PNN_FP64 if prec == "fp64" else pnn.PNN_FP32)
                roof["frac_of_measured_peak"] = ach / roof["alu_peak_measured"]
            except Exception as ex:
                roof["alu_peak_measured"] = None
        elif fam.startswith("gemm_"):
            ach = flops / per_s / 1e12
            roof = dict(kernel=fam, bound="tensor", achieved=ach, peak=peaks["bf16_sust"], unit="TFLOP/s",
                        frac=ach / peaks["bf16_sust"], traffic=measured_traffic(WORKLOAD_NAMES[args.workload], fam),
                        peak_source=peaks["source"] + " (sustained bf16)", algorithmic_bytes=byts)
        else:
            ach = byts / per_s / 1e9
            roof = dict(kernel=fam, bound="hbm", achieved=ach, peak=peaks["hbm"], unit="GB/s", frac=ach / peaks["hbm"],
                        traffic=measured_traffic(WORKLOAD_NAMES[args.workload], fam), peak_source=peaks["source"],
                        algorithmic_bytes=byts, tensor_flops=flops)
        # the runner-up family, for context (the two are within a few percent of the step on cfg2)
        others = sorted((f for f in cand if f != fam), key=lambda f: -kernels[f]["share"])
        if others and prec in ("fp32", "fp64"):
            f2 = others[0]
            fl2 = gemm_work(f2, N, mc, prec, main_res["forces"])[0] if f2.startswith("gemm_") else \
                algorithmic_work(f2, N, E, mc, prec, main_res["forces"])[0]
            if fl2:
                a2 = fl2 / (kernels[f2]["ms_per_launch"] * 1e-3) / 1e12
                roof["runner_up"] = dict(kernel=f2, achieved=a2, frac=a2 / ALU_PEAK_TFLOPS[prec],
                                         share_of_step=kernels[f2]["share"])
        roof["share_of_step"] = kernels[fam]["share"]

    line = dict(metric="painn_energy_force_structures_per_s", value=main_res["structures_per_s"], unit="structures/s",
                n_gpus=world, steps=args.steps, warmup=args.warmup, ms_per_step=main_res["ms_per_step"],
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype=DTYPE[prec], data="synthetic",
                config=dict(workload=WORKLOAD_NAMES[args.workload], structures_per_step=int(main_res["n_structs"]),
                            atoms_per_step=int(main_res["n_atoms"]), directed_edges_per_step=int(main_res["n_edges"]),
                            mean_degree=main_res["n_edges"] / max(main_res["n_atoms"], 1), F=mc.F, T=mc.T, K=mc.K,
                            H=mc.H, cutoff=mc.cutoff, outputs="energy+forces" if main_res["forces"] else "energy",
                            l2="flushed between timed steps (256 MB write)", parallelism=f"replica x{world}"),
                edges_per_s=main_res["edges_per_s"], clocks=main_res["clocks"], e2e=main_res["e2e"],
                gpu_launches=int(main_res["launches"]), roofline=roof, kernels=kernels,
                workspace_bytes=main_res["ws_bytes"])

    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        import oracle
        oracle.build()
        cfg_id, _, forces, _ = WORKLOADS[args.workload]
        # a bounded sample of the same workload, repeated until about 10 s of CPU work have been timed
        n_sample = {1: 8, 2: 256, 3: 2, 4: 512, 5: 1}[cfg_id]
        sb = gen.make_batch(cfg_id, 0, n_sample) if cfg_id != 5 else gen.make_batch(5, n_atoms=3000)
        wts = gen.make_weights(mc, cfg_id)
        oracle.evaluate(mc, wts, sb.select([0]), forces=forces)   # page in
        passes, t0 = 0, time.perf_counter()
        while True:
            o = oracle.evaluate(mc, wts, sb, forces=forces)
            passes += 1
            dt = time.perf_counter() - t0
            if dt >= 10.0 or passes >= 1000:
                break
        line["cpu_baseline"] = dict(value=passes * sb.n_structs / dt, unit="structures/s", cores=oracle.num_threads(),
                                    kind="oracle", edges_per_s=passes * o["n_edges"] / dt, seconds=dt,
                                    sample=f"{passes} passes over the first {sb.n_structs} structures ({sb.n_atoms} "
                                           f"atoms, {o['n_edges']} directed edges) of {WORKLOAD_NAMES[args.workload]}, "
                                           f"FP64 oracle")

    if not args.no_extra and world == 1:
        extra = {}
        for name in ("cfg1", "cfg2_blended", "cfg3_fp32", "cfg3_bf16", "cfg4", "cfg5"):
            if name == args.workload:
                continue
            try:
                r = run_workload(name, 5, 3, full=False)
                extra[WORKLOAD_NAMES[name]] = dict(ms_per_step=r["ms_per_step"], structures_per_s=r["structures_per_s"],
                                                   edges_per_s=r["edges_per_s"], atoms=int(r["n_atoms"]),
                                                   directed_edges=int(r["n_edges"]), launches_per_step=r["launches"] / 5)
            except Exception as ex:  # context only: never fail the headline line
                extra[WORKLOAD_NAMES[name]] = dict(error=str(ex)[:200])
        line["other_workloads"] = extra

    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
