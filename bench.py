#!/usr/bin/env python
"""bench.py — PaiNN energy+force throughput of the B200 path (BASELINE.json metric) on synthetic input.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg2|cfg3_fp32|cfg3_bf16|cfg4|cfg5|...]
                  [--impl reference] [--only-headline]

One step = one pass of the whole hot path (graph build + forward + analytic adjoint) over one batch.
Prints ONE JSON line (rank 0): the headline workload's contract keys plus `workloads`, one full record (>= 20 timed
steps, median of per-step CUDA-event times, clocks, per-kernel-family times, roofline of the dominant kernel family,
whole-step fraction of the SURVEY.md §8(d) roof, end-to-end leg) for each of BASELINE.json's configs: cfg2 FP32,
cfg3 FP32, cfg3 BF16, cfg4 BF16 (one resident batch, and the WHOLE 64-batch stream from pinned host memory through the
streaming driver), cfg5 FP64.  See DESIGN.md "Measurement" for every definition used here.
"""
from __future__ import annotations

import argparse
import dataclasses
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
    # the paper's own model settings and the second backbone on the cfg2 batch (context lines)
    "cfg2_pooled": (2, "fp32", True, None),
    "cfg2_cap20": (2, "fp32", True, None),
    "cfg2_schnet": (2, "fp32", True, None),
}
# model options that differ from the config's BASELINE.json model (gen.ModelCfg fields)
VARIANTS = {"cfg2_pooled": dict(head_type="pooled", head_d1=50, head_d2=776),
            "cfg2_cap20": dict(max_neighbors=20),
            "cfg2_schnet": dict(backbone="schnet")}
WORKLOAD_NAMES = {"cfg1": "cfg1_tiny_fp64", "cfg2": "cfg2_molecular_fp32", "cfg2_fp64": "cfg2_molecular_fp64",
                  "cfg2_blended": "cfg2_molecular_fp32_blended_heads",
                  "cfg3_fp32": "cfg3_crystals_fp32", "cfg3_bf16": "cfg3_crystals_bf16",
                  "cfg4": "cfg4_screening_bf16_batch16384", "cfg4_fp32": "cfg4_screening_fp32_batch16384",
                  "cfg5": "cfg5_large_fp64", "cfg2_pooled": "cfg2_molecular_fp32_pooled_heads_50_776",
                  "cfg2_cap20": "cfg2_molecular_fp32_max_neighbors_20", "cfg2_schnet": "cfg2_molecular_fp32_schnet"}
FULL_RECORDS = ("cfg2", "cfg3_fp32", "cfg3_bf16", "cfg4", "cfg5")   # BASELINE.json configs[1..4] (cfg3 in both precisions)
CFG4_STREAM_BATCHES = 64                                            # 1,048,576 structures / 16,384
STREAM_DEPTH = 2   # pipeline slots of the streaming driver (measured: 3 slots are not faster, 1.073 against 1.062 of resident)
DTYPE = {"fp64": "f64", "fp32": "f32", "bf16": "bf16"}
# plain-ALU peaks derived from the guide's unit counts and clocks:
# 148 SMs x 128 FP32 lanes x 2 flop x 1.965 GHz; FP64 at half the FP32 lane count.
ALU_PEAK_TFLOPS = {"fp32": 148 * 128 * 2 * 1.965e9 / 1e12, "fp64": 148 * 64 * 2 * 1.965e9 / 1e12}
TRAFFIC_FILE = os.path.join("profiles", "r02_traffic.csv")


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


# ------------------------------------------------------------------------------------------------ algorithmic work
def edge_work(family: str, N: int, E: int, mc: gen.ModelCfg, prec: str):
    """(flops, bytes) per LAUNCH of an edge kernel: what the METHOD requires (:461-469), not what the
    implementation chose to move.  flops: a4 6KF + 16F per edge, a7 12KF + 60F (filter value and derivative, the
    transposed contraction, the adjoint products); bytes: a4 N 11 F b + 20 E, a7 N 16 F b + 20 E (FP32 / FP64: b = 4 / 8);
    BF16 model (reading Q19: BF16 gathered payloads, FP32 residual and adjoint streams): a4 N 52 F + 20 E, a7 N 50 F + 20 E.
    The FP32 edge tape (24 F bytes per edge written by a4, read by a7) is NOT algorithmic: it appears in `traffic`."""
    F, K = mc.F, mc.K
    fl = E * (6 * K * F + 16 * F) if family == "edge_fwd" else E * (12 * K * F + 60 * F)
    if prec == "bf16":
        by = N * (52 if family == "edge_fwd" else 50) * F + 20 * E
    else:
        b = 8 if prec == "fp64" else 4
        by = N * (11 if family == "edge_fwd" else 16) * F * b + (4 + 4 * b) * E
    return float(fl), float(by)


def gemm_work(family: str, N: int, mc: gen.ModelCfg, prec: str, forces: bool):
    """(flops, bytes, launches) per launch, averaged over the launches of one GEMM family in a step: 2 M N K flop; operands
    and result once (the SiLU GEMMs' stored pre-activation and the accumulating ones' read of C are not counted)."""
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


def step_roof(N: int, E: int, mc: gen.ModelCfg, prec: str, forces: bool, peaks, alu_peak_tflops):
    """SURVEY.md §8(d) whole-step roof (the table at :474-480): forward flops T (30 F^2 N + (6KF + 16F) E) + (F^2 + F) N and
    compulsory bytes T (23 F b N + 20 E), x3 for energy + forces; t_roof = max over the applicable roofs (HBM; plain ALU
    for FP32 / FP64; BF16 tensor pipe for the BF16 model)."""
    F, T, K = mc.F, mc.T, mc.K
    b = {"fp64": 8, "fp32": 4, "bf16": 2}[prec]
    mult = 3 if forces else 1
    flops = mult * (T * (30.0 * F * F * N + (6 * K * F + 16 * F) * E) + (F * F + F) * N)
    byts = mult * T * (23.0 * F * b * N + 20.0 * E)
    gather = mult * T * 6.0 * F * b * E
    t_hbm = byts / (peaks["hbm"] * 1e9)
    if prec == "bf16":
        t_c, cname, cpeak = flops / (peaks["bf16_sust"] * 1e12), "tensor", peaks["bf16_sust"]
    else:
        t_c, cname, cpeak = flops / (alu_peak_tflops * 1e12), "alu", alu_peak_tflops
    binds = "hbm" if t_hbm >= t_c else cname
    return dict(flops=flops, compulsory_bytes=byts, gather_bytes=gather, t_hbm_ms=1e3 * t_hbm, t_compute_ms=1e3 * t_c,
                compute_roof=cname, compute_peak_tflops=cpeak, t_roof_ms=1e3 * max(t_hbm, t_c), binds=binds,
                t_hbm_if_all_gathers_miss_ms=1e3 * (byts + gather) / (peaks["hbm"] * 1e9))


def measured_traffic(workload: str, family: str):
    """(DRAM bytes per launch of a kernel family, source) from the committed ncu capture, or (None, None).  The number is
    a constant of that capture, not measured in this run: `traffic_source` says so."""
    try:
        with open(os.path.join(ROOT, TRAFFIC_FILE)) as fh:
            for line in fh:
                q = line.strip().split(",")
                if len(q) >= 4 and q[0] == workload and q[1] == family:
                    return int(q[2]), (f"{TRAFFIC_FILE}: ncu --set full capture of {','.join(q[3:])} (dram__bytes_read.sum + "
                                       "dram__bytes_write.sum; a constant of that capture, not measured in this run)")
    except Exception:
        pass
    return None, None


L2_PEAK_GBS = None   # measured once per run by pnn_measure_l2_peak (L2-resident reads, 512-byte rows per warp)


def gather_context(fam: str, per_s: float, E: int, mc, prec: str):
    """Context for the edge kernels, next to the SURVEY.md 8(d) roof: the sender rows a launch gathers (a4: phi_j and v_j,
    6 F payload elements per edge; a7 also the adjoint rows s-bar_j, v-bar_j, 4 F more) and the rate at which it does, against
    the measured bandwidth of L2-resident reads.  The rows are served by L1 and L2 (they are read deg times each), so this is
    not DRAM traffic and not the roof of the contract -- it shows how far a gather-bound kernel is from the cache it lives in."""
    pb = {"fp64": 8, "fp32": 4, "bf16": 2}[prec]
    ab = 8 if prec == "fp64" else 4
    g = E * mc.F * (6.0 * pb + (4.0 * ab if fam == "edge_bwd" else 0.0))
    out = dict(gather_bytes=g, gather_gbs=g / per_s / 1e9)
    if L2_PEAK_GBS:
        out["l2_peak_gbs_measured"] = L2_PEAK_GBS
        out["gather_frac_of_l2_peak"] = out["gather_gbs"] / L2_PEAK_GBS
    return out


def family_roofline(fam: str, per_s: float, N: int, E: int, mc, prec: str, forces: bool, peaks, wname: str,
                    alu_meas):
    r = _family_roofline(fam, per_s, N, E, mc, prec, forces, peaks, wname, alu_meas)
    if fam in ("edge_fwd", "edge_bwd"):
        r.update(gather_context(fam, per_s, E, mc, prec))
    return r


def _family_roofline(fam: str, per_s: float, N: int, E: int, mc, prec: str, forces: bool, peaks, wname: str,
                     alu_meas):
    if fam.startswith("gemm_"):
        flops, byts, _ = gemm_work(fam, N, mc, prec, forces)
    else:
        flops, byts = edge_work(fam, N, E, mc, prec)
    traffic, tsrc = measured_traffic(wname, fam)
    if prec in ("fp32", "fp64"):
        ach, peak = flops / per_s / 1e12, ALU_PEAK_TFLOPS[prec]
        r = dict(kernel=fam, bound="alu", achieved=ach, peak=peak, unit="TFLOP/s", frac=ach / peak, traffic=traffic,
                 traffic_source=tsrc, peak_source="derived: 148 SMs x lanes x 2 x 1.965 GHz (DESIGN.md)",
                 algorithmic_flops=flops, algorithmic_bytes=byts, hbm_achieved_gbs=byts / per_s / 1e9,
                 hbm_frac=byts / per_s / 1e9 / peaks["hbm"], hbm_peak_gbs=peaks["hbm"], hbm_peak_source=peaks["source"])
        if alu_meas:
            r["alu_peak_measured"] = alu_meas
            r["frac_of_measured_peak"] = ach / alu_meas
        if prec == "fp64":   # edge_dmma.cu / gemm_dmma.cu: the FP64 tensor instruction (DMMA) has the FP64 FMA peak
            r["pipe"] = "fp64 tensor path (mma.sync m8n8k4 f64) where F % 64 == 0; its measured peak equals the FP64 FMA peak (DESIGN.md section 6)"
        return r
    if fam.startswith("gemm_"):
        ach = flops / per_s / 1e12
        return dict(kernel=fam, bound="tensor", achieved=ach, peak=peaks["bf16_sust"], unit="TFLOP/s",
                    frac=ach / peaks["bf16_sust"], traffic=traffic, traffic_source=tsrc,
                    peak_source=peaks["source"] + " (sustained bf16)", algorithmic_flops=flops, algorithmic_bytes=byts,
                    hbm_achieved_gbs=byts / per_s / 1e9, hbm_frac=byts / per_s / 1e9 / peaks["hbm"])
    ach = byts / per_s / 1e9
    return dict(kernel=fam, bound="hbm", achieved=ach, peak=peaks["hbm"], unit="GB/s", frac=ach / peaks["hbm"],
                traffic=traffic, traffic_source=tsrc, peak_source=peaks["source"], algorithmic_bytes=byts,
                tensor_flops=flops)


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
    ap.add_argument("--no-extra", "--only-headline", dest="no_extra", action="store_true",
                    help="only the headline workload (skip the per-config records of the other configs)")
    ap.add_argument("--stream-batches", type=int, default=CFG4_STREAM_BATCHES)
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
    alu_meas = {}
    for pr, code in (("fp32", pnn.PNN_FP32), ("fp64", pnn.PNN_FP64)):
        try:   # the nominal ALU peak is also measured on the box (FMA micro-benchmark)
            alu_meas[pr] = pnn.pnn_measure_alu_peak(code)
        except Exception:
            alu_meas[pr] = None
    global L2_PEAK_GBS
    try:   # context for the gather-bound edge kernels (gather_context)
        L2_PEAK_GBS = pnn.pnn_measure_l2_peak()
    except Exception:
        L2_PEAK_GBS = None

    def run_workload(name: str, steps: int, warmup: int, full: bool):
        cfg_id, prec, forces, per_step = WORKLOADS[name]
        c = gen.CONFIGS[cfg_id]
        mc = dataclasses.replace(gen.model_cfg(cfg_id), **VARIANTS.get(name, {}))
        opts = dict(max_neighbors=mc.max_neighbors, head_type=mc.head_type, head_d1=mc.head_d1, head_d2=mc.head_d2,
                    backbone=mc.backbone)
        S = per_step or c["S"]
        # weak scaling: rank r evaluates its own structures [r*S, (r+1)*S) of the same recipe
        b = gen.make_batch(cfg_id, rank * S, S)
        w = gen.make_weights(mc, cfg_id)
        tt = lambda a: None if a is None else torch.from_numpy(np.ascontiguousarray(a)).to(dev)
        d = dict(Z=tt(b.Z), pos=tt(b.pos), sp=tt(b.struct_ptr), head=tt(b.head), cell=tt(b.cell), pbc=tt(b.pbc))
        # the workspace is sized from the batch's real edge count (a cheap graph-only pass with a generous bound), so that
        # the FP32 edge tape is as large as the workload needs and no larger
        deg_cap = 96 if cfg_id in (3, 5) else 40
        probe = pnn.PaiNN(mc.F, mc.T, mc.K, mc.H, w, precision=prec, cutoff=mc.cutoff, Zmax=mc.Zmax,
                          norm_eps=mc.norm_eps, max_atoms=b.n_atoms, max_edges=b.n_atoms * deg_cap,
                          max_structs=b.n_structs, forces=False, **dict(opts, max_neighbors=0))   # max_edges bounds the UNCAPPED count
        probe.build_graph(d["pos"], d["sp"], d["cell"], d["pbc"])
        _, _, _, E = pnn.pnn_graph_view(probe.ws)
        probe.close()
        del probe
        torch.cuda.empty_cache()
        max_edges = int(E * 1.02) + 1024
        net = pnn.PaiNN(mc.F, mc.T, mc.K, mc.H, w, precision=prec, cutoff=mc.cutoff, Zmax=mc.Zmax,
                        norm_eps=mc.norm_eps, max_atoms=b.n_atoms, max_edges=max_edges,
                        max_structs=b.n_structs, forces=forces, **opts)
        flush = torch.empty(256 * 1024 * 1024 // 4, dtype=torch.float32, device=dev)  # 256 MB > 126 MB L2
        st = torch.cuda.current_stream()

        blended = name.endswith("_blended")
        if blended:
            # the composition -> softmax router runs on the device inside every step (Fig. 5)
            net.set_branch_mlp(gen.BRANCH_MLP_WIDTHS, gen.make_branch_mlp())

        def step_eager():
            if blended:
                hw = net.branch_weights(d["Z"], d["sp"])
                return net.eval_blended(d["Z"], d["pos"], d["sp"], hw, d["cell"], d["pbc"], forces=forces,
                                        skip_below=0.01)
            return net.eval(d["Z"], d["pos"], d["sp"], d["head"], d["cell"], d["pbc"], forces=forces)

        # the timed step: graph build + evaluation replayed as ONE CUDA graph (pnn_eval_replay: same kernels, bit-identical
        # results, fixed output buffers); the blended pipeline has no recorded form and stays eager
        e_out = torch.empty(b.n_structs, dtype=net.out_dtype, device=dev)
        f_out = torch.empty((b.n_atoms, 3), dtype=net.out_dtype, device=dev) if forces else None

        def step():
            if blended:
                return step_eager()
            return net.eval_replay(d["Z"], d["pos"], d["sp"], d["head"], e_out, f_out, d["cell"], d["pbc"])

        for _ in range(warmup):
            flush.zero_()
            e, f = step()
        torch.cuda.synchronize()
        net.check()
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
        per_step_ms = [a.elapsed_time(z) for a, z in ev]
        # the same step launched kernel by kernel (pnn_build_graph + pnn_eval), a few steps, for comparison
        ev_e = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(min(steps, 10))]
        for a, z in ev_e:
            flush.zero_()
            a.record(st)
            step_eager()
            z.record(st)
        torch.cuda.synchronize()
        eager_ms = float(np.median([a.elapsed_time(z) for a, z in ev_e]))
        ms = sum(per_step_ms)
        tmax = torch.tensor([ms, float(np.median(per_step_ms))], dtype=torch.float64, device=dev)
        tot = torch.tensor([float(b.n_structs), float(E), float(b.n_atoms)], dtype=torch.float64, device=dev)
        if world > 1:
            dist.all_reduce(tmax, op=dist.ReduceOp.MAX)
            dist.all_reduce(tot, op=dist.ReduceOp.SUM)
        ms, med = float(tmax[0].item()), float(tmax[1].item())
        S_tot, E_tot, N_tot = (float(x) for x in tot.tolist())
        res = dict(name=name, prec=prec, forces=forces, mc=mc, batch=b, n_structs=S_tot, n_edges=E_tot, n_atoms=N_tot,
                   ms_per_step=ms / steps, ms_per_step_median=med, ms_per_step_min=min(per_step_ms), steps=steps,
                   structures_per_s=S_tot * steps / (ms * 1e-3), edges_per_s=E_tot * steps / (ms * 1e-3),
                   launches=launches, wall_s=t_wall, ws_bytes=pnn.pnn_workspace_bytes(net.ws), eager_ms=eager_ms,
                   launch_mode="eager" if blended else "CUDA graph replay (pnn_eval_replay)",
                   tape_bytes=pnn.pnn_workspace_edge_tape_bytes(net.ws))
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
            res["clocks"] = sampler.stop()
            ms2 = torch.tensor([sum(a.elapsed_time(z) for a, z in ev2)], dtype=torch.float64, device=dev)
            if world > 1:
                dist.all_reduce(ms2, op=dist.ReduceOp.MAX)
            h2d = sum(x.numel() * x.element_size() for x in (hz, hp, hs, hh, hc, hb) if x is not None)
            d2h = sum(x.numel() * x.element_size() for x in (eo, fo) if x is not None)
            res["e2e"] = dict(value=S_tot * steps / (float(ms2.item()) * 1e-3), unit="structures/s",
                              h2d_bytes_per_step=h2d, d2h_bytes_per_step=d2h,
                              ms_per_step=float(ms2.item()) / steps,
                              api="pnn_eval_host (pinned host buffers; H2D, graph build, evaluation, D2H, synchronise)")
            # ---- per-kernel-family CUDA-event timing (separate pass: the event pairs would perturb the step time)
            pnn.pnn_profile_enable(net.ws, True)
            for _ in range(steps):
                flush.zero_()
                step_eager()
            prof = pnn.pnn_profile_read(net.ws)
            pnn.pnn_profile_enable(net.ws, False)
            res["profile"] = prof
        res["net"] = net
        del flush
        return res

    def cfg4_stream(res, n_batches: int):
        """The WHOLE cfg4 stream (BASELINE.json configs[3]: 1,048,576 molecules in 64 batches of 16,384) from pinned host
        memory through the double-buffered streaming driver: host wall clock around submit ... drain."""
        net, mc = res["net"], res["mc"]
        S = 16384
        t_gen = time.perf_counter()
        try:
            import multiprocessing as mp
            with mp.get_context("spawn").Pool(min(16, os.cpu_count() or 1, n_batches)) as pool:
                batches = pool.starmap(gen.make_batch, [(4, (rank * n_batches + k) * S, S) for k in range(n_batches)])
        except Exception:
            batches = [gen.make_batch(4, (rank * n_batches + k) * S, S) for k in range(n_batches)]
        t_gen = time.perf_counter() - t_gen
        maxN = max(b.n_atoms for b in batches)
        pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
        hin = [(pin(b.Z), pin(b.pos), pin(b.struct_ptr), pin(b.head)) for b in batches]
        eo = [torch.empty(S, dtype=torch.float32).pin_memory() for _ in batches]
        sh = pnn.pnn_stream_create(net.model, maxN, int(maxN * 12.5), S, pnn.PNN_ENERGY, STREAM_DEPTH)
        try:
            def run(n):
                for k in range(n):
                    z, p, sp, h = hin[k]
                    pnn.pnn_stream_submit(sh, batches[k].n_atoms, S, z.numpy(), p.numpy(), sp.numpy(), h.numpy(), None,
                                          None, eo[k].numpy())
                pnn.pnn_stream_drain(sh)
            run(min(3, n_batches))                       # warm-up
            torch.cuda.synchronize()
            if world > 1:
                dist.barrier()
            l0 = pnn.pnn_stream_launch_count(sh)
            t0 = time.perf_counter()
            run(n_batches)
            dt = time.perf_counter() - t0
            if world > 1:   # replica streaming (P independent replicas): every rank streams its own
                tm = torch.tensor([dt], dtype=torch.float64, device=dev)   # batches; the job's time is the slowest rank's
                dist.all_reduce(tm, op=dist.ReduceOp.MAX)
                dt = float(tm.item())
            launches = pnn.pnn_stream_launch_count(sh) - l0
        finally:
            pnn.pnn_stream_destroy(sh)
        n_struct = S * n_batches * world
        h2d = sum(x.numel() * x.element_size() for hb in hin for x in hb)
        assert all(np.isfinite(e.numpy()).all() for e in eo)
        return dict(api=f"pnn_stream_submit / pnn_stream_drain (depth {STREAM_DEPTH}: one workspace and CUDA stream per slot, pinned host buffers)",
                    batches=n_batches * world, ranks=world, structures=n_struct, atoms=int(sum(b.n_atoms for b in batches)), seconds=dt,
                    structures_per_s=n_struct / dt, ms_per_batch=1e3 * dt / n_batches,
                    resident_ms_per_batch=res["ms_per_step_median"],
                    ratio_to_resident_batches=(1e3 * dt / n_batches) / res["ms_per_step_median"],
                    # the stream launches kernel by kernel (ragged batch sizes have no recorded form): against the resident
                    # batch launched the same way
                    resident_ms_per_batch_eager=res["eager_ms"],
                    ratio_to_resident_batches_eager=(1e3 * dt / n_batches) / res["eager_ms"],
                    h2d_bytes=h2d, d2h_bytes=4 * n_struct, gpu_launches=int(launches), input_generation_s=t_gen,
                    timing="host wall clock around submit ... drain after a device synchronise")

    def record(name: str, res) -> dict:
        """The full per-config record (the headline's contract keys are derived from the same dict)."""
        mc, prec, forces = res["mc"], res["prec"], res["forces"]
        N, E = int(res["n_atoms"] / world), int(res["n_edges"] / world)
        wname = WORKLOAD_NAMES[name]
        kernels, tot_ms = {}, sum(v[0] for v in res["profile"].values())
        for fam, (ms, nl) in sorted(res["profile"].items(), key=lambda kv: -kv[1][0]):
            kernels[fam] = dict(launches_per_step=nl / res["steps"], ms_per_launch=ms / max(nl, 1), share=ms / tot_ms)
        cand = [f for f in kernels if f.startswith("edge_") or f.startswith("gemm_")]
        roof, per_kernel = None, {}
        for fam in cand:
            per_kernel[fam] = family_roofline(fam, kernels[fam]["ms_per_launch"] * 1e-3, N, E, mc, prec, forces, peaks,
                                              wname, alu_meas.get(prec))
            per_kernel[fam]["share_of_step"] = kernels[fam]["share"]
        if prec == "fp32" and "edge_fwd" in per_kernel and "edge_bwd" in per_kernel and res["tape_bytes"]:
            # FP32 with the edge tape: the forward kernel also evaluates dw/dd (6KF of the reverse step's 12KF flop per edge)
            # and the reverse kernel streams it back, so each family's own fraction is skewed (reverse can exceed 1):
            # the pair is judged together
            fw, bw = per_kernel["edge_fwd"], per_kernel["edge_bwd"]
            t_pair = (kernels["edge_fwd"]["ms_per_launch"] + kernels["edge_bwd"]["ms_per_launch"]) * 1e-3
            ach = (fw["algorithmic_flops"] + bw["algorithmic_flops"]) / t_pair / 1e12
            note = ("edge tape: the forward kernel computes half of the reverse step's algorithmic flops; see "
                    "roofline_per_kernel['edge_fwd+edge_bwd']")
            fw["note"] = bw["note"] = note
            per_kernel["edge_fwd+edge_bwd"] = dict(kernel="edge_fwd+edge_bwd", bound="alu", achieved=ach, peak=fw["peak"],
                                                   unit="TFLOP/s", frac=ach / fw["peak"], peak_source=fw["peak_source"],
                                                   algorithmic_flops=fw["algorithmic_flops"] + bw["algorithmic_flops"],
                                                   share_of_step=kernels["edge_fwd"]["share"] + kernels["edge_bwd"]["share"])
        if cand:
            roof = per_kernel[max(cand, key=lambda f: kernels[f]["share"])]   # the dominant kernel family of the step
        sr = step_roof(N, E, mc, prec, forces, peaks, ALU_PEAK_TFLOPS.get(prec, 0.0))
        sr["frac"] = sr["t_roof_ms"] / res["ms_per_step_median"]
        out = dict(workload=wname, dtype=DTYPE[prec], outputs="energy+forces" if forces else "energy",
                   structures_per_step=int(res["n_structs"]), atoms_per_step=int(res["n_atoms"]),
                   directed_edges_per_step=int(res["n_edges"]), mean_degree=res["n_edges"] / max(res["n_atoms"], 1),
                   F=mc.F, T=mc.T, K=mc.K, H=mc.H, cutoff=mc.cutoff, steps=res["steps"],
                   ms_per_step=res["ms_per_step_median"], ms_per_step_mean=res["ms_per_step"],
                   ms_per_step_min=res["ms_per_step_min"], timing="median of per-step CUDA-event times, L2 flushed",
                   launch_mode=res["launch_mode"], ms_per_step_eager=res["eager_ms"],
                   structures_per_s=res["n_structs"] / (res["ms_per_step_median"] * 1e-3),
                   edges_per_s=res["n_edges"] / (res["ms_per_step_median"] * 1e-3), clocks=res.get("clocks"),
                   e2e=res.get("e2e"), gpu_launches_per_step=res["launches"] / res["steps"], roofline=roof,
                   roofline_per_kernel=per_kernel, step_roofline=sr, kernels=kernels,
                   workspace_bytes=res["ws_bytes"], edge_tape_bytes=res["tape_bytes"])
        return out

    def close(res):
        res["net"].close()
        res.pop("net")
        torch.cuda.empty_cache()

    main_res = run_workload(args.workload, args.steps, args.warmup, full=True)
    main_rec = record(args.workload, main_res)
    if args.workload == "cfg4" and not args.no_extra:
        main_rec["stream"] = cfg4_stream(main_res, args.stream_batches)
    close(main_res)
    mc, prec = main_res["mc"], main_res["prec"]

    line = dict(metric="painn_energy_force_structures_per_s", value=main_rec["structures_per_s"], unit="structures/s",
                n_gpus=world, steps=args.steps, warmup=args.warmup, ms_per_step=main_rec["ms_per_step"],
                higher_is_better=True, scaling="weak", vs_baseline=None, dtype=DTYPE[prec], data="synthetic",
                config=dict(workload=WORKLOAD_NAMES[args.workload], structures_per_step=main_rec["structures_per_step"],
                            atoms_per_step=main_rec["atoms_per_step"],
                            directed_edges_per_step=main_rec["directed_edges_per_step"],
                            mean_degree=main_rec["mean_degree"], F=mc.F, T=mc.T, K=mc.K, H=mc.H, cutoff=mc.cutoff,
                            outputs=main_rec["outputs"], l2="flushed between timed steps (256 MB write)",
                            timing="median of the per-step CUDA-event times", parallelism=f"replica x{world}",
                            launch=main_rec["launch_mode"], ms_per_step_eager=main_rec["ms_per_step_eager"]),
                edges_per_s=main_rec["edges_per_s"], clocks=main_rec["clocks"], e2e=main_rec["e2e"],
                gpu_launches=int(main_res["launches"]), roofline=main_rec["roofline"],
                roofline_per_kernel=main_rec["roofline_per_kernel"], step_roofline=main_rec["step_roofline"],
                kernels=main_rec["kernels"], workspace_bytes=main_rec["workspace_bytes"],
                edge_tape_bytes=main_rec["edge_tape_bytes"])

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
        # one full record per BASELINE.json config (per kernel per config the binding roof)
        recs = {WORKLOAD_NAMES[args.workload]: main_rec}
        for name in FULL_RECORDS:
            if name == args.workload:
                continue
            try:
                r = run_workload(name, 20, 3, full=True)
                rec = record(name, r)
                if name == "cfg4":
                    try:
                        rec["stream"] = cfg4_stream(r, args.stream_batches)
                    except Exception as ex:
                        rec["stream"] = dict(error=str(ex)[:300])
                close(r)
                recs[WORKLOAD_NAMES[name]] = rec
            except Exception as ex:  # never fail the headline line
                recs[WORKLOAD_NAMES[name]] = dict(error=str(ex)[:300])
        line["workloads"] = recs
        extra = {}
        for name in ("cfg1", "cfg2_blended", "cfg2_pooled", "cfg2_cap20", "cfg2_schnet"):   # context only: short timings
            try:
                r = run_workload(name, 5, 3, full=False)
                extra[WORKLOAD_NAMES[name]] = dict(ms_per_step=r["ms_per_step_median"],
                                                   structures_per_s=r["n_structs"] / (r["ms_per_step_median"] * 1e-3),
                                                   atoms=int(r["n_atoms"]), directed_edges=int(r["n_edges"]),
                                                   launches_per_step=r["launches"] / 5)
                close(r)
            except Exception as ex:
                extra[WORKLOAD_NAMES[name]] = dict(error=str(ex)[:200])
        line["other_workloads"] = extra

    if rank == 0:
        print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
