#!/usr/bin/env python
"""Benchmark of the BiP-PRISM on-atom contraction on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--workload cfg2] [--atoms A]

A *step* is one pass of the whole hot path (plane-loop driver, crop, de-tilt, NNW
reconstruction, probe GEMM, (.)H_n, detector GEMM, |a|^2 reduction) over one batch of ``--atoms`` ionised atoms of
the synthetic BASELINE.json configs[1] cell (512^2 grid, 40 slices, 300 kV, 25/40 mrad, parent factor 4, 9
channels, 48 x 48 windows, 64 x 64 scan, elemental-map output), all scan positions, channels and detector beams.
metric = scan-pos x atom x channel x detector-beam amplitudes per second.

  value   inputs resident in HBM, whole step timed on the device (CUDA events on the launching stream);
  e2e     the same through the host-buffer entry points: per step the edge (sites, H_n windows, detector beams,
          weight table) is copied host->device from pinned memory by bip_add_edge and the map is read back by
          bip_map_host;
  roofline  the detector-projection kernel (a7-a8, >= 90 % of the flops): algorithmic flops / its event time,
          against the fp32-equivalent ceiling of the arithmetic in use;
  cpu_baseline  the fp64 NumPy oracle, as it stands, on the host cores, on a bounded sample.

With N > 1 (torchrun) every rank runs the same step on its own atoms (independent problems, no data-path
collective): weak scaling, value = total amplitudes / max-over-ranks time.
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
sys.path.insert(0, os.path.join(ROOT, "tests"))

METRIC = "scan-pos x atom x channel x detector-beam amplitudes/s"
CONFIG_INDEX = {"cfg1": 0, "cfg2": 1, "cfg3": 2, "cfg4": 3, "cfg5": 4}
UNIT = "amplitudes/s"
SM_COUNT, FMA_LANES, = 148, 128


def load_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return d, "measured"
    return {"hbm_gbs": 6650.0, "bf16_tflops": 1590.0, "bf16_tflops_sustained": 1400.0, "sm_max_mhz": 1965.0}, "fallback"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "200"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.th = threading.Thread(target=self._read, daemon=True)
            self.th.start()
        except OSError:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append([x.strip() for x in line.split(",")])

    def stop(self):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
        self.th.join(timeout=2)
        sm = [float(r[0]) for r in self.rows if r and r[0].replace(".", "").isdigit()]
        mx = [float(r[1]) for r in self.rows if len(r) > 1 and r[1].replace(".", "").isdigit()]
        pw = [float(r[2]) for r in self.rows if len(r) > 2 and r[2].replace(".", "").isdigit()]
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(len(r) > 3 + k and r[3 + k].lower().startswith("active") for r in self.rows)]
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": max(mx) if mx else None,
                "power_w_max": max(pw) if pw else None, "samples": len(sm), "reasons": reasons}


def pinned(a: np.ndarray) -> np.ndarray:
    """Copy of ``a`` in page-locked host memory (numpy view of a pinned torch tensor)."""
    import torch
    t = torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    return t.numpy()


def shard_atoms(rank, atoms_per_rank, n_atoms_total):
    """Sites of rank ``rank``: a contiguous block of ``atoms_per_rank`` of the edge's slice-sorted site list (sites are
    independent problems, eq. 4/14: no data-path collective; weak scaling)."""
    lo = rank * atoms_per_rank
    return np.arange(min(lo, n_atoms_total), min(lo + atoms_per_rank, n_atoms_total))


def max_over_ranks(x, world, device="cuda"):
    """MAX all-reduce of one float over the job (the time every multi-GPU number is divided by)."""
    if world <= 1:
        return float(x)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def sample_sites(edge, rank, atoms, planes):
    """The sites of one step on rank ``rank``: ``atoms`` sites spread evenly over the first ``planes`` ionisation planes of
    the edge that hold sites ("atoms spread over planes"); inside a plane, rank r takes the r-th block of
    the plane's slice-sorted site list (sites are independent problems: no data-path collective)."""
    pl = np.unique(edge.slice)[: max(1, planes)]
    per = max(1, atoms // len(pl))
    idx = []
    for p in pl:
        of_plane = np.nonzero(edge.slice == p)[0]
        idx.extend(of_plane[shard_atoms(rank, per, len(of_plane))].tolist())
    return np.asarray(idx, dtype=np.int64)


def build_problem(args, rank):
    """Synthetic cell of the workload; every edge is sampled down to --atoms sites over its first --planes planes."""
    from bip_inputs.specimen import make_workload
    pf = (args.parent_factor, args.parent_factor) if args.parent_factor else None
    wl = make_workload(args.workload, scale=args.scale, parent_factor=pf)
    src = wl.edges if args.edges == "all" else wl.edges[:1]
    return wl, [e.take(sample_sites(e, rank, args.atoms, args.planes)) for e in src]


def run_ours(args):
    import torch
    import torch.distributed as dist
    import paper_2607_00756_b200 as B

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    assert world == args.gpus, f"--gpus {args.gpus} but WORLD_SIZE = {world}"
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (libbip has no CPU path)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    peaks, peak_src = load_peaks()
    prec = {"fp16x4": B.PREC_FP16X4, "fp16x3": B.PREC_FP16X3, "bf16x6": B.PREC_BF16X6, "tf32x3": B.PREC_TF32X3, "fp32_simt": B.PREC_FP32_SIMT}[args.precision]
    recon = {"linear": B.RECON_LINEAR, "magphase": B.RECON_MAGPHASE}[args.recon]

    mode = {"map": B.MODE_MAP, "qeels_x": B.MODE_QEELS_X, "cube": B.MODE_CUBE}[args.mode]
    wl, edges = build_problem(args, rank)
    edge = edges[0]
    g = B.Grid(wl.ny, wl.nx, wl.ly, wl.lx, wl.nz, wl.dz, wl.lam)
    geo = B.plan_geometry(g, wl.alpha_mrad, edge.det_mrad, wl.defocus, wl.parent_factor, prism=wl.prism)
    T_dev = torch.from_numpy(wl.T).cuda()
    ctx = B.Context(g, T_dev, geo.ap_h, geo.ap_c, geo.p1_h, geo.w1, geo.p2_h)
    if args.precision == "tf32x3":
        ctx.allow_tf32x3(True)                       # the A/B arithmetic: misses the 1e-6 summed bound (include/bip.h)
    ctx.build_S1()
    ctx.build_S2()
    ctx.set_scan(wl.scan)
    crop = (args.crop, args.crop) if args.crop else wl.crop
    ctx.set_crop(*crop)                              # PRISM crop mask of the workload ((1, 1) = none)
    ctx.set_association({"probe": B.ASSOC_PROBE, "coupling": B.ASSOC_COUPLING, "auto": B.ASSOC_AUTO}[args.assoc])
    eids = [ctx.add_edge(e.slice, e.centre, e.H, geo.det_h, geo.w2) for e in edges]
    torch.cuda.synchronize()
    t_build = ctx.get_timing()
    K = geo.det_h.shape[0]
    outs = [None]
    n_planes = len(set(int(s_) for e in edges for s_ in e.slice))

    def step():
        # one plane loop shared by all registered edges: the cursor walks forward through the sampled planes
        # (ADVANCETO / PEELTO inside the step) and goes back to the first of them at the start of the next step
        outs[0] = ctx.map_all(mode, recon, prec)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    for _ in range(args.warmup):
        step()
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    gemm2_ms, gemm2_launches, contract_ms, adv_ms, launches = 0.0, 0, 0.0, 0.0, 0
    barrier()
    torch.cuda.profiler.start()                      # ncu --profile-from-start off captures the timed steps only
    ev0.record()
    for _ in range(args.steps):
        step()
        t = ctx.get_timing()                         # synchronises; the spans are device event times
        gemm2_ms += t["gemm2_ms"]; gemm2_launches += t["gemm2_launches"]; contract_ms += t["contract_ms"]
        adv_ms += t["advance_peel_ms"]; launches += t["kernel_launches"]
    ev1.record()
    barrier()
    torch.cuda.profiler.stop()
    clocks = sampler.stop() if rank == 0 else None
    ms_total = ev0.elapsed_time(ev1)
    ms_total = max_over_ranks(ms_total, world)
    amps_step = float(ctx.get_timing()["amplitudes"])          # scan rows actually contracted (crop mask) x channels x beams
    value = amps_step * world * args.steps / (ms_total * 1e-3)
    map_dev = outs[0][0].cpu().numpy()
    out_bytes = sum(o.numel() * o.element_size() for o in outs[0])

    # ---- end to end through the host-buffer API: pinned inputs in, map out, every step ----
    h_edges = [(pinned(e.slice), pinned(e.centre), pinned(e.H)) for e in edges]
    h_det, h_idx, h_w = pinned(geo.det_h), pinned(geo.w2[0]), pinned(geo.w2[1])
    h2d = sum(sum(a.nbytes for a in he) + 2 * 4 * he[0].shape[0] + sum(a.nbytes for a in (h_det, h_idx, h_w)) + 2 * 4 * K for he in h_edges)
    d2h = out_bytes

    def step_e2e():
        ctx.clear_edges()
        ids = [ctx.add_edge(hs, hc, hH, h_det, (h_idx, h_w)) for hs, hc, hH in h_edges]
        res = [ctx.map_host(i, mode, recon, prec) for i in ids]     # the host-buffer entry point serves one edge per call
        return res[0]

    step_e2e()
    barrier()
    t0 = time.perf_counter()
    e2e_steps = max(1, min(args.steps, 3))
    for _ in range(e2e_steps):
        m_host = step_e2e()
    barrier()
    e2e_s = time.perf_counter() - t0
    e2e_s = max_over_ranks(e2e_s, world)
    e2e_value = amps_step * world * e2e_steps / e2e_s
    # the host-buffer path must reproduce the device path: same kernels on the same inputs.  MAP accumulates in fp64 (order-free to
    # ~1e-12); QEELS / CUBE accumulate with fp32 REDs whose order differs from run to run, and the plane cursor has walked S2 back
    # and forth a few more times (one c64 rounding per slice step), and eq. 11 divides by |sum_p w_p D_p|, which amplifies those roundings where the parents nearly cancel (7.9e-5 measured at
    # parent factor 8): those are held to 5e-4 of the brightest element -- a sanity check, parity is tests/test_gpu_parity*.py
    e2e_diff = float(np.abs(m_host - map_dev).max() / np.abs(map_dev).max())
    assert e2e_diff <= (1e-5 if args.mode == "map" else 5e-4), f"host-buffer path disagrees with the device path: {e2e_diff:.3e} of the maximum"

    # ---- roofline of the dominant kernel (a7-a8) ----
    flops_gemm2_step = 8.0 * edge.W * edge.W * amps_step          # a7: 8 W^2 real flops per amplitude (every edge here has the same W)
    n_b = geo.ap_h.shape[0]
    rows_total = amps_step / (K * sum(e.n_ch for e in edges) / len(edges)) if len(edges) == 1 else None
    assoc_ran = "probe"
    if args.assoc != "probe" and rows_total is not None:
        # which association the library ran (AUTO decides per edge): its flop count tells -- probe-first counts
        # 8 W^2 (rows B + amplitudes), the coupling association 8 N_ch K B (sites W^2 + rows)
        probe_flops = 8.0 * edge.W * edge.W * (rows_total * n_b + amps_step)
        if abs(float(ctx.get_timing()["flops"]) - probe_flops) > 1e-6 * probe_flops:
            assoc_ran = "coupling"
            flops_gemm2_step = 8.0 * n_b * amps_step               # the timed kernel is then a = A M^T: 8 B real flops per amplitude
    achieved = flops_gemm2_step * args.steps / (gemm2_ms * 1e-3) / 1e12 if gemm2_ms > 0 else 0.0
    n_sites_step = sum(e.n_atoms for e in edges)
    if args.precision in ("fp16x4", "fp16x3", "bf16x6"):
        # a kernel timed inside a seconds-long step under the power cap: the SUSTAINED measured tensor rate is the
        # denominator (B200_PROFILING.md); the fraction of the burst figure is printed beside it
        sus, burst = peaks["bf16_tflops_sustained"], peaks["bf16_tflops"]
        nprod = {"fp16x4": 4, "fp16x3": 3, "bf16x6": 6}[args.precision]
        roof = {"bound": "tensor", "achieved": achieved, "peak": sus / nprod, "unit": "TFLOP/s",
                "frac": achieved / (sus / nprod), "frac_burst": achieved / (burst / nprod), "traffic": None, "kernel": "k_sliced_contract<2>",
                "note": f"fp32-equivalent flops; the sliced 16-bit split issues {nprod} fp16/bf16 tensor flops per flop: ceiling = "
                        f"sustained bf16 rate {sus:.0f} / {nprod} of {peak_src} (fp16 = bf16 rate; burst figure {burst:.0f}: frac_burst); "
                        f"the denominators are cuBLAS measurements, so a fraction a little above 1 is possible; issued tensor rate "
                        f"{nprod * achieved:.1f} TFLOP/s",
                "avg_launch_ms": gemm2_ms / max(gemm2_launches, 1), "launches": gemm2_launches}
    elif args.precision == "tf32x3":
        tf32_peak = peaks["bf16_tflops_sustained"] * (1.1 / 2.25)          # nominal tf32 : bf16 ratio (B200_PROFILING.md)
        roof = {"bound": "tensor", "achieved": achieved, "peak": tf32_peak / 3.0, "unit": "TFLOP/s",
                "frac": achieved / (tf32_peak / 3.0), "traffic": None, "kernel": "k_gemm2_tc",
                "note": f"fp32-equivalent flops; 3xTF32 issues 3 tensor flops per flop: ceiling = tf32 peak {tf32_peak:.0f} / 3 "
                        f"(bf16 sustained x 1.1/2.25, {peak_src}); issued tensor rate {3 * achieved:.1f} TFLOP/s",
                "avg_launch_ms": gemm2_ms / max(gemm2_launches, 1), "launches": gemm2_launches}
    else:
        alu_peak = SM_COUNT * FMA_LANES * 2 * peaks.get("sm_max_mhz", 1965.0) * 1e6 / 1e12
        roof = {"bound": "alu", "achieved": achieved, "peak": alu_peak, "unit": "TFLOP/s", "frac": achieved / alu_peak,
                "traffic": None, "kernel": "k_gemm2_simt",
                "note": "fp32 FMA peak = 148 SMs x 128 lanes x 2 x max SM clock (reference CUDA-core path)",
                "avg_launch_ms": gemm2_ms / max(gemm2_launches, 1), "launches": gemm2_launches}
    # bytes per launch of the dominant kernel.  algorithmic_bytes is SURVEY 8(d)'s figure: the parent windows the method
    # itself has to read, (B_p1 + B_p2) W^2 8 per site, plus the output; operand_bytes is what THIS design streams into the
    # kernel (the materialised sliced operands Phi and R2); traffic is ncu's dram__bytes of the same kernel at the same
    # launch shape, from the committed capture named in traffic_source (regenerated whenever kernel or shape change).
    atoms_launch = n_sites_step * args.steps / max(gemm2_launches, 1)
    roof["algorithmic_bytes"] = atoms_launch * 8.0 * edge.W * edge.W * (ctx.n_p1 + ctx.n_p2) + out_bytes
    roof["operand_bytes"] = atoms_launch * 8.0 * edge.W * edge.W * (ctx.n_rho * edge.n_ch + K)
    traffic_file = os.path.join(ROOT, "profiles", "r02_gemm2_traffic.txt")
    if os.path.exists(traffic_file) and args.precision == "fp16x4" and args.workload == "cfg2" and args.mode == "map":
        kv = dict(l.split(None, 1) for l in open(traffic_file).read().splitlines() if l.strip() and not l.startswith("#"))
        roof["traffic"] = (float(kv["dram_bytes_read"]) + float(kv["dram_bytes_write"])) * atoms_launch / float(kv["atoms_per_launch"])
        roof["traffic_unit"] = "bytes per launch (ncu dram__bytes_read.sum + dram__bytes_write.sum, scaled to this launch's sites)"
        roof["traffic_source"] = f"profiles/r02_gemm2_traffic.txt, captured at commit {kv.get('commit', '?').strip()} ({kv.get('command', '?').strip()})"

    line = None
    if rank == 0:
        cpu = cpu_baseline(args) if world == 1 and not args.no_cpu_baseline else None
        extra = extra_legs(args) if world == 1 else None
        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
            "ms_per_step": ms_total / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
            "dtype": {"fp16x4": "fp16x4(c64)", "fp16x3": "fp16x3(c64)", "bf16x6": "bf16x6(c64)", "tf32x3": "tf32x3(c64)", "fp32_simt": "f32(c64)"}[args.precision], "data": "synthetic",
            "config": {"workload": f"BASELINE configs[{CONFIG_INDEX.get(args.workload, '?')}] ({wl.name}): {wl.ny}x{wl.nx} grid, {wl.nz} slices, "
                                   f"B={geo.ap_h.shape[0]}, K={K}, parents=({ctx.n_p1},{ctx.n_p2}), parent factor {wl.parent_factor[0]:g}, "
                                   f"W={edge.W}, N_ch={[e.n_ch for e in edges]}, N_rho={ctx.n_rho}, {args.mode} output, recon={args.recon}",
                       "association": args.assoc, "association_ran": assoc_ran, "crop_mask": list(crop),
                       "atoms_per_step_per_gpu": [e.n_atoms for e in edges], "planes_per_step": n_planes,
                       "sampled": f"sites spread evenly over the first {args.planes} ionisation plane(s) of each edge; the plane cursor walks "
                       f"through them inside the step; the full edges have {[e.n_atoms for e in (wl.edges if args.edges == 'all' else wl.edges[:1])]} sites",
                       "precision": args.precision,
                       "l2": "per-step working set (sliced operands, > 0.5 GB per atom, rewritten every step) exceeds the 126 MB L2: no flush needed",
                       "parallelism": f"atoms sharded over {world} GPU(s), no data-path collective"},
            "clocks": clocks, "gpu_launches": launches,
            "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
                    "steps": e2e_steps, "max_abs_diff_vs_device_path_rel": e2e_diff},
            "roofline": roof,
            "phases_ms_per_step": {"contract": contract_ms / args.steps, "gemm2": gemm2_ms / args.steps,
                                   "advance_peel": adv_ms / args.steps, "build_s1_once": t_build["build_s1_ms"],
                                   "build_s2_once": t_build["build_s2_ms"]},
            "fp32_equiv_tflops_contract": float(ctx.get_timing()["flops"]) * 1.0 / (contract_ms / args.steps * 1e-3) / 1e12 if contract_ms else None,
            "cpu_baseline": cpu,
        }
        if extra:
            line["extra"] = extra
        print(json.dumps(line))
    ctx.close()
    if world > 1:
        dist.destroy_process_group()
    return line


def run_alg3(args):
    """NEXT-3 leg: Algorithm 3 (bip_cube_alg3; S1-partitioned cube on all G exit beams, per-scan exit multislice) on --atoms
    sites of the workload.  One JSON line; amplitudes = scan positions x sites x channels x G exit beams."""
    import torch
    import paper_2607_00756_b200 as B
    assert torch.cuda.is_available()
    wl, edges = build_problem(args, 0)
    edge = edges[0]
    g = B.Grid(wl.ny, wl.nx, wl.ly, wl.lx, wl.nz, wl.dz, wl.lam)
    geo = B.plan_geometry(g, wl.alpha_mrad, edge.det_mrad, wl.defocus, wl.parent_factor, prism=wl.prism)
    ctx = B.Context(g, torch.from_numpy(wl.T).cuda(), geo.ap_h, geo.ap_c, geo.p1_h, geo.w1, geo.p2_h)
    ctx.build_S1()
    ctx.set_scan(wl.scan)
    ctx.add_edge(edge.slice, edge.centre, edge.H, geo.det_h, geo.w2)
    recon = {"linear": B.RECON_LINEAR, "magphase": B.RECON_MAGPHASE}[args.recon]
    out = torch.empty((ctx.n_rho, wl.ny, wl.nx), dtype=torch.float32, device="cuda")
    for _ in range(args.warmup):
        ctx.cube_alg3(0, recon, B.PREC_FP16X4, out=out)
    torch.cuda.synchronize()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    ev0.record()
    adv = con = 0.0
    for _ in range(args.steps):
        ctx.cube_alg3(0, recon, B.PREC_FP16X4, out=out)
        t = ctx.get_timing()
        adv += t["advance_peel_ms"]; con += t["contract_ms"]
    ev1.record()
    torch.cuda.synchronize()
    ms = ev0.elapsed_time(ev1) / args.steps
    amps = float(ctx.n_rho) * edge.n_atoms * edge.n_ch * wl.ny * wl.nx
    slices_below = float(np.mean(wl.nz - edge.slice))
    G = wl.ny * wl.nx
    line = {"metric": METRIC.replace("detector-beam", "exit-beam"), "value": amps / (ms * 1e-3), "unit": UNIT, "n_gpus": 1, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": ms, "higher_is_better": True, "dtype": "f32(c64) wavefields, fp16x4 probe contraction", "data": "synthetic",
            "config": {"workload": f"Algorithm 3 on BASELINE configs[{CONFIG_INDEX.get(args.workload, '?')}] ({wl.name}): {wl.ny}x{wl.nx} grid, {wl.nz} slices, "
                                   f"B={geo.ap_h.shape[0]}, parents={ctx.n_p1}, W={edge.W}, N_ch={edge.n_ch}, N_rho={ctx.n_rho}, all {G} exit beams",
                       "atoms_per_step": edge.n_atoms, "mean_slices_to_exit": slices_below},
            "phases_ms_per_step": {"s1_advance": adv / args.steps, "probe_exit_detect": con / args.steps},
            "wavefield_slice_steps_per_s": ctx.n_rho * edge.n_atoms * edge.n_ch * slices_below * args.steps / (con * 1e-3) if con else None,
            "hbm_GBps_of_slice_steps": (ctx.n_rho * edge.n_atoms * edge.n_ch * slices_below * G * 48.0 * args.steps / (con * 1e-3) / 1e9) if con else None}
    print(json.dumps(line))
    ctx.close()
    return line


def extra_legs(args):
    """Short legs on other BASELINE.json configs, each in a fresh process, embedded under "extra" of the main line (the driver
    parses the LAST line, which stays configs[1]).  Default: configs[3] in the paper's own regime (FePt nanoparticle, PRISM
    f = 8 beam lists + crop mask), the FP16X3 arithmetic on the default workload, Algorithm 3 on the
    configs[4] geometry, and configs[2] (five edges in one plane loop, the largest config that fits one GPU)."""
    out = {}
    for spec in [x for x in args.extra.split(",") if x and x != "none"]:
        name, _, n = spec.partition(":")
        base = [sys.executable, os.path.abspath(__file__), "--steps", "2", "--warmup", "1", "--no-cpu-baseline", "--extra", "none"]
        if name == "fp16x3":        # the three-product arithmetic (reduced outputs only) on the default workload
            cmd = base + ["--precision", "fp16x3", "--atoms", n or "16", "--planes", "2"]
        elif name == "alg3":        # NEXT-3: Algorithm 3 on the configs[4] geometry
            cmd = base + ["--workload", "cfg5", "--mode", "cube_alg3", "--atoms", n or "2", "--planes", "1"]
        elif name == "cfg3":        # five edges in one plane loop, the largest config that fits one GPU
            cmd = base + ["--workload", "cfg3", "--edges", "all", "--atoms", n or "2", "--planes", "1"]
        else:
            cmd = base + ["--workload", name, "--atoms", n or "256", "--planes", "8", "--assoc", "auto"]
        try:
            r = subprocess.run(cmd, capture_output=True, text=True, timeout=900, env=dict(os.environ, WORLD_SIZE="1", RANK="0", LOCAL_RANK="0"))
            lines = [l for l in r.stdout.splitlines() if l.startswith("{")]
            d = json.loads(lines[-1]) if r.returncode == 0 and lines else None
        except Exception as ex:                      # a leg that fails must not take the main line with it
            d, r = None, None
            out[name] = {"error": repr(ex)[:200]}
            continue
        if d is None:
            out[name] = {"error": (r.stderr or r.stdout)[-300:]}
            continue
        if name == "alg3":
            out[name] = {k: d[k] for k in ("value", "unit", "ms_per_step", "config", "phases_ms_per_step", "wavefield_slice_steps_per_s", "hbm_GBps_of_slice_steps")}
            continue
        out[name] = {"value": d["value"], "unit": d["unit"], "dtype": d["dtype"], "e2e": d["e2e"]["value"], "ms_per_step": d["ms_per_step"], "workload": d["config"]["workload"],
                     "association_ran": d["config"]["association_ran"], "crop_mask": d["config"]["crop_mask"],
                     "atoms_per_step": d["config"]["atoms_per_step_per_gpu"], "phases_ms_per_step": d["phases_ms_per_step"],
                     "roofline_frac": d["roofline"]["frac"], "gemm2_tflops_fp32_equiv": d["roofline"]["achieved"], "clocks": d["clocks"]}
    return out or None


def oracle_sample_setup(args, n_scan=256):
    """The bounded sample timed on the host cores (tests/helpers.OracleSample): ONE atom of the same cell geometry
    (same grid, beams, parents, window, channels, all detector beams), a regular subset of ``n_scan`` scan positions,
    slab truncated to its first two slices so that the (untimed) fp64 parent windows are cheap to build."""
    from helpers import OracleSample
    return OracleSample(args.workload, scale=args.scale, nz=2, n_atoms=1, n_scan=n_scan)


def oracle_sample_run(smp, recon):
    return smp.run(recon)["map"]


def _threads():
    try:
        from threadpoolctl import threadpool_info
        n = [p["num_threads"] for p in threadpool_info() if p.get("user_api") == "blas"]
        return max(n) if n else os.cpu_count()
    except Exception:
        return os.cpu_count()


def cpu_baseline(args):
    smp = oracle_sample_setup(args)
    wl, e, orc, A = smp.wl, smp.e, smp.orc, smp.A
    t0 = time.perf_counter()
    m = oracle_sample_run(smp, args.recon)
    dt = time.perf_counter() - t0
    amps = float(A.shape[0]) * 1 * e.n_ch * len(orc.det)
    return {"value": amps / dt, "unit": UNIT, "cores": _threads(), "host_cpus": os.cpu_count(), "kind": "oracle", "seconds": dt,
            "sample": f"1 atom x {A.shape[0]} scan positions x {e.n_ch} channels x {len(orc.det)} detector beams of the same cell "
                      f"(slab truncated to 2 slices for the untimed window build); steps a1-a8, NumPy complex128",
            "map_sum": float(m.sum())}


def run_reference(args):
    """The oracle as it stands, timed on the host cores (this tier's reference arm)."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return None
    smp = oracle_sample_setup(args, n_scan=64)          # ~5 s of host work per step: a 20-step run ends within minutes
    wl, e, orc, A = smp.wl, smp.e, smp.orc, smp.A
    for _ in range(min(args.warmup, 1)):
        oracle_sample_run(smp, args.recon)
    t0 = time.perf_counter()
    for _ in range(args.steps):
        oracle_sample_run(smp, args.recon)
    dt = time.perf_counter() - t0
    amps = float(A.shape[0]) * e.n_ch * len(orc.det)
    v = amps * args.steps / dt
    sample = (f"each step: 1 atom x {A.shape[0]} scan positions x {e.n_ch} channels x {len(orc.det)} detector beams of "
              f"BASELINE configs[1] geometry (slab truncated to 2 slices for the untimed fp64 window build)")
    line = {"impl": "reference", "metric": METRIC, "value": v, "unit": UNIT, "n_gpus": int(os.environ.get("WORLD_SIZE", "1")),
            "steps": args.steps, "warmup": min(args.warmup, 1), "ms_per_step": dt / args.steps * 1e3, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64(c128)", "data": "synthetic",
            "config": {"workload": f"BASELINE configs[1] ({wl.name}) sampled", "sample": sample, "recon": args.recon},
            "cpu_baseline": {"value": v, "unit": UNIT, "kind": "oracle", "cores": _threads(), "sample": sample},
            "e2e": {"value": v, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}, "gpu_launches": 0}
    print(json.dumps(line))
    return line


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=3)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="cfg2")
    ap.add_argument("--scale", type=int, default=1, help="shrink cells and grid together (debug; 1 = BASELINE size)")
    ap.add_argument("--atoms", type=int, default=32, help="ionised atoms per step per GPU (per edge)")
    ap.add_argument("--planes", type=int, default=2, help="ionisation planes the atoms of a step are spread over")
    ap.add_argument("--precision", default=os.environ.get("BIP_BENCH_PRECISION", "fp16x4"), choices=["fp16x4", "fp16x3", "bf16x6", "tf32x3", "fp32_simt"])
    ap.add_argument("--recon", default="magphase", choices=["linear", "magphase"])
    ap.add_argument("--mode", default="map", choices=["map", "qeels_x", "cube", "cube_alg3"])
    ap.add_argument("--edges", default="first", choices=["first", "all"], help="all: every edge of the workload shares one plane loop (configs[2])")
    ap.add_argument("--parent-factor", type=float, default=0.0, help="override the workload's parent factor (configs[4] sweeps 1/2/4/8)")
    ap.add_argument("--assoc", default="probe", choices=["probe", "coupling", "auto"], help="association of the contraction (bip_set_association)")
    ap.add_argument("--crop", type=int, default=0, help="override the workload's crop-mask factor (0 = the workload's own)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--extra", default=None, help="comma list of short extra legs embedded under 'extra' (workload[:atoms]); default cfg4:256 for "
                    "the default workload, none otherwise")
    args = ap.parse_args()
    if args.extra is None:
        args.extra = "cfg4:256,fp16x3:16,alg3:2,cfg3:2" if args.workload == "cfg2" and args.scale == 1 and args.precision == "fp16x4" else "none"
    if args.impl == "reference":
        run_reference(args)
        return
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        # plain `python bench.py --gpus N`: launch the N ranks ourselves, one per GPU (same command line the driver uses)
        import socket
        with socket.socket() as sk:
            sk.bind(("127.0.0.1", 0))
            port = sk.getsockname()[1]
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}", "--master-addr", "127.0.0.1",
               "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        sys.exit(subprocess.call(cmd))
    if args.mode == "cube_alg3":
        run_alg3(args)
        return
    if world != args.gpus:
        sys.exit(f"bench.py: --gpus {args.gpus} does not match WORLD_SIZE = {world} (launch with torchrun --nproc-per-node {args.gpus})")
    run_ours(args)


if __name__ == "__main__":
    main()
