#!/usr/bin/env python
"""bench.py — one JSON line for the fused gradient iteration of tensor tomography on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C5] [--impl ours|reference]

A step = one pass of the whole hot path (Joseph forward + basis map + residual +
weighted loss + basis^T + exact adjoint) over one synthetic data set, i.e. one `mm_loss_gradient` call.
Workload at N=1: BASELINE.json configs[4] ("C5": 256^3 voxels, l_max=8 -> K=45, 360 projections, 256^2 pixels,
D=8), the configuration the metric is quoted on; inputs (3.2 GB volume) exceed the 126 MB L2, so no flush.
The path does not shard inside the library (BASELINE.json north_star: one GPU, no collectives): --gpus N runs
N independent replicas ("replicas only") and reports the aggregate.

`--impl reference` times the CPU oracle (oracle/, test infrastructure) on a bounded sample of the same workload.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

from paper_2504_16446_b200 import synth  # noqa: E402

METRIC = "fused gradient iteration throughput (G voxel-channel-projections/s); ms per iteration in ms_per_step"
UNIT = "G vcp/s"


def algorithmic_bytes(cfg):
    """SURVEY.md §8(d) streaming model, unpadded K, 4 B each: forward streams the volume once per projection
    (4 B per vcp) + writes the D-channel sinogram; the fused gradient adds the gradient write and the data,
    weights, wr traffic."""
    N, K, P = cfg.n_voxels, cfg.K, cfg.P
    sino = P * cfg.det[0] * cfg.det[1] * cfg.D * 4
    fwd = P * N * K * 4 + sino
    fused = P * N * K * 4 + N * K * 4 + 4 * sino
    return fwd, fused


def source_sha16():
    """hash of the sources of the step's two kernels (john_forward_kernel, adjoint_brick_kernel) and of the headers they
    include: ties a stored ncu traffic figure to the code it was measured on"""
    import hashlib
    h = hashlib.sha256()
    for name in ("mm_adjoint_brick.cu", "mm_adjoint_brick_pair.cuh", "mm_internal.h", "mm_kernels.cu", "mm_ptx.cuh"):
        with open(os.path.join(ROOT, "paper_2504_16446_b200", "csrc", name), "rb") as fh:
            h.update(fh.read())
    return h.hexdigest()[:16]


def record_traffic(csv_path, cfg_name, command):
    """`--record-traffic`: read dram__bytes_{read,write}.sum per kernel from an `ncu --page raw --csv` export and store
    them, with the hash of the kernel sources, in profiles/r02_traffic.json"""
    import csv
    with open(csv_path) as f:
        rows = list(csv.reader(f))
    hdr = rows[0]
    ik, ir, iw = hdr.index("Kernel Name"), hdr.index("dram__bytes_read.sum"), hdr.index("dram__bytes_write.sum")
    unit = {"Gbyte": 1e9, "Mbyte": 1e6, "Tbyte": 1e12, "Kbyte": 1e3, "byte": 1.0}
    ent = {}
    for r in rows[2:]:
        if len(r) <= max(ir, iw):
            continue
        b = float(r[ir]) * unit[rows[1][ir]] + float(r[iw]) * unit[rows[1][iw]]
        if b != b:                                   # a launch ncu could not replay: no figure
            continue
        for key, match in (("john_forward_kernel", "john_forward_kernel"), ("adjoint_brick_kernel", "adjoint_brick")):
            if match in r[ik]:                       # adjoint_brick_kernel or adjoint_brick_pair_kernel
                ent[key + "_dram_bytes"] = int(b)
    out = os.path.join(ROOT, "profiles", "r02_traffic.json")
    tr = {}
    if os.path.exists(out):
        with open(out) as f:
            tr = json.load(f)
    if tr.get("source_sha16") != source_sha16():
        tr = {}
    tr["source_sha16"] = source_sha16()
    tr["command"] = command
    tr.setdefault(cfg_name, {}).update(ent)
    with open(out, "w") as f:
        json.dump(tr, f, indent=1)
    print(json.dumps(tr))


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index=0):
        self.proc, self.index = None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "100"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
        except OSError:
            self.proc = None

    def stop(self):
        if self.proc is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.proc.terminate()
        try:
            out, _ = self.proc.communicate(timeout=5)
        except subprocess.TimeoutExpired:
            self.proc.kill()
            out, _ = self.proc.communicate()
        sm, mx, reasons = [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for line in out.strip().splitlines():
            t = [x.strip() for x in line.split(",")]
            if len(t) < 7:
                continue
            try:
                sm.append(float(t[0])); mx.append(float(t[1]))
            except ValueError:
                continue
            for nm, val in zip(names, t[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(nm)
        # idle samples (before the first kernel) pull the median down: keep the upper half
        sm_load = sorted(sm)[len(sm) // 2:] if sm else []
        return {"sm_mhz": statistics.median(sm_load) if sm_load else None, "sm_max_mhz": max(mx) if mx else None,
                "reasons": sorted(reasons), "samples": len(sm)}


# -------------------------------------------------------------------------------------------------
# reference arm / cpu_baseline: the oracle on a bounded sample
# -------------------------------------------------------------------------------------------------
def oracle_sample(cfg, n_sample_proj):
    """stratified projection subset: full volume, full detector, n_sample_proj of the P projections — spread over the
    tilts first (projections are tilt-major) with the rotation staggered from tilt to tilt, so that a sample of
    n_tilts projections has one per tilt and sweeps the rotation range (all three major axes on configs 2-5)."""
    rot, tilt = synth.angles(cfg)
    n_t, n_r = len(cfg.tilts_deg), cfg.n_rot
    n = int(max(1, min(cfg.P, n_sample_proj)))
    if n >= cfg.P:
        return rot, tilt, np.arange(cfg.P)
    per_t = -(-n // n_t)                                   # samples per tilt (the last tilts may get one fewer)
    idx = []
    for i in range(n):
        t, m = (i % n_t, i // n_t) if n >= n_t else ((i * n_t + n_t // 2) // n, 0)
        r = int((m + 0.5) * n_r / per_t + (t * n_r) / (float(n_t) * per_t)) % n_r      # staggered from tilt to tilt
        idx.append(t * n_r + r)
    idx = np.unique(np.array(idx, dtype=int))
    return rot[idx], tilt[idx], idx


def major_axes(go, n):
    """how many of the n projections of an oracle geometry march along x, y, z"""
    m = [go.get(s)[3] for s in range(n)]
    return {"x": m.count(0), "y": m.count(1), "z": m.count(2)}


def run_oracle_step(ora, go, B, vol, data, w, K):
    t0 = time.perf_counter()
    ora.loss_gradient(go, B, vol, data, w, form="scatter", threads=1)
    return time.perf_counter() - t0


def oracle_setup(cfg, n_sample_proj, vol=None):
    from oracle import oracle as ora
    ora.build()
    rot, tilt, idx = oracle_sample(cfg, n_sample_proj)
    go = ora.Geometry(cfg.shape, cfg.det, rot, tilt)
    B = ora.basis_matrix(go, cfg.ell_max, *synth.segments(cfg.D)).astype(np.float32)
    if vol is None:
        vol = synth.make_volume(cfg, cfg.K)
    data = synth.surrogate_model(cfg)[idx]
    return ora, go, B, vol, data, idx


def proj_seconds(cfg):
    """estimated single-core oracle time of one projection's loss_gradient (forward + scatter adjoint): measured
    ~1.0e9 tap-FMAs/s on the B200 boxes' hosts (config 5: 6e9 tap-FMAs, 5.9 s)"""
    return cfg.det[0] * cfg.det[1] * max(cfg.shape) * 4 * cfg.K * 2 / 1.0e9


def sample_size_for(cfg, budget_s=55.0):
    """projections in the cpu_baseline sample: at least one per tilt where that fits the time budget (config 5: 9
    projections, ~55 s on one core), the whole config when it is small"""
    n = int(budget_s // max(proj_seconds(cfg), 1e-9))
    return int(max(1, min(cfg.P, n)))


def reference_arm(args, cfg):
    """`--impl reference`: the oracle as it stands, one host core.  Every step marches a bounded sample of the workload
    (whole volume and detector, a few projections) sized so that warm-up + steps end within a few minutes; successive
    steps take successive members of the one-per-tilt stratified set, so a run covers all tilts and major axes."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    per_step = max(1, min(cfg.P, int((150.0 / max(1, args.steps + args.warmup)) // max(proj_seconds(cfg), 1e-9))))
    pool_n = min(cfg.P, max(len(cfg.tilts_deg), per_step))
    ora, go, B, vol, data, idx = oracle_setup(cfg, pool_n)
    K = cfg.K
    groups = [np.arange(i, i + per_step) % len(idx) for i in range(0, len(idx), per_step)]

    def step(i):
        sel = np.unique(groups[i % len(groups)])
        g1 = ora.Geometry(cfg.shape, cfg.det, go.rot[sel], go.tilt[sel])
        return run_oracle_step(ora, g1, B[sel], vol[..., :K], data[sel], None, K), len(sel)

    for i in range(args.warmup):
        step(i)
    res = [step(args.warmup + i) for i in range(args.steps)]
    t = sum(r[0] for r in res) / len(res)
    nproj = sum(r[1] for r in res) / len(res)
    vcp = cfg.n_voxels * K * nproj
    val = vcp / t / 1e9
    sample = (f"{nproj:g} of {cfg.P} projections per step, drawn in turn from the stratified set {idx.tolist()} (one per tilt; "
              f"major axes {major_axes(go, len(idx))}), full {cfg.shape} volume and {cfg.det} detector")
    line = {"impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": t * 1e3, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "sample": sample},
            "cpu_baseline": {"value": val, "unit": UNIT, "cores": 1, "kind": "oracle", "sample": sample},
            "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def max_over_ranks(ms: float, world: int, device) -> float:
    """device-timed duration of the slowest rank (the contract's max-over-ranks); identity at world 1."""
    if world <= 1:
        return float(ms)
    import torch
    import torch.distributed as dist
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def aggregate_throughput(cfg, world: int, ms_step: float) -> float:
    """whole-job G vcp/s of `world` independent replicas ("replicas only") that each took ms_step."""
    return world * cfg.vcp / (ms_step * 1e-3) / 1e9


def workload_name(cfg):
    return (f"{cfg.name}: {cfg.shape[0]}x{cfg.shape[1]}x{cfg.shape[2]} voxels, l_max={cfg.ell_max} (K={cfg.K}), "
            f"P={cfg.P}, detector {cfg.det[0]}x{cfg.det[1]}, D={cfg.D}")


# -------------------------------------------------------------------------------------------------
# our arm
# -------------------------------------------------------------------------------------------------
def ours(args, cfg):
    import torch
    import torch.distributed as dist
    from paper_2504_16446_b200 import mm

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (no CPU fallback)")
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    mm.load()

    K, D, ldk = cfg.K, cfg.D, synth.ldk_for(cfg.K)
    rot, tilt = synth.angles(cfg)
    g = mm.Geometry(cfg.shape, cfg.det, rot, tilt)
    h_B = mm.mm_basis_sh_matrix(g, cfg.ell_max, *synth.segments(D))
    t0 = time.time()
    h_vol = torch.from_numpy(synth.make_volume(cfg, ldk)).pin_memory()
    h_w = None if cfg.weights == "unit" else torch.from_numpy(synth.make_weights(cfg)).pin_memory()
    gen_s = time.time() - t0
    vol, B = h_vol.cuda(), torch.from_numpy(h_B).cuda()
    w = None if h_w is None else h_w.cuda()
    # data = forward model + Poisson noise (BASELINE.json configs): model from the parity-tested GPU forward
    model = torch.empty(g.proj_shape(D), device="cuda")
    mm.mm_forward(g, B, vol, K, model)
    h_data = torch.from_numpy(synth.poisson_data(model.cpu().numpy(), cfg.counts, cfg.seed)).pin_memory()
    del model
    data = h_data.cuda()
    grad = torch.empty(g.vol_shape(ldk), device="cuda")
    wr = torch.empty(g.proj_shape(D), device="cuda")
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)

    def step():
        mm.mm_loss_gradient(g, B, vol, K, data, w, grad, loss, wr)
        if cfg.gd_iters > 1:
            mm.mm_axpy(vol, grad, 1e-9)

    for _ in range(max(args.warmup, 3)):
        step()
    torch.cuda.synchronize()
    ev0 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    evm = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    ev1 = [torch.cuda.Event(enable_timing=True) for _ in range(args.steps)]
    for e in evm:
        e.record()                       # creates the handle the library re-records between the two phases
    torch.cuda.synchronize()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    if world > 1:
        dist.barrier()
    torch.cuda.synchronize()
    launches0 = mm.mm_launch_count()
    start, end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    start.record()
    for i in range(args.steps):
        ev0[i].record()
        mm.mm_set_phase_event(evm[i])
        step()
        ev1[i].record()
    end.record()
    mm.mm_set_phase_event(None)
    torch.cuda.synchronize()
    if world > 1:
        dist.barrier()
    launches = mm.mm_launch_count() - launches0
    clocks = sampler.stop() if rank == 0 else None
    total_ms = max_over_ranks(start.elapsed_time(end), world, torch.device("cuda", local))
    ms_step = total_ms / args.steps
    fwd_ms = sum(a.elapsed_time(b) for a, b in zip(ev0, evm)) / args.steps
    adj_ms = sum(a.elapsed_time(b) for a, b in zip(evm, ev1)) / args.steps
    value = aggregate_throughput(cfg, world, ms_step)
    loss_val = loss.item()

    # ---- optional extra (not part of the step): the paper's bilinear back-projection (NEXT-1) of the residual
    extras = None
    if args.extras and rank == 0:
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        mm.mm_backproject(g, B, wr, K, grad)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(args.steps):
            mm.mm_backproject(g, B, wr, K, grad)
        e1.record()
        torch.cuda.synchronize()
        extras = {"mm_backproject_ms": e0.elapsed_time(e1) / args.steps,
                  "what": "basis^T + bilinear interpolation of the projection (PAPER.md:314), same wr as the step"}

        def timed_extra(fn):
            fn()
            torch.cuda.synchronize()
            e0.record()
            for _ in range(args.steps):
                fn()
            e1.record()
            torch.cuda.synchronize()
            return e0.elapsed_time(e1) / args.steps

        # NEXT-4: the Huber-regressor step and the per-voxel derived quantities (Eq. 10-12)
        delta = 3.0 * float(wr.abs().mean())
        extras["mm_loss_gradient_huber_ms"] = timed_extra(lambda: mm.mm_loss_gradient_huber(g, B, vol, K, data, w, delta, grad, loss, wr))
        n3 = tuple(cfg.shape)
        dq = [torch.empty(n3 + t, device="cuda") for t in ((), (6,), (3,), (3, 3), ())]
        extras["mm_derived_quantities_ms"] = timed_extra(lambda: mm.mm_derived_quantities(g, vol, K, *dq))
        del dq
        mm.mm_loss_gradient(g, B, vol, K, data, w, grad, loss, wr)          # leave grad / wr / loss as the step left them
        torch.cuda.synchronize()

    # ---- end to end through the host-buffer C-ABI call (H2D of every input, D2H of gradient + loss, inside)
    e2e = None
    if rank == 0:
        h_grad = torch.empty(g.vol_shape(ldk), dtype=torch.float32).pin_memory()
        del grad, wr
        torch.cuda.empty_cache()
        n_e2e = max(1, min(args.steps, 2))
        mm.mm_loss_gradient_host(g, h_B, h_vol, K, h_data, h_w, h_grad)      # warm-up (page-in, allocator)
        t0 = time.perf_counter()
        for _ in range(n_e2e):
            Lh = mm.mm_loss_gradient_host(g, h_B, h_vol, K, h_data, h_w, h_grad)
        te = (time.perf_counter() - t0) / n_e2e
        nsino = h_data.numel() * 4
        e2e = {"value": cfg.vcp / te / 1e9, "unit": UNIT, "ms_per_step": te * 1e3,
               "h2d_bytes_per_step": int(h_vol.numel() * 4 + nsino * (2 if h_w is not None else 1) + h_B.size * 4),
               "d2h_bytes_per_step": int(h_grad.numel() * 4 + 8), "steps": n_e2e,
               "loss_matches_device_path": bool(abs(Lh - loss_val) <= 1e-9 * abs(loss_val)) if cfg.gd_iters <= 1 else None}
    if rank != 0:
        return

    peak, peak_src = measured_peaks()
    fwd_bytes, fused_bytes = algorithmic_bytes(cfg)
    achieved = fwd_bytes / (fwd_ms * 1e-3) / 1e9
    roofline = {"kernel": "john_forward_kernel (phase 1 of mm_loss_gradient: Joseph march + basis + residual + loss)",
                "bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                "bound_note": "frac is the STREAMING MODEL (one volume pass per projection) against the HBM copy peak; "
                              "cross-projection L2 reuse keeps real DRAM traffic below the model (see dram_frac), and ncu "
                              "(profiles/r02_ncu_c5_v6.md) shows no saturated unit on config 5 - L1 data pipe 83 %, DRAM 50 %, "
                              "L2 37 %: the march is latency-bound at 16 warps per SM (DESIGN.md 5)",
                "traffic": None, "dram_frac": None, "peak_source": peak_src, "ms_per_launch": fwd_ms,
                "algorithmic_bytes_per_launch": fwd_bytes,
                "model": "streaming: 4 B per voxel-channel-projection + sinogram write (SURVEY.md 8d)",
                "fused_step": {"algorithmic_bytes": fused_bytes, "achieved": fused_bytes / (ms_step * 1e-3) / 1e9,
                               "frac": fused_bytes / (ms_step * 1e-3) / 1e9 / peak},
                "adjoint_kernel_ms": adj_ms}
    # measured DRAM bytes of that kernel (one ncu --set full capture, profiles/r02_traffic.json, written by
    # `bench.py --record-traffic <ncu raw csv>`); only trusted while the kernel sources are the ones it was measured on
    traffic_file = os.path.join(ROOT, "profiles", "r02_traffic.json")
    if os.path.exists(traffic_file):
        with open(traffic_file) as f:
            tr = json.load(f)
        ent = tr.get(cfg.name, {})
        if tr.get("source_sha16") == source_sha16() and ent.get("john_forward_kernel_dram_bytes"):
            roofline["traffic"] = ent["john_forward_kernel_dram_bytes"]
            roofline["dram_frac"] = roofline["traffic"] / (fwd_ms * 1e-3) / 1e9 / peak
            roofline["traffic_source"] = tr.get("command")
        else:
            roofline["traffic_source"] = "profiles/r02_traffic.json is stale (kernel sources changed since the capture): null"

    # ---- cpu_baseline: the oracle, single core, on a bounded projection sample of the same workload
    cpu = None
    if world == 1 and not args.no_cpu_baseline:
        n_s = sample_size_for(cfg)
        vol_np = h_vol.numpy()
        ora, go, Bo, _, data_s, idx = oracle_setup(cfg, n_s, vol=vol_np)
        t = run_oracle_step(ora, go, Bo, vol_np[..., :K], data_s, None, K)
        cpu = {"value": cfg.n_voxels * K * len(idx) / t / 1e9, "unit": UNIT, "cores": 1, "kind": "oracle",
               "seconds": t, "sample": f"{len(idx)} of {cfg.P} projections (indices {idx.tolist()}: stratified over the tilts, "
                                       f"major axes {major_axes(go, len(idx))}), full volume and detector",
               "host_cores_available": len(os.sched_getaffinity(0))}

    line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": max(args.warmup, 3),
            "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f32",
            "data": "synthetic",
            "config": {"workload": workload_name(cfg), "ldk": ldk, "l2": "inputs (%.1f GB volume) larger than L2; no flush" % (vol.numel() * 4 / 1e9),
                       "multi_gpu": "replicas only", "input_generation_s": round(gen_s, 1)},
            "clocks": clocks, "e2e": e2e, "gpu_launches": int(launches), "roofline": roofline, "cpu_baseline": cpu,
            "loss": loss_val, "phase_ms": {"forward_residual": fwd_ms, "adjoint": adj_ms}, "extras": extras}
    print(json.dumps(line), flush=True)


def iterate_extra(args):
    """`--iterate-extra`: NEXT-3 measurement (not the headline step).  The device-resident regularised Nesterov iteration
    `mm_iterate` on the configured workload (default C5): wall time per iteration for a run of `--steps` iterations with
    the Laplacian and L2 regularisers and the relative-change stop test every iteration (tol so small that it never
    fires), against the bare fused gradient timed the same way."""
    import torch
    from paper_2504_16446_b200 import mm
    torch.cuda.set_device(0)
    mm.load()
    cfg = synth.get_config(args.config)
    K, D, ldk = cfg.K, cfg.D, synth.ldk_for(cfg.K)
    rot, tilt = synth.angles(cfg)
    g = mm.Geometry(cfg.shape, cfg.det, rot, tilt)
    B = torch.from_numpy(mm.mm_basis_sh_matrix(g, cfg.ell_max, *synth.segments(D))).cuda()
    gen = torch.Generator(device="cuda")
    gen.manual_seed(cfg.seed)
    truth = torch.rand(g.vol_shape(ldk), device="cuda", generator=gen)
    truth[..., K:] = 0
    data = torch.empty(g.proj_shape(D), device="cuda")
    mm.mm_forward(g, B, truth, K, data)
    scale = float(data.abs().max())
    del truth
    n_it = max(2, args.steps)
    c = torch.zeros(g.vol_shape(ldk), device="cuda")
    v = torch.zeros_like(c)
    losses = torch.zeros(n_it, device="cuda", dtype=torch.float64)
    # step length: a fifth of the exact line-search step along the first gradient, ||g||^2 / ||A g||^2 >= 1 / ||A^T A||
    g0 = torch.empty_like(c)
    l0 = torch.zeros(1, device="cuda", dtype=torch.float64)
    wr0 = torch.empty_like(data)
    mm.mm_loss_gradient(g, B, c, K, data, None, g0, l0, wr0)
    mm.mm_forward(g, B, g0, K, wr0)
    eta = 0.2 * float((g0.double() ** 2).sum() / (wr0.double() ** 2).sum())
    del g0, wr0
    kw = dict(eta=eta, momentum=0.5, mu_laplacian=1e-3 * scale, mu_l2=1e-4 * scale, max_iter=n_it, tol=1e-30, check_every=1)
    mm.mm_iterate(g, B, K, data, None, c, v, torch.zeros(2, device="cuda", dtype=torch.float64), **{**kw, "max_iter": 2})   # warm-up (pool, clocks)
    torch.cuda.synchronize()
    c.zero_(); v.zero_()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    launches = mm.mm_launch_count()
    e0.record()
    done = mm.mm_iterate(g, B, K, data, None, c, v, losses, **kw)
    e1.record()
    torch.cuda.synchronize()
    launches = mm.mm_launch_count() - launches
    it_ms = e0.elapsed_time(e1) / done
    grad = torch.empty_like(c)
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)
    wr = torch.empty_like(data)
    for _ in range(3):
        mm.mm_loss_gradient(g, B, c, K, data, None, grad, loss, wr)
    torch.cuda.synchronize()
    e0.record()
    for _ in range(n_it):
        mm.mm_loss_gradient(g, B, c, K, data, None, grad, loss, wr)
    e1.record()
    torch.cuda.synchronize()
    grad_ms = e0.elapsed_time(e1) / n_it
    hist = losses.cpu().numpy()
    line = {"what": "NEXT-3 device-resident regularised Nesterov iteration (PAPER.md:262-264, 270-272, 336-340)", "data": "synthetic",
            "config": {"workload": workload_name(cfg), "regularisers": "Laplacian + L2", "momentum": 0.5, "eta": "0.2 x the exact line-search step of the first gradient", "stop_check_every": 1},
            "iterations": int(done), "ms_per_iteration": it_ms, "bare_gradient_ms": grad_ms, "overhead_ms": it_ms - grad_ms,
            "gpu_launches": int(launches), "host_syncs": "one 4-byte D2H per stop check",
            "loss_first": float(hist[0]), "loss_last": float(hist[int(done) - 1])}
    print(json.dumps(line))


def sparse_extra(args):
    """`--sparse-extra`: NEXT-2 measurement (not the headline step).  Table V's largest basis (N = 162 directions, NN
    indicator functions) on a 100^3 volume, 240 projections (6 tilts x 40), 100^2 detector, D = 8:
    dense fused forward / gradient against the sparse-plan calls on the same NN matrix."""
    import torch
    from paper_2504_16446_b200 import mm
    torch.cuda.set_device(0)
    mm.load()
    cfg = synth.get_config("C3", tilts_deg=(0.0, 9.0, 18.0, 27.0, 36.0, 45.0))
    K, D = 162, 8
    ldk = synth.ldk_for(K)
    rot, tilt = synth.angles(cfg)
    g = mm.Geometry(cfg.shape, cfg.det, rot, tilt)
    h_B = mm.mm_basis_grid_matrix(g, mm.MM_BASIS_NN, synth.grid_directions(K), *synth.segments(D), n_quad=8)
    plan = mm.SparsePlan(g, h_B)
    rng = np.random.default_rng(162)
    vol = torch.from_numpy(synth.pad_channels(rng.uniform(0, 1, cfg.shape + (K,)).astype(np.float32), ldk)).cuda()
    B = torch.from_numpy(h_B).cuda()
    sino = torch.empty(g.proj_shape(D), device="cuda")
    mm.mm_forward(g, B, vol, K, sino)
    data = sino * (1 + 0.03 * torch.randn_like(sino))
    grad = torch.empty(g.vol_shape(ldk), device="cuda")
    wr = torch.empty_like(sino)
    loss = torch.zeros(1, device="cuda", dtype=torch.float64)

    def timed(fn):
        for _ in range(max(3, args.warmup)):
            fn()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        torch.cuda.synchronize()
        e0.record()
        for _ in range(args.steps):
            fn()
        e1.record()
        torch.cuda.synchronize()
        return e0.elapsed_time(e1) / args.steps

    res = {"forward_dense_ms": timed(lambda: mm.mm_forward(g, B, vol, K, sino)),
           "forward_sparse_ms": timed(lambda: mm.mm_forward_sparse(g, plan, B, vol, K, sino)),
           "gradient_dense_ms": timed(lambda: mm.mm_loss_gradient(g, B, vol, K, data, None, grad, loss, wr)),
           "gradient_sparse_ms": timed(lambda: mm.mm_loss_gradient_sparse(g, plan, B, vol, K, data, None, grad, loss, wr)),
           "adjoint_dense_ms": timed(lambda: mm.mm_adjoint(g, B, wr, K, grad))}
    line = {"what": "NEXT-2 sparse reciprocal-space map vs dense, NN basis (PAPER.md:242, 274)", "data": "synthetic",
            "config": {"workload": f"100x100x100 voxels, K={K} NN directions (ldk {ldk}), P={g.P}, detector 100x100, D={D}, n_quad=8",
                       "active_channels_per_projection": {"max": plan.max_active, "mean": plan.mean_active}},
            "steps": args.steps, **res,
            "forward_speedup": res["forward_dense_ms"] / res["forward_sparse_ms"],
            "gradient_speedup": res["gradient_dense_ms"] / res["gradient_sparse_ms"]}
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", default="C5", choices=sorted(synth.CONFIGS))
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--extras", action="store_true", help="also time mm_backproject, mm_loss_gradient_huber and mm_derived_quantities (outside the step)")
    ap.add_argument("--iterate-extra", action="store_true", help="time the NEXT-3 device-resident iteration (mm_iterate) against the bare gradient and exit")
    ap.add_argument("--sparse-extra", action="store_true", help="time the NEXT-2 sparse-plan calls against the dense ones (K = 162 NN basis) and exit")
    ap.add_argument("--record-traffic", metavar="NCU_RAW_CSV", help="store the kernels' DRAM bytes from an ncu raw-page csv and exit")
    ap.add_argument("--traffic-command", default="ncu --set full --clock-control none -k regex:john_forward|adjoint_brick ... python bench.py --steps 1 --warmup 3 --no-cpu-baseline; ncu -i <rep> --page raw --csv")
    args = ap.parse_args()
    cfg = synth.get_config(args.config)
    if args.record_traffic:
        record_traffic(args.record_traffic, cfg.name, args.traffic_command)
        return
    if args.iterate_extra:
        iterate_extra(args)
        return
    if args.sparse_extra:
        sparse_extra(args)
        return
    if args.impl == "reference":
        reference_arm(args, cfg)
    else:
        ours(args, cfg)


if __name__ == "__main__":
    main()
