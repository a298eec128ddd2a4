#!/usr/bin/env python
"""bench.py -- electron-steps/s of the domain-batched real-time Kohn-Sham step on B200.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config C] [--gemm-mode M] [--impl reference]

A "step" is one Taylor-4 time step of EVERY domain of the config: four Horner stages (projection
GEMM, fused stencil pass, back-application GEMM) plus the density.  The default
workload is BASELINE.json configs[3] (64 PbTiO3-shaped domains, 48^3 grid, 224 orbitals, 240
projectors: the "throughput at HBM fill" config the metric is quoted on).  One JSON line is printed
by rank 0.  See DESIGN.md "Measurement" for the roofline arithmetic.
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

import workloads as W  # noqa: E402

PAPER_CONTEXT = {
    "t2s_s_per_electron_step": 1.11e-7, "sustained_eflops": 1.87, "gpus": 60000,
    "note": "PAPER.md L38-39, L298, L302: Aurora, 1,024-orbital domains of unstated mesh size; context only",
}
MODE_NAMES = {"fp32grade": 0, "fp64": 1, "bf16": 2, "tf32x1": 3, "simt": 4, "staged": 5}
CPU_STEPS = 8            # timed oracle steps of the cpu_baseline leg
STEP_NAMES = {"taylor": "Taylor-4 (full H, north_star)", "split": "Eq. (2) split (half-kick, Taylor-4 of h_loc, half-kick)",
              "richardson": "Eq. (2) split with the paper's own local solver (half-kick, block-diagonal split-operator on the "
                            "7-point operator, half-kick)"}
SPLIT_STEPS = ("split", "richardson")
# tensor peak as a multiple of the measured dense BF16 peak (B200_PROFILING.md nominal ratios:
# tf32 1.1 PF vs bf16 2.25 PF); 3xTF32 issues three TF32 MMAs per product.
# the opt-in low-precision mode stores beta and W as BF16 and issues tcgen05.mma.kind::f16: the BF16 peak itself
TF32_OVER_BF16 = 1.1 / 2.25     # nominal dense peaks (B200_PROFILING.md): tf32 1.1 PF, bf16 2.25 PF
# "staged" (MLMD_GEMM_FP32GRADE_STAGED, Taylor step): of the 8 GEMMs of a step the outermost 2 issue 3 products per MAC, the
# inner projections 1 and the inner back-applications 2: (2 x 3 + 3 x 1 + 3 x 2) / 8 = 1.875 products on average
TENSOR_RATIO = {"fp32grade": TF32_OVER_BF16 / 3.0, "tf32x1": TF32_OVER_BF16, "bf16": 1.0,
                "staged": TF32_OVER_BF16 / 1.875}
FP32_ALU_TFLOPS = 148 * 128 * 2 * 1.965e9 / 1e12   # 148 SMs x 128 FMA lanes x 2 flop x max SM clock
FP64_ALU_TFLOPS = 148 * 64 * 2 * 1.965e9 / 1e12    # nominal 64 DFMA lanes per SM (guide: ~40 TF)


def load_peaks():
    path = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(path):
        with open(path) as f:
            p = json.load(f)
        return {"hbm_gbs": p["hbm_gbs"], "bf16_burst": p["bf16_tflops"],
                "bf16_sustained": p.get("bf16_tflops_sustained", p["bf16_tflops"]), "source": "measured"}
    return {"hbm_gbs": 6650.0, "bf16_burst": 1590.0, "bf16_sustained": 1400.0, "source": "fallback"}


class ClockSampler(threading.Thread):
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        super().__init__(daemon=True)
        self.index, self.rows, self.stop_flag = index, [], threading.Event()

    def run(self):
        while not self.stop_flag.is_set():
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.index), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                parts = [x.strip() for x in out.strip().split(",")]
                if len(parts) == 7:
                    self.rows.append(parts)
            except Exception:
                pass
            self.stop_flag.wait(0.2)

    def summary(self):
        self.stop_flag.set()
        self.join(timeout=6)
        if not self.rows:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        sm = sorted(float(r[0]) for r in self.rows)
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        reasons = [n for k, n in enumerate(names) if any(r[3 + k] == "Active" for r in self.rows)]
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.rows[0][1]), "samples": len(sm),
                "power_w_max": max(float(r[2]) for r in self.rows), "reasons": reasons}


def algorithmic(c, gemm_real=True, step="taylor"):
    """Algorithmic bytes and flops per step of the whole batch.  step="split" (the literal
    Eq. (2) step, mlmd_propagate_split): two V_NL applications instead of four, no per-step norm pass (two
    norms ride on stencil passes, the third comes from the projector Gram matrix; one 8 B/element pass per
    CALL for the incoming norms and one 16 B/element rescaling pass per CALL are not counted: inside a call psi stays
    un-normalised and the density takes the scale through the occupations)."""
    elems = c.ndom * c.ngrid * c.norb
    # "richardson": three in-place passes (one per axis); no per-step norm pass either (norms from the projector Gram matrix)
    stage_bytes = [16, 16, 16] if step == "richardson" else [16, 24, 24, 24]
    split = step in SPLIT_STEPS
    density_b, norm_b, ngemm = (8, 0, 4) if split else (8, 0, 8)
    bytes_step = elems * (sum(stage_bytes) + density_b + norm_b) + c.ndom * c.ngrid * (4 * 4 + 4)
    gemm_flops_each = (2 if gemm_real else 4) * 2.0 * c.ndom * c.ngrid * c.nproj * c.norb   # one GEMM batch
    return {"elems": elems, "bytes_step": bytes_step, "stencil_bytes": [elems * b for b in stage_bytes],
            "density_bytes": elems * density_b, "norm_bytes": elems * 8, "gemm_flops_each": gemm_flops_each,
            "gemm_flops_step": ngemm * gemm_flops_each}


def ncu_traffic(c, kernel_class):
    """(dram__bytes_read.sum + dram__bytes_write.sum per launch of the class's kernel, where it comes from): read from
    the newest committed `ncu --set full` capture of the same workload (profiles/r*_traffic_cfg3.json, which names the
    commit it was taken at); (None, None) when there is none.  It is NOT measured by this run: ncu replays kernels."""
    import glob
    paths = sorted(glob.glob(os.path.join(ROOT, "profiles", "r*_traffic_cfg3.json")))
    if c.cfg != 3 or c.ndom != 64 or not paths:
        return None, None
    with open(paths[-1]) as f:
        j = json.load(f)
    t = j["dram_bytes_per_launch"]
    pick = {"stencil": ["stencil_tma_kernel<0, 0, 0>", "stencil_tma_kernel"], "proj": ["proj2_tc_kernel", "proj_tc_kernel"],
            "back": ["back2_tc_kernel", "back_tc_kernel"], "density": ["density_kernel"]}.get(kernel_class, [])
    src = "%s (ncu --set full at commit %s)" % (os.path.relpath(paths[-1], ROOT), j.get("commit", "?"))
    for name in pick:
        for key in t:
            if key == name or key.startswith(name + "<"):
                return t[key], src
    return None, None


def sample_for_oracle(c, d, norb_sample):
    """Domain 0, first norb_sample orbitals: the bounded sample the oracle is timed on."""
    n = min(norb_sample, c.norb)
    return {"psi": np.ascontiguousarray(d["psi"][:1, ..., :n]), "occ": np.ascontiguousarray(d["occ"][:1, :n]),
            "vloc": d["vloc"][:1], "beta": d["beta"][:1], "D": d["D"][:1]}


def time_oracle(c, s, A, steps, warmup, step="taylor"):
    from oracle import ref
    if step == "richardson":
        def prop(*a):
            return ref.propagate_split(*a, local="richardson")
    else:
        prop = ref.propagate_split if step == "split" else ref.propagate
    for _ in range(warmup):
        prop(s["psi"], s["occ"], s["vloc"], s["beta"], s["D"], A[:1], c.dt, c.h)
    t0 = time.perf_counter()
    psi = s["psi"]
    for k in range(steps):
        psi, _ = prop(psi, s["occ"], s["vloc"], s["beta"], s["D"], A[k:k + 1], c.dt, c.h)
    dt = time.perf_counter() - t0
    electrons = float(s["occ"].sum())
    return electrons * steps / dt, dt / steps, ref.num_threads(), electrons


def run_reference(args):
    """--impl reference: the FP64 oracle, as it stands, on the host cores, on a bounded sample."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    c = W.get_config(args.config)
    d1 = W.generate_domain(c, 0)
    d = {k: d1[k][None] for k in ("psi", "occ", "vloc", "beta", "D")}
    A = W.laser_samples(c, nsteps=max(args.steps, 1))
    s = sample_for_oracle(c, d, args.oracle_orbitals)
    value, sec_step, cores, electrons = time_oracle(c, s, A, args.steps, args.warmup, args.step)
    sample = "domain 0 of configs[%d], first %d of %d orbitals (%g electrons), all %d projectors, 1 %s step per bench step" % (
        c.cfg, s["psi"].shape[-1], c.norb, electrons, c.nproj, STEP_NAMES[args.step])
    line = {
        "impl": "reference", "metric": "electron-steps/s", "value": value, "unit": "electron-steps/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": sec_step * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": workload_config(c, args),
        "cpu_baseline": {"value": value, "unit": "electron-steps/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "electron-steps/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def workload_config(c, args):
    return {"workload": "configs[%d] %s: %d domains x %dx%dx%d grid x %d orbitals x %d projectors, dt=%g" % (
        c.cfg, c.name, c.ndom, *c.grid, c.norb, c.nproj, c.dt),
        "ndom_per_gpu": c.ndom, "step": STEP_NAMES[args.step], "gemm_mode": args.gemm_mode, "parallelism": "domains sharded, no collective",
        "l2": "working set (3 x %.1f GB psi buffers + beta) exceeds the 126 MB L2; no flush needed" % (
            c.ndom * c.ngrid * c.norb * 8 / 1e9) if c.ndom * c.ngrid * c.norb * 8 > 4e8 else
        "working set may fit L2: a 256 MB buffer is written between timed repetitions"}


def power_probe(c, dom, psi_dev, occ, vloc, A, dev):
    """--power: what 1000 W buy for each operation (profiles/r*_power_per_kernel.md).  One operation at a time is launched back
    to back for ~3 s while a host thread samples NVML power and clocks every 20 ms; the second half of the samples is averaged.
    Returns a list of rows.  Uses the public API only (the back-application alone is the step minus the rest)."""
    import torch
    import pynvml
    import paper_2509_00966_b200 as M
    pynvml.nvmlInit()
    H = pynvml.nvmlDeviceGetHandleByIndex(dev.index or 0)
    rows = []

    def run(name, fn, seconds=3.0):
        fn()
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        e0.record(dom.stream)
        fn()
        e1.record(dom.stream)
        torch.cuda.synchronize()
        n = max(2, int(seconds * 1e3 / max(e0.elapsed_time(e1), 1e-3)))
        samples, stop = [], threading.Event()

        def sample():
            while not stop.is_set():
                samples.append((pynvml.nvmlDeviceGetPowerUsage(H) / 1e3, pynvml.nvmlDeviceGetClockInfo(H, pynvml.NVML_CLOCK_SM)))
                stop.wait(0.02)
        th = threading.Thread(target=sample, daemon=True)
        th.start()
        e0.record(dom.stream)
        for _ in range(n):
            fn()
        e1.record(dom.stream)
        torch.cuda.synchronize()
        stop.set()
        th.join(timeout=5)
        half = samples[len(samples) // 2:] or [(0.0, 0.0)]
        w = float(np.mean([x[0] for x in half]))
        ms = e0.elapsed_time(e1) / n
        rows.append({"operation": name, "ms_per_launch": ms, "watt": w, "sm_mhz": float(np.median([x[1] for x in half])),
                     "joule_per_launch": w * ms * 1e-3, "launches": n, "samples": len(samples)})
        time.sleep(1.0)

    time.sleep(2.0)
    rows.append({"operation": "idle", "watt": pynvml.nvmlDeviceGetPowerUsage(H) / 1e3})
    with torch.cuda.stream(dom.stream):
        a = torch.empty(1 << 30, dtype=torch.bfloat16, device=dev)
        b = torch.empty_like(a)
        run("torch copy, 2 GiB read + 2 GiB written", lambda: b.copy_(a))
        del a, b
        x = torch.randn(8192, 8192, device=dev, dtype=torch.bfloat16)
        y = torch.randn(8192, 8192, device=dev, dtype=torch.bfloat16)
        run("cuBLAS bf16 8192^3", lambda: torch.matmul(x, y))
        xf, yf = x.float(), y.float()
        torch.backends.cuda.matmul.allow_tf32 = True
        run("cuBLAS tf32 8192^3", lambda: torch.matmul(xf, yf))
        del x, y, xf, yf
    torch.cuda.empty_cache()
    dom.set_orbitals(psi_dev, occ)
    run("one Taylor-4 step of the whole batch (mlmd_propagate, 3xTF32)", lambda: dom.propagate(1, c.dt, A[:1]), 5.0)
    E = torch.empty(c.ndom, dtype=torch.float64, device=dev)
    run("projection, 3xTF32 (mlmd_energy_nl: proj2_tc_kernel + a reduction)", lambda: M.mlmd_energy_nl(dom.handle, E))
    dom.set_gemm_mode(M.GEMM_FP32GRADE_STAGED)
    run("the same step, staged mode", lambda: dom.propagate(1, c.dt, A[:1]), 5.0)
    dom.set_gemm_mode(M.GEMM_LOWP_BF16)
    run("the same step, low-precision (BF16) mode", lambda: dom.propagate(1, c.dt, A[:1]), 5.0)
    dom.set_gemm_mode(M.GEMM_FP32GRADE)
    dom.set_orbitals(psi_dev, occ)
    run("Eq. (2) step, Taylor local solver (mlmd_propagate_split)", lambda: dom.propagate_split(1, c.dt, A[:1]), 4.0)
    dom.set_option(M.OPT_LOCAL_SOLVER, 1)
    run("Eq. (2) step, split-operator local solver", lambda: dom.propagate_split(1, c.dt, A[:1]), 4.0)
    dom.set_option(M.OPT_LOCAL_SOLVER, 0)
    # the local part alone: a second handle without projectors (four stencil passes + the density pass per step)
    loc = M.Domain(c.ndom, c.grid, c.h, c.norb, 0, device=str(dev), stream=dom.stream)
    loc.set_vloc(vloc)
    loc.set_projectors(None, None)
    loc.set_orbitals(psi_dev, occ)
    run("four stencil passes + the density pass (a handle without projectors)", lambda: loc.propagate(1, c.dt, A[:1]))
    loc.set_option(M.OPT_LOCAL_SOLVER, 1)
    run("three split-operator passes + the density pass (the same handle)", lambda: loc.propagate_split(1, c.dt, A[:1]))
    loc.close()
    return rows


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=3)
    ap.add_argument("--ndom", type=int, default=0, help="override the number of domains (debug)")
    ap.add_argument("--gemm-mode", default="fp32grade", choices=sorted(MODE_NAMES))
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--step", default="taylor", choices=sorted(STEP_NAMES),
                    help="taylor: mlmd_propagate (north_star hot path, the default bench line); split: mlmd_propagate_split (NEXT-1)")
    ap.add_argument("--oracle-orbitals", type=int, default=32)
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-observables", action="store_true")
    ap.add_argument("--no-staged", action="store_true", help="skip the extra timing of the same steps in the staged GEMM mode")
    ap.add_argument("--power", action="store_true",
                    help="instead of the bench line: board power / SM clock / energy per launch of each operation looping alone (NVML)")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import paper_2509_00966_b200 as M

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; libmlmd has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    c = W.get_config(args.config)
    if args.ndom:
        c = W.get_config(args.config, ndom=args.ndom)
    K, Wm = args.steps, args.warmup
    alg = algorithmic(c, step=args.step)
    peaks = load_peaks()

    # ---- inputs: seeded per (config, global domain index); generated in a thread pool, staged per domain
    dev = torch.device("cuda", local)
    psi_dev = torch.empty((c.ndom, *c.grid, c.norb), dtype=torch.complex64, device=dev)
    beta_dev = torch.empty((c.ndom, c.ngrid, c.nproj), dtype=torch.float32, device=dev)
    vloc = np.empty((c.ndom, *c.grid), dtype=np.float32)
    occ = np.empty((c.ndom, c.norb))
    D = np.empty((c.ndom, c.nproj))
    first = {}
    from concurrent.futures import ThreadPoolExecutor
    workers = max(1, min(8, (os.cpu_count() or 2) // (2 * max(1, min(world, 8)))))
    t_gen = time.perf_counter()
    with ThreadPoolExecutor(max_workers=workers) as ex:
        from paper_2509_00966_b200.shard import weak_scaling_block
        first_dom, last_dom = weak_scaling_block(c.ndom, rank)   # domains are the sharding unit: no collective
        for i, dd in enumerate(ex.map(lambda k: W.generate_domain(c, k), range(first_dom, last_dom))):
            psi_dev[i].copy_(torch.from_numpy(dd["psi"]))
            beta_dev[i].copy_(torch.from_numpy(dd["beta"]))
            vloc[i], occ[i], D[i] = dd["vloc"], dd["occ"], dd["D"]
            if i == 0:
                first = {k: dd[k][None] for k in ("psi", "occ", "vloc", "beta", "D")}
    t_gen = time.perf_counter() - t_gen
    A = W.laser_samples(c, nsteps=max(K, Wm, 1), t0=0.9)   # around the pulse maximum: A != 0 in every step

    dom = M.Domain(c.ndom, c.grid, c.h, c.norb, c.nproj, device=str(dev))
    dom.set_gemm_mode(MODE_NAMES[args.gemm_mode])
    dom.set_vloc(vloc)
    dom.set_projectors(beta_dev, D)
    dom.set_orbitals(psi_dev, occ)
    del beta_dev
    stream = dom.stream
    propagate = dom.propagate_split if args.step in SPLIT_STEPS else dom.propagate
    if args.step == "richardson":
        dom.set_option(M.OPT_LOCAL_SOLVER, 1)
    flush = torch.empty(64 * 1024 * 1024, dtype=torch.float32, device=dev) if alg["elems"] * 8 < 4e8 else None

    def barrier():
        if dist is not None:
            dist.barrier()
        torch.cuda.synchronize()

    if args.power:
        if rank == 0:
            print(json.dumps({"power_probe": power_probe(c, dom, psi_dev, occ, vloc, A, dev), "config": workload_config(c, args)}))
        return

    # ---- warm-up (W steps), then EXACTLY K timed steps in one mlmd_propagate call
    if Wm > 0:
        propagate(Wm, c.dt, A)
    if flush is not None:
        # small, launch-bound batches replay a CUDA graph of the step, which the library captures in the first call of
        # >= 4 steps: make sure that has happened before the timed region whatever W is (extra untimed steps)
        propagate(4, c.dt, np.concatenate([A, A, A, A])[:4])
    dom.set_orbitals(psi_dev, occ)         # state reset: timed steps start from Psi(0)
    if flush is not None:
        flush.fill_(1.0)
    barrier()
    sampler = ClockSampler(local) if rank == 0 else None
    if sampler:
        sampler.start()
    launches0 = dom.launch_count()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(stream)
    propagate(K, c.dt, A)            # the timed region: un-instrumented (the library's own launch path, CUDA graph included)
    e1.record(stream)
    barrier()
    ms = e0.elapsed_time(e1)
    launches = dom.launch_count() - launches0
    clocks = sampler.summary() if sampler else None
    gemm_path = dom.gemm_path()
    # second pass over the same K steps with mlmd_profile on: CUDA events around every launch on the library's
    # stream give the per-kernel-class table (this pass forces eager launches and is not what `value` is taken from)
    dom.set_orbitals(psi_dev, occ)
    if flush is not None:
        flush.fill_(1.0)
    torch.cuda.synchronize()
    dom.profile(True)
    p0, p1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    p0.record(stream)
    propagate(K, c.dt, A)
    p1.record(stream)
    torch.cuda.synchronize()
    ms_profiled = p0.elapsed_time(p1)
    dom.profile(False)
    kern = dom.profile_read()
    t = torch.tensor([ms], dtype=torch.float64, device=dev)
    if dist is not None:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    electrons = c.ndom * c.electrons_per_domain * world
    value = electrons * K / (ms * 1e-3)

    # ---- end to end through the C ABI with HOST buffers: per step the host sends V_loc (PAPER.md L145:
    # only Delta v_loc goes to the GPU per MD step; Psi stays resident) and A, and reads rho back.
    e2e = None
    if not args.no_e2e:
        vpin = torch.from_numpy(vloc).pin_memory()
        rpin = torch.empty((c.ndom, *c.grid), dtype=torch.float32).pin_memory()
        vnp, rnp = vpin.numpy(), rpin.numpy()
        dom.set_orbitals(psi_dev, occ)
        barrier()
        t0 = time.perf_counter()
        for k in range(K):
            dom.set_vloc(vnp)
            propagate(1, c.dt, A[k:k + 1])
            dom.density(rnp)
        torch.cuda.synchronize()
        sec = time.perf_counter() - t0
        tt = torch.tensor([sec], dtype=torch.float64, device=dev)
        if dist is not None:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        sec = float(tt.item())
        e2e = {"value": electrons * K / sec, "unit": "electron-steps/s", "h2d_bytes_per_step": int(vnp.nbytes + 24),
               "d2h_bytes_per_step": int(rnp.nbytes), "ms_per_step": sec / K * 1e3,
               "what": "per step: mlmd_set_vloc(host pinned) + %s(1, A host) + mlmd_density(host pinned); " % (
                   "mlmd_propagate_split" if args.step in SPLIT_STEPS else "mlmd_propagate") +
                       "Psi stays device-resident as in the paper's shadow dynamics (L130-132, L145)"}

    # ---- on-request observables (NEXT rows of SURVEY.md 8(f)): device time of one call each, CUDA events
    def time_call(fn, reps=3):
        fn()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        b.record(stream)
        torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    observables = None
    if rank == 0 and not args.no_observables:
        e_dev = torch.empty(c.ndom, dtype=torch.float64, device=dev)
        j_dev = torch.empty((c.ndom, 3), dtype=torch.float64, device=dev)
        elems = alg["elems"]
        t_e = time_call(lambda: M.mlmd_energy_nl(dom.handle, e_dev))
        t_j = time_call(lambda: M.mlmd_current(dom.handle, A[0], j_dev))
        observables = {
            "energy_nl": {"ms": t_e, "tflops": alg["gemm_flops_each"] / (t_e * 1e-3) / 1e12,
                          "what": "projection GEMM + reduction (mlmd_energy_nl), device buffers"},
            "current": {"ms": t_j, "gbs": elems * 8 / (t_j * 1e-3) / 1e9, "frac_hbm": elems * 8 / (t_j * 1e-3) / 1e9 / peaks["hbm_gbs"],
                        "what": "forward-neighbour pass over psi (mlmd_current), algorithmic bytes = one read of psi"},
        }

    # ---- the same K steps in the opt-in stage-adaptive GEMM mode, reported beside the default line
    also_staged = None
    if rank == 0 and world == 1 and args.step == "taylor" and args.gemm_mode == "fp32grade" and gemm_path == "tcgen05" and not args.no_staged:
        dom.set_gemm_mode(MODE_NAMES["staged"])
        propagate(min(Wm, 3) or 1, c.dt, A)
        dom.set_orbitals(psi_dev, occ)
        if flush is not None:
            flush.fill_(1.0)
        torch.cuda.synchronize()
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(stream)
        propagate(K, c.dt, A)
        s1.record(stream)
        torch.cuda.synchronize()
        ms_s = s0.elapsed_time(s1)
        also_staged = {"gemm_mode": "staged", "value": c.ndom * c.electrons_per_domain * K / (ms_s * 1e-3), "unit": "electron-steps/s",
                       "ms_per_step": ms_s / K, "n_gpus": 1,
                       "what": "mlmd_set_gemm_mode(MLMD_GEMM_FP32GRADE_STAGED): 3xTF32 in the outermost Horner stage, 1 (projection) / 2 "
                               "(back-application) TF32 products in the three inner ones; same FP32-grade tolerances, "
                               "tests/test_gpu_staged.py; this rank only"}
        dom.set_gemm_mode(MODE_NAMES[args.gemm_mode])

    if rank != 0:
        if dist is not None:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel class and of the whole step
    mode = args.gemm_mode
    if mode == "staged" and args.step in SPLIT_STEPS:
        mode = "fp32grade"      # the staged mode only changes mlmd_propagate's inner Horner stages
    tensor_peak_sus = peaks["bf16_sustained"] * TENSOR_RATIO.get(mode, TENSOR_RATIO["fp32grade"])
    tensor_peak_burst = peaks["bf16_burst"] * TENSOR_RATIO.get(mode, TENSOR_RATIO["fp32grade"])
    per_class = {}
    total_kernel_ms = sum(v[0] for v in kern.values()) or 1.0
    for name, (kms, n) in kern.items():
        avg = kms / n
        entry = {"ms_total": kms, "launches": n, "ms_avg": avg, "share": kms / total_kernel_ms}
        if name == "stencil":
            # the Taylor forms time one Horner stage per profiling scope, the split-operator solver its three passes together
            b = sum(alg["stencil_bytes"]) / (1.0 if args.step == "richardson" else 4.0)
            entry.update(bound="hbm", achieved=b / (avg * 1e-3) / 1e9, peak=peaks["hbm_gbs"], unit="GB/s")
        elif name == "density":
            entry.update(bound="hbm", achieved=alg["density_bytes"] / (avg * 1e-3) / 1e9, peak=peaks["hbm_gbs"], unit="GB/s")
        elif name == "norm":
            entry.update(bound="hbm", achieved=alg["norm_bytes"] / (avg * 1e-3) / 1e9, peak=peaks["hbm_gbs"], unit="GB/s")
        elif name in ("proj", "back", "nlp"):
            fl = alg["gemm_flops_each"] * (2 if name == "nlp" else 1)
            if gemm_path == "simt":
                pk = FP64_ALU_TFLOPS if mode == "fp64" else FP32_ALU_TFLOPS
                entry.update(bound="alu", achieved=fl / (avg * 1e-3) / 1e12, peak=pk, unit="TFLOP/s")
            else:
                entry.update(bound="tensor", achieved=fl / (avg * 1e-3) / 1e12, peak=tensor_peak_sus, unit="TFLOP/s")
        if "achieved" in entry:
            entry["frac"] = entry["achieved"] / entry["peak"]
        per_class[name] = entry
    top = max((n for n in per_class if "achieved" in per_class[n]), key=lambda n: per_class[n]["ms_total"])
    roof = {k: per_class[top][k] for k in ("bound", "achieved", "peak", "unit", "frac")}
    traffic, traffic_src = ncu_traffic(c, top) if args.step == "taylor" or top != "density" else (None, None)
    roof.update(kernel=top, traffic=traffic, traffic_source=traffic_src, peak_source="%s (%s)" % (
        "MEASURED_PEAKS.json" if peaks["source"] == "measured" else "B200_PROFILING.md fallback",
        "hbm copy" if roof["bound"] == "hbm" else
        "sustained bf16 x nominal ratio for the mode" if roof["bound"] == "tensor" else "derived FP32/FP64 ALU peak, DESIGN.md"))
    t_hbm = alg["bytes_step"] / (peaks["hbm_gbs"] * 1e9) * 1e3
    t_tc = alg["gemm_flops_step"] / (tensor_peak_sus * 1e12) * 1e3
    t_roof = max(t_hbm, t_tc)
    step_roof = {"t_hbm_ms": t_hbm, "t_tensor_ms": t_tc, "t_roof_ms": t_roof, "bound": "tensor" if t_tc > t_hbm else "hbm",
                 "frac": t_roof / (ms / K), "t_sum_ms": t_hbm + t_tc, "frac_of_sum": (t_hbm + t_tc) / (ms / K),
                 "tensor_peak_tflops": tensor_peak_sus, "tensor_peak_burst_tflops": tensor_peak_burst,
                 "hbm_peak_gbs": peaks["hbm_gbs"], "bytes_step": alg["bytes_step"], "gemm_flops_step": alg["gemm_flops_step"],
                 "definition": "max(stencil+density%s bytes / HBM peak, real-beta GEMM flops / tensor peak of the GEMM mode); "
                               "t_sum / frac_of_sum: the same two terms added, the bound for kernels that do not overlap "
                               "(at the power cap overlap buys little: DESIGN.md section 8)" % (
                     "+norm" if args.step in SPLIT_STEPS else "")}

    cpu = None
    if world > 1:
        cpu = {"value": None, "unit": "electron-steps/s", "cores": None, "kind": "oracle",
               "sample": "not timed at N > 1: the oracle is timed on rank 0 at N = 1 only"}
    elif not args.no_cpu_baseline:
        # a bounded sample sized for roughly 10 s of host work at configs[3] (1 warm-up + CPU_STEPS timed steps)
        s = sample_for_oracle(c, first, 2 * args.oracle_orbitals)
        v, sec_step, cores, el = time_oracle(c, s, W.laser_samples(c, nsteps=CPU_STEPS, t0=0.9), steps=CPU_STEPS, warmup=1, step=args.step)
        cpu = {"value": v, "unit": "electron-steps/s", "cores": cores, "kind": "oracle", "s_per_step": sec_step,
               "sample": "domain 0, first %d of %d orbitals (%g electrons), all %d projectors, %d timed %s steps" % (
                   s["psi"].shape[-1], c.norb, el, c.nproj, CPU_STEPS, "Eq. (2) split" if args.step in SPLIT_STEPS else "Taylor-4")}

    line = {
        "metric": "electron-steps/s", "value": value, "unit": "electron-steps/s", "n_gpus": world, "steps": K, "warmup": Wm,
        "ms_per_step": ms / K, "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "complex64",
        "data": "synthetic", "config": workload_config(c, args), "clocks": clocks, "e2e": e2e, "gpu_launches": launches,
        "roofline": roof, "cpu_baseline": cpu, "step_roofline": step_roof, "gemm_path": gemm_path,
        "kernels": per_class, "kernels_pass_ms_per_step": ms_profiled / K, "observables": observables,
        "orbital_steps_per_s": c.ndom * c.norb * world * K / (ms * 1e-3), "input_generation_s": t_gen,
        "paper_context": PAPER_CONTEXT, "also_staged": also_staged,
    }
    print(json.dumps(line))
    dom.close()
    if dist is not None:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
