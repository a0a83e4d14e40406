#!/usr/bin/env python
"""bench.py -- MLUPs of the fused HHRRLBM + wall-model step on B200 (BASELINE.json metric).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl ours|reference]

A "step" is one pass of Listing 3: rotor/porosity update, fused
collide-stream, wall model, per-element force reduction.  At N = 1 the workload is
BASELINE.json config 5: the 768x384x364 (~107 M cells) block holding one synthetic rotor of
radius 120 cells.  The path does not shard (north_star: one GPU, no collectives): with N > 1
every rank runs an independent replica ("replicas only", weak scaling), timed as the max
over ranks.  Prints ONE JSON line on rank 0.

--impl reference times the fp64 CPU oracle (oracle/) as it stands on the host cores, on a
bounded sample of the same recipe (there is no reference implementation to install; see
DESIGN.md "Reference arm").
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
sys.path.insert(0, str(ROOT))

from paper_2510_13726_b200 import inputs as I  # noqa: E402  (seeded input recipes only)

METRIC = "MLUPs (fused HHRRLBM+wall-model step) on 1 B200 and % of HBM peak GB/s"
BYTES_PER_CELL = 216.0  # D3Q27: 27 x 4 B read + 27 x 4 B write; D3Q19: 152 B


def bytes_per_cell(q: int) -> float:
    return 8.0 * q
FALLBACK_HBM_GBS = 6650.0  # /opt/skills/guides/B200_PROFILING.md fallback


def measured_peak():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            return float(json.loads(p.read_text())["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def workload(config: int, region_split: bool = False) -> tuple[I.Case, str]:
    case = I.baseline_config(config)
    if region_split:   # bulk RRLBM-LES outside boxes around the fringe / rotor / static geometry
        case = I.with_region_split(case)
    names = {1: "config1 TGV 32^3", 2: "config2 sphere channel 128x64x64", 3: "config3 half-channel 256x128x128",
             4: "config4 rotor R=80 512x256x256", 5: "config5 rotor R=120 768x384x364 (~107M cells)"}
    return case, names[config] + (" + bulk/FSI region split" if region_split else "")


# ------------------------------------------------------------------------------- clocks
class ClockSampler:
    """Samples nvidia-smi clocks / throttle reasons during the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.index, self.rows, self.proc = index, [], None

    def start(self):
        try:
            self.proc = subprocess.Popen(
                ["nvidia-smi", "-i", str(self.index), f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                 "-lms", "100"], stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.thread = threading.Thread(target=self._read, daemon=True)
            self.thread.start()
        except Exception:
            self.proc = None

    def _read(self):
        for line in self.proc.stdout:
            self.rows.append((time.time(), line.strip()))

    def stop(self, t0, t1):
        if not self.proc:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        time.sleep(0.15)
        self.proc.terminate()
        sm, smax, reasons = [], None, set()
        rows = [r for t, r in self.rows if t0 - 0.05 <= t <= t1 + 0.15] or [r for _, r in self.rows]
        for r in rows:
            c = [x.strip() for x in r.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0]))
                smax = float(c[1])
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": smax, "reasons": sorted(reasons),
                "samples": len(sm)}


# ------------------------------------------------------------------------------- CPU oracle leg
def oracle_sample(config: int, budget_s: float = 20.0, q: int = 27):
    """Times the oracle as it stands on a bounded sample of the config's recipe."""
    from oracle import oracle as O
    O.build()
    if q != 27:
        O = O.view(q)
    case, sample = reference_sample(config)
    p = O.make_params(case.nx, case.ny, case.nz, mode=case.mode, **case.params)
    L = O.Lattice(p)
    I.apply_case(case, L)
    L.step(1)  # warm-up (first-touch, geometry)
    t0 = time.perf_counter()
    steps = 0
    while True:
        L.step(1)
        steps += 1
        dt = time.perf_counter() - t0
        if dt > budget_s or steps >= 50:
            break
    L.close()
    mlups = case.n * steps / dt / 1e6
    return {"value": mlups, "unit": "MLUPs", "cores": O.threads(), "kind": "oracle",
            "sample": f"{sample}, {steps} steps in {dt:.1f} s"}, dt / steps


def reference_sample(config: int, shrink: int = 0):
    """The bounded sample of the config's recipe the oracle is timed on; shrink halves the scale again."""
    if config >= 4:
        k = 4 << shrink
        nx, ny, nz, R = 768 // k, 384 // k, 364 // k, 120.0 / k
        return (I.case_rotor(nx, ny, nz, R, 4, omega=0.002 * k),
                f"config-5 recipe scaled 1/{k} ({nx}x{ny}x{nz} cells, rotor R={R:g}, wall model + forces on)")
    if config == 3:
        return I.case_channel(128, 64, 64, 4), "config-3 recipe at 128x64x64"
    return I.baseline_config(config), f"config {config} at full size"


def run_reference(args, rank, world):
    """Reference arm: the oracle, as it stands, on the host cores (rank 0 only).  One step = one oracle
    time step (all of Listing 3) on the bounded sample lattice; W untimed warm-up steps, K timed."""
    if rank != 0:
        return
    _, wname = workload(args.config)
    from oracle import oracle as O
    O.build()
    if args.q != 27:
        O = O.view(args.q)
    # size the sample so that W + K oracle steps end within a few minutes on this host
    for shrink in range(4):
        case, sample = reference_sample(args.config, shrink)
        p = O.make_params(case.nx, case.ny, case.nz, mode=case.mode, **case.params)
        L = O.Lattice(p)
        I.apply_case(case, L)
        L.step(1)
        t0 = time.perf_counter()
        L.step(1)
        if (time.perf_counter() - t0) * (args.steps + args.warmup) <= 200.0 or shrink == 3 or args.config < 4:
            break
        L.close()
    L.step(max(0, args.warmup - 2))
    t0 = time.perf_counter()
    L.step(args.steps)
    dt = time.perf_counter() - t0
    L.close()
    value = case.n * args.steps / dt / 1e6
    cb = {"value": value, "unit": "MLUPs", "cores": O.threads(), "kind": "oracle",
          "sample": f"{sample}, {args.steps} steps in {dt:.1f} s"}
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": "MLUPs", "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": dt / args.steps * 1e3,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
            "data": "synthetic", "config": {"workload": wname, "lattice": args.lattice, "note": "each step = one oracle time step on the bounded sample"},
            "cpu_baseline": cb,
            "e2e": {"value": value, "unit": "MLUPs", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line), flush=True)


def run_ours(args, rank, world, local_rank):
    import torch
    import torch.distributed as dist
    from paper_2510_13726_b200 import binding as B, build, replicas

    build.build()
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device (the CUDA library is the only implementation)")
    torch.cuda.set_device(local_rank)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device(f"cuda:{local_rank}"))
    dev = f"cuda:{local_rank}"

    case, wname = workload(args.config, args.region_split)
    slab = None
    if args.decompose:
        # SURVEY 8(f)-3, the paper's weak-scaling layout: the ranks' blocks are stacked along z into
        # ONE periodic lattice of N x nz planes, one rotor per block; every rank holds its block plus a halo plane at
        # either end and exchanges Q planes per face after every step (paper_2510_13726_b200/slabs.py)
        import dataclasses
        from paper_2510_13726_b200 import slabs as S
        assert case.rotor is not None and case.phi is None, "--decompose: rotor recipes (configs 4, 5)"
        nzl = case.nz + 2
        rotor = dict(case.rotor, centre=(case.rotor["centre"][0], case.rotor["centre"][1], case.rotor["centre"][2] + 1.0))
        n_l = case.nx * case.ny * nzl
        u = np.zeros((3, n_l), np.float32)
        u[0] = case.fringe[2][0]
        boxes = None if case.fsi_boxes is None else [(b[0], b[1], b[2], b[3], b[4] + 1, b[5] + 1) for b in case.fsi_boxes]
        case = dataclasses.replace(case, nz=nzl, rotor=rotor, rho=np.ones(n_l, np.float32), u=u, fsi_boxes=boxes)
        wname += f" x{world} stacked along z, one block (+2 halo planes) per GPU"
    p = B.make_params(case.nx, case.ny, case.nz, mode=case.mode, **case.params)
    L = B.Lattice(p, rotor_shape=None if case.rotor is None else case.rotor["sdf"].shape, device=dev, q=args.q)
    BYTES_PER_CELL = bytes_per_cell(args.q)
    L.set_kernel_variant(args.variant)
    if args.chunk_planes or args.cluster:
        L.set_launch_shape(args.chunk_planes, args.cluster)
    I.apply_case(case, L)
    n = case.n
    if args.decompose:
        n = case.nx * case.ny * (case.nz - 2)          # real cells: halo planes are not counted as work
        slab = S.SlabLattice(L, rank, world, dist.group.WORLD if world > 1 else "self")
    stepper = slab if slab is not None else L

    def barrier():
        torch.cuda.synchronize()
        if world > 1:
            dist.barrier()
            torch.cuda.synchronize()

    stepper.step(args.warmup)
    barrier()
    sampler = ClockSampler(local_rank)
    if rank == 0:
        sampler.start()
        time.sleep(0.3)
    L.set_timing(True)
    launches0 = L.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    t_wall0 = time.time()
    ev0.record(L.stream)
    stepper.step(args.steps)
    ev1.record(L.stream)
    barrier()
    t_wall1 = time.time()
    ms = ev0.elapsed_time(ev1)
    launches = L.launch_count() - launches0
    k_ms, k_n = L.timing()
    L.set_timing(False)
    clocks = sampler.stop(t_wall0, t_wall1) if rank == 0 else None
    L.check_finite()
    ms = replicas.max_over_ranks(ms, device=dev)          # slowest replica
    value = replicas.aggregate_mlups(n, args.steps, ms, world)

    # end to end through the C ABI with HOST buffers: upload the populations from pinned host
    # memory, step, read moments and forces back -- all inside the timed region
    e2e_steps = args.steps
    h_f = torch.empty((args.q, n), dtype=torch.float32).pin_memory()
    h_rho = torch.empty(n, dtype=torch.float32).pin_memory()
    h_v = torch.empty((3, n), dtype=torch.float32).pin_memory()
    lib = B.lib(args.q)
    import ctypes as C
    L._check(lib.hhrr_get_populations(L.h, C.c_void_p(h_f.data_ptr())))
    barrier()
    e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    e0.record(L.stream)
    L._check(lib.hhrr_set_populations(L.h, C.c_void_p(h_f.data_ptr())))
    stepper.step(e2e_steps)
    L._check(lib.hhrr_get_moments(L.h, C.c_void_p(h_rho.data_ptr()), C.c_void_p(h_v.data_ptr())))
    F = L.forces(L.step_count() - min(e2e_steps, 1024), min(e2e_steps, 1024))
    e1.record(L.stream)
    barrier()
    e2e_ms = e0.elapsed_time(e1)
    e2e_ms = replicas.max_over_ranks(e2e_ms, device=dev)
    e2e = {"value": replicas.aggregate_mlups(n, e2e_steps, e2e_ms, world), "unit": "MLUPs",
           "h2d_bytes_per_step": h_f.numel() * 4 / e2e_steps,
           "d2h_bytes_per_step": (h_rho.numel() + h_v.numel()) * 4 / e2e_steps + F.nbytes / e2e_steps,
           "steps": e2e_steps, "ms_total": e2e_ms,
           "what": "hhrr_set_populations(pinned host) + hhrr_step + hhrr_get_moments(pinned host) + hhrr_get_forces"}
    thrust = float(F[-1, 1:5, 0].sum()) if case.rotor is not None else None
    # Definition 3 / Eq. 26: C_T = T / (0.5 rho pi r^2 U_inf^2), lattice units, rho = 1;
    # after a few hundred steps from rest it is a start-up value, not the converged one of the paper's Fig. 7
    # (hhrr_get_rotor_coefficients).  Torque of the rotor about its axis (+x) from hhrr_get_torques and the usual power
    # coefficient C_P = M_x Omega / (0.5 rho pi r^2 U_inf^3) (not defined in the paper, start-up value)
    c_t = torque = c_p = None
    if case.rotor is not None:
        torque = float(L.torques(L.step_count() - 1, 1)[0, 1:5, 0].sum())
        if case.fringe is not None:
            r_rot = 0.5 * (case.rotor["sdf"].shape[1] - 1) * case.rotor["spacing"] - 4.0   # grid half-extent minus its 4-cell margin
            ct, cp = L.rotor_coefficients(1.0, case.fringe[2][0], r_rot, L.step_count() - 1, 1)
            c_t, c_p = float(ct[0]), float(cp[0])

    # the same workload with the paper's bulk / FSI region split (Listing 2): reported beside the
    # headline, which keeps HHRRLBM in every cell
    split = None
    if not args.region_split and not args.no_region_split_leg and case.fringe is not None:
        boxes = I.with_region_split(case).fsi_boxes
        L.set_fsi_region(boxes)
        stepper.step(min(args.warmup, 20))
        barrier()
        L.set_timing(True)
        s0, s1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        s0.record(L.stream)
        stepper.step(args.steps)
        s1.record(L.stream)
        barrier()
        s_ms = replicas.max_over_ranks(s0.elapsed_time(s1), device=dev)
        sk_ms, sk_n = L.timing()
        L.set_timing(False)
        L.check_finite()
        split = {"value": replicas.aggregate_mlups(n, args.steps, s_ms, world), "unit": "MLUPs",
                 "ms_per_step": s_ms / args.steps, "kernel_ms": sk_ms / max(1, sk_n),
                 "kernel_frac_of_peak": n * BYTES_PER_CELL / (sk_ms / max(1, sk_n) * 1e-3) / 1e9 / measured_peak()[0],
                 "fsi_boxes": [list(map(int, b)) for b in boxes],
                 "what": "bulk RRLBM-LES (PAPER.md:215, Listing 2) outside the boxes, HHRRLBM + wall model inside"}

    if rank == 0:
        peak, peak_src = measured_peak()
        k_avg_ms = k_ms / max(1, k_n)
        achieved = n * BYTES_PER_CELL / (k_avg_ms * 1e-3) / 1e9
        roofline = {"bound": "hbm", "kernel": {0: "moments_kernel+collide_kernel", 2: "fused_ws_kernel", 5: "fused_xpull_kernel"}[args.variant],
                    "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak, "traffic": None,
                    "traffic_source": None,
                    "peak_source": peak_src, "kernel_ms": k_avg_ms, "kernel_launches_timed": k_n,
                    "kernel_share_of_step": k_ms / (ms * k_n / args.steps) if k_n else None,
                    "algorithmic_bytes_per_cell": BYTES_PER_CELL}
        # DRAM bytes per launch: NOT measured in this run -- the figure of the committed ncu capture of the same kernel,
        # lattice and launch configuration (profiles/r02_traffic.txt names the capture command); null if there is none
        tr = ROOT / "profiles" / "r02_traffic.txt"
        if tr.exists():
            try:
                for t in json.loads(tr.read_text()):
                    if (t.get("cells") == n and t.get("variant") == args.variant and t.get("lattice", "D3Q27") == args.lattice
                            and bool(t.get("region_split")) == bool(args.region_split)):
                        roofline["traffic"] = t["dram_bytes_per_launch"]
                        roofline["traffic_source"] = "committed ncu capture: " + t.get("source", "profiles/r02_traffic.txt")
            except Exception:
                pass
        cpu = None
        if world == 1 and not args.no_cpu_baseline:
            cpu, _ = oracle_sample(args.config, budget_s=15.0, q=args.q)
        line = {"metric": METRIC, "value": value, "unit": "MLUPs", "n_gpus": world, "steps": args.steps,
                "warmup": args.warmup, "ms_per_step": ms / args.steps, "higher_is_better": True,
                "scaling": "weak", "vs_baseline": None, "dtype": "f32", "data": "synthetic",
                "config": {"workload": wname, "cells_per_gpu": n, "lattice": args.lattice, "storage": "fp32 SoA A/B" + (", x-pull / yz-push" if L.population_storage() else ""),
                           "kernel_variant": args.variant, "chunk_planes": args.chunk_planes or "auto", "cluster": args.cluster or "auto",
                           "parallelism": (f"z-slabs x{world}: halo exchange of {args.q} planes per face and step (NCCL send/recv), "
                                           "per-element force all-reduce" if args.decompose else f"replicas x{world}"),
                           "l2": "inputs (%.1f GB per buffer) exceed the 126 MB L2; no flush needed" % (4e-9 * args.q * n)},
                "hbm_frac_of_peak_step": value * 1e6 * BYTES_PER_CELL / 1e9 / peak / world,
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": launches,
                "clocks": clocks, "thrust_last_step": thrust, "thrust_coefficient_last_step": c_t,
                "torque_last_step": torque, "power_coefficient_last_step": c_p,
                "region_split": split}
        print(json.dumps(line), flush=True)
    L.close()
    if world > 1:
        dist.destroy_process_group()


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=100)
    ap.add_argument("--config", type=int, default=5, choices=[1, 2, 3, 4, 5])
    ap.add_argument("--variant", type=int, default=5, choices=[0, 2, 5])
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--chunk-planes", type=int, default=0, help="planes per z-chunk of the default kernel (0: automatic)")
    ap.add_argument("--cluster", type=int, default=0, help="tiles per thread-block cluster of the default kernel (0: automatic)")
    ap.add_argument("--decompose", action="store_true",
                    help="N blocks stacked along z into one lattice with halo exchange (SURVEY 8(f)-3) instead of N replicas")
    ap.add_argument("--lattice", default="D3Q27", choices=["D3Q27", "D3Q19"],
                    help="velocity set: D3Q27 (BASELINE.json's configs, default) or the paper's own D3Q19 (PAPER.md:94)")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-region-split-leg", action="store_true", help="skip the extra region-split measurement")
    ap.add_argument("--region-split", action="store_true",
                    help="the paper's bulk / FSI region split (PAPER.md:215); default: HHRRLBM in every cell")
    args = ap.parse_args()
    args.q = 27 if args.lattice == "D3Q27" else 19
    args.warmup = max(args.warmup, 3) if args.impl == "ours" else args.warmup
    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        run_reference(args, rank, world)
    else:
        run_ours(args, rank, world, local_rank)


if __name__ == "__main__":
    main()
