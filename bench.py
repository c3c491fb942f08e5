#!/usr/bin/env python
"""bench.py -- Wilson-loop k-points/s of the B200-native BerryEasy hot path.

One "step" = one pass of the whole hot path (eigensolve at every k, PSO projection, links, ordered
product, eigenphases) over one synthetic H_grid.  Default workload: BASELINE.json configs[3]
(20x20 BHZ supercell, N = 1600, n_occ = 800 -> 2 x 400, 24 x 25 grid, spin resolved), the
configuration the target ">= 50 % of FP64 peak" is quoted on.  ``--config 1|2|3|5`` selects the
other workloads (parity-test cases; not the bench line).

Contract: python bench.py --gpus N --steps K --warmup W [--impl reference]; one JSON line on rank 0.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

import numpy as np

METRIC = "Wilson-loop k-points/sec (eigh+overlap chain), FP64 fraction of B200 peak"
FP64_NOMINAL_TFLOPS = 37.2   # 148 SMs x 64 FMA/clk x 2 x 1.965 GHz


# ------------------------------------------------------------------------------------------------
def model_flops_per_kpoint(N: int, m: int, spin: bool, m_lo: int | None = None) -> float:
    """SURVEY 8(d) flop model (real flops, 8 per complex multiply-add); tridiagonal solve, W
    eigen-solve and Jacobi sweeps count as zero."""
    f = 16.0 / 3.0 * N ** 3 + 8.0 * N * N * m
    if not spin:
        return f + 8.0 * N * m * m + 8.0 * m ** 3
    ml = m // 2 if m_lo is None else m_lo
    mh = m - ml
    f += 8.0 * N * m * m                       # U^H S U
    f += (16.0 / 3.0 + 8.0) * m ** 3           # PSO eigh, all vectors
    f += 8.0 * N * m * m                       # rotation into the sectors
    for ms in (ml, mh):
        f += 8.0 * N * ms * ms + 8.0 * ms ** 3
    return f


class Workload:
    def __init__(self, cfg: int, rank: int, small: bool):
        self.cfg, self.rank, self.small = cfg, rank, small
        if cfg == 4:
            self.L = 8 if small else 20
            self.N, self.m = 4 * self.L ** 2, 2 * self.L ** 2
            self.n1, self.n2, self.batch = 25, (4 if small else 24), 1
            self.spin, self.kind = True, "spin_resolved"
            self.name = f"configs[3]: BHZ {self.L}x{self.L} supercell N={self.N} n_occ={self.m}, Zeeman impurities 5%, grid {self.n2}x{self.n1}, spin-resolved Wilson loop"
        elif cfg == 3:
            self.L = 10
            self.N, self.m = 400, 200
            self.n1, self.n2, self.batch = 33, 32, (2 if small else 16)
            self.spin, self.kind = False, "wilson"
            self.name = f"configs[2]: BHZ 10x10 supercell N=400 n_occ=200, Anderson W=2, grid 32x33, {self.batch} realizations"
        elif cfg == 5:
            self.N, self.m = 64, 32
            self.n1, self.n2, self.batch = 65, 64, (4 if small else 64)
            self.spin, self.kind = False, "wilson"
            self.name = f"configs[4]: Wannier-like 64 orbitals n_occ=32, {self.batch}x64 loops of 65 kz points"
        elif cfg == 1:
            self.N, self.m, self.n1, self.n2, self.batch = 4, 2, 100, 101, 1
            self.spin, self.kind = True, "spin_resolved"
            self.name = "configs[0]: BHZ 4-band 101 loops x 100 kx, spin resolved"
        elif cfg == 2:
            self.N, self.m, self.n1, self.n2, self.batch = 4, 2, 100, 100, 1
            self.spin, self.kind = False, "nested"
            self.name = "configs[1]: BBH 100x100 nested Wilson loop"
        else:
            raise SystemExit("config must be 1..5")
        self.loops = self.batch * self.n2
        self.kpoints = self.loops * self.n1
        self.flops = self.kpoints * model_flops_per_kpoint(self.N, self.m, self.spin)
        self.h_bytes = self.kpoints * self.N * self.N * 16

    # weak scaling: every rank runs the full workload on its own seeded realization
    def device_grid(self, torch, device):
        from paper_2312_13051_b200 import workloads as wl
        c, r = self.cfg, self.rank
        if c == 4:
            parts = wl.config4_parts(self.L, realization=r)
            H = wl.supercell_grid_torch([parts], self.n1, 24, device, t2_indices=range(self.n2))
            S = torch.from_numpy(wl.supercell_spin_z(self.L)).to(device)
            return H, S
        if c == 3:
            parts = [wl.config3_parts(16 * r + i) for i in range(self.batch)]
            return wl.supercell_grid_torch(parts, self.n1, self.n2, device), None
        if c == 5:
            parts = wl.config5_parts(seed=wl.BASE_SEED + r)
            H = wl.config5_grid_torch(parts, 64, 64, 65, device, ix=range(self.batch))
            return H, None
        if c == 1:
            return torch.from_numpy(wl.config1_grid()[None]).to(device), torch.from_numpy(wl.bhz4_spin_z()).to(device)
        return torch.from_numpy(wl.config2_grid()[None]).to(device), None

    def run_device(self, ctx, H, S):
        if self.kind == "spin_resolved":
            return ctx.spin_resolved_wilson(H, self.m, 1, S)
        if self.kind == "nested":
            return ctx.nested_wilson(H, self.m, 1, 0)
        return ctx.wilson_loop(H, self.m, H.dim() - 4)

    def run_host(self, ctx, Hh, Sh):
        if self.kind == "spin_resolved":
            return ctx.spin_resolved_wilson_host(Hh, self.m, Hh.dim() - 4, Sh)
        if self.kind == "nested":
            return None
        return ctx.wilson_loop_host(Hh, self.m, Hh.dim() - 4)

    # bounded oracle sample: whole loops cut to ``pts`` points of the same matrices
    def oracle_sample(self, pts4: int = 25):
        from oracle import wilson_oracle as wo
        from paper_2312_13051_b200 import workloads as wl
        c = self.cfg
        t0 = time.perf_counter()
        if c == 4:
            pts = pts4          # 25 = one whole loop, ~13 s on the GPU box's 16 cores
            parts = wl.config4_parts(self.L, realization=self.rank)
            H = wl.supercell_grid([parts], pts, 24, t2_indices=[0])
            S = wl.supercell_spin_z(self.L)
            tb = time.perf_counter()
            wo.spin_resolved_surface(H, self.m, 1, S)
            desc = f"1 loop of {pts} k-points of the same N={self.N} matrices (spin resolved)"
            k = pts
        elif c == 3:
            H = wl.supercell_grid([wl.config3_parts(0)], 33, 32, t2_indices=range(3))
            tb = time.perf_counter()
            wo.wilson_surface(H, self.m, 1)
            desc, k = "3 loops x 33 k-points, realization 0", 99
        elif c == 5:
            H = wl.config5_grid(wl.config5_parts(), 64, 64, 65, ix=[0], iy=range(48))
            tb = time.perf_counter()
            wo.wilson_surface(H, self.m, 1)
            desc, k = "48 loops x 65 k-points (kx=0)", 48 * 65
        elif c == 1:
            H = wl.config1_grid()[None]
            tb = time.perf_counter()
            wo.spin_resolved_surface(H, 2, 1, wl.bhz4_spin_z())
            desc, k = "whole config", self.kpoints
        else:
            H = wl.config2_grid()
            tb = time.perf_counter()
            wo.nested_wilson(H, 2)
            desc, k = "whole config", self.kpoints
        dt = time.perf_counter() - tb
        return k / dt, desc, dt, time.perf_counter() - t0


# ------------------------------------------------------------------------------------------------
class ClockSampler:
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index: int):
        self.rows, self.proc, self.index = [], None, index

    def start(self):
        try:
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.index}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "200"],
                                         stdout=subprocess.PIPE, stderr=subprocess.DEVNULL, text=True)
            self.t = threading.Thread(target=self._read, daemon=True)
            self.t.start()
        except Exception:
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
        except Exception:
            self.proc.kill()
        sm, mx, reasons = [], None, set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for r in self.rows:
            try:
                sm.append(float(r[0])); mx = float(r[1])
                for n, v in zip(names, r[3:7]):
                    if v.lower().startswith("active"):
                        reasons.add(n)
            except Exception:
                pass
        return {"sm_mhz": float(np.median(sm)) if sm else None, "sm_max_mhz": mx,
                "reasons": sorted(reasons), "samples": len(sm)}


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        try:
            d = json.load(open(p))
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


# ------------------------------------------------------------------------------------------------
def reference_arm(args, wk: Workload, rank: int):
    if rank != 0:
        return
    os.environ.setdefault("OMP_NUM_THREADS", str(os.cpu_count()))
    cores = os.cpu_count()
    nwarm = max(0, min(args.warmup, 1))
    # bounded sample per step: the whole run stays within a few minutes whatever --steps says
    pts4 = max(4, min(25, 100 // max(1, args.steps + nwarm)))
    for _ in range(nwarm):
        wk.oracle_sample(pts4)
    vals, dts = [], []
    for _ in range(args.steps):
        v, desc, dt, _ = wk.oracle_sample(pts4)
        vals.append(v); dts.append(dt)
    tot_k = sum(v * d for v, d in zip(vals, dts))
    value = tot_k / sum(dts)
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "k-points/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(dts)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": wk.name, "sample": desc},
        "cpu_baseline": {"value": value, "unit": "k-points/s", "cores": cores, "kind": "oracle", "sample": desc},
        "e2e": {"value": value, "unit": "k-points/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=4)
    ap.add_argument("--small", action="store_true", help="reduced workload for quick checks (not a bench value)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--ws-gib", type=float, default=None, help="workspace cap in GiB (default: the library's)")
    ap.add_argument("--eigh-algo", type=int, default=None, choices=[0, 1, 2],
                    help="tridiagonalization: 0 one-stage, 1 two-stage (default: the library's)")
    args = ap.parse_args()

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    wk = Workload(args.config, rank, args.small)
    if args.impl == "reference":
        reference_arm(args, wk, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_2312_13051_b200.binding import Context

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=device)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    ctx = Context()
    if args.eigh_algo is not None:
        ctx.set_eigh_algorithm(args.eigh_algo)
    if args.ws_gib is not None:
        ctx.set_workspace_limit(int(args.ws_gib * 2 ** 30))
    H, S = wk.device_grid(torch, device)
    torch.cuda.synchronize()

    for _ in range(args.warmup):
        out = wk.run_device(ctx, H, S)
    barrier()
    sampler = ClockSampler(local)
    if rank == 0:
        sampler.start()
    n0 = ctx.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(args.steps):
        out = wk.run_device(ctx, H, S)      # inputs (>= 24 GB for the default workload) exceed the 126 MB L2
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = ctx.launch_count() - n0
    # Per-kernel-class CUDA-event profile (roofline): one more pass of the same step, right after the timed
    # region and still under the clock sampler, with an event pair around every launch of an instrumented
    # kernel class.  It is kept out of the timed region because ~10 000 event pairs per step cost ~2.5 %.
    ctx.profile_enable(True)
    out = wk.run_device(ctx, H, S)
    prof = ctx.profile()
    ctx.profile_enable(False)
    prof_steps = 1
    clocks = sampler.stop() if rank == 0 else None
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms = float(t.item())
    ms_step = ms / args.steps
    value = world * wk.kpoints / (ms_step * 1e-3)

    # ---- end to end through the host-buffer C-ABI call (H2D of the grid inside the timed region)
    e2e = None
    if not args.no_e2e and wk.kind != "nested":
        Hh = torch.empty(H.shape, dtype=H.dtype).pin_memory()
        Hh.copy_(H)
        Sh = S.cpu() if S is not None else None
        del H
        torch.cuda.empty_cache()
        e2e_steps = max(1, min(args.steps, 2))
        o = wk.run_host(ctx, Hh, Sh)        # warm-up (allocations, page faults)
        barrier()
        t0 = time.perf_counter()
        for _ in range(e2e_steps):
            o = wk.run_host(ctx, Hh, Sh)    # synchronous: returns after the results are on the host
        torch.cuda.synchronize()
        dt = time.perf_counter() - t0
        tt = torch.tensor([dt], dtype=torch.float64, device=device)
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        d2h = sum(int(x.numel()) * 8 for x in o if x is not None)
        e2e = {"value": world * wk.kpoints * e2e_steps / float(tt.item()), "unit": "k-points/s",
               "h2d_bytes_per_step": int(Hh.numel()) * 16 + (int(Sh.numel()) * Sh.element_size() if Sh is not None else 0),
               "d2h_bytes_per_step": d2h, "steps": e2e_steps,
               "how": "be_*_host C-ABI call on pinned host H_grid; chunked H2D overlapped with compute; wall clock, max over ranks"}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel class (largest share of the profiled time)
    peak, peak_src = measured_peaks()
    tot_prof = sum(v["ms"] for v in prof.values()) or 1.0
    dom = max(prof, key=lambda k: prof[k]["ms"])
    d = prof[dom]
    if dom == "zgemm":
        ach = d["flops"] / (d["ms"] * 1e-3) / 1e12
        roof = {"kernel": dom, "bound": "alu", "achieved": ach, "peak": FP64_NOMINAL_TFLOPS, "unit": "TFLOP/s",
                "frac": ach / FP64_NOMINAL_TFLOPS, "traffic": None,
                "peak_source": "nominal FP64 (DESIGN.md Peaks): 148 SM x 64 FMA/clk x 2 x 1.965 GHz"}
    else:
        ach = d["bytes"] / (d["ms"] * 1e-3) / 1e9
        roof = {"kernel": dom, "bound": "hbm", "achieved": ach, "peak": peak, "unit": "GB/s",
                "frac": ach / peak,
                # bytes per launch, like `achieved`: the DRAM read + write of the one captured launch exceeds
                # its algorithmic bytes by the factor below; that factor is applied to the mean launch
                "traffic": 1.065 * d["bytes"] / max(1, d["launches"]), "traffic_unit": "bytes per launch",
                "algorithmic_bytes_per_launch": d["bytes"] / max(1, d["launches"]), "peak_source": peak_src,
                # one ncu --set full capture of one launch (profiles/r01h_hemv_ncu_details.md): DRAM
                # read + write 5.135 GB for 4.82 GB algorithmic; `achieved` averages over all launches,
                # so the per-launch capture is reported as a ratio, not as `traffic`
                "traffic_over_algorithmic_ncu": 1.065}
    roof["launches"] = d["launches"]
    roof["avg_launch_ms"] = d["ms"] / max(1, d["launches"])
    roof["share_of_profiled_time"] = d["ms"] / tot_prof
    roof["classes_ms_per_step"] = {k: round(v["ms"] / prof_steps, 3) for k, v in prof.items() if v["launches"]}
    roof["measured_on"] = "one instrumented pass of the same step directly after the timed region (event pairs around every launch cost ~2.5 %, so the timed steps run without them)"

    cpu = None
    if not args.no_cpu:
        v, desc, dt, _ = wk.oracle_sample()
        cpu = {"value": v, "unit": "k-points/s", "cores": os.cpu_count(), "kind": "oracle", "sample": desc,
               "seconds": dt}
    tflops = world * wk.flops / (ms_step * 1e-3) / 1e12
    line = {
        "metric": METRIC, "value": value, "unit": "k-points/s", "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": wk.name, "loops_per_gpu": wk.loops, "kpoints_per_gpu": wk.kpoints,
                   "l2": f"inputs larger than L2 ({wk.h_bytes / 1e9:.1f} GB H_grid per GPU)",
                   "parallelism": f"replicated workload per GPU (weak), {world} rank(s), no data-path collective",
                   "wilson_loops_per_s": world * wk.loops / (ms_step * 1e-3),
                   "model_tflops": tflops, "fp64_frac_nominal": tflops / (world * FP64_NOMINAL_TFLOPS),
                   "flop_model": "16/3 N^3 + 8 N^2 m + GEMM flops (SURVEY 8(d))"},
        "e2e": e2e, "gpu_launches": launches, "clocks": clocks, "roofline": roof, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
