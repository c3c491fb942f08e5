#!/usr/bin/env python
"""bench.py -- Wilson-loop k-points/s of the B200-native BerryEasy hot path.

One "step" = one pass of the whole hot path (eigensolve at every k, PSO projection, links, ordered
product, eigenphases) over one synthetic H_grid.  The bench line is BASELINE.json configs[3]
(20x20 BHZ supercell, N = 1600, n_occ = 800 -> 2 x 400, 24 x 25 grid, spin resolved), the
configuration the target ">= 50 % of FP64 peak" is quoted on.  The default invocation then runs the other
four configs for a few steps each and attaches them as ``config.other_workloads`` (north_star: "throughput
on the five synthetic workloads"); ``--config 1|2|3|5`` times one of them alone (not the bench line).

Contract: python bench.py --gpus N --steps K --warmup W [--impl reference]; one JSON line on rank 0.
Launched bare with --gpus N > 1 it re-launches itself under torch.distributed.run with N ranks.
Multi-GPU: the Wilson loops are independent problems; the job is N x 24 loops, rank r owns the loops
sharding.shard_range gives it (= its own seeded realization), no data-path collective, one all-gather of
the phase arrays at the end (weak scaling: per-GPU work fixed).
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
# kernel classes of the library's CUDA-event profile and the roofline that bounds each
CLASS_BOUND = {"hemv": "hbm", "colw": "hbm", "zgemm": "alu", "fused": "alu", "q2": "alu", "panel": "latency",
               "chase": "latency", "bisect": "latency", "invit": "latency", "cluster_orth": "latency",
               "hessenberg": "latency", "hqr": "latency", "jacobi": "hbm", "misc": "hbm"}
CLASS_KERNEL = {"hemv": "k_hemv", "colw": "k_colw", "zgemm": "zgemm_async_kernel", "fused": "k_fused", "q2": "k_q2",
                "panel": "k_ysum + k_mc + k_wupd + k_panel", "chase": "k_chase4", "bisect": "k_bisect", "invit": "k_invit",
                "cluster_orth": "cluster_orth.cu", "hessenberg": "k_hessenberg", "hqr": "k_hqr", "jacobi": "k_jacobi / k_small_loop",
                "misc": "k_tridiag_smem"}


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

    # rank r owns its own seeded realization(s): the job of N ranks is N x (this workload)
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
            return ctx.nested_wilson_host(Hh, self.m, 1, 0)
        return ctx.wilson_loop_host(Hh, self.m, Hh.dim() - 4)

    # bounded oracle sample: whole loops of the same matrices
    def oracle_sample(self, budget: str = "full"):
        from oracle import wilson_oracle as wo
        from paper_2312_13051_b200 import workloads as wl
        c = self.cfg
        t0 = time.perf_counter()
        if c == 4:
            # one whole loop of 25 k-points, ~13 s on the GPU box's 16 cores
            parts = wl.config4_parts(self.L, realization=self.rank)
            H = wl.supercell_grid([parts], 25, 24, t2_indices=[0])
            S = wl.supercell_spin_z(self.L)
            tb = time.perf_counter()
            wo.spin_resolved_surface(H, self.m, 1, S)
            desc = f"1 whole loop of 25 k-points of the same N={self.N} matrices (spin resolved)"
            k = 25
        elif c == 3:
            nl = 3 if budget == "full" else 2
            H = wl.supercell_grid([wl.config3_parts(0)], 33, 32, t2_indices=range(nl))
            tb = time.perf_counter()
            wo.wilson_surface(H, self.m, 1)
            desc, k = f"{nl} loops x 33 k-points, realization 0", nl * 33
        elif c == 5:
            nl = 48 if budget == "full" else 24
            H = wl.config5_grid(wl.config5_parts(), 64, 64, 65, ix=[0], iy=range(nl))
            tb = time.perf_counter()
            wo.wilson_surface(H, self.m, 1)
            desc, k = f"{nl} loops x 65 k-points (kx=0)", nl * 65
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
    """The oracle as it stands on the box's host cores, on whole loops of the same workload (config 4: one loop
    of 25 k-points of N = 1600 per sample, ~13 s).  At most ``MAX_SAMPLES`` samples are timed whatever --steps
    says, so that the run ends within a few minutes; the value is k-points per second over what was timed."""
    if rank != 0:
        return
    os.environ.setdefault("OMP_NUM_THREADS", str(os.cpu_count()))
    cores = os.cpu_count()
    MAX_SAMPLES = 8
    nwarm = 1 if args.warmup > 0 else 0
    nsamp = max(1, min(args.steps, MAX_SAMPLES))
    for _ in range(nwarm):
        wk.oracle_sample()
    vals, dts = [], []
    desc = ""
    for _ in range(nsamp):
        v, desc, dt, _ = wk.oracle_sample()
        vals.append(v); dts.append(dt)
    tot_k = sum(v * d for v, d in zip(vals, dts))
    value = tot_k / sum(dts)
    sample = f"{desc}; {nsamp} such sample(s) timed after {nwarm} warm-up"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": "k-points/s", "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * float(np.mean(dts)),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "config": {"workload": wk.name, "sample": sample, "timed_samples": nsamp},
        "cpu_baseline": {"value": value, "unit": "k-points/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": "k-points/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
def class_rooflines(prof, peaks, hbm_peak, hbm_src):
    """One roofline entry per profiled kernel class: achieved = the class's algorithmic flops (alu) or bytes
    (hbm) over its summed CUDA-event time in the instrumented pass."""
    out = {}
    for k, v in prof.items():
        if not v["launches"] or v["ms"] <= 0:
            continue
        bound = CLASS_BOUND.get(k, "latency")
        e = {"kernel": CLASS_KERNEL.get(k, k), "bound": bound, "ms": round(v["ms"], 3), "launches": v["launches"]}
        if bound == "alu":
            ach = v["flops"] / (v["ms"] * 1e-3) / 1e12
            pk = peaks["dfma_3operand"] if k == "q2" else peaks["dmma"]
            e.update(achieved=ach, peak=pk, unit="TFLOP/s", frac=ach / pk,
                     peak_source=("measured in this run: DFMA chain with three distinct register operands (what a reflector "
                                  "application issues)" if k == "q2" else "measured in this run: DMMA.8x8x4 chain (be_probe_fp64)"))
        elif bound == "hbm":
            ach = v["bytes"] / (v["ms"] * 1e-3) / 1e9
            e.update(achieved=ach, peak=hbm_peak, unit="GB/s", frac=ach / hbm_peak, peak_source=hbm_src)
        out[k] = e
    return out


def measure(ctx, wk, torch, dist, device, world, steps, warmup, sampler=None):
    """W warm-up passes, K timed passes bracketed by barrier + synchronize (CUDA events on the launching stream),
    one more instrumented pass for the per-class profile, the FP64 probes right after it."""
    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    H, S = wk.device_grid(torch, device)
    torch.cuda.synchronize()
    out = None
    for _ in range(warmup):
        out = wk.run_device(ctx, H, S)
    barrier()
    if sampler:
        sampler.start()
    n0 = ctx.launch_count()
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    ev0.record()
    for _ in range(steps):
        out = wk.run_device(ctx, H, S)      # inputs are either larger than the 126 MB L2 or (configs 1-2) tiny by definition
    ev1.record()
    barrier()
    ms = ev0.elapsed_time(ev1)
    launches = ctx.launch_count() - n0
    # Per-kernel-class CUDA-event profile: one more pass of the same step, right after the timed region and still
    # under the clock sampler, with an event pair around every launch of an instrumented kernel class (kept out
    # of the timed region: the event pairs cost time).
    ctx.profile_enable(True)
    out = wk.run_device(ctx, H, S)
    prof = ctx.profile()
    ctx.profile_enable(False)
    peaks = ctx.probe_fp64()
    t = torch.tensor([ms], dtype=torch.float64, device=device)
    if world > 1:
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
    ms_step = float(t.item()) / steps
    return {"H": H, "S": S, "out": out, "ms_step": ms_step, "launches": launches, "prof": prof, "peaks": peaks}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=2)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--config", type=int, default=None, help="time one config alone (default: 4 = the bench line, then the others)")
    ap.add_argument("--small", action="store_true", help="reduced workload for quick checks (not a bench value)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-others", action="store_true", help="skip configs 1, 2, 3, 5 after the bench line")
    ap.add_argument("--ws-gib", type=float, default=None, help="workspace cap in GiB (default: the library's)")
    ap.add_argument("--eigh-algo", type=int, default=None, choices=[0, 1, 2],
                    help="tridiagonalization: 0 one-stage, 1 two-stage, 2 auto (default: the library's = 2)")
    args = ap.parse_args()

    if args.gpus > 1 and "WORLD_SIZE" not in os.environ and args.impl == "ours":
        # launched bare: one rank per GPU under torchrun (the driver launches it this way itself)
        import socket
        s = socket.socket(); s.bind(("127.0.0.1", 0)); port = s.getsockname()[1]; s.close()
        cmd = [sys.executable, "-m", "torch.distributed.run", "--nnodes=1", f"--nproc-per-node={args.gpus}",
               "--master-addr", "127.0.0.1", "--master-port", str(port), os.path.abspath(__file__)] + sys.argv[1:]
        raise SystemExit(subprocess.call(cmd))

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    cfg = 4 if args.config is None else args.config
    wk = Workload(cfg, rank, args.small)
    if args.impl == "reference":
        reference_arm(args, wk, rank)
        return

    import torch
    import torch.distributed as dist
    from paper_2312_13051_b200.binding import Context
    from paper_2312_13051_b200 import sharding

    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device (the product has no CPU fallback)")
    torch.cuda.set_device(local)
    device = torch.device("cuda", local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", rank=rank, world_size=world, device_id=device)
    # the job: world x wk.loops independent loops; this rank's share (its own realization)
    lo_loop, hi_loop = sharding.shard_range(world * wk.loops, rank, world)
    assert hi_loop - lo_loop == wk.loops and lo_loop == rank * wk.loops

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    ctx = Context()
    if args.eigh_algo is not None:
        ctx.set_eigh_algorithm(args.eigh_algo)
    if args.ws_gib is not None:
        ctx.set_workspace_limit(int(args.ws_gib * 2 ** 30))
    sampler = ClockSampler(local)
    r = measure(ctx, wk, torch, dist, device, world, args.steps, args.warmup, sampler if rank == 0 else None)
    clocks = sampler.stop() if rank == 0 else None
    H, S, prof, peaks, ms_step = r["H"], r["S"], r["prof"], r["peaks"], r["ms_step"]
    value = world * wk.kpoints / (ms_step * 1e-3)
    # results of all ranks on every rank (KB): the only collective of the job
    if world > 1 and wk.kind != "nested":
        allph = sharding.gather_phases(r["out"][0].reshape(wk.loops, -1), world * wk.loops, rank, world)
        assert allph.shape[0] == world * wk.loops

    # ---- end to end through the host-buffer C-ABI call (H2D of the grid inside the timed region)
    e2e = None
    if not args.no_e2e:
        Hh = torch.empty(H.shape, dtype=H.dtype).pin_memory()
        Hh.copy_(H)
        Sh = S.cpu() if S is not None else None
        del H
        r["H"] = None
        torch.cuda.empty_cache()
        e2e_steps = max(1, min(args.steps, 2))
        for _ in range(2):
            o = wk.run_host(ctx, Hh, Sh)    # warm-up (allocations, page faults; the staging buffers settle on the second call)
        barrier()
        t0 = time.perf_counter()
        copied0 = ctx.host_grid_bytes_copied()
        for _ in range(e2e_steps):
            o = wk.run_host(ctx, Hh, Sh)    # synchronous: returns after the results are on the host
        torch.cuda.synchronize()
        grid_bytes = (ctx.host_grid_bytes_copied() - copied0) // e2e_steps
        dt = time.perf_counter() - t0
        tt = torch.tensor([dt], dtype=torch.float64, device=device)
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        d2h = sum(int(x.numel()) * 8 for x in o if x is not None)
        e2e = {"value": world * wk.kpoints * e2e_steps / float(tt.item()), "unit": "k-points/s",
               "h2d_bytes_per_step": int(grid_bytes) + (int(Sh.numel()) * Sh.element_size() if Sh is not None else 0),
               "host_grid_bytes": int(Hh.numel()) * 16, "host_schedule": ctx.host_schedule(),
               "d2h_bytes_per_step": d2h, "steps": e2e_steps,
               "how": "be_*_host C-ABI call on pinned host H_grid; chunked H2D overlapped with compute; h2d_bytes_per_step counts the bytes the library copies (for N >= 256 only the upper triangle of the Hermitian matrices, in 8 row blocks); wall clock, max over ranks"}
        del Hh
    else:
        del H
        r["H"] = None
    torch.cuda.empty_cache()
    ctx.release_workspace()     # the next workloads' grids (43 GB for config 3) need the memory

    # ---- configs 1, 2, 3, 5 (rank 0's numbers; every rank runs them so that the ranks stay in step)
    others = None
    if args.config is None and not args.no_others and not args.small:
        hbm_peak, hbm_src = measured_peaks()
        others = []
        for c in (1, 2, 3, 5):
            w2 = Workload(c, rank, False)
            r2 = measure(ctx, w2, torch, dist, device, world, max(2, min(args.steps, 3)), 2)
            r2["H"] = None; r2["S"] = None
            torch.cuda.empty_cache()
            ctx.release_workspace()
            roofs = class_rooflines(r2["prof"], r2["peaks"], hbm_peak, hbm_src)
            dom = max(roofs, key=lambda k: roofs[k]["ms"]) if roofs else None
            tfl = w2.flops / (r2["ms_step"] * 1e-3) / 1e12
            entry = {"workload": w2.name, "ms_per_step": r2["ms_step"], "kpoints_per_s": world * w2.kpoints / (r2["ms_step"] * 1e-3),
                     "wilson_loops_per_s": world * w2.loops / (r2["ms_step"] * 1e-3), "model_tflops": world * tfl,
                     "fp64_frac_nominal": tfl / FP64_NOMINAL_TFLOPS, "fp64_frac_measured": tfl / r2["peaks"]["dmma"],
                     "gpu_launches": r2["launches"], "l2": ("inputs larger than L2" if w2.h_bytes > 2 ** 27 else
                                                            "2.6 MB of input: L2 resident by the definition of the workload"),
                     "dominant_kernel": roofs[dom] if dom else None}
            if rank == 0 and not args.no_cpu:
                v, desc, dt, _ = w2.oracle_sample("short")
                entry["cpu_baseline"] = {"value": v, "unit": "k-points/s", "cores": os.cpu_count(), "kind": "oracle",
                                         "sample": desc, "seconds": dt}
            others.append(entry)
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # ---- roofline of the dominant kernel class (largest share of the profiled time)
    hbm_peak, hbm_src = measured_peaks()
    roofs = class_rooflines(prof, peaks, hbm_peak, hbm_src)
    tot_prof = sum(v["ms"] for v in prof.values()) or 1.0
    dom = max(roofs, key=lambda k: roofs[k]["ms"])
    d = prof[dom]
    roof = dict(roofs[dom])
    roof["kernel_class"] = dom
    if roof["bound"] == "alu":
        roof["traffic"] = None   # not the bound; DRAM bytes of the captured launches are in profiles/ (ncu)
        if dom == "zgemm":
            roof["note"] = ("achieved counts 8 M N K model flops per complex GEMM; the kernel forms a complex product from three "
                            "real DMMAs (Karatsuba), i.e. executes 3/4 of them, so frac can approach 4/3")
    else:
        # bytes the launches request from the memory system, counted by the library from the shapes of every launch
        # (matrix, panel block columns, row partials); the DRAM counters of one captured launch are in profiles/
        roof["traffic"] = d["bytes"] / max(1, d["launches"])
        roof["traffic_unit"] = "bytes per launch (requested, counted by the library per launch)"
    roof["avg_launch_ms"] = d["ms"] / max(1, d["launches"])
    roof["share_of_profiled_time"] = d["ms"] / tot_prof
    roof["classes_ms_per_step"] = {k: round(v["ms"], 3) for k, v in prof.items() if v["launches"]}
    roof["classes"] = {k: {kk: (round(vv, 4) if isinstance(vv, float) else vv) for kk, vv in e.items() if kk != "peak_source"}
                       for k, e in roofs.items()}
    roof["measured_on"] = ("one instrumented pass of the same step directly after the timed region (an event pair around every "
                           "launch costs time, so the timed steps run without them)")

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
                   "parallelism": f"{world} rank(s) x {wk.loops} independent loops (rank r: realization r), no data-path collective, "
                                  "one all-gather of the phases",
                   "wilson_loops_per_s": world * wk.loops / (ms_step * 1e-3),
                   "model_tflops": tflops, "fp64_frac_nominal": tflops / (world * FP64_NOMINAL_TFLOPS),
                   "fp64_peak_measured_tflops": peaks, "fp64_frac_measured": tflops / (world * peaks["dmma"]),
                   "fp64_peak_how": "be_probe_fp64 right after the instrumented pass, same process, same clocks",
                   "flop_model": "16/3 N^3 + 8 N^2 m + GEMM flops (SURVEY 8(d))",
                   "other_workloads": others},
        "e2e": e2e, "gpu_launches": r["launches"], "clocks": clocks, "roofline": roof, "cpu_baseline": cpu,
    }
    print(json.dumps(line), flush=True)
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
