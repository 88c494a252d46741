#!/usr/bin/env python
"""bench.py -- cell-updates/s per full RK2 step of the AMR finite-volume hot path on B200.

One "step" = one pass of the whole hot path over one level/hierarchy: CFL reduction, ghost
fill, RK stage 1, ghost fill, RK stage 2 (plus restriction/refluxing on AMR workloads).
Default workload: BASELINE.json configs[4] (512^3 uniform periodic Euler stress test, 32768
patches of 16^3), the configuration the metric is quoted on, in fp64; the same workload in fp32
is timed right after it and reported as the sub-record "fp32" of the same JSON line (the
configuration names both precisions).  Inputs are seeded and synthetic
(paper_0910_5547_b200/workloads.py).  Prints ONE JSON line on rank 0: value (device-resident),
e2e (host buffers through amrhydro_advance_host), roofline of the stage kernel (algorithmic
bytes / CUDA-event time / measured HBM peak, plus the ncu DRAM bytes and the issue / FP64-pipe
fractions), cpu_baseline (the oracle on the host cores), clocks (NVML samples in the timed region).
--workload cfg3 (AMR) runs amrhydro_advance as one CUDA-graph replay per coarse step.
Single-level workloads are built in the "zstrip" table order (--order; workloads.build_hierarchy): the launch order in
which sibling halos hit in L2 (real DRAM traffic 1.2x instead of 1.44x the algorithmic bytes; any order gives the same bits).
--gpus N (torchrun): N independent replicas, weak scaling, max-over-ranks timing.
--impl reference: the CPU oracle on a bounded sample (there is no reference implementation).

  python bench.py [--gpus N] [--steps K] [--warmup W] [--dtype f64|f32] [--impl ours|reference]
                  [--workload cfg5|cfg2|cfg4|cfg4g|cfg3] [--size S] [--halo 0|1] [--graph 0|1] [--no-fp32]
                  [--order zstrip|morton|linear]
"""
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

from paper_0910_5547_b200 import workloads as wl  # noqa: E402

# dram__bytes_read.sum + dram__bytes_write.sum per rk_stage launch from the `ncu --set full`
# capture summarised under profiles/ (None until a capture of this configuration exists).
NCU_TRAFFIC = {}
try:
    with open(os.path.join(ROOT, "profiles", "traffic.json")) as _f:
        NCU_TRAFFIC = json.load(_f)
except Exception:
    pass


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--dtype", default="f64", choices=["f64", "f32"])
    ap.add_argument("--workload", default="cfg5", choices=["cfg5", "cfg2", "cfg4", "cfg4g", "cfg3"])
    ap.add_argument("--size", type=int, default=0, help="cells per side (default: the config's own size)")
    ap.add_argument("--halo", type=int, default=1, help="1: rk_stage reads sibling interiors directly")
    ap.add_argument("--kernel", type=int, default=3, help="3 = k_rk_stage_pair (nvars = 5; k_rk_stage_march otherwise), 2 = k_rk_stage_march, 0 = reference")
    ap.add_argument("--zsplit", type=int, default=2, help="AMRHYDRO_OPT_ZSPLIT (2 = automatic)")
    ap.add_argument("--fuse-cfl", type=int, default=2, help="AMRHYDRO_OPT_FUSE_CFL (2 = library default)")
    ap.add_argument("--graph", type=int, default=1, help="AMRHYDRO_OPT_GRAPH for the AMR workload (cfg3): one CUDA-graph replay per coarse step")
    ap.add_argument("--order", default="zstrip", help="patch order of the single-level workloads: zstrip (strips of 8 rows, z outermost: "
                    "sibling halos hit in L2), morton, linear")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-fp32", action="store_true", help="skip the fp32 sub-record of the default fp64 run (cfg5, cfg2)")
    ap.add_argument("--e2e-steps", type=int, default=2)
    return ap.parse_args()


WORKLOADS = {
    "cfg5": dict(size=512, gamma=1.4, nv=5, cfl=0.3, name="cfg5_euler_stress_512^3_periodic"),
    "cfg2": dict(size=256, gamma=5.0 / 3.0, nv=5, cfl=0.3, name="cfg2_kelvin_helmholtz_256^3_periodic"),
    "cfg4": dict(size=128, gamma=5.0 / 3.0, nv=8, cfl=0.3, name="cfg4_mhd_turbulence_128^3_periodic"),
    "cfg4g": dict(size=128, gamma=5.0 / 3.0, nv=9, cfl=0.3, name="cfg4_glm_mhd_9var_128^3_periodic (NEXT-1: psi = 0 initially, c_h = 1, c_r = 0.18)"),
    "cfg3": dict(size=64, gamma=1.4, nv=5, cfl=0.3, name="cfg3_sedov_amr_64^3+4levels, criterion-built hierarchy (S16: 64+64+160+432+1880 patches)"),
}


def make_workload(name, size, seed_shift=0, order="zstrip"):
    """Returns (hierarchy, U[npatch][nv][16][16][16] float64, cell-updates per coarse step)."""
    w = WORKLOADS[name]
    n = size or w["size"]
    if name == "cfg3":
        # reading S16: the hierarchy built by the configuration's own criterion (tests/golden/make_cfg3_hierarchy.py,
        # oracle only); the nested-ball stand-in only when --size asks for another base grid
        if n == w["size"]:
            h = wl.blocks_hierarchy(os.path.join(ROOT, "tests", "golden", "cfg3_blocks.txt"), n // 16)
        else:
            h = wl.ball_hierarchy(n // 16, 5, bc=(1,) * 6)
        U = wl.sedov_hierarchy_state(h, gamma=w["gamma"])
        upd = sum(int((h["level"] == l).sum()) * 4096 * (1 << l) for l in range(h["nlevels"]))
        return h, U, upd
    h = wl.uniform_hierarchy(n // 16, periodic=True, order=order)
    if name == "cfg5":
        G = wl.stress_global(n, gamma=w["gamma"], seed=20005 + seed_shift)
    elif name == "cfg2":
        G = wl.kelvin_helmholtz_global(n, gamma=w["gamma"], seed=20002 + seed_shift)
    else:
        G = wl.mhd_turbulence_global(n, gamma=w["gamma"], seed=20004 + seed_shift)
        if name == "cfg4g":
            G = np.concatenate([G, np.zeros_like(G[:1])])
    U = wl.split_global(h, G)
    del G
    return h, U, n ** 3


class ClockSampler:
    """SM clock, power and throttle reasons sampled through NVML every ~5 ms by a thread while the
    timed region runs (the recipe's nvidia-smi line starts too slowly for a region of ~0.1 s)."""

    def __init__(self, index):
        import threading
        self.rows, self.stop_flag, self.err = [], False, None
        try:
            import pynvml as nv
            nv.nvmlInit()
            self.nv = nv
            self.h = nv.nvmlDeviceGetHandleByIndex(index)
            self.max = float(nv.nvmlDeviceGetMaxClockInfo(self.h, nv.NVML_CLOCK_SM))
        except Exception as e:      # no NVML: report no samples rather than invent them
            self.nv, self.err = None, repr(e)
            return
        self.t = threading.Thread(target=self._run, daemon=True)
        self.t.start()

    def _run(self):
        nv = self.nv
        while not self.stop_flag:
            try:
                self.rows.append((float(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)),
                                  nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0,
                                  int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                                  if hasattr(nv, "nvmlDeviceGetCurrentClocksEventReasons")
                                  else int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))))
            except Exception as e:
                self.err = repr(e)
                break
            time.sleep(0.005)

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.nv is None:
            out["error"] = self.err
            return out
        self.stop_flag = True
        self.t.join(timeout=2)
        nv = self.nv
        names = {"hw_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwSlowdown", 0x8),
                 "hw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonHwThermalSlowdown", 0x40),
                 "sw_thermal_slowdown": getattr(nv, "nvmlClocksThrottleReasonSwThermalSlowdown", 0x20),
                 "sw_power_cap": getattr(nv, "nvmlClocksThrottleReasonSwPowerCap", 0x4)}
        if self.rows:
            allr = 0
            for _, _, r in self.rows:
                allr |= r
            out.update(sm_mhz=float(np.median([r[0] for r in self.rows])), sm_max_mhz=self.max,
                       reasons=sorted(k for k, bit in names.items() if allr & bit), samples=len(self.rows),
                       power_w_max=float(max(r[1] for r in self.rows)))
        return out


def peaks():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs)"
    except Exception:
        return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


def cpu_oracle_rate(name, size, seconds=10.0, dtype="f64"):
    """The oracle as it stands on the host cores, on a bounded sample of the same workload:
    a contiguous 64^3 block (4x4x4 patches) of the workload's initial data, periodic on the
    block; full RK2 steps until `seconds` of wall time have elapsed (at least 2 steps)."""
    import oracle
    w = WORKLOADS[name]
    cores = os.cpu_count() or 1
    if name == "cfg3":
        h, U, upd = make_workload("cfg3", size)
        sample = "whole cfg3 hierarchy (%d patches), coarse steps" % len(h["level"])
    else:
        h, U, upd = make_workload(name, 64)
        sample = "64^3 block (64 patches) generated by the same recipe, periodic, full RK2 steps"
    o = oracle.Oracle(h, w["gamma"], w["nv"], bits=64, threads=cores)
    o.upload(0, U)
    if name != "cfg3":
        o.advance(w["cfl"])  # warm-up (page-in); a coarse step of cfg3 alone is ~10-25 s of CPU work
    t0 = time.perf_counter()
    n = 0
    while n < (1 if name == "cfg3" else 2) or time.perf_counter() - t0 < seconds:
        o.advance(w["cfl"])
        n += 1
    dt = time.perf_counter() - t0
    return upd * n / dt, cores, sample + ", %d steps in %.1f s" % (n, dt), dt / n


def max_over_ranks(x, dist=None, device="cpu"):
    """Multi-GPU timing rule: every duration is the MAX over ranks (one process per GPU)."""
    if dist is None:
        return float(x)
    import torch
    t = torch.tensor([float(x)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def whole_job_rate(units_per_rank_step, world, steps, ms):
    """Weak scaling over independent replicas: units all ranks processed / the slowest rank's time."""
    return units_per_rank_step * world * steps / (ms * 1e-3)


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w = WORKLOADS[args.workload]
    rate, cores, sample, per_step = cpu_oracle_rate(args.workload, args.size, seconds=max(5.0, 2.0 * args.steps))
    line = {
        "impl": "reference", "metric": "cell-updates/sec per RK2 step", "value": rate, "unit": "cell-updates/s",
        "n_gpus": args.gpus, "steps": args.steps, "warmup": args.warmup, "ms_per_step": per_step * 1e3,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "config": {"workload": w["name"], "note": "CPU oracle (oracle/amr_oracle.cpp) on a bounded sample"},
        "cpu_baseline": {"value": rate, "unit": "cell-updates/s", "cores": cores, "kind": "oracle", "sample": sample},
        "e2e": {"value": rate, "unit": "cell-updates/s", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line))


def run_ours(args):
    import torch
    from paper_0910_5547_b200 import binding

    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: the amrhydro path has no CPU fallback")
    torch.cuda.set_device(local)
    dist = None
    if world > 1:
        import torch.distributed as dist
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    w = WORKLOADS[args.workload]
    nv, gamma, cfl = w["nv"], w["gamma"], w["cfl"]
    h, U, upd_per_step = make_workload(args.workload, args.size, seed_shift=rank, order=args.order)
    npatch = len(h["level"])
    single = h["nlevels"] == 1
    esz = 8 if args.dtype == "f64" else 4
    npdt = np.float64 if args.dtype == "f64" else np.float32
    g = binding.AmrHydro(h, gamma, nv, dtype=args.dtype, halo=args.halo, kernel=args.kernel, zsplit=args.zsplit, fuse_cfl=args.fuse_cfl,
                         graph=0 if single else args.graph, device="cuda:%d" % local)
    host_in = torch.empty((npatch, nv, 16, 16, 16), dtype=torch.float64 if esz == 8 else torch.float32, pin_memory=True)
    host_in.numpy()[...] = U.astype(npdt, copy=False)
    del U
    g.upload_ptr(0, 0, npatch, host_in.data_ptr())
    g.sync()

    ev = lambda: torch.cuda.Event(enable_timing=True)

    def barrier():
        torch.cuda.synchronize()
        if dist is not None:
            dist.barrier()
            torch.cuda.synchronize()

    def measure(g, dtype):
        """W warm-up steps, then K timed steps (CUDA events on the library's stream = torch's current stream, barrier +
        synchronize on both sides, max over ranks); per-stage events inside the timed region for the roofline."""
        esz = 8 if dtype == "f64" else 4
        stage_ev = []

        def step(record=False):
            if single:
                dt = g.cfl_dt(0, 0, cfl)
                g.fill_ghosts(0, 0)
                if record:
                    e0, e1, e2, e3 = ev(), ev(), ev(), ev()
                    e0.record()
                g.rk_stage(0, 0, 0, 1, 0.0, 1.0, dt)
                if record:
                    e1.record()
                g.fill_ghosts(0, 1)
                if record:
                    e2.record()
                g.rk_stage(0, 1, 0, 0, 0.5, 0.5, dt)
                if record:
                    e3.record()
                    stage_ev.append((e0, e1, e2, e3))
            else:
                g.advance(cfl, want_dt=False)          # (no host read of dt: with the graph the step does not synchronise)

        for _ in range(max(3, args.warmup)):
            step()
        barrier()
        g.get_counter(binding.CNT_LAUNCHES, reset=True)
        sampler = ClockSampler(local) if rank == 0 else None
        t0, t1 = ev(), ev()
        t0.record()
        for _ in range(args.steps):
            step(record=True)
        t1.record()
        barrier()
        ms = t0.elapsed_time(t1)
        clocks = sampler.stop() if sampler else {}
        launches = g.get_counter(binding.CNT_LAUNCHES)
        ms = max_over_ranks(ms, dist, "cuda")
        ms_per_step = ms / args.steps
        value = whole_job_rate(upd_per_step, world, args.steps, ms)

        # finiteness of the state after the timed run (S4 warning): sample the first patches
        chk = g.download(0, 0, min(npatch, 64))
        finite = bool(np.isfinite(chk).all())

        # roofline of the dominant kernel (rk_stage): algorithmic bytes / measured launch time
        peak, peak_src = peaks()
        roof = None
        if stage_ev:
            s1 = float(np.mean([a.elapsed_time(b) for a, b, _, _ in stage_ev]))
            s2 = float(np.mean([c.elapsed_time(d) for _, _, c, d in stage_ev]))
            cells = npatch * 4096
            b1, b2 = 2 * nv * esz * cells, 3 * nv * esz * cells       # stage 1: read U write U1; stage 2: + read Un
            avg_ms = 0.5 * (s1 + s2)
            ach = 0.5 * (b1 + b2) / (avg_ms * 1e-3) / 1e9
            key = "%s_%s" % (args.workload, dtype) if not args.size else "%s_%d_%s" % (args.workload, args.size, dtype)
            traffic = NCU_TRAFFIC.get(key)
            roof = {"bound": "hbm", "kernel": {0: "k_rk_stage_ref", 2: "k_rk_stage_march", 3: "k_rk_stage_pair" if nv == 5 else "k_rk_stage_march"}[args.kernel],
                    "achieved": ach, "peak": peak, "unit": "GB/s", "frac": ach / peak,
                    "traffic": traffic, "peak_source": peak_src,
                    "algorithmic_bytes_per_launch": 0.5 * (b1 + b2),
                    # the same launches in real DRAM bytes (ncu dram__bytes_read + write per launch, profiles/traffic.json)
                    "dram_frac": (traffic / (avg_ms * 1e-3) / 1e9 / peak) if traffic else None,
                    "stage1": {"ms": s1, "GB/s": b1 / (s1 * 1e-3) / 1e9, "bytes_per_cell": 2 * nv * esz},
                    "stage2": {"ms": s2, "GB/s": b2 / (s2 * 1e-3) / 1e9, "bytes_per_cell": 3 * nv * esz},
                    "share_of_step": (s1 + s2) / ms_per_step,
                    "frac_of_nominal_8TBs": ach / 8000.0}
            # the arithmetic side of the same kernel: executed thread-instructions
            # per cell and stage from the committed ncu capture / the SM's issue and FP64-pipe rates
            ipc = (NCU_TRAFFIC.get("instr_per_cell_stage") or {}).get(key)
            if ipc:
                clk = (clocks.get("sm_mhz") or 1965.0) * 1e6
                alu = {"bound": "alu", "unit": "G thread-instr/s", "sm_mhz": clk / 1e6,
                       "issue": {"instr_per_cell_stage": ipc["total"], "achieved": ipc["total"] * cells / (avg_ms * 1e-3) / 1e9,
                                 "peak": 148 * 128 * clk / 1e9}}
                alu["issue"]["frac"] = alu["issue"]["achieved"] / alu["issue"]["peak"]
                if "fp64" in ipc:
                    alu["fp64_pipe"] = {"instr_per_cell_stage": ipc["fp64"], "achieved": ipc["fp64"] * cells / (avg_ms * 1e-3) / 1e9,
                                        "peak": 148 * 64 * clk / 1e9}
                    alu["fp64_pipe"]["frac"] = alu["fp64_pipe"]["achieved"] / alu["fp64_pipe"]["peak"]
                roof["alu"] = alu
        return dict(value=value, ms_per_step=ms_per_step, roofline=roof, clocks=clocks, launches=int(launches), finite=finite)

    m = measure(g, args.dtype)
    value, ms_per_step, roof, clocks, launches, finite = (m[k] for k in ("value", "ms_per_step", "roofline", "clocks", "launches", "finite"))

    # the other precision the configuration names (BASELINE.json configs[1] and [4]: "run in fp32 and fp64"): the same
    # workload, steps and timing rules in fp32, reported as a sub-record; the top-level value stays fp64
    fp32 = None
    if args.dtype == "f64" and args.workload in ("cfg5", "cfg2") and not args.no_fp32:
        g32 = binding.AmrHydro(h, gamma, nv, dtype="f32", halo=args.halo, kernel=args.kernel, zsplit=args.zsplit, fuse_cfl=args.fuse_cfl, device="cuda:%d" % local)
        h32 = torch.empty((npatch, nv, 16, 16, 16), dtype=torch.float32, pin_memory=True)
        h32.numpy()[...] = host_in.numpy()
        g32.upload_ptr(0, 0, npatch, h32.data_ptr())
        g32.sync()
        m32 = measure(g32, "f32")
        fp32 = {"value": m32["value"], "unit": "cell-updates/s", "ms_per_step": m32["ms_per_step"], "dtype": "f32",
                "roofline": m32["roofline"], "clocks": m32["clocks"], "gpu_launches": m32["launches"], "finite": m32["finite"]}
        finite = finite and m32["finite"]
        launches += m32["launches"]
        del g32, h32
        torch.cuda.empty_cache()

    # end to end through the C ABI with host buffers (H2D of all interiors, one step, D2H)
    e2e = None
    if not args.no_e2e:
        host_out = torch.empty(host_in.shape, dtype=host_in.dtype, pin_memory=True)   # (empty_like would drop the pinning)
        hb = npatch * nv * 4096 * esz
        g.advance_host(cfl, 0.0, 1, host_in.data_ptr(), host_out.data_ptr())      # warm-up
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.e2e_steps):
            g.advance_host(cfl, 0.0, 1, host_in.data_ptr(), host_out.data_ptr())
        torch.cuda.synchronize()
        el = time.perf_counter() - t0
        el = max_over_ranks(el, dist, "cuda")
        e2e = {"value": whole_job_rate(upd_per_step, world, args.e2e_steps, el * 1e3), "unit": "cell-updates/s",
               "h2d_bytes_per_step": hb, "d2h_bytes_per_step": hb, "steps": args.e2e_steps,
               "api": "amrhydro_advance_host (pinned host buffers)"}
        finite = finite and bool(np.isfinite(host_out.numpy()[:8]).all())

    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu:
        rate, cores, sample, _ = cpu_oracle_rate(args.workload, args.size)
        cpu = {"value": rate, "unit": "cell-updates/s", "cores": cores, "kind": "oracle", "sample": sample}

    if rank == 0:
        line = {
            "metric": "cell-updates/sec per RK2 step", "value": value, "unit": "cell-updates/s",
            "n_gpus": world, "steps": args.steps, "warmup": max(3, args.warmup), "ms_per_step": ms_per_step,
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": args.dtype,
            "data": "synthetic",
            "config": {"workload": w["name"] if not args.size or args.size == w["size"] else
                       w["name"] + " (REDUCED to %d cells per side by --size)" % args.size, "patches": npatch, "cells": npatch * 4096, "nvars": nv,
                       "cfl": cfl, "halo": "direct sibling reads" if args.halo else "materialised ghosts",
                       "patch_order": "criterion-built table (Morton)" if args.workload == "cfg3" else args.order,
                       "l2_policy": "working set (%.1f GB per slot) far exceeds the 126 MB L2" % (npatch * nv * 4096 * esz / 1e9)
                       if npatch * nv * 4096 * esz > 4 * 126e6 else "working set fits L2 (small config)",
                       "parallelism": "replicas, one per GPU" if world > 1 else "single GPU",
                       **({} if single else {"cuda_graph": bool(args.graph), "graph_replays": int(g.get_counter(binding.CNT_GRAPH_REPLAYS))})},
            "roofline": roof, "fp32": fp32, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": int(launches),
            "clocks": clocks, "finite": finite,
            "paper_context": "paper reports 8-10x vs one 3 GHz core on a Quadro FX 5600, fp32 (PAPER.md:274)",
        }
        print(json.dumps(line))
    if dist is not None:
        dist.destroy_process_group()
    if not finite:
        raise SystemExit("non-finite state after the timed run")


if __name__ == "__main__":
    a = parse()
    if a.impl == "reference":
        run_reference(a)
    else:
        run_ours(a)
