#!/usr/bin/env python
"""bench.py -- throughput of the tet-mesh -> solid-bit-grid hot path on B200.

One "step" = one vox_run (K1 count, K2 scan, K3 scatter, K4 brick voxelizer incl. the
large-tet path; every word of the grid written) over one synthetic mesh of the workload.
Default workload = BASELINE.json configs[3] ("cfg4": ~4.8M tets, 1024^3 grid), the
configuration the metric is quoted on.  DESIGN.md "Measurement" defines every number.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg4] [--impl reference]

Prints ONE JSON line (rank 0).  With --gpus N > 1 it expects to be launched by
torch.distributed.run (one rank per GPU): every rank voxelizes its own replica of the
workload (seed + rank), no data-path collective ("replicas only").
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

METRIC = "Gvoxel-samples/s"
UNIT = "Gvoxel-samples/s"
# INT32 model frozen in DESIGN.md "Roofline": ops the method itself must execute
OPS_PER_SAMPLE = 11.0
OPS_PER_PAIR = 150.0
# alu-pipe peak: 148 SMs x 64 INT32 lanes/clk x clocks.max.sm (B300_MICROARCH "Pipe rates":
# IADD3/LOP3/SHF rt_SMSP = 2 -> 16 lanes/clk/SMSP -> 64/SM); DESIGN.md "Roofline"
ALU_LANES_PER_SM = 64


def _args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=30)
    ap.add_argument("--warmup", type=int, default=5)
    ap.add_argument("--impl", default="b200", choices=["b200", "reference"])
    ap.add_argument("--workload", default="cfg4")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--e2e-steps", type=int, default=20)
    ap.add_argument("--e2e-depth", type=int, default=3)
    ap.add_argument("--variant", type=int, default=0)
    ap.add_argument("--input", default="tets", choices=["tets", "lattice"],
                    help="lattice: the timed steps take the mesh as lattice vertices + keep mask (vox_lattice; "
                         "--variant 0 = the library's choice, 1 = through the binning passes, 2 = fused path) instead of a tet array")
    ap.add_argument("--tile", type=int, nargs=2, default=None)
    return ap.parse_args()


def candidate_samples(m):
    """Sum over tets of |closed bbox(t) /\\ voxel-centre lattice| (PAPER.md:98's unit of work).

    Pure bookkeeping on the input arrays (min/max, floor division); culled slivers count 0,
    degenerate tets count their bbox like any other (the GPU has to look at them too)."""
    import numpy as np

    total = 0
    step = 1 << 20
    for s in range(0, m.T, step):
        v = m.verts[m.tets[s : s + step]].astype(np.int64)  # [t][4][3]
        lo, hi = v.min(axis=1), v.max(axis=1)
        cnt = np.ones(len(v), dtype=np.int64)
        for a in range(3):
            h = m.extent[a] // m.grid[a]
            i0 = np.maximum(-((h - 2 * lo[:, a]) // (2 * h)), 0)
            i1 = np.minimum((2 * hi[:, a] - h) // (2 * h), m.grid[a] - 1)
            cnt *= np.maximum(i1 - i0 + 1, 0)
        total += int(cnt.sum())
    return total


def rank_seed(workload, rank):
    """Replicas: rank r voxelizes its own mesh of the same recipe, seed = default seed + r."""
    from meshgen.kuhn import _CONFIGS

    return _CONFIGS[workload][1] + rank


def reduce_over_ranks(dist, ms, samples, tets, device):
    """(max over ranks of the device time, sum over ranks of the work).  No data-path collective:
    this is the only communication of a multi-rank run."""
    if dist is None:
        return float(ms), float(samples), float(tets)
    import torch

    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    w = torch.tensor([float(samples), float(tets)], dtype=torch.float64, device=device)
    dist.all_reduce(w, op=dist.ReduceOp.SUM)
    return float(t[0]), float(w[0]), float(w[1])


def workload_config(m, input_kind, samples, stride, grid_words):
    """The `config` object of the JSON line: what identifies the workload, and nothing about how an arm maps it to
    hardware, so that the CUDA arm and --impl reference print the same keys (and, when the oracle runs the whole
    workload per step, the same values).  Arm-specific facts (pairs, tile) sit under `binning` in the CUDA line."""
    mb = (16 * m.T + 12 * m.V + 4 * grid_words) / 1e6
    return {"workload": m.name, "input": input_kind, "tets": m.T, "verts": m.V, "grid": list(m.grid), "batch": m.batch,
            "candidate_samples": int(samples), "bounded_sample_stride": int(stride),
            "l2": f"no flush between steps; one step streams {mb:.0f} MB of tets+verts+grid "
                  f"({'>' if mb > 126 else '<='} 126 MB L2)",
            "multi_gpu": "replicas only (seed + rank), no collective"}


def kernel_source_sha256():
    """sha256 over the CUDA sources the library is built from (every file under csrc/, by name): ties a committed ncu
    capture (profiles/traffic.csv, column capture_sha256) to the code being timed."""
    import hashlib

    d = os.path.join(ROOT, "paper_2106_01326_b200", "csrc")
    h = hashlib.sha256()
    for name in sorted(os.listdir(d)):
        if name.endswith((".cu", ".cuh", ".h")):
            h.update(name.encode() + b"\0" + open(os.path.join(d, name), "rb").read())
    return h.hexdigest()


def ncu_traffic(workload, kernel):
    """dram__bytes_read.sum + dram__bytes_write.sum per launch of `kernel` on `workload`, from the
    committed ncu --set full capture (profiles/traffic.csv names the capture); None if absent."""
    path = os.path.join(ROOT, "profiles", "traffic.csv")
    try:
        best = None
        for ln in open(path).read().splitlines():
            f = [x.strip() for x in ln.split(",")]
            if len(f) >= 5 and f[0] == workload and f[1] == kernel:
                best = {"bytes": float(f[2]) + float(f[3]), "source": "profiles/" + f[4]}
                if len(f) >= 7:  # the same capture's warp instructions and issue-slot utilisation
                    best["ncu"] = {"warp_inst_executed": float(f[5]), "issue_active_pct": float(f[6]),
                                   "gpu_time_ms": float(f[7]) if len(f) >= 8 else None,
                                   "thread_inst_per_warp_inst": float(f[8]) if len(f) >= 9 else None,
                                   "shared_wavefronts": float(f[9]) if len(f) >= 10 else None,
                                   "shared_bank_conflicts": float(f[10]) if len(f) >= 11 else None}
                best["capture_sha256"] = f[11] if len(f) >= 12 else None
        return best
    except OSError:
        return None


class ClockSampler:
    """Samples SM clock and throttle reasons through NVML while the timed region runs."""

    def __init__(self, index, period=0.004):
        self.index, self.period = index, period
        self.sm, self.reasons, self.power = [], set(), []
        self.sm_max = None
        self._stop = threading.Event()
        self._thr = None
        try:
            import pynvml

            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM)
        except Exception as e:  # pragma: no cover
            self.nv = None
            self.err = repr(e)

    _NAMES = {
        0x2: "applications_clocks_setting", 0x4: "sw_power_cap", 0x8: "hw_slowdown", 0x10: "sync_boost",
        0x20: "sw_thermal_slowdown", 0x40: "hw_thermal_slowdown", 0x80: "hw_power_brake_slowdown",
        0x100: "display_clock_setting",
    }

    def _loop(self):
        nv = self.nv
        while not self._stop.is_set():
            try:
                self.sm.append(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM))
                r = nv.nvmlDeviceGetCurrentClocksEventReasons(self.h) if hasattr(
                    nv, "nvmlDeviceGetCurrentClocksEventReasons") else nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h)
                for bit, name in self._NAMES.items():
                    if r & bit:
                        self.reasons.add(name)
                self.power.append(nv.nvmlDeviceGetPowerUsage(self.h) / 1000.0)
            except Exception:  # pragma: no cover
                pass
            time.sleep(self.period)

    def __enter__(self):
        if self.nv is not None:
            self._thr = threading.Thread(target=self._loop, daemon=True)
            self._thr.start()
        return self

    def __exit__(self, *a):
        self._stop.set()
        if self._thr is not None:
            self._thr.join()

    def summary(self):
        if self.nv is None or not self.sm:
            return {"sm_mhz": None, "sm_max_mhz": self.sm_max, "reasons": [], "note": "nvml unavailable"}
        return {
            "sm_mhz": statistics.median(self.sm), "sm_min_mhz": min(self.sm), "sm_max_mhz": self.sm_max,
            "reasons": sorted(self.reasons), "samples": len(self.sm),
            "power_w_max": max(self.power) if self.power else None,
        }


# ------------------------------------------------------------------------------------------
# the oracle timed on the host cores (cpu_baseline leg and --impl reference)
# ------------------------------------------------------------------------------------------
def time_oracle(m, target_s=12.0, repeats=1):
    """Times oracle.voxelize as it stands on a bounded sample: every `stride`-th tet of the
    workload (the oracle's own tet_stride argument).  Returns (samples/s, info dict)."""
    import oracle

    cores = oracle.num_threads()
    # two-point calibration (the fixed cost of zero-filling the grid cancels), then aim for target_s
    def once(stride):
        t0 = time.perf_counter()
        _, s = oracle.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets,
                               tet_stride=stride, return_samples=True)
        return s, time.perf_counter() - t0

    sa, ta = once(max(1, m.T // 4096))
    sb, tb = once(max(1, m.T // 65536))
    rate0 = (sa - sb) / max(ta - tb, 1e-4) if sa > sb else max(sa, 1) / max(ta, 1e-4)
    total = candidate_samples(m)
    want = rate0 * target_s
    stride = max(1, int(total / max(want, 1.0)))
    best = None
    for _ in range(repeats):
        t0 = time.perf_counter()
        _, s = oracle.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets,
                               tet_stride=stride, return_samples=True)
        dt = time.perf_counter() - t0
        if best is None or dt < best[0]:
            best = (dt, s)
    dt, s = best
    info = {
        "kind": "oracle", "cores": cores,
        "sample": f"every {stride}th tet of {m.name} ({-(-m.T // stride)} of {m.T} tets, {s} candidate samples, "
                  f"{dt:.2f} s wall incl. zero-filling the grid)",
        "seconds": dt, "samples": s, "stride": stride,
    }
    return s / dt, info


def oracle_whole(m, repeats=3, budget_s=30.0):
    """oracle.voxelize as it stands on the WHOLE workload: returns (grid, candidate samples, best seconds, runs).
    Repeats while the accumulated time stays within budget_s (at least one run)."""
    import oracle

    best, grid, samples, spent, runs = None, None, 0, 0.0, 0
    for _ in range(repeats):
        t0 = time.perf_counter()
        grid, samples = oracle.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets,
                                        return_samples=True)
        dt = time.perf_counter() - t0
        runs += 1
        spent += dt
        best = dt if best is None else min(best, dt)
        if spent + best > budget_s:
            break
    return grid, samples, best, runs


def run_reference(args):
    """--impl reference: the oracle (unmodified) on the host cores, same metric/config."""
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    import meshgen
    import oracle

    m = meshgen.make_config(args.workload)
    total = candidate_samples(m)
    # size a step so that warmup+steps finish in ~2-3 minutes
    per_step_s = max(1.0, min(15.0, 150.0 / max(1, args.steps + args.warmup)))
    rate, info = time_oracle(m, target_s=per_step_s)
    stride = info["stride"]
    if total / max(rate, 1.0) <= 8.0:  # the whole workload fits a step: same config as the CUDA arm
        stride = 1
    times, samples = [], 0
    for i in range(args.warmup + args.steps):
        t0 = time.perf_counter()
        _, s = oracle.voxelize(m.verts, m.tets, m.grid, m.extent, tet_offsets=m.tet_offsets,
                               tet_stride=stride, return_samples=True)
        dt = time.perf_counter() - t0
        if i >= args.warmup:
            times.append(dt)
            samples += s
    tsum = sum(times)
    value = samples / tsum / 1e9
    info["sample"] = (f"each step = the whole of {m.name} ({m.T} tets, {samples // max(1, args.steps)} candidate samples)"
                      if stride == 1 else
                      f"each step = every {stride}th tet of {m.name} ({-(-m.T // stride)} of {m.T} tets, "
                      f"{samples // max(1, args.steps)} candidate samples)")
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tsum / max(1, args.steps),
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int64",
        "data": "synthetic",
        "config": workload_config(m, "tets", total, stride, m.batch * m.grid[2] * m.grid[1] * (m.grid[0] // 32)),
        "mtets_per_s": (-(-m.T // stride)) * args.steps / tsum / 1e6,
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": info["cores"], "kind": "oracle",
                         "sample": info["sample"]},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------
# the CUDA path
# ------------------------------------------------------------------------------------------
def run_b200(args):
    import numpy as np
    import torch

    import meshgen
    import paper_2106_01326_b200 as pkg

    rank = int(os.environ.get("RANK", "0"))
    local_rank = int(os.environ.get("LOCAL_RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    if not torch.cuda.is_available():
        raise RuntimeError("bench.py needs a CUDA device: the product has no CPU fallback")
    if not os.path.exists(pkg.lib_path()):  # a fresh checkout: compile the extension (no-op otherwise)
        from paper_2106_01326_b200.build import build as _build

        if local_rank == 0:
            _build()
        else:  # the other ranks of the node wait for rank 0's build
            for _ in range(600):
                if os.path.exists(pkg.lib_path()):
                    break
                time.sleep(0.5)
    pkg.load_library()  # fail loudly if libvox.so is missing
    torch.cuda.set_device(local_rank)
    dist = None
    if world > 1:
        import torch.distributed as dist

        dist.init_process_group("nccl", device_id=torch.device("cuda", local_rank))

    # replicas: rank r voxelizes its own mesh of the same recipe (default seed + r)
    base = meshgen.make_config(args.workload, None) if rank == 0 else None
    m = base if rank == 0 else meshgen.make_config(args.workload, rank_seed(args.workload, rank))
    samples = candidate_samples(m)

    stream = torch.cuda.Stream()
    off_np = m.tet_offsets if m.batch > 1 else None
    with torch.cuda.stream(stream):
        d_verts = torch.from_numpy(m.verts).cuda()
        d_tets = torch.from_numpy(m.tets).cuda()
        d_off = torch.from_numpy(off_np).cuda() if off_np is not None else None
        vz = pkg.Voxelizer(m.grid, m.extent, m.batch, tile=args.tile, variant=args.variant)
        if args.input == "lattice":
            if getattr(m, "cells", None) is None:
                raise SystemExit(f"--input lattice: workload {args.workload} is not a background lattice")
            d_keep_main = torch.from_numpy(meshgen.lattice_form(m, m.cells)).cuda()
            vz.set_lattice(d_verts, m.cells, d_keep_main)
        else:
            vz.set_tets(d_verts, d_tets, d_off)
        pairs = vz.plan(stream)  # exact workspace sizing: outside the timed region (one sync)
        vz.alloc_workspace()
        nx, ny, nz = m.grid
        out = torch.empty((m.batch, nz, ny, nx // 32), dtype=torch.int32, device="cuda")
        vz.timing_enable(args.steps)

        def barrier():
            if dist is not None:
                dist.barrier()

        for _ in range(args.warmup):
            vz.run(out, stream)
        stream.synchronize()
        st = vz.status(stream)
        vz.timing_enable(0)  # the timed steps run WITHOUT the per-kernel events (they cost ~15 us per step: visible on
        barrier()            # the small configs); the kernel shares come from a second, instrumented pass below
        torch.cuda.synchronize()
        e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        launches0 = pkg.kernel_launches()
        with ClockSampler(local_rank) as clk:
            e0.record(stream)
            for _ in range(args.steps):
                vz.run(out, stream)
            e1.record(stream)
            barrier()
            torch.cuda.synchronize()
        gpu_launches = pkg.kernel_launches() - launches0  # counted by the library, not derived (vox_kernel_launches)
        ms_total = e0.elapsed_time(e1)
        vz.timing_enable(args.steps)  # instrumented pass: the same steps again with an event after every kernel
        for _ in range(args.steps):
            vz.run(out, stream)
        stream.synchronize()
        per = [vz.timing_read(i) for i in range(args.steps)]
        vz.timing_enable(0)
        popcount = None
        got_grid = None
        if rank == 0:
            got_grid = out.cpu().numpy().view(np.uint32).copy()  # the timed steps' output, compared with the oracle below
            popcount = int(np.unpackbits(got_grid.view(np.uint8)).sum())

        # max over ranks of the device time; sum over ranks of the work
        tmax, ssum, tsum = reduce_over_ranks(dist, ms_total, samples, m.T, "cuda")
        sec = tmax * 1e-3
        value = ssum * args.steps / sec / 1e9

        # ---- e2e: HOST buffers in, HOST grid out, through the public vox_pipe_* calls.  Every step
        # copies that step's mesh from pinned host memory (H2D), runs the hot path and copies the
        # grid back (D2H); `depth` meshes are in flight so step k's copies overlap step k+-1's
        # kernels.  Also reported: the unpipelined vox_run_host call (one mesh, fully serialised).
        e2e = None
        if not args.no_e2e:
            hv = torch.from_numpy(m.verts).pin_memory()
            ht = torch.from_numpy(m.tets).pin_memory()
            ho = torch.from_numpy(off_np).pin_memory() if off_np is not None else None
            depth = args.e2e_depth
            houts = [torch.empty((m.batch, nz, ny, nx // 32), dtype=torch.int32).pin_memory() for _ in range(depth)]
            pipe = pkg.Pipe(m.grid, m.extent, m.batch, depth=depth, max_V=m.V, max_T=m.T, tile=args.tile,
                            variant=args.variant, max_pairs=pairs)

            def pipe_steps(k):
                tickets = []
                for i in range(k):
                    if i >= depth:
                        pipe.wait(tickets[i - depth])
                    tickets.append(pipe.submit(hv, ht, houts[i % depth], ho))
                for t in tickets[max(0, k - depth):]:
                    pipe.wait(t)

            pipe_steps(max(3, depth))  # warm-up
            barrier()
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            pipe_steps(args.e2e_steps)
            torch.cuda.synchronize()
            e2e_ms = (time.perf_counter() - t0) * 1e3  # host wall clock around submit..wait of all steps
            e2e_ms = reduce_over_ranks(dist, e2e_ms, 0, 0, "cuda")[0]
            same = bool(rank != 0 or all(torch.equal(h, out.cpu()) for h in houts[:min(depth, args.e2e_steps)]))
            # sparse output through the same pipeline (vox_pipe_submit_sparse): same steps, the grid
            # leaves the GPU as a tile table + the mixed tiles K4 stores straight into pinned memory
            ts = pipe.tile_shape
            nb = m.batch * ts["nbx"] * ts["nby"] * ts["nbz"]
            cap_tiles = int(st["nonempty_tiles"])  # a tile without tets cannot be mixed
            htabs = [torch.zeros(nb, dtype=torch.int32).pin_memory() for _ in range(depth)]
            hpays = [torch.zeros((cap_tiles, ts["tz"], ts["ty"]), dtype=torch.int32).pin_memory() for _ in range(depth)]

            def pipe_steps_sparse(k):
                tickets, last = [], None
                for i in range(k):
                    if i >= depth:
                        pipe.wait(tickets[i - depth])
                    tickets.append(pipe.submit_sparse(hv, ht, htabs[i % depth], hpays[i % depth], cap_tiles, ho))
                for t in tickets[max(0, k - depth):]:
                    last = pipe.wait(t)
                return last

            pipe_steps_sparse(max(3, depth))
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            sp_stats = pipe_steps_sparse(args.e2e_steps)
            torch.cuda.synchronize()
            sp_ms = (time.perf_counter() - t0) * 1e3
            sp_ms = reduce_over_ranks(dist, sp_ms, 0, 0, "cuda")[0]
            e2e_sparse = {"value": ssum * args.e2e_steps / (sp_ms * 1e-3) / 1e9, "unit": UNIT,
                          "ms_per_step": sp_ms / args.e2e_steps, "h2d_bytes_per_step": None,
                          "d2h_bytes_per_step": nb * 4 + 256 + sp_stats["mixed_tiles"] * ts["ty"] * ts["tz"] * 4,
                          "mixed_tiles": sp_stats["mixed_tiles"], "full_tiles": sp_stats["full_tiles"], "tiles": nb,
                          "api": f"vox_pipe_submit_sparse/vox_pipe_wait, depth {depth}; payload stored by K4 "
                                 "into pinned host memory"}
            # lattice input through the same pipeline (vox_pipe_submit_lattice): the mesh travels as lattice
            # vertices + one keep byte per cell, no tet array (f4); sparse output as above
            e2e_lattice = None
            if getattr(m, "cells", None) is not None:
                import meshgen as _mg

                cells = m.cells
                hk = torch.from_numpy(_mg.lattice_form(m, cells)).pin_memory()
                lat_T = m.batch * 6 * cells[0] * cells[1] * cells[2]
                d_keep = hk.cuda()
                e2e_lattice = {"unit": UNIT, "h2d_bytes_per_step": hv.numel() * 4 + hk.numel(), "cells": list(cells),
                               "api": f"vox_pipe_submit_lattice/vox_pipe_wait, depth {depth}",
                               "paths": "binned = the implied tets through K1-K3 (vox_lattice's default for ordinary cells); fused = "
                                        "vox_set_variant(2): K0 slabs + K4 enumerating its candidate cells, no K1-K3, no "
                                        "pair list (the default's own choice only for giant cells)"}
                for path, lvar in (("fused", 2), ("binned", 1)):
                    # device step of this path on resident inputs (its own tile: the implicit tet count picks it);
                    # the plan gives the binned path's exact pair count (outside the timing)
                    vzl = pkg.Voxelizer(m.grid, m.extent, m.batch, tile=args.tile, variant=lvar)
                    vzl.set_lattice(d_verts, cells, d_keep)
                    lat_pairs = vzl.plan(stream)
                    lout = torch.empty_like(out)
                    for _ in range(3):
                        vzl.run(lout, stream)
                    l0, l1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
                    l0.record(stream)
                    for _ in range(10):
                        vzl.run(lout, stream)
                    l1.record(stream)
                    stream.synchronize()
                    lat_dev_ms = l0.elapsed_time(l1) / 10
                    lst0 = vzl.status(stream)
                    lat_cap = max(int(lst0["nonempty_tiles"]), 1)
                    ltile = vzl.tile_shape
                    lat_ws = vzl.workspace_bytes
                    same_dev = bool(torch.equal(lout, out))
                    vzl.close()
                    del lout
                    lpipe = pkg.Pipe(m.grid, m.extent, m.batch, depth=depth, max_V=m.V, max_T=lat_T,
                                     tile=(ltile["ty"], ltile["tz"]), variant=lvar, max_pairs=lat_pairs)
                    lts = lpipe.tile_shape
                    lnb = m.batch * lts["nbx"] * lts["nby"] * lts["nbz"]
                    ltabs = [torch.zeros(lnb, dtype=torch.int32).pin_memory() for _ in range(depth)]
                    lpays = [torch.zeros((lat_cap, lts["tz"], lts["ty"]), dtype=torch.int32).pin_memory()
                             for _ in range(depth)]

                    def lat_steps(k, sparse_out):
                        tickets, last = [], None
                        for i in range(k):
                            if i >= depth:
                                lpipe.wait(tickets[i - depth])
                            if sparse_out:
                                tickets.append(lpipe.submit_lattice(hv, cells, hk, ltabs[i % depth], lpays[i % depth], lat_cap))
                            else:
                                tickets.append(lpipe.submit_lattice(hv, cells, hk, houts[i % depth]))
                        for t in tickets[max(0, k - depth):]:
                            last = lpipe.wait(t)
                        return last

                    res = {}
                    for key, sp in (("dense", False), ("sparse", True)):
                        lat_steps(max(3, depth), sp)
                        torch.cuda.synchronize()
                        t0 = time.perf_counter()
                        lst = lat_steps(args.e2e_steps, sp)
                        torch.cuda.synchronize()
                        lms = (time.perf_counter() - t0) * 1e3
                        res[key] = {"value": ssum * args.e2e_steps / (lms * 1e-3) / 1e9, "ms_per_step": lms / args.e2e_steps}
                    lat_steps(1, False)
                    same_l = bool(torch.equal(houts[0], out.cpu()))
                    e2e_lattice[path] = {"device_ms_per_step": lat_dev_ms,
                                         "device_value": float(samples) / (lat_dev_ms * 1e-3) / 1e9,
                                         "dense_output": res["dense"], "sparse_output": res["sparse"],
                                         "same_result": bool(same_l and same_dev), "pairs": lst["pairs"],
                                         "tile": [32, ltile["ty"], ltile["tz"]], "workspace_bytes": lat_ws}
                    lpipe.close()
                    del ltabs, lpays
                del d_keep
            pipe.close()
            del htabs, hpays
            # unpipelined single call
            vz2 = pkg.Voxelizer(m.grid, m.extent, m.batch, tile=args.tile, variant=args.variant)
            # vox_host_arena_bytes sizes the pair list by an estimate; add room for the planned count
            arena = torch.empty(vz2.host_arena_bytes(m.V, m.T) + 4 * pairs, dtype=torch.uint8, device="cuda")
            for _ in range(2):
                vz2.run_host(hv, ht, houts[0], arena, ho, stream)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            for _ in range(3):
                vz2.run_host(hv, ht, houts[0], arena, ho, stream)  # synchronises each call
            sync_ms = (time.perf_counter() - t0) * 1e3 / 3
            vz2.close()
            del arena
            h2d = hv.numel() * 4 + ht.numel() * 4 + (ho.numel() * 8 if ho is not None else 0)
            d2h = houts[0].numel() * 4 + 256  # grid + the status header
            e2e = {"value": ssum * args.e2e_steps / (e2e_ms * 1e-3) / 1e9, "unit": UNIT,
                   "h2d_bytes_per_step": h2d, "d2h_bytes_per_step": d2h, "ms_per_step": e2e_ms / args.e2e_steps,
                   "steps": args.e2e_steps, "api": f"vox_pipe_submit/vox_pipe_wait, depth {depth}",
                   "same_result": same,
                   "unpipelined_vox_run_host": {"ms_per_call": sync_ms,
                                                "value": float(samples) / (sync_ms * 1e-3) / 1e9},
                   "sparse_output": e2e_sparse, "lattice_input": e2e_lattice}
            e2e_sparse["h2d_bytes_per_step"] = h2d

        if rank != 0:
            vz.close()
            if dist is not None:
                dist.destroy_process_group()
            return

        # ---- roofline of the dominant kernel (K4), from the live per-kernel events
        k4 = statistics.mean(p["k4"] for p in per)
        shares = {k: statistics.mean(p[k] for p in per) for k in ("k1", "k2", "k3", "k4", "total")}
        sm_max = clk.sm_max or 1965
        peak_alu = 148 * ALU_LANES_PER_SM * sm_max * 1e6 / 1e12  # Tops/s
        ops = OPS_PER_SAMPLE * samples + OPS_PER_PAIR * pairs
        achieved = ops / (k4 * 1e-3) / 1e12
        try:
            probe = {k: pkg.probe_int32(kind=i) / 1e12 for i, k in enumerate(("alu_lop3", "fma_imad", "mixed"))}
        except Exception as e:  # pragma: no cover
            probe = {"error": repr(e)}
        peaks = {}
        try:
            peaks = json.load(open(os.path.join(ROOT, "MEASURED_PEAKS.json")))
        except Exception:
            pass
        hbm_peak = peaks.get("hbm_gbs", 6650.0)
        min_bytes = 16.0 * m.T + 12.0 * m.V + 4.0 * vz.grid_words
        k4_bytes = 4.0 * vz.grid_words + pairs * (4.0 + 16.0 + 48.0)  # grid + per pair: id, tet, 4 verts
        tr = ncu_traffic(args.workload + ("_lattice" if vz.path == "lattice_fused" else ""), "k4_flat")
        # what the kernel EXECUTES (as opposed to the frozen model of what a brute-force incremental test would):
        # thread instructions per launch from the committed ncu capture of this code (profiles/traffic.csv) over the
        # K4 time measured live in this run, against (i) the in-run mixed alu+fma probe and (ii) the issue slots
        executed = None
        ncu = (tr or {}).get("ncu")
        # the capture must belong to the code being timed: profiles/traffic.csv carries the sha256 of csrc/ at capture
        # time; any difference (or no capture of this workload at all) nulls every figure derived from it
        src_sha = kernel_source_sha256()
        stale = None
        if not ncu:
            stale = "no committed ncu capture of this workload"
        elif (tr or {}).get("capture_sha256") != src_sha:
            stale = "stale capture: profiles/traffic.csv was taken from other kernel sources than the ones timed"
        if ncu and not stale and ncu.get("thread_inst_per_warp_inst"):
            tinst = ncu["warp_inst_executed"] * ncu["thread_inst_per_warp_inst"]
            issue_peak = 148 * 4 * sm_max * 1e6  # warp instructions per second: one per cycle per SM sub-partition
            executed = {
                "thread_inst_per_launch": tinst, "warp_inst_per_launch": ncu["warp_inst_executed"],
                "source": (tr or {}).get("source"),
                "achieved_winst_per_s": ncu["warp_inst_executed"] / (k4 * 1e-3) / 1e9,
                "issue_peak_winst_per_s": issue_peak / 1e9,
                "frac_issue": ncu["warp_inst_executed"] / (k4 * 1e-3) / issue_peak,
                "issue_active_pct_ncu": ncu["issue_active_pct"],
                # secondary: ALL thread instructions (LDS/ATOMS/branches included) over the alu+fma-only probe: numerator
                # and denominator are different populations, so this over-states pipe use; kept for continuity
                "achieved_tinst_per_s": tinst / (k4 * 1e-3) / 1e12,
                "frac_mixed_probe_all_inst": (tinst / (k4 * 1e-3) / 1e12 / probe["mixed"]) if probe.get("mixed") else None,
                "unit": "G warp-instructions/s against 148 SMs x 4 issue slots x clocks.max.sm",
            }
        # The fraction that BOUNDS the kernel is the share of the SMs' issue slots it fills: warp instructions per
        # launch (ncu smsp__inst_executed.sum of the committed capture of THIS code, guarded by the source hash) over
        # the K4 time measured live, against one warp instruction per cycle per SM sub-partition.  Numerator and
        # denominator count the same thing (every issued instruction), and ncu's own smsp__issue_active of the same
        # capture is printed beside it.  The frozen 11/150 model of SURVEY.md 8(d) is what a per-sample incremental
        # test would execute; the row-span kernel executes far less, so that figure is an EFFECTIVE one (> 1) and is
        # reported under its own name.
        effective = {
            "achieved": achieved, "peak": peak_alu, "unit": "Tops/s (INT32, modelled)", "frac": achieved / peak_alu,
            "model": f"{OPS_PER_SAMPLE:g} ops/candidate sample + {OPS_PER_PAIR:g} ops/(tet,tile) pair", "ops_per_launch": ops,
            "peak_source": "derived: 148 SMs x 64 alu-pipe lanes x clocks.max.sm (DESIGN.md Roofline)",
            "note": "algorithmic ops of the frozen model over measured time and the alu-pipe peak: a speed-up over the "
                    "brute-force incremental method, not a roofline position (it exceeds 1)",
        }
        roofline = {
            "bound": "alu", "kernel": "k4_flat",
            "achieved": (executed or {}).get("achieved_winst_per_s"), "peak": 148 * 4 * sm_max * 1e6 / 1e9,
            "unit": "G warp-instructions/s (issue slots: the integer alu/fma/lsu pipes all drain through them)",
            "frac": (executed or {}).get("frac_issue"),
            "reason": stale,
            "peak_source": "derived: 148 SMs x 4 sub-partitions x 1 warp instruction per cycle x clocks.max.sm "
                           "(DESIGN.md Roofline); in-run pipe probes under peak_probe_tops",
            "frac_issue": (executed or {}).get("frac_issue"),
            "issue_active_pct_ncu": (ncu or {}).get("issue_active_pct") if not stale else None,
            "capture_sha256": (tr or {}).get("capture_sha256"), "source_sha256": src_sha,
            "traffic": (tr or {}).get("bytes") if not stale else None, "traffic_source": (tr or {}).get("source"),
            "ncu": ncu if not stale else None,
            "executed": executed,
            "note": "achieved = warp instructions per K4 launch (profiles/traffic.csv: ncu smsp__inst_executed.sum of the "
                    "committed capture, valid only while capture_sha256 == source_sha256) / K4 time measured live with CUDA "
                    "events on the launching stream.  frac, traffic and ncu are null (see reason) when the capture is "
                    "missing or was taken from other sources.  The SURVEY 8(d) model figure is under "
                    "effective_vs_bruteforce_model.",
            "effective_vs_bruteforce_model": effective,
            "kernel_ms": k4,
            "peak_probe_tops": probe,
            "hbm": {"achieved_gbs": k4_bytes / (k4 * 1e-3) / 1e9, "peak_gbs": hbm_peak,
                    "frac": k4_bytes / (k4 * 1e-3) / 1e9 / hbm_peak,
                    "peak_source": "MEASURED_PEAKS.json (measured)" if peaks else "fallback",
                    "k4_bytes_per_launch": k4_bytes, "whole_path_min_bytes": min_bytes,
                    "whole_path_frac": min_bytes / (shares["total"] * 1e-3) / 1e9 / hbm_peak},
        }

        # ---- occupancy fold (f2): this step's grid read as the k = 2 fine grid of a half-resolution model
        occ = None
        if nx % 64 == 0 and ny % 2 == 0 and nz % 2 == 0:
            cgrid = (nx // 2, ny // 2, nz // 2)
            counts = torch.empty((m.batch, cgrid[2], cgrid[1], cgrid[0]), dtype=torch.uint8, device="cuda")
            for _ in range(3):
                pkg.occupancy(out, cgrid, 2, batch=m.batch, out=counts, stream=stream)
            o0, o1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            o0.record(stream)
            for _ in range(20):
                pkg.occupancy(out, cgrid, 2, batch=m.batch, out=counts, stream=stream)
            o1.record(stream)
            stream.synchronize()
            oms = o0.elapsed_time(o1) / 20
            obytes = out.numel() * 4 + counts.numel()
            occ = {"k": 2, "coarse_grid": list(cgrid), "ms": oms, "bytes": obytes, "bound": "hbm",
                   "achieved_gbs": obytes / (oms * 1e-3) / 1e9, "peak_gbs": hbm_peak,
                   "frac": obytes / (oms * 1e-3) / 1e9 / hbm_peak,
                   "note": f"20 launches back to back on the same {obytes / 1e6:.0f} MB (L2 holds 126 MB); "
                           f"sum(counts) == popcount: {int(counts.sum(dtype=torch.int64)) == popcount}"}

        # ---- "bit-exact" (BASELINE.json's metric, third clause): the WHOLE grid of the timed steps against the
        # oracle run on the whole workload; the same oracle runs are the cpu_baseline (best of up to 3)
        cpu = None
        bit_exact = None
        if not args.no_cpu_baseline:
            import oracle

            exp, osamples, odt, oruns = oracle_whole(base, repeats=3, budget_s=30.0)
            same_grid = bool(np.array_equal(got_grid, exp))
            bit_exact = {"equal": same_grid, "words": int(exp.size), "popcount_gpu": popcount,
                         "popcount_oracle": int(np.unpackbits(exp.view(np.uint8)).sum()),
                         "candidate_samples_oracle": int(osamples),
                         "samples_agree": bool(int(osamples) == int(samples)),
                         "how": "np.array_equal of the whole uint32 grid: last timed vox_run vs oracle.voxelize on the whole workload"}
            if not same_grid:
                bad = np.argwhere(got_grid != exp)
                b = tuple(int(v) for v in bad[0])
                bit_exact.update({"differing_words": int(len(bad)), "first_diff_mzyx": list(b),
                                  "gpu_word": int(got_grid[b]), "oracle_word": int(exp[b])})
            cpu = {"value": osamples / odt / 1e9, "unit": UNIT, "cores": oracle.num_threads(), "kind": "oracle",
                   "sample": f"the whole of {base.name} ({base.T} tets, {osamples} candidate samples), best of {oruns} "
                             f"runs, {odt:.2f} s each incl. zero-filling the grid",
                   "seconds": odt}
            del exp

        line = {
            "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": tmax / args.steps, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "int32/int64 (exact integer)", "data": "synthetic",
            "config": workload_config(m, args.input + (f" (variant {args.variant})" if args.input == "lattice" else ""),
                                      samples, 1, vz.grid_words),
            "path": vz.path,
            "binning": {"pairs": pairs, "tile": [32, vz.tile_shape["ty"], vz.tile_shape["tz"]],
                        "step_bytes_incl_ranges_and_pair_list": 16 * m.T + 12 * m.V + 8 * m.T + 4 * pairs * 2 + 4 * vz.grid_words},
            "mtets_per_s": tsum * args.steps / sec / 1e6,
            "gvoxels_per_s": world * m.batch * nx * ny * nz * args.steps / sec / 1e9,
            "kernel_ms": shares, "status": st, "popcount": popcount,
            "gpu_launches": gpu_launches, "gpu_launches_whole_run": pkg.kernel_launches(),
            "bit_exact": (bit_exact or {}).get("equal"), "bit_exact_detail": bit_exact,
            "clocks": clk.summary(), "roofline": roofline, "occupancy_fold": occ, "cpu_baseline": cpu, "e2e": e2e,
        }
        print(json.dumps(line), flush=True)
        vz.close()
    if dist is not None:
        dist.destroy_process_group()


def main():
    args = _args()
    if args.impl == "reference":
        run_reference(args)
    else:
        run_b200(args)


if __name__ == "__main__":
    main()
