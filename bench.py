#!/usr/bin/env python
"""bench.py -- throughput of the B200-native Poisson solve (arxiv 1211.5244 hot path).

    python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--config c1] [--headline-only]

One "step" = one full solve (all five fused passes F1,F2,F3,I2,I1 of DESIGN.md) of the workload
BASELINE.json's metric is quoted on: configs[1], free BCs, fp64, 128^3 physical -> 256^3 padded
("fp64, free BC 256^3": the paper labels grids by padded FFT size).  Rank 0 prints ONE
JSON line.  `value` / `ms_per_step` = poisson_solve (the north-star call) back to back on ONE stream; the batched
route (poisson_solve_batch) is reported under `batched`.  N > 1 (launched by torch.distributed.run, one rank per GPU) runs N independent replicas
("replicas only": a solve does not shard without an all-to-all, and the north star is
one GPU); value = all ranks' solves / max-over-ranks device time.

--impl reference times the CPU oracle (oracle/, test infrastructure) on the host cores: there is
no reference implementation for this paper, the oracle is the stand-in (rank 0 only).
"""
from __future__ import annotations

import argparse
import json
import math
import os
import subprocess
import sys
import tempfile
import time
from pathlib import Path

import numpy as np

ROOT = Path(__file__).resolve().parent
if str(ROOT) not in sys.path:
    sys.path.insert(0, str(ROOT))

from workloads import generators as gen  # noqa: E402

METRIC = "poisson_solves_per_sec"
UNIT = "solves/s"
BATCH = 32            # solves per poisson_solve_batch call
L2_BYTES = 126e6
WORKLOAD_TEXT = {
    "c0": "configs[0]: free BCs, fp64, 32^3 -> 64^3 padded, h=0.3, 4 seeded Gaussians, K=1/(4 pi r)",
    "c1": "configs[1]: free BCs, fp64, 128^3 physical -> 256^3 padded, h=0.2, 32 seeded Gaussians, K=1/(4 pi r)",
    "c2": "configs[2]: surface BCs (periodic x,y; free z), fp64, 128^3 -> 128x128x256, 32 Gaussians, image-sum kernel",
    "c3": "configs[3]: wire BCs (periodic z; free x,y), fp64, 96x96x256 -> 192x192x256, chain of 64 Gaussians",
    "c4a": "configs[4]: free BCs, fp64, 256^3 physical -> 512^3 padded, 256 Gaussians",
    "c4b": "configs[4]: free BCs, fp32, 256^3 physical -> 512^3 padded, 256 Gaussians",
    "c4p": "configs[4] companion: fully periodic 256^3, fp64, K_f=-1/k^2",
}


# ------------------------------------------------------------------ helpers
def measured_peaks():
    p = ROOT / "MEASURED_PEAKS.json"
    if p.exists():
        try:
            d = json.loads(p.read_text())
            return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json)"
        except Exception:
            pass
    return 6650.0, "fallback (B200_PROFILING.md)"


def nominal_flops(info) -> float:
    """5 n log2 n per complex 1D FFT, 2.5 for the real ones, 2 per K^F multiply."""
    rows, length = list(info.rows), list(info.length)
    f = 0.0
    for q, w in ((0, 2.5), (4, 2.5), (1, 5.0), (3, 5.0)):
        f += rows[q] * w * length[q] * math.log2(length[q])
    f += rows[2] * (2 * 5.0 * length[2] * math.log2(length[2]) + 2.0 * length[2])
    return f


def build_inputs(key):
    """Seeded synthetic density + kernel spectrum for a named config (recipe: DESIGN.md 'Input recipe').
    K_f is prepared from the real-space Green's function with numpy's FFT: input preparation outside the
    timed region (the values do not influence timing; parity for these inputs is checked in tests/)."""
    cfg = gen.get_config(key)
    rho = gen.gaussian_density(cfg)
    if cfg.kernel == "periodic_k2":
        kf = gen.periodic_kernel_spectrum(cfg.n, cfg.h)
    else:
        K = gen.green_kernel_realspace(cfg.n, cfg.bc, cfg.h, cfg.images)
        kf = np.ascontiguousarray(np.fft.rfftn(K).real)
        del K
    return cfg, rho, kf


class ClockSampler:
    """nvidia-smi clocks/throttle reasons sampled DURING the timed regions (B200_PROFILING.md)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")
    NAMES = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap")

    def __init__(self, device_index: int):
        self.proc = None
        self.file = None
        try:
            import torch
            uuid = str(torch.cuda.get_device_properties(device_index).uuid)
            self.ident = uuid if uuid.startswith("GPU-") else "GPU-" + uuid
        except Exception:
            self.ident = str(device_index)

    def start(self):
        try:
            self.file = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
            self.proc = subprocess.Popen(["nvidia-smi", f"--id={self.ident}", f"--query-gpu={self.Q}",
                                          "--format=csv,noheader,nounits", "-lms", "50"],
                                         stdout=self.file, stderr=subprocess.DEVNULL)
        except Exception:
            self.proc = None

    def stop(self):
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        if self.proc is None:
            return out
        time.sleep(0.06)
        self.proc.terminate()
        try:
            self.proc.wait(timeout=5)
        except Exception:
            self.proc.kill()
        self.file.flush()
        self.file.seek(0)
        sm, mx, reasons, power = [], [], set(), []
        for line in self.file.read().splitlines():
            parts = [x.strip() for x in line.split(",")]
            if len(parts) < 7:
                continue
            try:
                sm.append(float(parts[0])); mx.append(float(parts[1])); power.append(float(parts[2]))
            except ValueError:
                continue
            for name, val in zip(self.NAMES, parts[3:7]):
                if val.lower().startswith("active"):
                    reasons.add(name)
        try:
            os.unlink(self.file.name)
        except OSError:
            pass
        if sm:
            out.update(sm_mhz=float(np.median(sm)), sm_max_mhz=float(max(mx)), reasons=sorted(reasons),
                       samples=len(sm), power_w_max=float(max(power)))
        return out


def dist_setup(n_gpus: int):
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        import torch
        import torch.distributed as dist
        torch.cuda.set_device(local)
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group(backend="nccl", device_id=torch.device("cuda", local))
    return world, rank, local


def reduce_max(value: float, device=None) -> float:
    """Max over ranks of a per-rank time (every multi-GPU number is the slowest rank's)."""
    import torch
    import torch.distributed as dist
    if not (dist.is_available() and dist.is_initialized()) or dist.get_world_size() == 1:
        return float(value)
    t = torch.tensor([float(value)], dtype=torch.float64, device=device if device is not None else "cpu")
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    return float(t.item())


def barrier():
    import torch.distributed as dist
    if dist.is_available() and dist.is_initialized() and dist.get_world_size() > 1:
        dist.barrier()


# ------------------------------------------------------------------ CPU oracle timing (cpu_baseline / --impl reference)
class OracleTimer:
    """Times the oracle as it stands (oracle/poisson_oracle.c: naive O(n^2) DFT per axis on the explicitly padded grid).
    A step is ONE WHOLE oracle.solve call of the workload (padding, six DFT sweeps, K_f multiply, scaling, crop) whenever
    the requested number of steps fits the time budget; only if it does not, a step is a bounded slab sample of the six
    sweeps scaled to the whole grid, and the result is flagged `extrapolated`."""

    def __init__(self, cfg, rho, kf):
        import oracle
        self.oracle, self.cfg = oracle, cfg
        self.rho = np.ascontiguousarray(rho, dtype=np.float64)
        self.kf = np.ascontiguousarray(kf, dtype=np.float64)
        self.pad = None

    def whole_solve(self) -> float:
        t0 = time.perf_counter()
        self.oracle.solve(self.rho, self.kf, self.cfg.bc)
        return time.perf_counter() - t0

    def _sweeps(self, m):
        pad, dft = self.pad, self.oracle.dft_axis
        tx = ty = tz = 0.0
        for sign in (-1, +1):
            t0 = time.perf_counter(); dft(pad[:m], 2, sign); tx += time.perf_counter() - t0      # x sweep, m z-planes
            t0 = time.perf_counter(); dft(pad[:m], 1, sign); ty += time.perf_counter() - t0      # y sweep, m z-planes
            t0 = time.perf_counter(); dft(pad[:, :m], 0, sign); tz += time.perf_counter() - t0   # z sweep, m y-planes
        return tx, ty, tz

    def slab_sample(self, budget_s: float, per_plane_s: float):
        """(seconds per solve scaled from a slab of m planes per sweep, fraction f, description)."""
        sx, sy, sz = self.cfg.s
        nx, ny, nz = self.cfg.n
        if self.pad is None:
            self.pad = np.zeros((sz, sy, sx), dtype=np.complex128)
            self.pad[:nz, :ny, :nx] = self.rho
        m = int(max(1, min(min(sy, sz), budget_s / max(per_plane_s, 1e-9))))
        tx, ty, tz = self._sweeps(m)
        f = m / float(min(sy, sz))
        full = tx * sz / m + ty * sz / m + tz * sy / m
        desc = (f"EXTRAPOLATED: oracle naive-DFT sweeps on {m} of {min(sy, sz)} planes per sweep (f={f:.4f}) of the padded "
                f"{sx}x{sy}x{sz} grid, 6 sweeps, scaled by 1/f; K_f multiply and padding copy not included")
        return full, f, desc


def oracle_steps(cfg, rho, kf, steps: int, warmup: int, budget_s: float):
    """Runs warmup + steps oracle steps inside about budget_s seconds.  Returns (seconds per solve [mean over the timed
    steps], description, threads, extrapolated, sample_fraction, steps actually timed as whole solves or samples)."""
    timer = OracleTimer(cfg, rho, kf)
    threads = timer.oracle.n_threads()
    first = timer.whole_solve()                      # also warms the library; counts as the first warm-up step
    total = warmup + steps
    sx, sy, sz = cfg.s
    if first * total <= budget_s:
        times = [first]
        for _ in range(total - 1):
            times.append(timer.whole_solve())
        timed = times[warmup:] if warmup < len(times) else times[-1:]
        desc = (f"{len(timed)} whole oracle.solve calls ({warmup} warm-up) on the padded {sx}x{sy}x{sz} grid: padding, six "
                "naive-DFT sweeps, K_f multiply, scaling, crop")
        return float(np.mean(timed)), desc, threads, False, 1.0, len(timed)
    per_plane = first / float(min(sy, sz))
    slab_budget = max(0.5, (budget_s - first) / total)
    times, f, desc = [], 1.0, ""
    for i in range(total):
        sec, f, desc = timer.slab_sample(slab_budget, per_plane)
        if i >= warmup:
            times.append(sec)
    return float(np.mean(times)), desc, threads, True, f, len(times)


def pruned_fft_cpu_times(cfg, rho, kf, budget_s: float = 25.0):
    """The timed CPU baseline of SURVEY.md 8d "CPU side (ii)" / BASELINE.md section 3: baseline/cpu_fft.cpp, the paper's
    customised FFT on the host (own Stockham FFT, OpenMP), best of 3 at 1 thread and at all cores, same seeded inputs.
    The analogue of the paper's "CPU implementation of the same method".  Returns a dict or None."""
    if cfg.precision != "fp64":
        return None
    try:
        import baseline
        out = {"kind": "pruned_fft", "source": "baseline/cpu_fft.cpp (g++ -O3 -march=native -fcx-limited-range -fopenmp; workspace kept between calls)", "unit": UNIT}
        nmax = baseline.max_threads()
        baseline.solve(rho, kf, cfg.bc, threads=nmax)     # untimed: allocates the workspace, warms the caches
        t_start = time.perf_counter()
        for label, th in (("all_cores", nmax), ("one_thread", 1)):
            best = None
            for rep in range(3):
                t0 = time.perf_counter()
                baseline.solve(rho, kf, cfg.bc, threads=th)
                dt = time.perf_counter() - t0
                best = dt if best is None else min(best, dt)
                if time.perf_counter() - t_start > budget_s:
                    break
            out[label] = {"threads": th, "ms_per_solve": best * 1e3, "value": 1.0 / best}
            if time.perf_counter() - t_start > budget_s and label == "all_cores":
                break
        return out
    except Exception as e:   # a missing compiler must not take the GPU numbers down with it
        return {"kind": "pruned_fft", "error": str(e)[:200]}


def config_dict(key, cfg, info_s, order, world):
    """The `config` object of the JSON line: the same keys and values in both arms (ours / reference)."""
    return {"workload": WORKLOAD_TEXT[key], "physical_grid": list(cfg.n), "padded_grid": list(info_s),
            "bc_xyz": ["free" if b == 0 else "periodic" for b in cfg.bc], "axis_order": list(order),
            "l2": "inputs larger than L2: rho/V rotate over a ring of device buffers whose footprint exceeds the 126 MB L2",
            "replicas": world}


def reference_axis_order(bc):
    """The planner's axis-order rule restated (tests/test_plan_host.py checks it against poisson_plan_describe)."""
    per = [b != 0 for b in bc]
    a = 2 if per[2] else (1 if per[1] else 2)
    o = 1 if a == 2 else 2
    b, c = ((0, o) if per[0] else (o, 0)) if per[0] != per[o] else (o, 0)
    return [a, b, c]


def run_reference(args):
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    cfg, rho, kf = build_inputs(args.config)
    steps, warmup = max(1, args.steps), max(0, args.warmup)
    sec, desc, threads, extrap, frac, ntimed = oracle_steps(cfg, rho, kf, steps, warmup, 170.0)
    val = 1.0 / sec
    # Same `config` keys as the main arm WITHOUT loading the product library (this arm must map oracle/ only): the padded
    # grid is S_i = N_i B_i, and the axis order is the planner's documented rule (include/poisson.h: periodic axes first,
    # free axes last, never x first, the contiguous axis last on a tie) restated here.
    s_pad = list(gen.padded_shape(cfg.n, cfg.bc))
    order = reference_axis_order(cfg.bc)
    line = {
        "impl": "reference", "metric": METRIC, "value": val, "unit": UNIT, "n_gpus": args.gpus, "steps": steps,
        "warmup": warmup, "ms_per_step": sec * 1e3, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64", "data": "synthetic",
        "config": config_dict(args.config, cfg, s_pad, order, world),
        "extrapolated": extrap, "sample_fraction": frac, "steps_timed": ntimed,
        "note": "CPU oracle (naive O(n^2) DFT per axis, test infrastructure), not a tuned baseline",
        "cpu_baseline": {"value": val, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc},
        "e2e": {"value": val, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "world_size_seen": world,
    }
    print(json.dumps(line))
    return 0


# ------------------------------------------------------------------ GPU timing
def time_periodic_same_fft_size(pk, torch, cfg, steps, warmup):
    """A fully periodic fp64 solve on the PADDED shape of `cfg` (the same FFT size, nothing skipped): the denominator of the
    paper's Fig. 1 ratios.  Timing does not depend on the values: random density, K^F = 1."""
    s = gen.padded_shape(cfg.n, cfg.bc)
    plan = pk.PoissonPlan(s, (pk.PERIODIC,) * 3, cfg.h, pk.FP64)
    try:
        plan.set_kernel(torch.ones(plan.kernel_dims, dtype=torch.float64, device="cuda"))
        nbuf = max(2, int(math.ceil(300e6 / (8.0 * s[0] * s[1] * s[2]))))      # rho / V ring larger than the 126 MB L2
        rhos = [torch.randn((s[2], s[1], s[0]), dtype=torch.float64, device="cuda") for _ in range(nbuf)]
        Vs = [torch.empty_like(r) for r in rhos]
        for i in range(warmup):
            plan.solve(rhos[i % nbuf], Vs[i % nbuf])
        torch.cuda.synchronize()
        best = []
        for rep in range(5):
            e0, e1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            e0.record()
            for i in range(steps):
                plan.solve(rhos[i % nbuf], Vs[i % nbuf])
            e1.record()
            torch.cuda.synchronize()
            best.append(e0.elapsed_time(e1) / steps)
        best.sort()
        return {"ms": best[len(best) // 2], "padded_grid": list(s), "bytes_total": plan.info.bytes_total}
    finally:
        plan.close()


def time_config(pk, torch, key, steps, warmup, with_e2e=True, with_cold=True, with_profile=True, inputs=None, even_kernel=False):
    cfg, rho_np, kf_np = inputs if inputs is not None else build_inputs(key)
    prec = pk.FP64 if cfg.precision == "fp64" else pk.FP32
    np_dt = np.float64 if prec == pk.FP64 else np.float32
    torch.cuda.synchronize()
    t_create = time.perf_counter()
    plan = pk.PoissonPlan(cfg.n, cfg.bc, cfg.h, prec)       # allocates, uploads tables, and TIMES the launch modes / graph shapes
    torch.cuda.synchronize()
    plan_create_ms = (time.perf_counter() - t_create) * 1e3
    info = plan.info
    # even_kernel: the folded K^F copy (poisson_set_kernel_even; every BASELINE kernel is even along each axis)
    (plan.set_kernel_even if even_kernel else plan.set_kernel)(torch.from_numpy(np.ascontiguousarray(kf_np.astype(np_dt))).cuda())
    rho_bytes = rho_np.size * np.dtype(np_dt).itemsize
    nbuf = max(2, int(math.ceil(1.1 * L2_BYTES / (2 * rho_bytes))))    # rho+V ring larger than L2
    nbuf = min(max(nbuf, min(BATCH, 8 if rho_bytes > 64e6 else BATCH)), 64)
    rho0 = torch.from_numpy(np.ascontiguousarray(rho_np.astype(np_dt))).cuda()
    rhos = [rho0.clone() for _ in range(nbuf)]
    vs = [torch.empty_like(rho0) for _ in range(nbuf)]
    stream = torch.cuda.current_stream()

    def timed_once(body, n):
        """n solves between two CUDA events on the launching stream; ms per solve (max over ranks)."""
        torch.cuda.synchronize()
        barrier()
        a, b = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        a.record(stream)
        body(n)
        b.record(stream)
        torch.cuda.synchronize()
        barrier()
        return reduce_max(a.elapsed_time(b), device="cuda") / n

    def timed(body, n, est_ms):
        """The timed region is EXACTLY n solves; it is repeated (>= 5 regions, up to 50, until about 0.25 s are covered) and
        the MEDIAN region is reported with the spread, so that a 20-step region of a 100 us solve is not a 2 ms one-off."""
        regions = int(min(50, max(5, math.ceil(250.0 / max(n * est_ms, 1e-3)))))
        vals = sorted(timed_once(body, n) for _ in range(regions))
        return {"ms": float(np.median(vals)), "min": vals[0], "max": vals[-1], "regions": regions}

    def one_by_one(n):
        for i in range(n):
            plan.solve(rhos[i % nbuf], vs[i % nbuf])

    bsz = min(BATCH, nbuf)
    # pointer arrays marshalled BEFORE any timed region, one per batch size the loop below uses (what a C caller holds)
    ptr_batches = {m: plan.pointer_batch(rhos[:m], vs[:m]) for m in {bsz, steps % bsz, max(3, warmup) % bsz} if m > 0}

    def batched(n):          # poisson_solve_batch: ceil(n / bsz) calls, exactly n solves
        done = 0
        while done < n:
            m = min(bsz, n - done)
            plan.solve_pointer_batch(ptr_batches[m])
            done += m

    one_by_one(max(3, warmup))
    est = timed_once(one_by_one, max(3, min(steps, 20)))
    single = timed(one_by_one, steps, est)
    pass_ms = None
    if with_profile:
        nprof = min(max(steps, 50), 256)
        for i in range(nprof):
            plan.solve_profiled(rhos[i % nbuf], vs[i % nbuf])
        ms_sum, cnt = plan.profile_read()
        pass_ms = [m / cnt for m in ms_sum]

    batched(max(3, warmup))
    batch = timed(batched, steps, est)
    mode, tune_ms = plan.launch_mode()
    res = {"key": key, "single": single, "batch": batch, "batch_size": bsz,
           "info": info, "nbuf": nbuf, "rho_bytes": rho_bytes,
           "launch_mode": mode, "tune_ms": tune_ms, "graph_shape": list(plan.graph_shape()), "lanes": plan.batch_lanes(bsz),
           "width": plan.batch_width(bsz), "launches_per_solve": plan.launches_per_solve(), "workspace_bytes": plan.workspace_bytes()}
    res["plan_create_ms"] = plan_create_ms
    if pass_ms is not None:
        res["pass_ms"] = pass_ms

    if with_cold:
        # cold-L2 variant: a 512 MB scratch write between solves, each solve timed by its own event pair
        scratch = torch.empty(512 * 1024 * 1024, dtype=torch.uint8, device="cuda")
        ncold = min(steps, 20)
        evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(ncold)]
        for i in range(ncold):
            scratch.fill_(i & 0xFF)
            evs[i][0].record(stream)
            plan.solve(rhos[i % nbuf], vs[i % nbuf])
            evs[i][1].record(stream)
        torch.cuda.synchronize()
        res["cold_ms_per_step"] = float(np.median([a.elapsed_time(b) for a, b in evs]))
        del scratch

    if with_e2e:
        # end to end through the C ABI with HOST buffers: poisson_solve_batch_host copies every rho H2D, runs the
        # passes and copies every V D2H inside the call (pinned host memory), overlapping neighbouring solves
        # (batch size: the pipeline's fill and drain -- first H2D, last D2H -- are paid once per call)
        nh = 8 if rho_bytes > 64e6 else 32
        hr = [torch.from_numpy(np.ascontiguousarray(rho_np.astype(np_dt))).pin_memory() for _ in range(nh)]
        hv = [torch.empty_like(hr[0]).pin_memory() for _ in range(nh)]
        ne2e = max(nh, min(steps, 96) // nh * nh)

        def host_batches(n):
            for _ in range(n // nh):
                plan.solve_batch_host(hr, hv)

        def host_single(n):
            for i in range(n):
                plan.solve_host(hr[i % nh], hv[i % nh])

        for fn, name in ((host_batches, "e2e_ms_per_step"), (host_single, "e2e_single_ms_per_step")):
            fn(nh)
            torch.cuda.synchronize()
            barrier()
            t0 = time.perf_counter()
            fn(ne2e)                                   # synchronous calls: wall clock is the honest timer here
            wall = (time.perf_counter() - t0) * 1e3
            barrier()
            res[name] = reduce_max(wall, device="cuda") / ne2e
        res["e2e_steps"] = ne2e
        res["e2e_batch"] = nh
    plan.close()
    return res


def run_ours(args):
    import torch
    import paper_1211_5244_b200 as pk
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device -- the solve has no CPU fallback (use --impl reference for the oracle)")
    pk.load_library()
    world, rank, local = dist_setup(args.gpus)
    if world == 1:
        torch.cuda.set_device(0)
    steps, warmup = max(1, args.steps), max(3, args.warmup)
    peak, peak_src = measured_peaks()

    inputs = build_inputs(args.config)
    sampler = ClockSampler(local)
    sampler.start()
    res = time_config(pk, torch, args.config, steps, warmup, inputs=inputs, even_kernel=args.even_kernel)
    clocks = sampler.stop()
    if rank != 0:
        return 0

    info = res["info"]
    cfg = inputs[0]
    ms = res["single"]["ms"]                          # the north-star call: poisson_solve back to back on one stream
    value = world * 1e3 / ms
    bms = res["batch"]["ms"]
    n_phys = cfg.n[0] * cfg.n[1] * cfg.n[2]
    n_pad = info.s[0] * info.s[1] * info.s[2]
    flops = nominal_flops(info)
    alu_peak = pk.poisson_measure_fma_peak(pk.FP64 if cfg.precision == "fp64" else pk.FP32)
    fused = res["launch_mode"] == "fused"
    dom = int(np.argmax(res["pass_ms"]))
    if fused:   # one kernel does the whole solve: it is the dominant (only) kernel, timed by the solve's own events
        dom_name, dom_kernel, dom_bytes = "solve", "solve_kernel<...> (all five passes in one cooperative launch)", info.bytes_total
        dom_us = ms * 1e3
    else:
        dom_name, dom_kernel, dom_bytes = pk.PASS_NAMES[dom], f"pass {pk.PASS_NAMES[dom]} (pass_kernel<..., KIND={dom}>)", info.bytes[dom]
        dom_us = res["pass_ms"][dom] * 1e3
    dom_gbs = dom_bytes / (dom_us * 1e-6) / 1e9
    traffic, traffic_src = None, None
    tfile = ROOT / "profiles" / "dram_traffic.csv"     # ncu dram__bytes_read.sum + dram__bytes_write.sum per launch
    if tfile.exists():
        try:
            import csv
            for row in csv.DictReader(tfile.open()):
                if row["config"] == args.config and row["pass"] == dom_name:
                    traffic = int(row["dram_bytes_read"]) + int(row["dram_bytes_write"])
                    traffic_src = f"ncu --set full (L2 flushed before the launch: cold-L2 DRAM bytes), capture {row['source']}"
        except Exception:
            traffic = None
    # executed FP64-pipe instructions of the dominant kernel (north_star: "evidenced by ncu counters"), from the tracked launch list
    inst_fp64, inst_all, inst_src = None, None, None
    ifile = ROOT / "profiles" / "inst_fp64.csv"
    if ifile.exists():
        try:
            import csv
            for row in csv.DictReader(ifile.open()):
                if row["config"] == args.config and row["pass"] == dom_name:
                    inst_fp64, inst_all = int(row["sm__inst_executed_pipe_fp64.sum"]), int(row["smsp__inst_executed.sum"])
                    inst_src = f"ncu --metrics sm__inst_executed_pipe_fp64.sum,smsp__inst_executed.sum per launch (warp-level counts), {row['source']}"
        except Exception:
            inst_fp64 = None
    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": steps, "warmup": warmup,
        "ms_per_step": ms, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
        "dtype": "f64" if cfg.precision == "fp64" else "f32", "data": "synthetic",
        "config": config_dict(args.config, cfg, info.s, info.order, world),     # identical keys and values in --impl reference
        "api": "poisson_solve (include/poisson.h), one call per solve, back to back on one stream",
        "l2_policy": (f"rho/V rotated over {res['nbuf']}+{res['nbuf']} device buffers "
                      f"({2 * res['nbuf'] * res['rho_bytes'] / 1e6:.0f} MB > 126 MB L2); the plan's A1/A2/K^F workspace "
                      f"({info.workspace_bytes / 1e6:.0f} MB) is reused every step (the paper's repeated-solve usage, "
                      "PAPER.md:53,89); cold_l2 below flushes L2 with a 512 MB write between solves"),
        "timing": {"timed_regions": res["single"]["regions"], "region": f"exactly {steps} solves between two CUDA events on the launching stream",
                   "statistic": "median region", "ms_per_step_min": res["single"]["min"], "ms_per_step_max": res["single"]["max"]},
        "grid_points_per_sec_physical": value * n_phys, "grid_points_per_sec_padded": value * n_pad,
        "solve_hbm": {"algorithmic_bytes": info.bytes_total, "achieved_gbs": info.bytes_total / (ms * 1e-3) / 1e9,
                      "peak_gbs": peak, "peak_source": peak_src, "frac": info.bytes_total / (ms * 1e-3) / 1e9 / peak,
                      "note": "effective bandwidth on ALGORITHMIC bytes (B_5 of SURVEY.md 8d) over the measured HBM copy peak; on grids whose "
                              "intermediates sit in the 126 MB L2 the DRAM traffic is lower (see roofline.traffic) and the figure can exceed 1"},
        "alu": {"nominal_gflop_per_solve": flops / 1e9, "achieved_nominal_tflops": flops / (ms * 1e-3) / 1e12,
                "peak_fma_tflops_measured": alu_peak, "frac": flops / (ms * 1e-3) / 1e12 / alu_peak,
                "note": "nominal 5 n log2 n flops per complex 1D FFT (2.5 real, 2 per K^F multiply) against the plain FMA peak "
                        "measured live by poisson_measure_fma_peak (FMA = 2 flops); the executed instruction count is lower "
                        "(radix-16 butterflies), see profiles/ for sm__inst_executed_pipe_fp64"},
        "batched": {"ms_per_step": bms, "solves_per_sec": world * 1e3 / bms, "hbm_frac": info.bytes_total / (bms * 1e-3) / 1e9 / peak,
                    "ms_per_step_min": res["batch"]["min"], "ms_per_step_max": res["batch"]["max"],
                    "api": (f"poisson_solve_batch, {res['batch_size']} resident densities per call, lanes={res['lanes']}, "
                            f"densities per launch={res['width']} (SURVEY.md 8f-1; pointer arrays marshalled before the timed region)")},
        "pass_us": {pk.PASS_NAMES[q]: res["pass_ms"][q] * 1e3 for q in range(5)},
        "pass_gbs": {pk.PASS_NAMES[q]: info.bytes[q] / (res["pass_ms"][q] * 1e-3) / 1e9 for q in range(5)},
        "pass_hbm_frac": {pk.PASS_NAMES[q]: info.bytes[q] / (res["pass_ms"][q] * 1e-3) / 1e9 / peak for q in range(5)},
        "plan_create_ms": res["plan_create_ms"],
        "plan_create_note": "wall clock of poisson_plan_create: allocation, tables and the launch-mode / graph-shape timing runs (POISSON_TUNE=0 skips those)",
        "pass_us_note": ("poisson_solve_profiled: the five passes as five STREAM launches with a CUDA event between each (launch gaps "
                         "included), not the launch mode poisson_solve uses; their sum exceeds ms_per_step"),
        "cold_l2": {"ms_per_step": res["cold_ms_per_step"],
                    "frac": info.bytes_total / (res["cold_ms_per_step"] * 1e-3) / 1e9 / peak},
        "roofline": {"bound": "hbm", "kernel": dom_kernel,
                     "achieved": dom_gbs, "peak": peak, "unit": "GB/s", "frac": dom_gbs / peak, "traffic": traffic,
                     "traffic_source": traffic_src,
                     "inst_fp64": inst_fp64, "inst_executed": inst_all, "inst_source": inst_src,
                     "fp64_thread_inst_per_s": (inst_fp64 * 32 / (dom_us * 1e-6)) if inst_fp64 else None,
                     "dram_frac": (traffic / (dom_us * 1e-6) / 1e9 / peak) if traffic else None,
                     "algorithmic_bytes_per_launch": dom_bytes, "peak_source": peak_src,
                     "duration_us": dom_us, "duration_source": "CUDA events around the kernel's stream launch (pass_us)"},
        "launch_mode": {"chosen": res["launch_mode"], "ms_per_solve_at_plan_creation": res["tune_ms"],
                        "graph_shape": {"plane_chains": res["graph_shape"][0], "x_chains": res["graph_shape"][1]},
                        "note": "poisson_plan_create times {five launches, five + programmatic dependent launch, one fused "
                                "cooperative launch, the five passes as one CUDA graph, that graph with PDL edges} and keeps the fastest; "
                                "the graph's passes are split into parallel chains over ranges of k_a planes and of x "
                                "(poisson_plan_graph_shape): the same tiles by the same kernels, only the dependencies are finer"},
        "e2e": {"value": world * 1e3 / res["e2e_ms_per_step"], "unit": UNIT, "h2d_bytes_per_step": res["rho_bytes"],
                "d2h_bytes_per_step": res["rho_bytes"], "ms_per_step": res["e2e_ms_per_step"], "steps": res["e2e_steps"],
                "api": (f"poisson_solve_batch_host, {res['e2e_batch']} pinned host densities per call: every rho copied H2D, five passes, "
                        "every V copied D2H, stream sync, all inside the timed region (wall clock, max over ranks)"),
                "single_call_ms_per_step": res["e2e_single_ms_per_step"],
                "single_call_api": "poisson_solve_host (one density per call: H2D + 5 passes + D2H + sync, nothing overlapped)"},
        "gpu_launches": int(res["launches_per_solve"] * steps),
        "gpu_launches_note": f"{res['launches_per_solve']} kernels per solve x {steps} solves in ONE timed region ({res['single']['regions']} regions were timed)",
        "clocks": clocks,
    }
    if args.even_kernel:
        line["config"]["kernel_storage"] = "folded: poisson_set_kernel_even (K^F kept for k_b <= S_b/2 only)"
    elif world == 1:
        # SURVEY.md 8f-2 (less K^F traffic): the same solves with the folded K^F copy, timed the same way
        try:
            ev = time_config(pk, torch, args.config, steps, warmup, with_e2e=False, with_cold=False, with_profile=False, inputs=inputs,
                             even_kernel=True)
            line["even_kernel"] = {"ms_per_step": ev["single"]["ms"], "solves_per_sec": 1e3 / ev["single"]["ms"],
                                   "workspace_bytes": ev["workspace_bytes"], "workspace_bytes_full_kernel": res["workspace_bytes"],
                                   "api": "poisson_set_kernel_even + poisson_solve: K^F stored for k_b <= S_b/2 only (kernels even along every axis)"}
        except pk.PoissonError as e:   # e.g. EUNSUPPORTED: pass F3 of this grid runs the any-length kernel
            line["even_kernel"] = {"unavailable": str(e), "status": e.status}
    if world == 1 and not args.no_cpu_baseline:
        sec, desc, threads, extrap, frac, ntimed = oracle_steps(cfg, inputs[1], inputs[2], 3, 0, 30.0)
        line["cpu_baseline"] = {"value": 1.0 / sec, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": desc,
                                "extrapolated": extrap, "sample_fraction": frac}
        # beside it: the same METHOD on the host cores (the paper's own comparison) -- a reported baseline
        line["cpu_pruned_fft"] = pruned_fft_cpu_times(cfg, inputs[1], inputs[2])
    if world == 1 and not args.headline_only:
        others = {}
        for key in ("c0", "c2", "c3", "c4a", "c4b", "c4p"):
            if key == args.config:
                continue
            smp = ClockSampler(local)
            smp.start()
            r = time_config(pk, torch, key, min(steps, 200), 5, with_e2e=True, with_cold=False)
            clk = smp.stop()
            i2 = r["info"]
            others[key] = {"workload": WORKLOAD_TEXT[key], "ms_per_step": r["single"]["ms"],
                           "ms_per_step_min": r["single"]["min"], "ms_per_step_max": r["single"]["max"], "timed_regions": r["single"]["regions"],
                           "clocks": clk,
                           "solves_per_sec": 1e3 / r["single"]["ms"],
                           "hbm_frac": i2.bytes_total / (r["single"]["ms"] * 1e-3) / 1e9 / peak,
                           "batched_ms_per_step": r["batch"]["ms"],
                           "batched_hbm_frac": i2.bytes_total / (r["batch"]["ms"] * 1e-3) / 1e9 / peak,
                           "e2e_ms_per_step": r["e2e_ms_per_step"], "launch_mode": r["launch_mode"], "graph_shape": r["graph_shape"],
                           "pass_us": {pk.PASS_NAMES[q]: r["pass_ms"][q] * 1e3 for q in range(5)},
                           # each pass's algorithmic bytes over its event-bracketed stream launch, as a fraction of the HBM peak
                           "pass_hbm_frac": {pk.PASS_NAMES[q]: (i2.bytes[q] / (r["pass_ms"][q] * 1e-3) / 1e9 / peak) if r["pass_ms"][q] > 0 else None
                                             for q in range(5)},
                           "plan_create_ms": r.get("plan_create_ms")}
        line["other_configs"] = others
        # The paper's Fig. 1 comparison: a free / wire / surface solve against the FULLY PERIODIC solve of the
        # SAME FFT size (free and wire: 58 %, surface: 66 % of the periodic time there).  Equal-size pairs: c1 (128^3 -> 256^3)
        # against c4p (periodic 256^3); c2 / c3 against periodic runs of their padded shapes.
        zs = {"paper_ratio": {"free": 0.58, "wire": 0.58, "surface": 0.66}, "cite": "PAPER.md:79", "pairs": {}}
        ms_of = {args.config: ms}
        ms_of.update({k: v["ms_per_step"] for k, v in others.items()})
        bytes_of = {args.config: info.bytes_total}
        bytes_of.update({k: pk.poisson_plan_describe(*gen.get_config(k).n, gen.get_config(k).bc, pk.FP64).bytes_total for k in others})
        if "c1" in ms_of and "c4p" in ms_of:
            zs["pairs"]["free_256"] = {"padded_grid": [256, 256, 256], "ms": ms_of["c1"], "periodic_ms": ms_of["c4p"],
                                       "ratio_time": ms_of["c1"] / ms_of["c4p"], "ratio_bytes_model": bytes_of["c1"] / bytes_of["c4p"]}
        for key, kind in (("c2", "surface"), ("c3", "wire")):
            if key not in ms_of:
                continue
            try:
                pr = time_periodic_same_fft_size(pk, torch, gen.get_config(key), min(steps, 200), 5)
                zs["pairs"][f"{kind}_{key}"] = {"padded_grid": pr["padded_grid"], "ms": ms_of[key], "periodic_ms": pr["ms"],
                                                "ratio_time": ms_of[key] / pr["ms"], "ratio_bytes_model": bytes_of[key] / pr["bytes_total"]}
            except pk.PoissonError as e:
                zs["pairs"][f"{kind}_{key}"] = {"unavailable": str(e)}
        line["zero_skipping"] = zs
    print(json.dumps(line))
    return 0


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)
    ap.add_argument("--warmup", type=int, default=20)
    ap.add_argument("--impl", choices=("ours", "reference"), default="ours")
    ap.add_argument("--config", default="c1", choices=sorted(WORKLOAD_TEXT))
    ap.add_argument("--headline-only", action="store_true", help="skip the other configs' timings")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--even-kernel", action="store_true", help="install K^F with poisson_set_kernel_even (folded storage) instead of poisson_set_kernel")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)
    return run_ours(args)


if __name__ == "__main__":
    sys.exit(main())
