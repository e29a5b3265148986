#!/usr/bin/env python
"""bench.py -- the headline measurement of the s-step PCG hot path (BASELINE.json):
microseconds per OUTER iteration on the 320^3 7-point fp64 Poisson system (config 4), achieved HBM GB/s vs the
measured peak, GDOF*iter/s; with the CPU oracle timed beside it.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--impl ours|reference] [--s 4] [--grid 320] [--sweep 1,2,4,8]

A "step" is one outer iteration (s Jacobi-fused SpMVs, fused Gram + on-device solves, fused block update) replayed
as one CUDA graph on the live solver state.  Every `restart_every` steps the solve is re-initialised from x0 = 0
inside the timed region (reading A19 in DESIGN.md: 200 outer iterations at s = 8 would run far past convergence),
so the timed region holds exactly K outer iterations plus ceil(K/restart_every) cheap re-initialisations.
Multi-GPU (torchrun): replicas only -- the north_star forbids sharding; every rank runs the same workload and the
job value aggregates them.
"""
from __future__ import annotations

import argparse
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import sstep_inputs as gen  # noqa: E402

METRIC = "sstep_pcg_us_per_outer_iteration"
NOMINAL_HBM_GBS = 8000.0          # north_star's "~8 TB/s"
FALLBACK_HBM_GBS = 6650.0         # /opt/skills/guides/B200_PROFILING.md fallback


# ----------------------------------------------------------------------------------------------- byte model
def model_bytes(n: int, nnz: int, s: int, form: int = 0) -> dict:
    """Algorithmic (compulsory) HBM bytes of one outer iteration, SURVEY.md §8(d) / DESIGN.md "Byte model".
    form 1 (moment form): the moments ride on the SpMV epilogues, so there is no Gram pass."""
    csr = 12 * nnz + 4 * (n + 1)
    mpk = s * csr + 8 * n * (3 * s - 1)       # s matrix sweeps, s gathers + s AR writes + (s-1) R writes
    gram = 0 if form else 8 * n * (3 * s + 1)  # R, AR, AP blocks + r
    update = 8 * n * (6 * s + 5)              # 4 block reads, 2 block writes, x, r read+write, R1 write
    return dict(mpk=mpk, gram=gram, update=update, total=mpk + gram + update, spmv_per_launch=mpk / s)


def c_default_grid(config: int) -> int:
    return {1: 32, 2: 128, 3: 160, 4: 320, 5: 256, 6: 250}[config]


def measured_peak():
    try:
        with open(os.path.join(ROOT, "MEASURED_PEAKS.json")) as f:
            return float(json.load(f)["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    except Exception:
        return FALLBACK_HBM_GBS, "fallback (B200_PROFILING.md)"


def ncu_traffic(config: int, s: int, prefix: str = "spmv"):
    """Per-launch DRAM bytes (read + write) of the kernels whose name starts with `prefix`, from the committed ncu
    summary profiles/ncu_traffic.csv (launch-weighted mean), or None if that workload was not captured."""
    try:
        tot = cnt = 0.0
        with open(os.path.join(ROOT, "profiles", "ncu_traffic.csv")) as f:
            next(f)
            for ln in f:
                c, ss, k, w, rd, wr = ln.split(",")[:6]
                if int(c) == config and int(ss) == s and k.startswith(prefix):
                    tot += float(w) * (float(rd) + float(wr))
                    cnt += float(w)
        return tot / cnt if cnt else None
    except Exception:
        return None


def workload_string(config: int, N: int, n: int, nnz: int, s: int, name: str = "") -> str:
    """config.workload -- the SAME string in both arms (ours / --impl reference), so the driver can tell they ran the same job."""
    if config == 4:
        return (f"config 4: 3-D Poisson 7-point {N}^3 (n={n}, nnz={nnz}), CSR fp64/int32, b=A x*, x*~U[-1,1] seed 3, "
                f"x0=0, Jacobi, s={s}, rtol=0 (fixed iteration count)")
    return (f"config {config} ({name}): grid {N}^3 (n={n}, nnz={nnz}), CSR fp64/int32, x0=0, Jacobi, "
            f"s={s}, rtol=0 (fixed iteration count)")


def restart_every_for(s: int) -> int:
    return max(1, 100 // s)       # <= 100 CG-equivalent steps per restart: far from convergence at 320^3


# ----------------------------------------------------------------------------------------------- clocks
class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled every 20 ms from before the warm-up to the end of the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, device_index: int):
        self.idx = device_index
        self.proc = None
        self.path = None

    def __enter__(self):
        try:
            fd, self.path = tempfile.mkstemp(suffix=".csv")
            os.close(fd)
            self.proc = subprocess.Popen(["nvidia-smi", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                          "-lms", "20", "-i", str(self.idx)], stdout=open(self.path, "w"),
                                         stderr=subprocess.DEVNULL)
            for _ in range(100):                 # nvidia-smi takes a moment to start: wait for its first sample
                if os.path.getsize(self.path) > 0:
                    break
                time.sleep(0.02)
        except Exception:
            self.proc = None
        return self

    def __exit__(self, *exc):
        if self.proc is not None:
            self.proc.terminate()
            try:
                self.proc.wait(timeout=5)
            except Exception:
                self.proc.kill()

    def summary(self) -> dict:
        out = {"sm_mhz": None, "sm_max_mhz": None, "reasons": [], "samples": 0}
        try:
            rows = [ln.split(",") for ln in open(self.path).read().strip().splitlines() if ln.strip()]
            rows = [r for r in rows if len(r) >= 9]          # (a sample cut off by terminate())
            sm = [float(r[1]) for r in rows]
            out["samples"] = len(sm)
            if sm:
                pw = np.array([float(r[3]) for r in rows])
                load = pw >= 0.5 * (pw.min() + pw.max())   # samples taken while the kernels ran (power well above idle)
                out["samples_under_load"] = int(load.sum())
                out["sm_mhz"] = float(np.median(np.array(sm)[load])) if load.any() else float(np.median(sm))
                out["sm_mhz_min"] = float(np.min(np.array(sm)[load])) if load.any() else float(np.min(sm))
                out["sm_max_mhz"] = float(rows[0][2])
                out["power_w_max"] = float(pw.max())
                out["sample_period_ms"] = 20
            names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
            for j, nm in enumerate(names):
                if any(r[5 + j].strip().lower().startswith("active") for r in rows):
                    out["reasons"].append(nm)
            os.unlink(self.path)
        except Exception as e:  # nvidia-smi missing or unparsable: say so instead of inventing numbers
            out["error"] = str(e)
        return out


# ----------------------------------------------------------------------------------------------- distributed plumbing
def dist_env():
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    return world, rank, local


def dist_ops(world: int, backend: str, device):
    """(reduce_max, barrier) of the job: identities at world 1, else torch.distributed over `backend`
    ("nccl" on the GPUs; "gloo" in the CPU test of this host logic).  Used only for timing, never on the data path."""
    if world == 1:
        return (lambda v: v), (lambda: None)
    import torch
    import torch.distributed as dist
    if not dist.is_initialized():
        kw = {"device_id": device} if backend == "nccl" else {}
        dist.init_process_group(backend, **kw)

    def reduce_max(v):
        t = torch.tensor([v], dtype=torch.float64, device=device)
        dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item())

    return reduce_max, dist.barrier


def aggregate_replicas(elapsed_ms: float, k_steps: int, world: int, reduce_max) -> dict:
    """Job-level numbers of N independent replicas: time = max over ranks, units = all ranks' outer iterations."""
    t = reduce_max(elapsed_ms)
    return dict(ms_total=t, ms_per_step=t / k_steps, us_per_outer_job=1e3 * t / (k_steps * world))


# ----------------------------------------------------------------------------------------------- our arm
def time_outer_iterations(torch, h, b, s, k_steps, warmup, barrier):
    """CUDA-event time (ms) of exactly k_steps outer iterations (graph replays) on the solver's stream."""
    R = restart_every_for(s)
    resident = h.get_info("resident") == 1      # whole loop in one cooperative launch: init + 1 launch per restart
    kpo = h.get_info("kernels_per_outer")
    h.solve_begin(b, None, 0.0)
    h.iterate(warmup)
    _, res = h.solve_end(want_x=False)
    assert res["status"] != 2, f"breakdown during warm-up: {res}"
    ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    barrier()
    torch.cuda.synchronize()
    ev0.record()
    done, launches = 0, 0
    while done < k_steps:
        k = min(R, k_steps - done)
        h.solve_begin(b, None, 0.0)
        h.iterate(k)
        done += k
        launches += 2 if resident else 1 + k * kpo
    ev1.record()
    torch.cuda.synchronize()
    barrier()
    ms = ev0.elapsed_time(ev1)
    _, res = h.solve_end(want_x=False)
    last = k_steps - (k_steps - 1) // R * R
    assert res["status"] == 1 and res["outer_iters"] == last, f"timed region did not run all iterations: {res}"
    assert np.isfinite(res["relres"]), res      # (the 2-norm of a CG residual need not fall monotonically)
    return ms, launches, res


def per_iteration_stats(torch, h, b, s, k_steps):
    """Median / min / max device time of single outer iterations (an event between consecutive graph replays), in a
    pass of its own so that the headline region stays one event pair ("median and min")."""
    R = restart_every_for(s)
    k = min(k_steps, R)
    h.solve_begin(b, None, 0.0)
    h.iterate(1)
    evs = [torch.cuda.Event(enable_timing=True) for _ in range(k + 1)]
    evs[0].record()
    for i in range(k):
        h.iterate(1)
        evs[i + 1].record()
    torch.cuda.synchronize()
    h.solve_end(want_x=False)
    us = np.array([1e3 * evs[i].elapsed_time(evs[i + 1]) for i in range(k)])
    return dict(iterations=int(k), median=float(np.median(us)), min=float(us.min()), max=float(us.max()))


def run_ours(args):
    import torch

    import paper_2501_03743_b200 as cg

    world, rank, local = dist_env()
    assert torch.cuda.is_available(), "bench.py needs a GPU: the hot path has no CPU fallback"
    torch.cuda.set_device(local)
    reduce_max, barrier = dist_ops(world, "nccl", torch.device("cuda", local))

    s0 = args.s
    t0 = time.time()
    c = gen.make_config(args.config, N=args.grid if args.config == 4 else (args.grid_override or None))
    N = c["N"]
    t_gen = time.time() - t0
    n, nnz = c["n"], c["nnz"]
    dev = lambda a: torch.from_numpy(np.ascontiguousarray(a)).cuda(local)
    rp, ci, va, b = dev(c["rowptr"]), dev(c["colidx"]), dev(c["vals"]), dev(c["b"])
    peak, peak_src = measured_peak()

    sweep = {}
    primary = None
    sustained = None
    read_peak = None
    s_list = [s0] + [int(t) for t in args.sweep.split(",") if t and int(t) != s0] if args.sweep else [s0]
    runs = [(0, s) for s in s_list] + ([(1, s) for s in s_list] if args.moment_form else [])
    moment = {}
    for form, s in runs:
        with cg.SStepCG(local, form=form, resident=1, **args.extra) as h:      # graph path: one launch per kernel, per-kernel times
            torch.cuda.synchronize()
            t_setup = time.perf_counter()
            h.setup(rp, ci, va, s)
            torch.cuda.synchronize()
            t_setup = time.perf_counter() - t_setup
            info = {k: h.get_info(k) for k in ("lanes", "spmv_bulk", "spmv_cta", "spmv_grid", "gram_grid", "update_grid", "reordered", "cm_levels", "pdl")}
            info["setup_seconds"] = t_setup      # validation, dinv, (auto) Cuthill-McKee reordering, workspaces, graph capture
            if s == s0 and form == 0:
                with ClockSampler(local) as clk:
                    ms, launches, res = time_outer_iterations(torch, h, b, s, args.steps, args.warmup, barrier)
                clocks = clk.summary()
                # sustained: the same step for >= 2 s (the headline region of a short --steps run is a burst at boost clocks;
                # a long solve runs under the power cap), its own clock samples beside it
                if args.sustained_s > 0:
                    R = restart_every_for(s)
                    k_sus = int(np.ceil(args.sustained_s * 1e3 / (ms / args.steps) / R)) * R
                    with ClockSampler(local) as clk2:
                        ms2, _, _ = time_outer_iterations(torch, h, b, s, k_sus, args.warmup, barrier)
                    us2 = 1e3 * reduce_max(ms2) / k_sus
                    mbs = model_bytes(n, nnz, s, form)["total"]
                    sustained = dict(us_per_outer=us2, steps=k_sus, seconds=ms2 / 1e3, achieved_gbs=mbs / (us2 * 1e-6) / 1e9,
                                     frac_of_measured_peak=mbs / (us2 * 1e-6) / 1e9 / peak, clocks=clk2.summary())
                # read-side and copy bandwidth of this box from the library's own streaming kernels (csrc/measure.cuh)
                if args.read_peak:
                    big = 8 << 30
                    rp_ldg = h.measure_bandwidth(0, big, 1, 5)
                    # bulk-copy path by the number of copies an SM keeps in flight (variants 3, 1, 5, 4 = 96, 48, 32, 24): HBM and L2
                    inflight = {96: 3, 48: 1, 32: 5, 24: 4}
                    bulk_hbm = {k: h.measure_bandwidth(v, big, 1, 3)[0] for k, v in inflight.items()}
                    bulk_l2 = {k: h.measure_bandwidth(v, 48 << 20, 64, 3)[0] for k, v in inflight.items()}
                    rp_bulk = max(bulk_hbm.values())
                    cp = h.measure_bandwidth(2, big // 2, 1, 5)
                    l2 = h.measure_bandwidth(0, 48 << 20, 64, 5)
                    read_peak = dict(read_ldg_gbs=rp_ldg[0], read_bulk_gbs=rp_bulk, read_peak_gbs=max(rp_ldg[0], rp_bulk),
                                     copy_gbs=cp[0], l2_read_48mb_gbs=max(l2[0], max(bulk_l2.values())),
                                     bulk_by_copies_in_flight_per_sm=dict(hbm_gbs=bulk_hbm, l2_gbs=bulk_l2),
                                     mean=dict(read_ldg=rp_ldg[1], copy=cp[1], l2_ldg=l2[1]),
                                     how="sstep_cg_measure_bandwidth: 8 GiB zero-filled buffer read once per launch (copy: 4 GiB "
                                         "read + 4 GiB written), best / mean of 3-5 launches; l2 = a 48 MiB buffer read 64 times in one launch")
            else:
                ms, launches, res = time_outer_iterations(torch, h, b, s, args.steps, args.warmup, barrier)
            agg = aggregate_replicas(ms, args.steps, world, reduce_max)
            mb = model_bytes(n, nnz, s, form)
            us = 1e3 * agg["ms_per_step"]
            entry = dict(s=s, form="moment" if form else "gram", us_per_outer=us, us_per_cg_equiv_iter=us / s, model_gb_per_outer=mb["total"] / 1e9,
                         achieved_gbs=mb["total"] / (us * 1e-6) / 1e9,
                         frac_of_measured_peak=mb["total"] / (us * 1e-6) / 1e9 / peak,
                         frac_of_nominal_8tbs=mb["total"] / (us * 1e-6) / 1e9 / NOMINAL_HBM_GBS,
                         gdof_iter_per_s=world * n * s / (us * 1e-6) / 1e9, relres_at_end=res["relres"], **info)
            # per-kernel device times (un-graphed, CUDA events around every launch, on the live solve state)
            h.solve_begin(b, None, 0.0)
            h.iterate(3)
            reps = max(2, min(10, restart_every_for(s) - 4))
            t_spmv, t_gram, t_upd = h.profile_outer(reps)
            h.solve_end(want_x=False)
            k_us = dict(spmv=1e3 * t_spmv / (reps * s), gram=1e3 * t_gram / reps, update=1e3 * t_upd / reps)
            entry["kernel_us"] = k_us
            entry["kernel_gbs"] = dict(spmv=mb["spmv_per_launch"] / k_us["spmv"] / 1e3, gram=mb["gram"] / k_us["gram"] / 1e3,
                                       update=mb["update"] / k_us["update"] / 1e3)
            if form:
                k_us["sw"] = k_us.pop("gram")          # the one-block scalar-work kernel takes the Gram kernel's place
                entry["kernel_gbs"].pop("gram")
            entry["kernel_frac_of_measured_peak"] = {k: v / peak for k, v in entry["kernel_gbs"].items()}
            t_all = s * k_us["spmv"] + sum(v for k, v in k_us.items() if k != "spmv")
            entry["kernel_share_of_step"] = {k: (v * (s if k == "spmv" else 1)) / t_all for k, v in k_us.items()}
            if not form and h.get_info("resident") == 0:
                entry["us_per_outer_stats"] = per_iteration_stats(torch, h, b, s, args.steps)
            if form:
                moment[str(s)] = entry
                continue
            sweep[str(s)] = entry
            if s == s0:
                primary = dict(entry, launches=launches, agg=agg, mb=mb)
    # the textbook PCG of Alg. 1 as its own kernel sequence (option method = 1): the classical
    # two-reduction comparator on the same workload; one "outer iteration" = one CG iteration
    pcg = None
    if args.pcg:
        with cg.SStepCG(local, method=1, **args.extra) as h:
            h.setup(rp, ci, va, 1)
            ms, launches, res = time_outer_iterations(torch, h, b, 1, args.steps, args.warmup, barrier)
            agg = aggregate_replicas(ms, args.steps, world, reduce_max)
            us = 1e3 * agg["ms_per_step"]
            bytes_it = 12 * nnz + 4 * (n + 1) + 8 * n * 12      # CSR + p, s | p, s, x, r -> x, r, u | u, p -> p
            h.solve_begin(b, None, 0.0)
            h.iterate(3)
            t_spmv, t_upd, t_dir = h.profile_outer(10)
            h.solve_end(want_x=False)
            pcg = dict(us_per_iteration=us, model_gb_per_iteration=bytes_it / 1e9, achieved_gbs=bytes_it / (us * 1e-6) / 1e9,
                       frac_of_measured_peak=bytes_it / (us * 1e-6) / 1e9 / peak, gdof_iter_per_s=world * n / (us * 1e-6) / 1e9,
                       kernel_us=dict(spmv=1e2 * t_spmv, update=1e2 * t_upd, direction=1e2 * t_dir), launches=launches,
                       note="Alg. 1 PCG-HS (PAPER.md:48-73), 3 kernels and 2 reductions per iteration; compare with "
                            "us_per_cg_equiv_iter of the s-step entries")
    # resident path: what sstep_cg_solve runs by default when every CTA's rows fit shared memory
    resident = None
    with cg.SStepCG(local, **args.extra) as h:
        h.setup(rp, ci, va, s0)
        if h.get_info("resident") == 1:
            ms, launches, res = time_outer_iterations(torch, h, b, s0, args.steps, args.warmup, barrier)
            agg = aggregate_replicas(ms, args.steps, world, reduce_max)
            resident = dict(s=s0, us_per_outer=1e3 * agg["ms_per_step"], launches=launches, grid=h.get_info("resident_grid"),
                            rows_per_cta=h.get_info("resident_rows_per_block"), smem_bytes=h.get_info("resident_smem_bytes"),
                            gdof_iter_per_s=world * n * s0 / (1e3 * agg["ms_per_step"] * 1e-6) / 1e9, relres_at_end=res["relres"],
                            sync=("tagged-word exchange between the CTAs, no grid barrier" if h.get_info("resident_sync") == 0
                                  else "s + 1 grid barriers per outer iteration"),
                            note="whole loop in one cooperative launch per restart (csrc/resident.cuh)")
    return dict(world=world, rank=rank, local=local, c=c, n=n, nnz=nnz, N=N, sweep=sweep, moment=moment, primary=primary, clocks=clocks,
                resident=resident, pcg=pcg, sustained=sustained, read_peak=read_peak,
                peak=peak, peak_src=peak_src, t_gen=t_gen, dev=(rp, ci, va, b))


def run_e2e(args, ctx):
    """The same metric through the C-ABI call with HOST buffers, as a user makes it: ONE sstep_cg_solve_host call that
    uploads the pinned CSR arrays and b, runs setup and the WHOLE solve to the config's own tolerance (config 4:
    rtol = 1e-8, 125 outer iterations at s = 4) and downloads x -- all inside the timed region.  value = that time
    divided by the outer iterations executed."""
    import torch

    import paper_2501_03743_b200 as cg
    c, s = ctx["c"], args.s
    rtol = float(c.get("rtol", 1e-8))
    pin = lambda a: torch.from_numpy(np.ascontiguousarray(a)).pin_memory()
    rp, ci, va, b = pin(c["rowptr"]), pin(c["colidx"]), pin(c["vals"]), pin(c["b"])
    x = torch.empty(c["n"], dtype=torch.float64).pin_memory()
    best = None
    with cg.SStepCG(ctx["local"], **args.extra) as h:
        # first pass warms allocator / graph instantiation paths; report the fastest of the next two -- or, for solves of a
        # few milliseconds (configs 1, 2), of as many as fit into ~0.3 s: after python-side gaps the GPU sits in a low
        # power state and single short passes were seen anywhere between 2 and 40 ms
        passes, spent = 0, 0.0
        for it in range(40):
            if it >= 3 and spent > 300.0:
                break
            ev0, ev1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
            torch.cuda.synchronize()
            t0 = time.perf_counter()
            ev0.record()
            _, res = h.solve_host(rp, ci, va, b, s, rtol=rtol, maxit=2000, x_out=x)
            ev1.record()
            torch.cuda.synchronize()
            wall_ms = 1e3 * (time.perf_counter() - t0)
            cur = dict(ms=max(ev0.elapsed_time(ev1), wall_ms), res=res)
            spent += cur["ms"]
            passes += 1
            if it >= 1 and (best is None or cur["ms"] < best["ms"]):
                best = cur
    k = best["res"]["outer_iters"]
    assert k >= 1 and best["res"]["status"] in (0, 1, 2), best
    # for reading the number: the same four uploads alone (pinned -> device), outside the timed region
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    tmp = [a.cuda(ctx["local"], non_blocking=True) for a in (rp, ci, va, b)]
    torch.cuda.synchronize()
    h2d_ms = 1e3 * (time.perf_counter() - t0)
    del tmp
    xerr = None
    if "xstar" in c and c["xstar"] is not None:
        xs = np.asarray(c["xstar"])
        xerr = float(np.linalg.norm(x.numpy() - xs) / np.linalg.norm(xs))
    h2d = rp.numel() * 4 + ci.numel() * 4 + va.numel() * 8 + b.numel() * 8
    return dict(value=1e3 * best["ms"] / k, unit="us", h2d_bytes_per_step=h2d / k, d2h_bytes_per_step=x.numel() * 8 / k,
                outer_iters=k, status=best["res"]["status_name"], relres=best["res"]["relres"], rtol=rtol, total_ms=best["ms"],
                rel_error_vs_xstar=xerr, h2d_alone_ms=h2d_ms, passes=passes,
                note="one sstep_cg_solve_host call: pinned host CSR+b -> device, setup (validation, dinv, reordering if "
                     f"needed, graph capture), the whole solve to rtol={rtol:g} ({k} outer iterations), x -> host; all "
                     "inside the timed region; value = total / outer iterations")


def run_cpu_baseline(args, ctx):
    """The oracle as it stands, on the host cores of this box, on a bounded sample of the same workload: `iters` outer
    iterations at full size, clocked inside the C loop (start-up excluded), (1) single-threaded as written and (2) the
    same source built with -fopenmp on all cores this process may use (SURVEY.md 8(d) "Oracle timed beside it")."""
    import oracle
    c, s = ctx["c"], args.s
    iters = args.cpu_iters
    mb = model_bytes(ctx["n"], ctx["nnz"], s)["total"]
    cores = len(os.sched_getaffinity(0))
    per_omp, start_omp, _ = oracle.sstep_timed(c["rowptr"], c["colidx"], c["vals"], c["b"], s, iters, omp=True)
    per_1, start_1, _ = oracle.sstep_timed(c["rowptr"], c["colidx"], c["vals"], c["b"], s, iters, omp=False)
    threads = oracle.omp_threads()
    leg = lambda per: dict(us_per_outer=1e6 * per, gdof_iter_per_s=ctx["n"] * s / per / 1e9, effective_gbs=mb / per / 1e9)
    # (value = the all-core leg; should a box's CPU quota make it the slower one, the single-thread leg is reported instead)
    best_is_omp = per_omp <= per_1
    return dict(value=1e6 * (per_omp if best_is_omp else per_1), unit="us", cores=threads if best_is_omp else 1, kind="oracle",
                value_leg="all_cores" if best_is_omp else "single_thread",
                sample=f"{iters} outer iterations (s={s}) of the same {ctx['N']}^3 system at full size, the oracle's start-up "
                       f"(dinv, r0) excluded; value = oracle/sstep_oracle.c built with -fopenmp on {threads} threads "
                       f"(sched_getaffinity: {cores} cores), single_thread = the same file as the parity tests use it",
                all_cores=leg(per_omp), single_thread=dict(leg(per_1), cores=1), iterations=iters,
                startup_seconds=dict(all_cores=start_omp, single_thread=start_1),
                note="a reported baseline, not the target: a deliberately plain program (long double inner products)")


# ----------------------------------------------------------------------------------------------- reference arm
def run_reference(args):
    """--impl reference: the oracle (oracle/sstep_oracle.c, as it stands) on this box's host cores.
    A step is ONE oracle outer iteration on a bounded sample of config 4: the 7-point operator on a
    grid x grid x nz z-slab (same plane size, same nnz/row; nz = grid, i.e. the whole system, when the budget allows),
    nz sized so that warm-up + K steps end within ~2.5 minutes; a value measured on a slab is scaled by grid/nz to the
    rows of the full workload.  value = the -fopenmp build of the same source on all cores; the single-threaded build
    (the one the parity tests use) is timed beside it on the same slab for a few iterations."""
    import oracle
    world, rank, _ = dist_env()
    if rank != 0:
        return None
    N, s, K, W = args.grid, args.s, args.steps, args.warmup
    R = restart_every_for(s)

    def slab(nz):
        if nz == N:                          # the full workload itself
            c = gen.make_config(4, N=N)
            return c["rowptr"], c["colidx"], c["vals"], c["b"]
        rp, ci, va = gen.poisson7_box(N, N, nz)
        xs = np.random.default_rng(3).uniform(-1.0, 1.0, N * N * nz)
        return rp, ci, va, gen.apply_poisson7_box(N, N, nz, xs)

    rp, ci, va, b = slab(4)
    per_row = oracle.sstep_timed(rp, ci, va, b, s, 2, omp=True)[0] / (N * N * 4)
    budget = float(os.environ.get("SSTEP_REF_BUDGET_S", "120"))
    nz = int(max(2, min(N, budget / ((K + W) * per_row * N * N))))
    rp, ci, va, b = slab(nz)

    def run(k, omp):
        done, t = 0, 0.0
        while done < k:
            kk = min(R, k - done)
            per, _, res = oracle.sstep_timed(rp, ci, va, b, s, kk, omp=omp)
            assert res["iters"] == kk and res["status"] == 1, res
            t += per * kk
            done += kk
        return t

    run(W, True)
    t = run(K, True)
    k1 = max(1, min(K, 3))
    t1 = run(k1, False)
    threads, cores = oracle.omp_threads(), len(os.sched_getaffinity(0))
    us_full_1 = 1e6 * t1 / k1 * N / nz
    value_leg = "all_cores"
    if t1 / k1 < t / K:      # a CPU quota below the visible core count: the single-thread leg is the better baseline
        t, K_eff, threads_used, value_leg = t1, k1, 1, "single_thread"
    else:
        K_eff, threads_used = K, threads
    us_sample = 1e6 * t / K_eff
    us_full = us_sample * N / nz
    n, nnz = N ** 3, 7 * N ** 3 - 6 * N ** 2
    mb = model_bytes(n, nnz, s)["total"]
    sample = (f"{K} oracle outer iterations (s={s}) on the {N}x{N}x{nz} z-slab of the {N}^3 7-point system"
              + (" (the whole system)" if nz == N else f"; value scaled by {N}/{nz} to the full row count")
              + f", oracle/sstep_oracle.c built with -fopenmp on {threads} threads (sched_getaffinity: {cores} cores), start-up "
              f"excluded, restarted from x0=0 every {R} iterations; single_thread = the plain build, {k1} iterations on the same slab; "
              f"value = the {value_leg} leg")
    return {
        "metric": METRIC, "value": us_full, "unit": "us", "n_gpus": args.gpus, "steps": K, "warmup": W,
        "ms_per_step": us_full / 1e3, "higher_is_better": False, "scaling": "weak", "vs_baseline": None, "dtype": "f64",
        "data": "synthetic", "impl": "reference",
        "config": {"workload": workload_string(4, N, n, nnz, s), "s": s, "grid": N, "restart_every": R, "sample": sample},
        "cpu_baseline": {"value": us_full, "unit": "us", "cores": threads_used, "kind": "oracle", "sample": sample, "value_leg": value_leg,
                         "measured_us_per_step_on_sample": us_sample, "effective_gbs": mb / (us_full * 1e-6) / 1e9,
                         "single_thread": {"us_per_outer": us_full_1, "cores": 1, "effective_gbs": mb / (us_full_1 * 1e-6) / 1e9}},
        "e2e": {"value": us_full, "unit": "us", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
        "gdof_iter_per_s": n * s / (us_full * 1e-6) / 1e9,
    }


# ----------------------------------------------------------------------------------------------- main
def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=200)       # config 4: "fixed 200 outer iterations for timing"
    ap.add_argument("--warmup", type=int, default=10)
    ap.add_argument("--impl", choices=["ours", "reference"], default="ours")
    ap.add_argument("--s", type=int, default=0, help="block size of the headline value (0 = the config's own: 2, 4, 4, 4, 8 for "
                                                     "configs 1-5, 4 for the paper-shaped config 6; the paper uses s <= 5)")
    ap.add_argument("--grid", type=int, default=320, help="grid edge N of config 4 (N^3 unknowns)")
    ap.add_argument("--config", type=int, default=4, choices=[1, 2, 3, 4, 5, 6],
                    help="BASELINE.json config (4 = the headline workload; the others fill BASELINE.md's table; 6 = the "
                         "paper's own 250^3, b = 1 problem).  The reference arm and the roofline always describe what ran.")
    ap.add_argument("--grid-override", type=int, default=0, help="grid edge for --config != 4 (0 = the config's own)")
    ap.add_argument("--sweep", type=str, default="1,2,4,8", help="block sizes also reported (config 4's sweep); '' = none")
    ap.add_argument("--no-moment-form", dest="moment_form", action="store_false",
                    help="skip the extra lines for the moment form (option form = 1) of the same block sizes")
    ap.add_argument("--no-pcg", dest="pcg", action="store_false", help="skip the Alg. 1 (PCG-HS) comparator line")
    ap.add_argument("--sustained-s", type=float, default=2.0, help="length in seconds of the extra sustained pass (0 = skip)")
    ap.add_argument("--no-read-peak", dest="read_peak", action="store_false", help="skip the read-side / copy / L2 bandwidth probes")
    ap.add_argument("--no-cpu-baseline", action="store_true")
    ap.add_argument("--cpu-iters", type=int, default=5, help="oracle outer iterations timed per cpu_baseline leg")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=INT",
                    help="extra solver option for every handle of the run (sstep_cg_set_option), e.g. --opt pdl=0; repeatable")
    args = ap.parse_args()
    args.extra = {kv.split("=", 1)[0]: int(kv.split("=", 1)[1]) for kv in args.opt}
    args.warmup = max(args.warmup, 3)
    if args.s == 0:
        args.s = {1: 2, 2: 4, 3: 4, 4: 4, 5: 8, 6: 4}[args.config]

    if args.impl == "reference":
        line = run_reference(args)
        if line is not None:
            print(json.dumps(line), flush=True)
        return

    ctx = run_ours(args)
    world, rank = ctx["world"], ctx["rank"]
    if world != args.gpus and rank == 0:
        print(f"[bench] note: --gpus {args.gpus} but WORLD_SIZE={world}; reporting n_gpus={world}", file=sys.stderr)
    e2e = None
    if not args.no_e2e:
        e2e = run_e2e(args, ctx)          # every rank runs it (replicas); rank 0 reports its own
    cpu = None
    if rank == 0 and world == 1 and not args.no_cpu_baseline:
        cpu = run_cpu_baseline(args, ctx)
    if world > 1:
        import torch.distributed as dist
        dist.barrier()
        dist.destroy_process_group()
    if rank != 0:
        return
    p, s, N, n, nnz = ctx["primary"], args.s, ctx["N"], ctx["n"], ctx["nnz"]
    mb = p["mb"]
    k_us = p["kernel_us"]["spmv"]
    line = {
        "metric": METRIC,
        "value": p["agg"]["us_per_outer_job"],
        "unit": "us",
        "n_gpus": world, "steps": args.steps, "warmup": args.warmup,
        "ms_per_step": p["agg"]["ms_per_step"],
        "higher_is_better": False,
        "scaling": "weak",
        "vs_baseline": None,             # BASELINE.md holds no published number for this metric/workload
        "dtype": "f64",
        "data": "synthetic",
        "config": {
            "workload": workload_string(args.config, N, n, nnz, s, ctx["c"]["name"]),
            "s": s, "grid": N, "restart_every": restart_every_for(s), "options": args.extra, "pdl": p.get("pdl"),
            "l2": "inputs larger than L2: one outer iteration streams %.1f GB >> 126 MB" % (mb["total"] / 1e9),
            "parallelism": "replicas only (north_star: one GPU, no sharding)" if world > 1 else "single GPU",
        },
        "us_per_outer_stats": p.get("us_per_outer_stats"),   # single outer iterations (separate pass): median / min / max
        "gdof_iter_per_s": p["gdof_iter_per_s"],
        "achieved_gbs": p["achieved_gbs"],
        "iteration_roofline": {"bound": "hbm", "achieved": p["achieved_gbs"], "peak": ctx["peak"], "unit": "GB/s",
                               "frac": p["frac_of_measured_peak"], "frac_of_nominal_8tbs": p["frac_of_nominal_8tbs"],
                               "algorithmic_bytes_per_outer": mb["total"]},
        "roofline": {"bound": "hbm", "kernel": ("spmv_cta_kernel" if p.get("spmv_cta") else "spmv_bulk_kernel" if p["spmv_bulk"] else "spmv_vec_kernel")
                     + " (Jacobi-fused CSR SpMV, s launches per outer iteration)",
                     "achieved": mb["spmv_per_launch"] / k_us / 1e3, "peak": ctx["peak"], "unit": "GB/s",
                     "frac": mb["spmv_per_launch"] / k_us / 1e3 / ctx["peak"], "peak_source": ctx["peak_src"],
                     "read_peak": ctx["read_peak"]["read_peak_gbs"] if ctx["read_peak"] else None,
                     "frac_of_read_peak": (mb["spmv_per_launch"] / k_us / 1e3 / ctx["read_peak"]["read_peak_gbs"]) if ctx["read_peak"] else None,
                     "algorithmic_bytes_per_launch": mb["spmv_per_launch"], "avg_launch_us": k_us,
                     "share_of_step": p["kernel_share_of_step"]["spmv"],
                     "traffic": ncu_traffic(args.config, s) if N == c_default_grid(args.config) else None,
                     "traffic_source": "profiles/ncu_traffic.csv (ncu --set full, dram__bytes_read.sum + dram__bytes_write.sum per launch)"},
        "kernels": {"us": p["kernel_us"], "gbs": p["kernel_gbs"], "frac_of_measured_peak": p["kernel_frac_of_measured_peak"],
                    "share_of_step": p["kernel_share_of_step"],
                    # the SpMV is 87 % reads and the Gram kernel 99.9 %: against the READ-side wall of this box
                    "frac_of_read_peak": ({k: p["kernel_gbs"][k] / ctx["read_peak"]["read_peak_gbs"] for k in ("spmv", "gram")
                                           if k in p["kernel_gbs"]} if ctx["read_peak"] else None)},
        "read_peak": ctx["read_peak"],
        "sustained": ctx["sustained"],
        "sweep": ctx["sweep"],
        "pcg_hs": ctx["pcg"],             # Alg. 1 as its own kernel sequence (comparator, not the headline)
        "resident_path": ctx["resident"],  # only for problems that fit shared memory (config 1), else null
        "moment_form": ctx["moment"],     # same solver with Alg. 5 + Alg. 6 (no Gram pass); not the headline
        "clocks": ctx["clocks"],
        "gpu_launches": p["launches"],
        "e2e": e2e,
        "cpu_baseline": cpu,
        "host_generation_seconds": ctx["t_gen"],
    }
    print(json.dumps(line), flush=True)


if __name__ == "__main__":
    main()
