#!/usr/bin/env python
"""bench.py -- one JSON line: grid points/s of the whole pointwise path on one config.

A "step" = one pass of the whole hot path (crf_thermo + crf_production_rates + crf_mix_transport,
SURVEY.md §8(a) rows a1-a13) over all points of the workload.  Default workload: C5 (BASELINE.json
configs[4], Ns=118/Nr=720, 2 097 152 points), the configuration BASELINE.json's target is quoted on
("on the largest mechanism"); ``--workload C2|C3|C4`` times the others.

  value     points/s with T, p, Y resident in HBM (CUDA events, K steps, max over ranks)
  e2e       the same through crf_step_host with pinned HOST buffers (H2D + kernels + D2H per step)
  roofline  the dominant kernel (largest share of the step), algorithmic flops / measured duration
  cpu_baseline  the oracle (oracle/crf_oracle.c, OpenMP) on a prefix of the same workload

``--impl reference`` times the oracle alone (this tier's reference arm).
N > 1 (torchrun): weak scaling, each rank owns its own full-size field; no data-path collective.
"""
from __future__ import annotations

import argparse
import json
import os
import statistics
import subprocess
import sys
import tempfile
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

METRIC = "grid points/s (fp64 omega_k + mix-avg transport)"
UNIT = "points/s"


def parse():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="C5", choices=["C1", "C2", "C3", "C4", "C5"])
    ap.add_argument("--points", type=int, default=0, help="override the number of points (debug)")
    ap.add_argument("--cpu-points", type=int, default=0, help="oracle sample size (default: ~10-30 s of CPU)")
    ap.add_argument("--path", default="three", choices=["three", "rhs", "jv", "sem"],
                    help="three: crf_thermo + crf_production_rates + crf_mix_transport (the default step); rhs: one "
                         "crf_rhs_pointwise call (SURVEY 8(f)1); jv: one crf_production_rates_jv call (8(f)2); sem: one "
                         "crf_sem_diffusion call on the outputs of crf_rhs_pointwise (8(f)3)")
    ap.add_argument("--plan", nargs="*", default=[], metavar="KEY=VALUE",
                    help="explicit kernel plan (crf_plan_options of include/crf_diag.h, e.g. thermo_sets=2); default: the "
                         "library's automatic plan.  Recorded in config.plan")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    return ap.parse_args()


# oracle sample sizes: ~10-30 s on 8 cores at the measured oracle rates (C5: ~6 k points/s)
CPU_SAMPLE = {"C1": 512, "C2": 1 << 20, "C3": 1 << 19, "C4": 1 << 18, "C5": 1 << 16}


CALLS = {"three": ["crf_thermo", "crf_production_rates", "crf_mix_transport"], "rhs": ["crf_rhs_pointwise"],
         "jv": ["crf_production_rates_jv"], "sem": ["crf_sem_diffusion"]}


def config_dict(name, n, world, path="three"):
    from paper_2409_06404_b200 import workloads as wl
    c = wl.CONFIGS[name]
    return {"workload": f"{name} (BASELINE.json configs[{int(name[1]) - 1}])", "Ns": c["Ns"], "Nr": c["Nr"],
            "N3": c["N3"], "Nt": c["Nt"], "points_per_gpu": n, "elements_per_gpu": n // 512,
            "state": c["state"], "seed": c["seed"], "parallelism": f"points x{world} (no collective)",
            "calls_per_step": CALLS[path],
            "l2": "inputs exceed L2 (no flush needed)" if n * 8 * (c["Ns"] + 2) > 126e6 * 2 else "flushed between steps"}


def run_oracle_sample(name, m_points):
    """The oracle as it stands on the first m points: returns (points/s, threads, seconds)."""
    from oracle import crf_oracle
    from paper_2409_06404_b200 import workloads as wl
    desc = wl.make_mechanism(name)
    st = wl.make_state(name, n=m_points, total=wl.config_points(name))
    o = crf_oracle.Oracle(desc)
    o.thermo(T=st["T"][:64], p=st["p"][:64], Y=st["Y"][:, :64].copy())  # spin up the OpenMP team
    t0 = time.perf_counter()
    o.thermo(**st)
    o.production_rates(**st)
    o.mix_transport(**st)
    dt = time.perf_counter() - t0
    return m_points / dt, crf_oracle.max_threads(), dt


def run_oracle_one_core(name, m_points):
    """The same oracle sample on ONE host core ('all cores ... and additionally 1 core'): a child
    process with OMP_NUM_THREADS=1, so that the OpenMP team of this process is left alone."""
    code = ("import sys, json; sys.path.insert(0, %r); import bench; "
            "v, c, dt = bench.run_oracle_sample(%r, %d); print(json.dumps([v, c, dt]))" % (ROOT, name, m_points))
    env = dict(os.environ, OMP_NUM_THREADS="1")
    try:
        out = subprocess.run([sys.executable, "-c", code], env=env, capture_output=True, text=True, timeout=600)
        v, c, dt = json.loads(out.stdout.strip().splitlines()[-1])
        return v, int(c), dt
    except Exception:  # noqa: BLE001  (a reported baseline: never fail the bench line over it)
        return None, 1, None


def reference_arm(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return 0
    from paper_2409_06404_b200 import workloads as wl
    name = args.workload
    full = args.points or wl.config_points(name)
    m = min(full, args.cpu_points or max(512, CPU_SAMPLE[name] // 8))
    for _ in range(max(args.warmup, 0)):
        run_oracle_sample(name, min(m, 2048))
    rates, secs, cores = [], [], 1
    for _ in range(max(args.steps, 1)):
        r, cores, dt = run_oracle_sample(name, m)
        rates.append(r)
        secs.append(dt)
    value = m * len(secs) / sum(secs)
    sample = f"first {m} points of {name} per step, thermo+rates+transport, gcc -O2 OpenMP"
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
            "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * sum(secs) / len(secs),
            "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(name, full, 1),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": cores, "kind": "oracle", "sample": sample},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))
    return 0


def ncu_counters(workload, kernel):
    """Counters of one launch of `kernel` on `workload` from the committed ncu --set full summary
    (profiles/r02_ncu_counters.csv: measured under the profiler on the build named there, not by this run):
    dict(traffic = dram__bytes_read.sum + dram__bytes_write.sum, fp64_inst = thread-level FP64 pipe instructions
    executed, inst = thread-level instructions executed) or None."""
    path = os.path.join(ROOT, "profiles", "r02_ncu_counters.csv")
    try:
        with open(path) as f:
            rows = [r.split(",") for r in f.read().splitlines() if r and not r.startswith("#")]
        hdr = rows[0]
        for c in rows[1:]:
            d = dict(zip(hdr, c))
            if d.get("workload") == workload and d.get("call") == kernel:
                return dict(traffic=float(d["dram_read_bytes"]) + float(d["dram_write_bytes"]),
                            fp64_inst=float(d["fp64_thread_inst"]), inst=float(d["thread_inst"]), build=d.get("build"))
    except (OSError, KeyError, ValueError, IndexError):
        pass
    return None


class ClockSampler:
    """nvidia-smi clocks / throttle reasons during the timed region (B200_PROFILING.md recipe)."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,"
         "clocks_event_reasons.hw_thermal_slowdown,clocks_event_reasons.sw_thermal_slowdown,"
         "clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", "-i", str(index), f"--query-gpu={self.Q}",
                                       "--format=csv,noheader,nounits", "-lms", "20"], stdout=self.f,
                                      stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except subprocess.TimeoutExpired:
            self.p.kill()
        self.f.flush()
        self.f.seek(0)
        sm, mx, pw, reasons = [], [], [], set()
        names = ["hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"]
        for row in self.f.read().splitlines():
            c = [x.strip() for x in row.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])), mx.append(float(c[1])), pw.append(float(c[2]))
            except ValueError:
                continue
            for nm, v in zip(names, c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(nm)
        self.f.close()
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        return {"sm_mhz": statistics.median(sm), "sm_max_mhz": max(mx), "power_w_max": max(pw),
                "samples": len(sm), "reasons": sorted(reasons)}


def host_cores_for_the_oracle():
    """torchrun exports OMP_NUM_THREADS=1 to every rank.  The CPU baseline is defined on the box's host cores and only
    rank 0 runs it, so that setting is dropped before any OpenMP runtime is loaded (torch's or the oracle's)."""
    if "TORCHELASTIC_RUN_ID" in os.environ and os.environ.get("OMP_NUM_THREADS") == "1":
        os.environ.pop("OMP_NUM_THREADS")


def other_path(args, mech, dev, out, n, name, world, rank, local, barrier, flush, stream):
    """--path rhs | jv: the SURVEY 8(f) calls on the same workload, with the separate-call equivalent timed beside
    them in the same run (CUDA events on the launching stream, K steps each, max over ranks)."""
    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2409_06404_b200 import binding, rooflines
    from paper_2409_06404_b200 import workloads as wl
    Ns = mech.Ns
    f64 = dict(dtype=torch.float64, device="cuda")
    cfg = wl.CONFIGS[name]
    n_eff = int(mech.tables.arrays["eff_ptr"][-1])
    w_th, w_ra, w_tr = (rooflines.thermo_work(Ns), rooflines.rates_work(Ns, cfg["Nr"], cfg["N3"], cfg["Nt"], n_eff),
                        rooflines.transport_work(Ns))
    if args.path == "rhs":
        out.update(cpk=torch.empty(Ns, n, **f64), rho=torch.empty(n, **f64), Wbar=torch.empty(n, **f64))

        def fused():
            mech.rhs_pointwise(dev["T"], dev["p"], dev["Y"], out)

        def separate():  # what a caller does without the fused call: the three calls (no rho, Wbar, c_pk at all)
            mech.thermo(dev["T"], dev["p"], dev["Y"], out["cp"], out["h"])
            mech.production_rates(dev["T"], dev["p"], dev["Y"], out["omega"], out["qdot"])
            mech.mix_transport(dev["T"], dev["p"], dev["Y"], out["mu"], out["lam"], out["rhoD"])
        flops = w_th["F"] + w_ra["F"] + w_tr["F"]
        alg_bytes = 8 * (Ns + 2) + 8 * (3 * Ns + 7)  # one read of T, p, Y; omega, rhoD, c_pk rows and 7 scalar fields
        sep_name, sep_note = "three_calls", "crf_thermo + crf_production_rates + crf_mix_transport (no rho, Wbar, c_pk)"
    elif args.path == "sem":
        rhs = mech.rhs_pointwise(dev["T"], dev["p"], dev["Y"], want_cpk=False)
        nel = n // 512
        h3 = torch.from_numpy(np.random.default_rng(7 + rank).uniform(0.2e-3, 1.5e-3, (nel, 3))).cuda()
        dYo, dTo = torch.empty(Ns, n, **f64), torch.empty(n, **f64)
        gY = torch.empty(3, n, **f64)

        def fused():
            mech.sem_diffusion(h3, dev["T"], rhs["Wbar"], dev["Y"], rhs["lam"], rhs["rhoD"], dYo, dTo)

        def separate():  # the pure stream of the same bytes: what a copy kernel needs for this operator's traffic
            dYo.copy_(dev["Y"])
            out["omega"].copy_(rhs["rhoD"])
            dTo.copy_(dev["T"])
            gY[0].copy_(rhs["lam"])
            gY[1].copy_(rhs["Wbar"])
        # algorithmic minimum per node and field: 24 FMA for the gradient (ONCE: the kernel's second evaluation in pass 2 is
        # its own choice, not the method's), 24 for the weak divergence, ~20 pointwise
        flops = 2 * ((24 + 24 + 20) * Ns + 24 + 24 + 10)
        alg_bytes = 8 * (3 * Ns + 4)  # Y, rho D in, dY out; T, lambda, Wbar in, dT out
        sep_name, sep_note = "copy_calls", "torch copies of the operator's algorithmic bytes (3 Ns + 4 fields in + out): the HBM stream it is bounded by"
    else:
        gen = torch.Generator(device="cuda").manual_seed(1234 + rank)
        v = {k: dev[k] * (2 * torch.rand(dev[k].shape, generator=gen, **f64) - 1) for k in ("T", "p", "Y")}
        sigma = 1e-6
        Jo, Jq = torch.empty(Ns, n, **f64), torch.empty(n, **f64)
        pert = {k: torch.empty_like(dev[k]) for k in ("T", "p", "Y")}
        om2, qd2 = torch.empty(Ns, n, **f64), torch.empty(n, **f64)

        def fused():
            mech.production_rates_jv(dev["T"], dev["p"], dev["Y"], v["T"], v["p"], v["Y"], sigma,
                                     out=(out["omega"], out["qdot"], Jo, Jq))

        def separate():  # perturb (3 axpy), two crf_production_rates calls, two quotients
            for k in ("T", "p", "Y"):
                torch.add(dev[k], v[k], alpha=sigma, out=pert[k])
            mech.production_rates(dev["T"], dev["p"], dev["Y"], out["omega"], out["qdot"])
            mech.production_rates(pert["T"], pert["p"], pert["Y"], om2, qd2)
            torch.sub(om2, out["omega"], out=Jo).div_(sigma)
            torch.sub(qd2, out["qdot"], out=Jq).div_(sigma)
        flops = 2 * w_ra["F"]
        alg_bytes = 8 * 2 * (Ns + 2) + 8 * 2 * (Ns + 1)
        sep_name, sep_note = "separate_calls", "3 axpy + 2 crf_production_rates + 2 quotient kernels (torch elementwise)"

        def with_base():  # the base values in hand (what an integrator has): only the perturbed state is evaluated
            mech.production_rates_jv_base(dev["T"], dev["p"], dev["Y"], v["T"], v["p"], v["Y"], sigma,
                                          out["omega"], out["qdot"], out=(Jo, Jq))
        extra = ("with_base", with_base, "crf_production_rates_jv_base: omega(y), qdot(y) given, one state evaluated",
                 w_ra["F"], 8 * 2 * (Ns + 2) + 8 * 2 * (Ns + 1))

    K = max(args.steps, 1)

    def timed(fn):
        for _ in range(max(args.warmup, 3)):
            fn()
        barrier()
        ev = [torch.cuda.Event(enable_timing=True) for _ in range(K + 1)]
        ev[0].record(stream)
        for k in range(K):
            if flush is not None:
                flush.add_(1)
            fn()
            ev[k + 1].record(stream)
        barrier()
        ms = np.array([ev[k].elapsed_time(ev[k + 1]) for k in range(K)])
        t = torch.tensor([float(ms.mean())], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(t, op=dist.ReduceOp.MAX)
        return float(t.item()), float(np.median(ms)), float(ms.min())

    clocks = ClockSampler(local) if rank == 0 else None
    launches0 = binding.launch_count()
    ms, med, best = timed(fused)
    launches = (binding.launch_count() - launches0) * K // (K + max(args.warmup, 3))
    clock_info = clocks.stop() if clocks else None
    sep_ms, sep_med, sep_best = timed(separate)
    extra_out = None
    if args.path == "jv":
        x_ms, x_med, x_best = timed(extra[1])
        extra_out = {"ms_per_step": x_ms, "ms_median": x_med, "ms_best": x_best, "what": extra[2],
                     "frac_of_fp64_roofline": extra[3] * n / (rooflines.FP64_PEAK_TFLOPS * 1e12) / (x_ms * 1e-3)}
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0
    peaks = rooflines.measured_peaks(ROOT)
    t_alu = flops * n / (rooflines.FP64_PEAK_TFLOPS * 1e12)
    t_hbm = alg_bytes * n / (peaks["hbm_gbs"] * 1e9)
    call = CALLS[args.path][0]
    hbm_bound = t_hbm > t_alu
    roof = {"bound": "hbm" if hbm_bound else "alu", "kernel": call,
            "achieved": alg_bytes * n / (ms * 1e-3) / 1e9 if hbm_bound else flops * n / (ms * 1e-3) / 1e12,
            "peak": peaks["hbm_gbs"] if hbm_bound else rooflines.FP64_PEAK_TFLOPS, "unit": "GB/s" if hbm_bound else "TFLOP/s",
            "frac": max(t_alu, t_hbm) / (ms * 1e-3), "traffic": None,
            "peak_source": "148 SM x 64 FP64 lanes x 1.965 GHz x 2 (DESIGN.md); FMA = 2 flops",
            "flops_per_point": flops, "bytes_per_point": alg_bytes, "t_hbm_ms": 1e3 * t_hbm, "t_alu_ms": 1e3 * t_alu}
    line = {"metric": METRIC, "value": world * n / (ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": max(args.warmup, 3), "ms_per_step": ms, "ms_median": med, "ms_best": best, "higher_is_better": True,
            "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": config_dict(name, n, world, args.path), "clocks": clock_info, "e2e": None,
            "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": None,
            sep_name: {"ms_per_step": sep_ms, "ms_median": sep_med, "ms_best": sep_best, "what": sep_note,
                       "fused_over_separate": ms / sep_ms}}
    if extra_out:
        line[extra[0]] = extra_out
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


def main():
    args = parse()
    host_cores_for_the_oracle()
    if args.impl == "reference":
        return reference_arm(args)

    import numpy as np
    import torch
    import torch.distributed as dist

    from paper_2409_06404_b200 import binding, rooflines, shard
    from paper_2409_06404_b200 import workloads as wl

    rank = int(os.environ.get("RANK", "0"))
    world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if not torch.cuda.is_available():
        raise SystemExit("bench.py needs a CUDA device: there is no CPU fallback for the product path")
    torch.cuda.set_device(local)
    if world > 1:
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    name = args.workload
    n = args.points or wl.config_points(name)
    offset, n, total = shard.weak_range(n, rank, world)
    desc = wl.make_mechanism(name)
    plan = {k: (int(v) if v.lstrip("-").isdigit() else v) for k, v in (kv.split("=", 1) for kv in args.plan)}
    mech = binding.Mechanism(desc, plan or None)
    Ns = mech.Ns
    st = wl.make_state(name, n=n, offset=offset, total=total)
    host = {k: torch.from_numpy(v).pin_memory() for k, v in st.items()}
    dev = {k: v.cuda(non_blocking=True) for k, v in host.items()}
    f64 = dict(dtype=torch.float64, device="cuda")
    out = dict(cp=torch.empty(n, **f64), h=torch.empty(n, **f64), omega=torch.empty(Ns, n, **f64),
               qdot=torch.empty(n, **f64), mu=torch.empty(n, **f64), lam=torch.empty(n, **f64),
               rhoD=torch.empty(Ns, n, **f64))
    flush = None
    if n * 8 * (Ns + 2) <= 126e6 * 2:
        flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda")  # > 126 MB L2
    stream = torch.cuda.current_stream()

    def step(ev=None):
        if flush is not None:
            flush.add_(1)
        if ev:
            ev[0].record(stream)
        mech.thermo(dev["T"], dev["p"], dev["Y"], out["cp"], out["h"])
        if ev:
            ev[1].record(stream)
        mech.production_rates(dev["T"], dev["p"], dev["Y"], out["omega"], out["qdot"])
        if ev:
            ev[2].record(stream)
        mech.mix_transport(dev["T"], dev["p"], dev["Y"], out["mu"], out["lam"], out["rhoD"])
        if ev:
            ev[3].record(stream)

    if args.path != "three":
        return other_path(args, mech, dev, out, n, name, world, rank, local, barrier, flush, stream)

    for _ in range(max(args.warmup, 3)):
        step()
    barrier()
    fp64_inst = binding.fp64_probe(4096) if rank == 0 else 0.0   # measured sustained DFMA rate
    barrier()

    K = max(args.steps, 1)
    evs = [[torch.cuda.Event(enable_timing=True) for _ in range(4)] for _ in range(K)]
    clocks = ClockSampler(local) if rank == 0 else None
    launches0 = binding.launch_count()
    barrier()
    t_start, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    t_start.record(stream)
    for k in range(K):
        step(evs[k])
    t_end.record(stream)
    barrier()
    launches = binding.launch_count() - launches0
    clock_info = clocks.stop() if clocks else None
    total_ms = t_start.elapsed_time(t_end)
    flush_ms = 0.0
    per_kernel = np.array([[e[i].elapsed_time(e[i + 1]) for i in range(3)] for e in evs])  # [K,3] ms
    if flush is not None:  # the flush is not part of the step: time the three calls only
        total_ms = float(per_kernel.sum())
    kern_ms = per_kernel.mean(axis=0)
    kern_med, kern_best = np.median(per_kernel, axis=0), per_kernel.min(axis=0)

    # ---- end to end through crf_step_host: pinned host in, pinned host out
    e2e = None
    if not args.no_e2e:
        hout = dict(cp=torch.empty(n, dtype=torch.float64).pin_memory(), h=torch.empty(n, dtype=torch.float64).pin_memory(),
                    omega=torch.empty(Ns, n, dtype=torch.float64).pin_memory(),
                    qdot=torch.empty(n, dtype=torch.float64).pin_memory(), mu=torch.empty(n, dtype=torch.float64).pin_memory(),
                    lam=torch.empty(n, dtype=torch.float64).pin_memory(),
                    rhoD=torch.empty(Ns, n, dtype=torch.float64).pin_memory())
        mech.step_host(host["T"], host["p"], host["Y"], hout)  # warm-up (allocates the pipeline)
        barrier()
        Ke = max(2, min(K, 5))
        t0 = time.perf_counter()
        for _ in range(Ke):
            mech.step_host(host["T"], host["p"], host["Y"], hout)  # synchronous
        torch.cuda.synchronize()
        e2e_s = (time.perf_counter() - t0) / Ke
        e2e_t = torch.tensor([e2e_s], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(e2e_t, op=dist.ReduceOp.MAX)
        e2e = {"value": world * n / float(e2e_t.item()), "unit": UNIT,
               "h2d_bytes_per_step": 8 * n * (Ns + 2), "d2h_bytes_per_step": 8 * n * (2 * Ns + 5),
               "ms_per_step": 1e3 * float(e2e_t.item()), "steps": Ke,
               "how": "crf_step_host: pinned host buffers, chunked H2D -> 3 kernels -> D2H over 3 streams, host wall clock"}
        del hout
        # the mixed-precision variant (crf_step_host_f32: double arithmetic, outputs rounded to float on the device)
        h32 = {k: torch.empty(sh, dtype=torch.float32).pin_memory() for k, sh in
               dict(cp=(n,), h=(n,), omega=(Ns, n), qdot=(n,), mu=(n,), lam=(n,), rhoD=(Ns, n)).items()}
        mech.step_host(host["T"], host["p"], host["Y"], h32)
        barrier()
        t0 = time.perf_counter()
        for _ in range(Ke):
            mech.step_host(host["T"], host["p"], host["Y"], h32)
        torch.cuda.synchronize()
        s32 = torch.tensor([(time.perf_counter() - t0) / Ke], device="cuda", dtype=torch.float64)
        if world > 1:
            dist.all_reduce(s32, op=dist.ReduceOp.MAX)
        e2e["f32_outputs"] = {"value": world * n / float(s32.item()), "unit": UNIT, "ms_per_step": 1e3 * float(s32.item()),
                              "d2h_bytes_per_step": 4 * n * (2 * Ns + 5),
                              "how": "crf_step_host_f32: the same path, outputs stored in single precision (half the D2H bytes)"}
        del h32

    tt = torch.tensor([total_ms], device="cuda", dtype=torch.float64)
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    total_ms = float(tt.item())
    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return 0

    # ---- roofline of the dominant kernel
    cfg = wl.CONFIGS[name]
    n_eff = int(mech.tables.arrays["eff_ptr"][-1])
    work = {"crf_thermo": rooflines.thermo_work(Ns),
            "crf_production_rates": rooflines.rates_work(Ns, cfg["Nr"], cfg["N3"], cfg["Nt"], n_eff),
            "crf_mix_transport": rooflines.transport_work(Ns)}
    names = list(work)
    peaks = rooflines.measured_peaks(ROOT)
    kernels = {}
    for i, nm in enumerate(names):
        w, ms = work[nm], float(kern_ms[i])
        t_alu = w["F"] * n / (rooflines.FP64_PEAK_TFLOPS * 1e12)
        t_hbm = w["B"] * n / (peaks["hbm_gbs"] * 1e9)
        t_inst = w["I"] * n / rooflines.FP64_PEAK_INST
        kernels[nm] = {"ms": ms, "ms_median": float(kern_med[i]), "ms_best": float(kern_best[i]),
                       "share": ms / float(kern_ms.sum()), "points_per_s": n / (ms * 1e-3),
                       "bound": "alu" if t_alu >= t_hbm else "hbm", "tflops": w["F"] * n / (ms * 1e-3) / 1e12,
                       "gbs": w["B"] * n / (ms * 1e-3) / 1e9, "frac_of_roofline": max(t_alu, t_hbm) / (ms * 1e-3),
                       # the same fraction with the algorithmic work counted in FP64 instructions instead of flops
                       "frac_instr_basis": max(t_inst, t_hbm) / (ms * 1e-3)}
        ctr = ncu_counters(name, nm)
        if ctr:  # what the shipped kernel executes (ncu, committed): FP64 pipe issue rate against the pipe's peak
            kernels[nm]["frac_executed_fp64"] = ctr["fp64_inst"] / rooflines.FP64_PEAK_INST / (ms * 1e-3)
            kernels[nm]["fp64_share_of_executed_inst"] = ctr["fp64_inst"] / ctr["inst"]
            kernels[nm]["dram_traffic_over_algorithmic"] = ctr["traffic"] / (w["B"] * n) if args.points == 0 else None
    dom = max(names, key=lambda k: kernels[k]["ms"])
    ctr = ncu_counters(name, dom)
    traffic = ctr["traffic"] if ctr and args.points == 0 else None
    kd = kernels[dom]
    if kd["bound"] == "alu":
        roof = {"bound": "alu", "kernel": dom, "achieved": kd["tflops"], "peak": rooflines.FP64_PEAK_TFLOPS,
                "unit": "TFLOP/s", "frac": kd["tflops"] / rooflines.FP64_PEAK_TFLOPS, "traffic": traffic,
                "peak_source": "148 SM x 64 FP64 lanes x 1.965 GHz x 2 (DESIGN.md); FMA = 2 flops",
                "peak_measured_dfma": 2 * fp64_inst / 1e12,
                "frac_of_measured_dfma": kd["tflops"] / (2 * fp64_inst / 1e12) if fp64_inst else None,
                "flops_per_point": work[dom]["F"], "fp64_instr_per_point": work[dom]["I"]}
    else:
        roof = {"bound": "hbm", "kernel": dom, "achieved": kd["gbs"], "peak": peaks["hbm_gbs"], "unit": "GB/s",
                "frac": kd["gbs"] / peaks["hbm_gbs"], "traffic": traffic, "peak_source": peaks["source"],
                "bytes_per_point": work[dom]["B"]}

    cpu = None
    if not args.no_cpu:
        m = min(n, args.cpu_points or CPU_SAMPLE[name])
        v, cores, dt = run_oracle_sample(name, m)
        m1 = max(512, m // max(cores, 1))
        v1, _, dt1 = run_oracle_one_core(name, m1)
        cpu = {"value": v, "unit": UNIT, "cores": cores, "kind": "oracle",
               "sample": f"first {m} points of {name}, thermo+rates+transport, gcc -O2 OpenMP, {dt:.1f} s",
               "value_1core": v1, "sample_1core": f"first {m1} points of {name}, OMP_NUM_THREADS=1"
                                                  + (f", {dt1:.1f} s" if dt1 else " (failed)")}

    line = {"metric": METRIC, "value": world * n * K / (total_ms * 1e-3), "unit": UNIT, "n_gpus": world, "steps": K,
            "warmup": max(args.warmup, 3), "ms_per_step": total_ms / K, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": dict(config_dict(name, n, world), plan=plan or "automatic", plan_info=mech.plan_info()),
            "clocks": clock_info, "e2e": e2e, "gpu_launches": int(launches), "roofline": roof, "cpu_baseline": cpu,
            "kernels": kernels}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()
    return 0


if __name__ == "__main__":
    sys.exit(main())
