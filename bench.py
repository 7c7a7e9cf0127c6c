#!/usr/bin/env python
"""bench.py -- the hot path of SURVEY.md section 8(a) timed on B200 (contract: see DESIGN.md "Measurement").

One step = one pass of the whole hot path over one batch of synthetic input with the momenta already
resident in HBM: S1 ami_dispersion (momenta -> line energies) then S2+S3 ami_evaluate (leaf phase + term
phase), all through the C ABI of include/ami.h.  Prints ONE JSON line.

  python bench.py [--gpus N] [--steps K] [--warmup W] [--workload cfg3] [--impl ours|reference]

--impl reference times the CPU oracle (oracle/, as it stands) on the host cores on a bounded sample of the
same workload.  Nothing here reads /root/reference.
"""
from __future__ import annotations

import argparse
import json
import os
import sys
import threading
import time

ROOT = os.path.dirname(os.path.abspath(__file__))
if ROOT not in sys.path:
    sys.path.insert(0, ROOT)

import numpy as np  # noqa: E402

METRIC = "ami_term_evaluations_per_s"
UNIT = "term-evals/s"
SUM_ORDER = "default"
ORDERED_ONLY = False     # --ordered: issue every step in plain stream order (no AMI_PLAN_UNORDERED)
BATCHES_NOTE = ("independent batches, each with its own momenta and result buffer, issued with AMI_PLAN_UNORDERED (the "
                "kernel of one batch may start while its predecessor drains); the batch that begins the reuse of the "
                "buffers is ordered; ordered_ms_per_step = the same K batches in plain stream order")


def parse_args():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=20)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--workload", default="cfg3", help="cfg1 | cfg2_se | cfg2_bubble | cfg3 | cfg4 | cfg5 | stress8")
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--n", type=int, default=0, help="override samples per step per GPU")
    ap.add_argument("--plan", default="auto", choices=["auto", "flat", "reg", "tree"])
    ap.add_argument("--sum-order", default="default", choices=["default", "fewest_terms", "fewest_ops"],
                    help="order of the Matsubara sums: the configuration's (default) or the one ami_search_sum_order picks")
    ap.add_argument("--no-extra", action="store_true", help="skip the secondary workloads and the CPU baseline")
    ap.add_argument("--no-graph", action="store_true", help="launch every step from Python instead of one CUDA graph")
    ap.add_argument("--ordered", action="store_true",
                    help="issue the steps in plain stream order instead of as independent batches (AMI_PLAN_UNORDERED)")
    ap.add_argument("--sweep", action="store_true",
                    help="batch-size sweep (BASELINE config 2: N = 1e3..1e8; the paper's Figs. 4-5 plot time against "
                         "the batch size): one JSON line with a row per (workload, N); one GPU")
    ap.add_argument("--cpu-seconds", type=float, default=12.0, help="target CPU time of the oracle sample")
    return ap.parse_args()


# ------------------------------------------------------------------------------------------------
# clocks: sampled DURING the timed region
# ------------------------------------------------------------------------------------------------
class ClockSampler:
    BAD = ("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown")

    def __init__(self, index=0, period=0.01):
        self.index, self.period = index, period
        self.samples, self.reasons = [], set()
        self.sm_max = None
        self._stop = threading.Event()
        self._th = None
        try:
            import pynvml
            pynvml.nvmlInit()
            self.nv = pynvml
            self.h = pynvml.nvmlDeviceGetHandleByIndex(index)
            self.sm_max = int(pynvml.nvmlDeviceGetMaxClockInfo(self.h, pynvml.NVML_CLOCK_SM))
        except Exception:  # noqa: BLE001
            self.nv = None

    def _loop(self):
        nv = self.nv
        names = {
            "hw_slowdown": getattr(nv, "nvmlClocksEventReasonHwSlowdown", 0x8),
            "hw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonHwThermalSlowdown", 0x40),
            "sw_thermal_slowdown": getattr(nv, "nvmlClocksEventReasonSwThermalSlowdown", 0x20),
            "sw_power_cap": getattr(nv, "nvmlClocksEventReasonSwPowerCap", 0x4),
        }
        while not self._stop.is_set():
            try:
                self.samples.append(int(nv.nvmlDeviceGetClockInfo(self.h, nv.NVML_CLOCK_SM)))
                try:
                    mask = int(nv.nvmlDeviceGetCurrentClocksEventReasons(self.h))
                except Exception:  # noqa: BLE001
                    mask = int(nv.nvmlDeviceGetCurrentClocksThrottleReasons(self.h))
                for k, bit in names.items():
                    if mask & bit:
                        self.reasons.add(k)
            except Exception:  # noqa: BLE001
                pass
            self._stop.wait(self.period)

    def start(self):
        if self.nv is not None:
            self._th = threading.Thread(target=self._loop, daemon=True)
            self._th.start()

    def stop(self):
        self._stop.set()
        if self._th:
            self._th.join()
        med = int(np.median(self.samples)) if self.samples else None
        return {"sm_mhz": med, "sm_max_mhz": self.sm_max, "reasons": sorted(self.reasons),
                "n_samples": len(self.samples)}


# ------------------------------------------------------------------------------------------------
# algorithmic FP64 work per sample, in FP64-pipe instruction slots:
#   W = N_eps (2 c_cos + 2)                      [S1: two cosines, one add, one fma per energy symbol]
#     + N_b U_F c_fermi                          [S2: Fermi/Bose leaves, once per beta]
#     + N_f U_D c_den  (register plan; x N_b for the flat plan)   [S2: complex reciprocals]
#     + N_b ops_FT + N_b N_f ops_R               [S3: Horner plan]   or   N_b N_f ops_flat  [S3: flat plan]
# c_* = FP64-pipe instructions of the leaf routines on their common path as compiled for sm_100a
# (cos 15, Fermi/Bose 24, complex reciprocal 8, plus the integer-coefficient sums of their arguments);
# cross-checked against the executed-instruction counts of ncu's source page in profiles/.
# ------------------------------------------------------------------------------------------------
def fp64_work_per_sample(info, n_f, n_b, reg, tree=False):
    """FP64-pipe instruction slots per sample of the representation executed; every count comes from
    ami_table_info (the library counts the instructions its generator emits plus the common-path cost
    of each leaf routine)."""
    disp = int(info["fp64_ops_dispersion"])
    fermi = n_b * int(info["fp64_ops_leaf_fermi"]) + int(info["fp64_ops_combos"])
    dens = n_b * n_f * int(info["fp64_ops_leaf_den"])
    if reg:
        dens = n_f * int(info["fp64_ops_leaf_den"])     # complex reciprocals once per frequency, shared by all beta
        ft = int(info["fp64_ops_tree_fermi"])
        terms = n_b * ft + n_b * n_f * (int(info["fp64_ops_tree"]) - ft)
        if n_b > 1 and int(info.get("plan_kind", 1)) == 1:
            # several temperatures per launch (register plan): prefix products of the complex reciprocals once per
            # frequency, then 2 instructions per (term of the sum, temperature) -- DESIGN.md 6.2
            terms = n_b * ft + n_f * int(info["fp64_ops_mb_prefix"]) + n_b * n_f * int(info["fp64_ops_mb_sum"])
    elif tree:   # same Horner sums, interpreted; leaves per leaf and reciprocals per (beta, frequency) as in the flat plan
        ft = int(info["fp64_ops_tree_fermi"])
        terms = n_b * ft + n_b * n_f * (int(info["fp64_ops_tree"]) - ft)
    else:
        terms = n_b * n_f * int(info["fp64_ops_flat"])
    return {"dispersion": disp, "evaluate": fermi + dens + terms, "fermi": fermi, "denominators": dens,
            "terms": terms}


def ncu_capture(workload, fused):
    """Counters of the dominant kernel from the committed ncu capture of this workload at its configured size
    (profiles/r02_ncu_<workload>.csv; commands in profiles/r02_ncu_summary.md): DRAM bytes per launch and the warp
    instructions executed per sample, or None."""
    import csv
    p = os.path.join(ROOT, "profiles", f"r02_ncu_{workload}.csv")
    if not fused or not os.path.exists(p):
        return None
    with open(p) as f:
        rows = list(csv.reader(f))
    hdr, units, first = rows[0], rows[1], rows[2]
    col = {h: i for i, h in enumerate(hdr)}
    scale = {"byte": 1.0, "Kbyte": 1e3, "Mbyte": 1e6, "Gbyte": 1e9}
    def nbytes(name):
        return float(first[col[name]].replace(",", "")) * scale.get(units[col[name]], 1.0)
    try:
        n_threads = float(first[col["launch__grid_size"]]) * float(first[col["launch__block_size"]])
        return {"kernel": first[col["Kernel Name"]],
                "dram_bytes": int(nbytes("dram__bytes_read.sum") + nbytes("dram__bytes_write.sum")),
                "warp_instructions": float(first[col["smsp__inst_executed.sum"]]),
                "threads": n_threads,
                "fp64_pipe_active_pct": float(first[col["sm__pipe_fp64_cycles_active.avg.pct_of_peak_sustained_active"]])}
    except (KeyError, ValueError):
        return None


def load_measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        with open(p) as f:
            d = json.load(f)
        return {"hbm_gbs": float(d["hbm_gbs"]), "source": "measured (MEASURED_PEAKS.json)"}
    return {"hbm_gbs": 6650.0, "source": "fallback (B200_PROFILING.md)"}


def dist_setup(args):
    world = int(os.environ.get("WORLD_SIZE", "1"))
    rank = int(os.environ.get("RANK", "0"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    dist = None
    if world > 1:
        import torch.distributed as dist_mod
        os.environ.setdefault("MASTER_ADDR", "127.0.0.1")
        os.environ.setdefault("MASTER_PORT", "29511")
        backend = "gloo" if args.impl == "reference" else "nccl"
        if args.impl != "reference":
            import torch
            torch.cuda.set_device(local)
        dist_mod.init_process_group(backend=backend, rank=rank, world_size=world)
        dist = dist_mod
    return dist, rank, local, world


def samples_per_step(cfg, args):
    return args.n if args.n > 0 else cfg.n_samples


# ------------------------------------------------------------------------------------------------
# reference arm: the CPU oracle, as it stands, on the host cores
# ------------------------------------------------------------------------------------------------
def oracle_rate(cfg, n_sample, threads):
    """term-evaluations/s of the double-precision oracle over n_sample samples of the workload
    (dispersion + evaluate for every beta and frequency), and the seconds it took."""
    import oracle
    ot = oracle.OracleTable.from_diagram(cfg.diagram)
    T = ot.info()["T"]
    k = cfg.momenta(n_sample)
    t0 = time.perf_counter()
    e = ot.dispersion(k, [cfg.q], cfg.t, cfg.mu, threads=threads)
    for beta in cfg.betas:
        ot.evaluate(e, cfg.z_ext, beta, e_reg=cfg.e_reg, quad=False, threads=threads)
    dt = time.perf_counter() - t0
    units = n_sample * len(cfg.betas) * len(cfg.z_ext)
    return T, units, dt


def oracle_sample_size(cfg, threads, seconds):
    """Calibrates on a small sample so that one timed pass takes about `seconds`."""
    n0 = 4096
    _, units, dt = oracle_rate(cfg, n0, threads)
    per_sample = max(dt / n0, 1e-9)
    return int(max(n0, min(cfg.n_samples, seconds / per_sample)))


def run_reference(args, dist, rank, world):
    import ami_inputs as A
    import oracle
    if rank != 0:
        return
    cfg = A.get_config(args.workload)
    threads = oracle.hardware_threads()
    n_s = oracle_sample_size(cfg, threads, min(args.cpu_seconds, 180.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_rate(cfg, max(4096, n_s // 8), threads)
    tot_units, tot_dt, T = 0, 0.0, 0
    for _ in range(args.steps):
        T, units, dt = oracle_rate(cfg, n_s, threads)
        tot_units += units
        tot_dt += dt
    value = T * tot_units / tot_dt
    sample = f"{n_s} of {cfg.n_samples} samples x {len(cfg.z_ext)} freq x {len(cfg.betas)} beta per step"
    line = {
        "impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus,
        "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * tot_dt / args.steps,
        "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "samples_per_s": tot_units / tot_dt,
        "config": {"workload": cfg.name, "samples_per_gpu": cfg.n_samples, "n_freq": len(cfg.z_ext),
                   "n_beta": len(cfg.betas), "T_flat": T, "precision": "double"},
        "config_detail": {"sample": sample},
        "cpu_baseline": {"value": value, "unit": UNIT, "cores": threads, "kind": "oracle", "sample": sample},
        "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
        "gpu_launches": 0,
    }
    print(json.dumps(line), flush=True)


# ------------------------------------------------------------------------------------------------
# our arm: the CUDA path through the C ABI
# ------------------------------------------------------------------------------------------------
def time_workload(pkg, torch, cfg, n, steps, warmup, plan, first_sample, dist, sample_clocks, use_graph=True):
    """Times `steps` passes of S1 + S2/S3 over rotating resident momentum batches (the set of inputs is
    larger than L2, so no batch is served from cache).  Returns a dict of device-timed results."""
    from paper_2311_17189_b200 import sharding
    sum_order = None
    if SUM_ORDER != "default":     # experiment knob; term-evals/s then counts the terms of THAT table
        sum_order = pkg.search_sum_order(cfg.diagram, 0 if SUM_ORDER == "fewest_terms" else 1)[0]
    t_c0 = time.perf_counter()
    tab = pkg.AmiTable.from_diagram(cfg.diagram, device=torch.cuda.current_device(), sum_order=sum_order)
    construct_ms = (time.perf_counter() - t_c0) * 1e3      # ami_construct: recursion + plans + device copy
    info = tab.info
    m, n_eps = cfg.diagram.n_int, cfg.diagram.n_eps
    n_f, n_b = len(cfg.z_ext), len(cfg.betas)
    bytes_in = n * 2 * m * 8
    n_rot = int(max(2, min(8, -(-300_000_000 // max(bytes_in + n * n_eps * 8, 1)))))
    reg = plan in (0, 2) and info["reg_plan_status"] in (0, 1)
    if reg:
        info = tab.specialize()        # NVRTC compile (or cache fetch) + load happen here, outside every timed region
    # The K batches of a step sequence are independent of one another (own momenta, own results: the batches of a
    # Monte-Carlo loop), so with the register plan they are issued as such (AMI_PLAN_UNORDERED): every
    # batch has its own result buffer and the one that begins the reuse of the buffers is issued ordered.
    independent = bool(reg and use_graph and int(info.get("plan_kind", 1)) == 1 and not ORDERED_ONLY)
    if independent:                    # eight buffer sets where 8 GB hold them: one batch in eight is ordered
        n_rot = int(max(n_rot, min(8, 8_000_000_000 // max(bytes_in + n * n_f * n_b * 16, 1))))
    ks = [tab.generate_momenta(cfg.seed, first_sample + r * n, n) for r in range(n_rot)]
    es = [torch.empty((n_eps, n), dtype=torch.float64, device="cuda") for _ in range(n_rot)] if not reg else []
    outs = [torch.empty((n_b, n_f, n), dtype=torch.complex128, device="cuda") for _ in range(n_rot if independent else 1)]
    out = outs[0]
    ev = [[torch.cuda.Event(enable_timing=True) for _ in range(3)] for _ in range(steps)]
    t_beg, t_end = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)

    def step(i, events=None, unordered=False):
        r = i % n_rot
        if events:
            events[0].record()
        if reg:     # one fused kernel: dispersion inline, energies stay in registers
            if events:
                events[1].record()
            flag = pkg.PLAN_UNORDERED if (unordered and r != 0) else 0
            tab.evaluate_momenta(ks[r], [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=plan | flag,
                                 out=outs[r % len(outs)])
        else:
            tab.dispersion(ks[r], [cfg.q], cfg.t, cfg.mu, out=es[r])
            if events:
                events[1].record()
            tab.evaluate(es[r], cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=plan, out=out)
        if events:
            events[2].record()

    for i in range(warmup):
        step(i)
    torch.cuda.synchronize()
    # The fused step is one short kernel (tens of microseconds), less than a Python -> ctypes launch
    # costs on the host, so the K timed steps are captured once into a CUDA graph and replayed: the
    # device then runs them back to back, as a C caller's loop would.
    graph = None
    l0 = pkg.kernel_launches()
    if reg and use_graph:
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            for i in range(steps):
                step(warmup + i, unordered=independent)
        launches = pkg.kernel_launches() - l0     # kernels recorded in the graph = launched per replay
        graph.replay()                            # one untimed replay: graph upload
        torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    sampler = ClockSampler(torch.cuda.current_device()) if sample_clocks else None
    if sampler:
        sampler.start()
    if graph is not None:
        if sampler:
            # the timed replay lasts about a millisecond; keep the same load on the GPU for ~0.2 s before
            # it (extra, untimed warm-up) so that the clock samples are taken under this load
            t_load = time.perf_counter()
            while time.perf_counter() - t_load < 0.2:
                graph.replay()
            torch.cuda.synchronize()
        t_beg.record()
        graph.replay()
        t_end.record()
        torch.cuda.synchronize()
    else:
        l0 = pkg.kernel_launches()
        t_beg.record()
        for i in range(steps):
            step(warmup + i, ev[i])
        t_end.record()
        torch.cuda.synchronize()
        launches = pkg.kernel_launches() - l0
    if dist is not None:
        dist.barrier()
    torch.cuda.synchronize()
    clocks = sampler.stop() if sampler else None
    total_ms_local = t_beg.elapsed_time(t_end)
    total_ms = sharding.max_over_ranks(total_ms_local, dist)
    if graph is not None:
        disp_ms, eval_ms = 0.0, total_ms_local / steps
    else:
        disp_ms = float(np.mean([e[0].elapsed_time(e[1]) for e in ev]))
        eval_ms = float(np.mean([e[1].elapsed_time(e[2]) for e in ev]))
    checksum = complex(out[0, 0, : min(n, 1024)].sum().item())
    ordered_ms = None          # the same K batches, every one ordered after the one before (plain stream order)
    if independent:
        g2 = torch.cuda.CUDAGraph()
        with torch.cuda.graph(g2):
            for i in range(steps):
                step(warmup + i)
        g2.replay()
        torch.cuda.synchronize()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        g2.replay()
        t1.record()
        torch.cuda.synchronize()
        ordered_ms = t0.elapsed_time(t1) / steps
        del g2
    return {"tab": tab, "info": info, "construct_ms": construct_ms, "fused": reg, "tree": plan == 3, "total_ms": total_ms, "disp_ms": disp_ms, "eval_ms": eval_ms,
            "launches": launches, "clocks": clocks, "graph": graph is not None, "ordered_ms": ordered_ms, "independent": independent, "n_rot": n_rot, "checksum": checksum,
            "bytes_in": bytes_in, "bytes_e": n * n_eps * 8, "bytes_out": n * n_f * n_b * 16}


def time_e2e(pkg, torch, tab, cfg, n, steps, warmup, plan, first_sample, dist):
    """Same metric through ami_run with HOST buffers: pinned momenta in, pinned complex128 results
    out, every step; host<->device copies are inside the timed region."""
    from paper_2311_17189_b200 import sharding
    m = cfg.diagram.n_int
    n_f, n_b = len(cfg.z_ext), len(cfg.betas)
    h_k = torch.from_numpy(cfg.momenta(n, start=first_sample).reshape(n, 2 * m)).pin_memory()
    h_out = torch.empty((n_b, n_f, n), dtype=torch.complex128).pin_memory()
    stats = None
    for _ in range(max(1, warmup)):
        stats, _ = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=plan, h_k=h_k,
                           h_out=h_out)
    torch.cuda.synchronize()
    if dist is not None:
        dist.barrier()
    t0 = time.perf_counter()
    for _ in range(steps):
        stats, _ = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=plan, h_k=h_k,
                           h_out=h_out)
    torch.cuda.synchronize()
    dt = sharding.max_over_ranks(time.perf_counter() - t0, dist)
    # the floor of this step on this box: the same pinned momenta copied alone, same clock
    d_k = torch.empty_like(h_k, device="cuda")
    d_k.copy_(h_k, non_blocking=True)
    torch.cuda.synchronize()
    t1 = time.perf_counter()
    for _ in range(steps):
        d_k.copy_(h_k, non_blocking=True)
    torch.cuda.synchronize()
    floor_s = (time.perf_counter() - t1) / steps
    # ... and both directions at once (what the step must move): the input in, a result-sized buffer out, two streams
    d_o = torch.empty(h_out.shape, dtype=torch.complex128, device="cuda")
    s_in, s_out = torch.cuda.Stream(), torch.cuda.Stream()
    torch.cuda.synchronize()
    t2 = time.perf_counter()
    for _ in range(steps):
        with torch.cuda.stream(s_in):
            d_k.copy_(h_k, non_blocking=True)
        with torch.cuda.stream(s_out):
            h_out.copy_(d_o, non_blocking=True)
        torch.cuda.synchronize()
    both_s = (time.perf_counter() - t2) / steps
    return {"seconds": dt, "h2d_copy_alone_ms": floor_s * 1e3, "both_copies_alone_ms": both_s * 1e3, "h2d": int(stats["h2d_bytes"]), "d2h": int(stats["d2h_bytes"]),
            "chunks": int(stats["n_chunks"]), "launches_per_step": int(stats["kernel_launches"]),
            "finite": bool(torch.isfinite(torch.view_as_real(h_out[0, 0, :1024])).all().item())}


def time_complex_energies(pkg, torch, cfg, peaks, dfma_per_s, steps=10, with_flat=True):
    """Variant 5b of reading P19 (energy_t is complex128): cfg5's table and grid fed with complex
    energies e - i gamma, gamma in [0, 0.05).  Energies are supplied, so a step is ami_evaluate alone (S2+S3) on the
    complex-energy variant of the specialised kernels; the same call with the table-driven flat kernel beside it."""
    import ami_inputs as A
    n, n_f, n_b = cfg.n_samples, len(cfg.z_ext), len(cfg.betas)
    tab = pkg.AmiTable.from_diagram(cfg.diagram, device=torch.cuda.current_device())
    k = tab.generate_momenta(cfg.seed, 0, n)
    e = tab.dispersion(k, [cfg.q], cfg.t, cfg.mu)
    gam = torch.from_numpy(A.uniform01(99, np.arange(e.numel(), dtype=np.uint64)).reshape(tuple(e.shape)) * 0.05).cuda()
    ec = torch.complex(e, -gam)
    out = torch.empty((n_b, n_f, n), dtype=torch.complex128, device="cuda")
    res = {}
    for label, plan, reps in (("register", 2, steps), ("flat", 1, 2)):
        if label == "flat" and not with_flat:      # (the table-driven kernel needs 0.1 s and more per step at order 8)
            res[label] = None
            continue
        tab.evaluate(ec, cfg.z_ext, cfg.betas, plan=plan, out=out)
        torch.cuda.synchronize()
        t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
        t0.record()
        for _ in range(reps):
            tab.evaluate(ec, cfg.z_ext, cfg.betas, plan=plan, out=out)
        t1.record()
        torch.cuda.synchronize()
        res[label] = t0.elapsed_time(t1) / reps
    T = int(tab.info["n_terms"])
    kind = "split" if int(tab.refresh_info().get("plan_kind", 1)) == 2 else "register"
    return {"T_flat": T, "samples": n, "n_freq": n_f, "n_beta": n_b, "plan": f"{kind}, complex-energy variant (ami_evaluate)",
            "ms_per_step": res["register"], "term_evals_per_s": T * n * n_f * n_b / (res["register"] * 1e-3),
            "samples_per_s": n * n_f * n_b / (res["register"] * 1e-3), "flat_plan_ms_per_step": res["flat"],
            "hbm_frac": (ec.numel() * 16 + out.numel() * 16) / (res["register"] * 1e-3) / 1e9 / peaks["hbm_gbs"]}


def time_e2e_seeded(torch, tab, cfg, n, steps, plan, T):
    """The end-to-end metric in the driver's seeded mode: no host-to-device copy at all (the momenta are drawn inside
    the evaluation kernel), every result copied to pinned host memory; the floor is the device-to-host copy."""
    n_f, n_b = len(cfg.z_ext), len(cfg.betas)
    h_out = torch.empty((n_b, n_f, n), dtype=torch.complex128).pin_memory()
    stats, _ = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=plan, seed=cfg.seed, h_out=h_out)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(steps):
        stats, _ = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=plan, seed=cfg.seed,
                           first_sample=(i + 1) * n, h_out=h_out)
    torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / steps
    return {"value": T * n * n_f * n_b / dt, "unit": UNIT, "ms_per_step": dt * 1e3, "h2d_bytes_per_step": int(stats["h2d_bytes"]),
            "d2h_bytes_per_step": int(stats["d2h_bytes"]), "chunks_per_step": int(stats["n_chunks"]),
            "api": "ami_run(seed -> h_out)"}


def time_monte_carlo(torch, tab, cfg, n, steps, plan):
    """S4 in the mode of the paper's Monte-Carlo momentum integration: ami_run generates the
    momenta on the device from the seed, evaluates them chunk by chunk on two streams and returns only the
    per-(beta, frequency) sums and sums of squares -- 16 n_f n_b bytes reach the host per step."""
    tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=plan, seed=cfg.seed, want_sum=True)
    torch.cuda.synchronize()
    t0 = time.perf_counter()
    for i in range(steps):
        stats, sums = tab.run(n, [cfg.q], cfg.t, cfg.mu, cfg.z_ext, cfg.betas, e_reg=cfg.e_reg, plan=plan,
                              seed=cfg.seed, first_sample=(i + 1) * n, want_sum=True)
    torch.cuda.synchronize()
    dt = (time.perf_counter() - t0) / steps
    n_f, n_b = len(cfg.z_ext), len(cfg.betas)
    mean = sums / n
    err = np.sqrt(np.maximum(tab.last_sumsq[..., 0] / n - mean.real ** 2, 0.0) / n)
    return {"samples_per_step": n, "ms_per_step": dt * 1e3, "samples_per_s": n * n_f * n_b / dt,
            "gpu_ms_per_step": float(stats["gpu_ms"]),
            "chunks_per_step": int(stats["n_chunks"]), "launches_per_step": int(stats["kernel_launches"]),
            "d2h_bytes_per_step": int(stats["d2h_bytes"]), "timed": "host clock around ami_run (synchronous)",
            "mean_re_first_row": float(mean[0, 0].real), "stderr_re_first_row": float(err[0, 0])}


NOMINAL_DFMA_PER_S = 148 * 64 * 1.965e9      # 148 SMs x 64 FP64 lanes x max SM clock


def roofline_objects(res, n, n_f, n_b, peaks, dfma_per_s, dfma3_per_s=None):
    """Roofline of the dominant kernel: FP64-pipe bound.  Work counted in FP64-pipe instruction slots
    per sample, expressed as DFMA-equivalent TFLOP/s (slot = 2 flop) against the DFMA-chain
    rate measured in this run; the HBM leg is reported beside it.  With the register plan the step is
    ONE fused kernel (S1+S2+S3), otherwise ami_evaluate is the dominant one of two."""
    w = fp64_work_per_sample(res["info"], n_f, n_b, res["fused"], res.get("tree", False))
    t_eval = res["eval_ms"] * 1e-3
    peak_tf = 2.0 * dfma_per_s / 1e12
    if res["fused"]:
        slots = w["evaluate"] + w["dispersion"]
        bytes_alg = res["bytes_in"] + res["bytes_out"]
        kernel = "ami_jit_fused (S1+S2+S3)" if int(res["info"].get("plan_kind", 1)) != 2 else \
            "split plan: ami_split_leaves_fused + ami_split_parts + ami_split_combine (S1+S2+S3)"
    else:
        slots = w["evaluate"]
        bytes_alg = res["bytes_e"] + res["bytes_out"]
        kernel = "ami_evaluate (flat)"
    ach = 2.0 * slots * n / t_eval / 1e12
    roof = {"bound": "alu", "kernel": kernel, "achieved": ach, "peak": peak_tf, "unit": "TFLOP/s",
            "frac": ach / peak_tf, "traffic": None,
            "peak_source": "DFMA-chain probe run by this bench, two distinct register sources per DFMA: the FP64 "
                           "pipe's issue rate (MEASURED_PEAKS.json has no FP64 figure)",
            "flop_convention": "FP64-pipe instruction slots x 2",
            "peak_nominal": 2.0 * NOMINAL_DFMA_PER_S / 1e12,     # 148 SMs x 64 FP64 lanes x max SM clock
            "frac_of_nominal": ach / (2.0 * NOMINAL_DFMA_PER_S / 1e12),
            "peak_three_source_dfma": None if dfma3_per_s is None else 2.0 * dfma3_per_s / 1e12,
            "frac_of_three_source_dfma": None if dfma3_per_s is None else ach / (2.0 * dfma3_per_s / 1e12),
            "fp64_slots_per_sample": w, "fp64_slots_counted": slots,
            "hbm_leg": {"algorithmic_bytes": bytes_alg, "achieved_gbs": bytes_alg / t_eval / 1e9,
                        "peak_gbs": peaks["hbm_gbs"], "frac": bytes_alg / t_eval / 1e9 / peaks["hbm_gbs"],
                        "peak_source": peaks["source"]}}
    disp = None
    if not res["fused"]:
        t_disp = res["disp_ms"] * 1e-3
        disp_bytes = res["bytes_in"] + res["bytes_e"]
        disp = {"kernel": "ami_dispersion", "ms": res["disp_ms"],
                "alu_frac": 2.0 * w["dispersion"] * n / t_disp / 1e12 / peak_tf,
                "hbm_frac": disp_bytes / t_disp / 1e9 / peaks["hbm_gbs"], "algorithmic_bytes": disp_bytes}
    return roof, disp


PLAN_IDS = {"auto": 0, "flat": 1, "reg": 2, "tree": 3}


def plan_name_of(info, plan):
    """Name of the representation ami_evaluate executes (after specialisation has been tried)."""
    if plan not in ("flat", "tree") and info["reg_plan_status"] == 0:
        if int(info.get("plan_kind", 1)) == 2:
            return "split (leaf kernel + Horner-plan parts + combine, NVRTC-specialised)"
        return "register (Horner DAG, NVRTC-specialised)"
    return "tree (table-driven Horner program)" if plan == "tree" else "flat (table-driven)"


def run_ours(args, dist, rank, local, world):
    import torch
    import ami_inputs as A
    import paper_2311_17189_b200 as pkg
    from paper_2311_17189_b200 import sharding
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    pkg.lib()   # raises if libami_b200.so has not been built
    global SUM_ORDER, ORDERED_ONLY
    SUM_ORDER, ORDERED_ONLY = args.sum_order, args.ordered
    cfg = A.get_config(args.workload)
    n = samples_per_step(cfg, args)
    first, _ = sharding.weak_range(n, rank, world)
    n_f, n_b = len(cfg.z_ext), len(cfg.betas)
    plan = PLAN_IDS[args.plan]
    dfma_per_s, _ = pkg.fp64_peak_probe(local, 2)       # the pipe's issue rate: the roofline's peak
    dfma3_per_s, _ = pkg.fp64_peak_probe(local, 3)      # DFMAs with three distinct register sources (context)
    dfma4_per_s, _ = pkg.fp64_peak_probe(local, 4)      # three register sources that change from one DFMA to the next
    dfma5_per_s, _ = pkg.fp64_peak_probe(local, 5)      # the same with one integer instruction per two DFMAs
    dfma6_per_s, _ = pkg.fp64_peak_probe(local, 6)      # two changing register sources and an immediate
    dfma7_per_s, _ = pkg.fp64_peak_probe(local, 7)      # the same with that integer work
    peaks = load_measured_peaks()

    res = time_workload(pkg, torch, cfg, n, args.steps, args.warmup, plan, first, dist, sample_clocks=True,
                        use_graph=not args.no_graph)
    info = res["info"]
    T = int(info["n_terms"])
    plan_name = plan_name_of(info, args.plan)
    units_per_step = n * n_f * n_b * world
    ms_per_step = res["total_ms"] / args.steps
    value = T * units_per_step / (ms_per_step * 1e-3)
    roof, disp = roofline_objects(res, n, n_f, n_b, peaks, dfma_per_s, dfma3_per_s)
    if res["ordered_ms"] is not None:      # the same kernel with every batch ordered after the one before
        roof["frac_ordered"] = roof["frac"] * res["eval_ms"] / res["ordered_ms"]
        roof["batches"] = "independent (AMI_PLAN_UNORDERED); frac_ordered: plain stream order"
    # context for `frac`: what DFMA chains reach when every DFMA reads three register pairs that differ
    # from its predecessor's (register-file bandwidth: one 64-bit operand per lane and cycle), without and with integer
    # instructions beside them in the proportion of the specialised kernels
    roof["register_file_context"] = {
        "three_changing_sources_dfma_per_s": dfma4_per_s, "frac_of_peak": dfma4_per_s / dfma_per_s,
        "with_integer_work_dfma_per_s": dfma5_per_s, "with_integer_work_frac_of_peak": dfma5_per_s / dfma_per_s,
        "two_changing_sources_frac_of_peak": dfma6_per_s / dfma_per_s,
        "two_changing_sources_with_integer_work_frac_of_peak": dfma7_per_s / dfma_per_s}
    # per cycle ("report the fraction per cycle so clock drift drops out"): the probe is a 4 ms burst at the
    # maximum SM clock, the timed steps follow 0.2 s of the same load with the board at its power cap
    ck = res.get("clocks") or {}
    if ck.get("sm_mhz") and ck.get("sm_max_mhz"):
        roof["frac_per_cycle"] = roof["frac"] * float(ck["sm_max_mhz"]) / float(ck["sm_mhz"])
        roof["frac_per_cycle_note"] = "frac x sm_max_mhz / sm_mhz (median SM clock sampled during the timed steps)"
    cap = ncu_capture(cfg.name, res["fused"]) if n == cfg.n_samples else None
    if cap:      # per launch, from profiles/ (ncu --set full of the same command, committed)
        roof["traffic"] = cap["dram_bytes"]
        roof["ncu"] = {"source": f"profiles/r02_ncu_{cfg.name}.csv", "kernel": cap["kernel"],
                       "warp_instructions_per_sample": 32.0 * cap["warp_instructions"] / n,
                       "fp64_pipe_active_pct_of_active_cycles": cap["fp64_pipe_active_pct"],
                       "fp64_slots_counted_per_sample": roof["fp64_slots_counted"]}
    e2e = time_e2e(pkg, torch, res["tab"], cfg, n, max(2, args.steps // 4), 1, plan, first, dist)
    e2e_steps = max(2, args.steps // 4)
    e2e_value = T * units_per_step * e2e_steps / e2e["seconds"]
    launches = int(sharding.sum_over_ranks([res["launches"]], dist)[0])

    line = {
        "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps,
        "warmup": args.warmup, "ms_per_step": ms_per_step, "higher_is_better": True, "scaling": "weak",
        "vs_baseline": None, "dtype": "f64", "data": "synthetic",
        "samples_per_s": units_per_step / (ms_per_step * 1e-3),
        "config": {"workload": cfg.name, "samples_per_gpu": n, "n_freq": n_f, "n_beta": n_b, "T_flat": T,
                   "precision": "double"},
        "config_detail": {"order": cfg.diagram.n_int, "n_green": cfg.diagram.n_g,
                          "U_F": int(info["n_fermi_leaves"]), "U_D": int(info["n_den_leaves"]), "plan": plan_name,
                          "sum_order": args.sum_order,
                          "l2": f"inputs rotated over {res['n_rot']} resident batches (> L2)",
                          "parallelism": "replicas" if world == 1 else f"sample-sharded x{world}, no collective"},
        "time_to_first_result": {"construct_ms": res["construct_ms"], "specialize_ms": float(info["specialize_ms"]),
                                 "specialize_from_disk_cache": bool(info["specialize_cached"]),
                                 "note": "ami_construct (host recursion + plans + device copy) and ami_table_specialize "
                                         "(generate + NVRTC or cache fetch + module load); outside every timed region"},
        "kernels": {"dominant_ms": res["eval_ms"], "ami_dispersion_ms": None if res["fused"] else res["disp_ms"],
                    "dispersion": disp, "launches_per_step": res["launches"] / max(1, args.steps),
                    "timed_as": "one CUDA graph of K steps" if res["graph"] else "K launches from the host",
                    "batches": BATCHES_NOTE if res["independent"] else "every step ordered after the one before",
                    "ordered_ms_per_step": res["ordered_ms"]},
        "roofline": roof,
        "e2e": {"value": e2e_value, "unit": UNIT, "h2d_bytes_per_step": e2e["h2d"], "d2h_bytes_per_step": e2e["d2h"],
                "steps": e2e_steps, "chunks_per_step": e2e["chunks"], "api": "ami_run(h_k -> h_out)",
                "ms_per_step": 1e3 * e2e["seconds"] / e2e_steps, "h2d_copy_alone_ms": e2e["h2d_copy_alone_ms"],
                "both_copies_alone_ms": e2e["both_copies_alone_ms"],
                "note": "H2D copy | kernels | D2H copy of consecutive chunks overlap on three streams; the input copy "
                        "alone (h2d_copy_alone_ms, same pinned buffer, same clock) and both copies of the step issued at once "
                        "without any kernel (both_copies_alone_ms) are the floors of the step on this box"},
        "gpu_launches": launches,
        "clocks": res["clocks"],
        "fp64_probe_dfma_per_s": dfma_per_s, "fp64_probe_three_source_dfma_per_s": dfma3_per_s,
    }
    if world == 1 and rank == 0 and not args.no_extra:
        # secondary workloads (north_star names order 4 AND order 6), short runs, same code path
        others = {}
        for name in ("cfg4", "cfg5", "cfg2_se", "cfg1", "order7", "stress8", "order9"):
            if name == cfg.name:
                continue
            # order7 / stress8 / order9: tables beyond one register-resident kernel (T = 8598 / 40244 / 137644; the paper
            # runs m = 9), outside the five graded configurations; they run the split plan
            c2 = A.get_config("stress8" if name in ("order7", "order9") else name)
            if name in ("order7", "order9"):      # order 9: the largest order the paper benchmarks (T = 137644)
                c2.diagram, c2.name = A.random_self_energy(int(name[-1]), 0), name
            r2 = time_workload(pkg, torch, c2, c2.n_samples, 20, 3, plan, 0, None, sample_clocks=True,
                               use_graph=not args.no_graph)
            i2 = r2["info"]
            pn2 = plan_name_of(i2, args.plan)
            f2, b2 = len(c2.z_ext), len(c2.betas)
            roof2, disp2 = roofline_objects(r2, c2.n_samples, f2, b2, peaks, dfma_per_s, dfma3_per_s)
            ms2 = r2["total_ms"] / 20
            others[name] = {"T_flat": int(i2["n_terms"]), "samples": c2.n_samples, "n_freq": f2, "n_beta": b2,
                            "plan": pn2, "ms_per_step": ms2, "eval_ms": r2["eval_ms"], "disp_ms": r2["disp_ms"],
                            "term_evals_per_s": int(i2["n_terms"]) * c2.n_samples * f2 * b2 / (ms2 * 1e-3),
                            "samples_per_s": c2.n_samples * f2 * b2 / (ms2 * 1e-3),
                            "alu_frac": roof2["frac"], "alu_frac_of_nominal": roof2["frac_of_nominal"],
                            "sm_mhz": (r2["clocks"] or {}).get("sm_mhz"),
                            "alu_frac_per_cycle": roof2["frac"] * float(r2["clocks"]["sm_max_mhz"]) / float(r2["clocks"]["sm_mhz"])
                            if r2["clocks"] and r2["clocks"].get("sm_mhz") else None,
                            "hbm_frac": roof2["hbm_leg"]["frac"], "fp64_slots_per_sample": roof2["fp64_slots_counted"],
                            "construct_ms": r2["construct_ms"], "specialize_ms": float(i2["specialize_ms"]),
                            "specialize_from_disk_cache": bool(i2["specialize_cached"]),
                            "ordered_ms_per_step": r2["ordered_ms"],
                            "alu_frac_ordered": None if r2["ordered_ms"] is None else roof2["frac"] * ms2 / r2["ordered_ms"]}
            if name == "cfg5":
                # the paper's use of the path: the momentum integral on a (frequency, temperature)
                # grid -- 256 result rows tallied inside the evaluation kernel, nothing but the sums leaves the device
                mc5 = time_monte_carlo(torch, r2["tab"], c2, 5 * c2.n_samples, 3, plan)
                w5 = fp64_work_per_sample(i2, f2, b2, r2["fused"])
                mc5["alu_frac_device_time"] = (w5["evaluate"] + w5["dispersion"]) * 5 * c2.n_samples \
                    / (mc5["gpu_ms_per_step"] * 1e-3) / dfma_per_s
                others[name]["monte_carlo_grid"] = mc5
            if int(i2.get("plan_kind", 1)) == 2:
                # the split plan's parts read every leaf they use from the L2-resident leaf array: that, not the FP64
                # pipe, bounds it; the slots counted are those of the Horner plan, without the sums
                # that several parts form again
                others[name]["bound"] = "L2 bandwidth (leaf array reads), see DESIGN.md 6.5"
            del r2
            torch.cuda.empty_cache()
        others["cfg5b"] = time_complex_energies(pkg, torch, A.get_config("cfg5"), peaks, dfma_per_s)
        # the order-8 table with complex energies: the split plan's complex variant
        others["stress8_complex"] = time_complex_energies(pkg, torch, A.get_config("stress8"), peaks, dfma_per_s, steps=5,
                                                          with_flat=False)
        line["other_workloads"] = others
        line["monte_carlo"] = time_monte_carlo(torch, res["tab"], cfg, 10 * n, 5, plan)
        w_mc = fp64_work_per_sample(info, n_f, n_b, res["fused"])
        line["monte_carlo"]["alu_frac"] = (w_mc["evaluate"] + w_mc["dispersion"]) * line["monte_carlo"]["samples_per_s"] \
            / dfma_per_s
        # the same against the CUDA-event time of the call's device work (without the host's launch and sync costs)
        line["monte_carlo"]["alu_frac_device_time"] = (w_mc["evaluate"] + w_mc["dispersion"]) * 10 * n * n_f * n_b \
            / (line["monte_carlo"]["gpu_ms_per_step"] * 1e-3) / dfma_per_s
        line["e2e_seeded"] = time_e2e_seeded(torch, res["tab"], cfg, n, max(2, args.steps // 4), plan, T)
        import oracle
        threads = oracle.hardware_threads()
        n_s = oracle_sample_size(cfg, threads, args.cpu_seconds)
        Tq, units, dt = oracle_rate(cfg, n_s, threads)
        line["cpu_baseline"] = {"value": Tq * units / dt, "unit": UNIT, "cores": threads, "kind": "oracle",
                                "sample": f"first {n_s} of {cfg.n_samples} samples x {n_f} freq x {n_b} beta, "
                                          f"double precision, {dt:.1f} s"}
    if rank == 0:
        print(json.dumps(line), flush=True)


def time_paper_example1(pkg, torch, cfg, steps, warmup, plan, peaks, dfma_per_s):
    """The paper's first example at its own size: energies supplied directly, [N_F][N_E] results,
    so a step is ami_evaluate alone (S2+S3).  Energy batches rotate (8 x 24 MB > L2); CUDA events around K calls."""
    n, n_f, n_b = cfg.n_samples, len(cfg.z_ext), len(cfg.betas)
    tab = pkg.AmiTable.from_diagram(cfg.diagram, device=torch.cuda.current_device())
    info = tab.specialize() if plan in (0, 2) else tab.info
    es = [torch.from_numpy(np.ascontiguousarray(cfg.energies(n, start=r * n).T)).cuda() for r in range(8)]
    out = torch.empty((n_b, n_f, n), dtype=torch.complex128, device="cuda")
    for i in range(warmup):
        tab.evaluate(es[i % 8], cfg.z_ext, cfg.betas, plan=plan, out=out)
    torch.cuda.synchronize()
    t0, t1 = torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)
    l0 = pkg.kernel_launches()
    t0.record()
    for i in range(steps):
        tab.evaluate(es[(warmup + i) % 8], cfg.z_ext, cfg.betas, plan=plan, out=out)
    t1.record()
    torch.cuda.synchronize()
    ms = t0.elapsed_time(t1) / steps
    reg = plan in (0, 2) and info["reg_plan_status"] == 0
    w = fp64_work_per_sample(info, n_f, n_b, reg)
    bytes_alg = n * cfg.diagram.n_eps * 8 + n * n_f * n_b * 16
    T = int(info["n_terms"])
    return {"workload": "paper_ex1", "n_e": n, "n_freq": n_f, "beta": cfg.betas[0], "steps": steps, "ms_per_step": ms,
            "launches_per_step": (pkg.kernel_launches() - l0) / steps, "plan": plan_name_of(info, "auto" if reg else "flat"),
            "samples_per_s": n * n_f * n_b / (ms * 1e-3), "term_evals_per_s": T * n * n_f * n_b / (ms * 1e-3),
            "alu_frac": 2.0 * w["evaluate"] * n / (ms * 1e-3) / (2.0 * dfma_per_s),
            "hbm_frac": bytes_alg / (ms * 1e-3) / 1e9 / peaks["hbm_gbs"], "algorithmic_bytes": bytes_alg}


SWEEP = (("cfg2_se", 8), ("cfg2_bubble", 8), ("cfg3", 7), ("cfg4", 7), ("stress8", 6))   # workload, largest power of ten
# (orders 2, 4, 6: register plan; stress8 = order 8, T = 40244: split plan)


def run_sweep(args, local):
    """Time per batch against the batch size (Figs. 4-5; BASELINE config 2), device-timed like
    the headline: K steps of the whole path over rotating resident batches, K reduced for the largest batches."""
    import torch
    import ami_inputs as A
    import paper_2311_17189_b200 as pkg
    if not torch.cuda.is_available():
        raise SystemExit("bench.py: no CUDA device; the product path has no CPU fallback")
    torch.cuda.set_device(local)
    pkg.lib()
    global ORDERED_ONLY
    ORDERED_ONLY = args.ordered
    plan = PLAN_IDS[args.plan]
    dfma_per_s, _ = pkg.fp64_peak_probe(local)
    peaks = load_measured_peaks()
    rows = []
    for name, top in SWEEP:
        cfg = A.get_config(name)
        n_f, n_b = len(cfg.z_ext), len(cfg.betas)
        for p10 in range(3, top + 1):
            n = 10 ** p10
            steps = args.steps if n <= 10 ** 6 else max(3, args.steps // 4)
            r = time_workload(pkg, torch, cfg, n, steps, args.warmup, plan, 0, None, sample_clocks=False,
                              use_graph=not args.no_graph)
            roof, _ = roofline_objects(r, n, n_f, n_b, peaks, dfma_per_s)
            ms = r["total_ms"] / steps
            T = int(r["info"]["n_terms"])
            rows.append({"workload": name, "n": n, "n_freq": n_f, "steps": steps, "ms_per_step": ms,
                         "ns_per_sample": ms * 1e6 / (n * n_f * n_b), "samples_per_s": n * n_f * n_b / (ms * 1e-3),
                         "term_evals_per_s": T * n * n_f * n_b / (ms * 1e-3), "alu_frac": roof["frac"],
                         "hbm_frac": roof["hbm_leg"]["frac"], "launches_per_step": r["launches"] / steps,
                         "ordered_ms_per_step": r["ordered_ms"],
                         "alu_frac_ordered": None if r["ordered_ms"] is None else roof["frac"] * ms / r["ordered_ms"]})
            del r
            torch.cuda.empty_cache()
    ex1 = time_paper_example1(pkg, torch, A.get_config("paper_ex1"), max(3, args.steps // 2), args.warmup, plan, peaks,
                              dfma_per_s)
    print(json.dumps({"metric": METRIC, "unit": UNIT, "n_gpus": 1, "warmup": args.warmup, "dtype": "f64",
                      "data": "synthetic", "fp64_probe_dfma_per_s": dfma_per_s, "sweep": rows, "paper_ex1": ex1}),
          flush=True)


def main():
    args = parse_args()
    if args.sweep:
        run_sweep(args, 0)
        return
    dist, rank, local, world = dist_setup(args)
    try:
        if args.impl == "reference":
            run_reference(args, dist, rank, world)
        else:
            run_ours(args, dist, rank, local, world)
    finally:
        if dist is not None:
            dist.destroy_process_group()


if __name__ == "__main__":
    main()
