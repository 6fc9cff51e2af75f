#!/usr/bin/env python
"""bench.py -- throughput of the hot path on B200 (contract: see README / DESIGN.md "Measurement").

Default workload = BASELINE.json configs[4] (C5): synthetic 360-species / 2172-reaction mechanism,
2^18 fp64 states, CONP, sparse Jacobian in CSR value order.  One "step" = one pass of the whole hot
path (steps a1-a11: concentrations, thermo, rate constants, falloff, rates of progress, per-reaction
partials, species rows, T/E rows, store) over the batch = one pyjac_jacobian_sparse call.

    python bench.py [--gpus N] [--steps K] [--warmup W] [--config 5] [--impl reference] [--peaks]

Prints ONE JSON line.  `--impl reference` times the CPU oracle (oracle/) on the host cores instead.  `--gpus N` with
N > 1 outside torchrun spawns N ranks itself (one process per GPU).  `--peaks` prints the machine peaks measured by the
library's own microbenchmarks (pyjac_measure_peak: DFMA/s, HBM write / read / copy, L2 read, shared-memory load).
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

import mechgen as mg  # noqa: E402
from mechgen.mechanism import CONFIGS, pack_phi  # noqa: E402

METRIC = "sparse Jacobian evals/s (states/s) and achieved HBM GB/s vs roofline"
UNIT = "states/s"


def measured_peaks():
    p = os.path.join(ROOT, "MEASURED_PEAKS.json")
    if os.path.exists(p):
        d = json.load(open(p))
        return float(d["hbm_gbs"]), "measured (MEASURED_PEAKS.json hbm_gbs, copy read+write)"
    return 6650.0, "fallback (B200_PROFILING.md 6.65 TB/s)"


TRAFFIC_CSV = os.path.join("profiles", "r02_traffic.csv")


def ncu_traffic(config, kernel):
    """dram bytes (read + write) per launch of the timed kernel from the committed ncu summary profiles/r02_traffic.csv
    (columns: config,kernel,n_states,dram_bytes_per_launch,capture), scaled to this run's states by the caller.  It is
    a constant from an earlier `ncu --set full` capture, NOT measured by this run: `traffic_source` says which."""
    p = os.path.join(ROOT, TRAFFIC_CSV)
    if os.path.exists(p):
        for line in open(p):
            f = line.strip().split(",")
            if len(f) >= 5 and f[0] == "c%d" % config and f[1] == kernel:
                return {"n_states": int(f[2]), "dram_bytes": float(f[3]), "source": "%s, ncu --set full capture %s" % (TRAFFIC_CSV, f[4])}
    return None


def fp64_model_ops(mech, what):
    """A-priori DFMA-equivalent count per state from the mechanism alone (SURVEY.md section 8d "Algorithmic FP64 ops";
    DESIGN.md section 8): not from the kernel's SASS.  exp = 24, log = 28, divide = 10 DFMA slots.
    what: "source" | "sparse" | "dense" (the Jacobian count includes everything the source terms need)."""
    EXP, LOG, DIV = 24, 28, 10
    ns, nr = int(mech["n_species"]), int(mech["n_reactions"])
    ty = np.asarray(mech["type"]); rev = np.asarray(mech["reversible"]).astype(bool)
    jac = what != "source"
    ops = (15 + (4 if jac else 0)) * ns + 2 * LOG
    n_re = np.diff(mech["reac_ptr"]); n_pr = np.diff(mech["prod_ptr"])
    n_eff = np.diff(mech["eff_ptr"])
    for i in range(nr):
        o = 2 + EXP + 5 + 4                                   # k_f, mass action, omega
        if rev[i]:
            o += 5 + EXP
        t = int(ty[i])
        if t in (2, 3, 4):
            o += EXP + 2 * DIV
        if t == 3:
            o += 4 * EXP + 2 * LOG + EXP
        if t == 4:
            o += 2 * EXP + 2 * LOG + EXP
        if t == 5:
            o += 15
        if t == 6:
            o += 50
        if t in (1, 2, 3, 4):
            o += 2 * int(n_eff[i])
        if jac:
            rows = int(len(set(mech["reac_species"][mech["reac_ptr"][i]:mech["reac_ptr"][i + 1]]) |
                           set(mech["prod_species"][mech["prod_ptr"][i]:mech["prod_ptr"][i + 1]])))
            cols = int(n_re[i]) + (int(n_pr[i]) if rev[i] else 0) + (int(n_eff[i]) if t in (1, 2, 3, 4) else 0)
            o += 19 + rows * (cols + 2) + 2 * (cols + 2)
        ops += o
    return int(ops)


class ClockSampler:
    """Samples nvidia-smi SM clocks and throttle reasons during the timed region."""
    Q = ("index,clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.active,"
         "clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, gpu_index):
        self.idx = gpu_index
        self.samples = []
        self.stop = False
        self.th = threading.Thread(target=self._run, daemon=True)

    def _run(self):
        while not self.stop:
            try:
                out = subprocess.run(["nvidia-smi", "-i", str(self.idx), "--query-gpu=" + self.Q,
                                      "--format=csv,noheader,nounits"], capture_output=True, text=True, timeout=5).stdout
                f = [x.strip() for x in out.strip().split(",")]
                if len(f) >= 9:
                    self.samples.append(f)
            except Exception:
                pass
            time.sleep(0.1)

    def __enter__(self):
        self.th.start()
        return self

    def __exit__(self, *a):
        self.stop = True
        self.th.join(timeout=6)

    def summary(self):
        if not self.samples:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["unsampled"]}
        sm = sorted(float(s[1]) for s in self.samples)
        reasons = set()
        for s in self.samples:
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), s[5:9]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        return {"sm_mhz": sm[len(sm) // 2], "sm_max_mhz": float(self.samples[0][2]), "reasons": sorted(reasons),
                "samples": len(sm), "power_w_max": max(float(s[3]) for s in self.samples)}


def oracle_rate(c, mode, what, target_s=12.0):
    """Times the oracle as it stands on a bounded sample; returns (states/s, threads, n_sample)."""
    from oracle import Oracle
    o = Oracle(mg.config_mechanism(c))
    n = 2 * o.threads
    while True:
        st = mg.config_states(c, n)
        phi, par = o.pack(st, mode)
        t0 = time.perf_counter()
        if what == "sparse":
            o.jacobian_sparse(mode, mg.CSR, phi, par)
        elif what == "dense":
            o.jacobian_dense(mode, phi, par)
        else:
            o.source(mode, phi, par)
        dt = time.perf_counter() - t0
        if dt >= 0.25 * target_s or n >= (1 << 16):
            return n / dt, o.threads, n, dt
        n = int(min(1 << 16, max(2 * n, n * 0.6 * target_s / max(dt, 1e-3))))


def run_reference(args, rank, world):
    if rank != 0:
        return
    c = args.config
    cfg = CONFIGS[c]
    what = "dense" if c in (1, 4) else "sparse"
    vals, info = [], None
    for i in range(args.warmup + args.steps):
        r, threads, n, dt = oracle_rate(c, cfg["mode"], what, target_s=max(2.0, 40.0 / (args.warmup + args.steps)))
        if i >= args.warmup:
            vals.append((n, dt))
        info = (threads, n)
    tot_n = sum(v[0] for v in vals); tot_t = sum(v[1] for v in vals)
    value = tot_n / tot_t
    line = {"impl": "reference", "metric": METRIC, "value": value, "unit": UNIT, "n_gpus": args.gpus, "steps": args.steps,
            "warmup": args.warmup, "ms_per_step": 1e3 * tot_t / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "f64", "data": "synthetic",
            "config": workload_config(c, what, None, None),
            "cpu_baseline": {"value": value, "unit": UNIT, "cores": info[0], "kind": "oracle",
                             "sample": "%d states of the workload per step (oracle/, OpenMP over states)" % info[1]},
            "e2e": {"value": value, "unit": UNIT, "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0},
            "gpu_launches": 0}
    print(json.dumps(line))


def workload_config(c, what, tile, S, N=None, mode=None):
    cfg = CONFIGS[c]
    N = cfg["n_states"] if N is None else N
    mode = cfg["mode"] if mode is None else mode
    return {"workload": "C%d: synthetic %d-species / %d-reaction mechanism, %d fp64 states, %s, %s Jacobian%s" % (
        c, cfg["ns"], cfg["nr"], N, "CONP" if mode == mg.CONP else "CONV", what,
        " (CSR value order)" if what == "sparse" else " (row-major)"),
        "n_states_per_gpu": N, "layout_tile": tile, "states_per_cta": S,
        "l2": "inputs+outputs larger than L2 (no flush needed)" if N * 8 * 1000 > 126e6 else "l2_flush_between_steps"}


def parse_args(argv=None):
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=10)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--config", type=int, default=5)
    ap.add_argument("--impl", default="b200")
    ap.add_argument("--states", type=int, default=None, help="override states per GPU (sweeps)")
    ap.add_argument("--tile", type=int, default=None, help="override layout tile (default: states per CTA)")
    ap.add_argument("--mode", choices=["conp", "conv"], default=None, help="override the config's mode (sweeps)")
    ap.add_argument("--pair-kernel", action="store_true", help="force the pair-of-states Jacobian kernel (PYJAC_PAIR_KERNEL)")
    ap.add_argument("--peaks", action="store_true", help="print the machine peaks measured by pyjac_measure_peak and exit")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--no-cpu", action="store_true")
    ap.add_argument("--no-fd", action="store_true", help="skip the finite-difference comparison")
    return ap.parse_args(argv)


PEAK_NAMES = ("dfma_per_s", "hbm_write_Bps", "hbm_read_Bps", "hbm_copy_Bps", "l2_read_Bps", "lds_Bps")


def measure_peaks(pj, device, kinds=range(6), reps=5, tries=3):
    """best of `tries` x (`reps` back-to-back launches, CUDA-event timed inside the library)"""
    return {PEAK_NAMES[k]: max(pj.pyjac_measure_peak(k, device, reps) for _ in range(tries)) for k in kinds}


def run_peaks(args):
    import torch
    import paper_1809_01029_b200 as pj
    assert torch.cuda.is_available(), "bench.py --peaks needs a CUDA device"
    with ClockSampler(0) as clk:
        peaks = measure_peaks(pj, 0)
    sm = torch.cuda.get_device_properties(0).multi_processor_count
    mhz = clk.summary().get("sm_mhz") or 0.0
    line = {"peaks": peaks, "n_sm": sm, "clocks": clk.summary(),
            "dfma_per_clk_per_sm": peaks["dfma_per_s"] / (sm * mhz * 1e6) if mhz else None,
            "how": "pyjac_measure_peak (csrc/pyjac_peaks.cu): DFMA = 8 independent chains x 2048 threads/SM; HBM = 4 GiB streams, "
                   "16-byte accesses; L2 = every CTA sweeps one 32 MiB window (ld.global.cg); LDS = conflict-free 16-byte loads; "
                   "best of 3 x 5 launches, CUDA events"}
    print(json.dumps(line))


def spawn_ranks(n, worker, args, port=None):
    """`python bench.py --gpus N` outside torchrun: N ranks, one process per GPU (torch.multiprocessing.spawn), the same
    environment torchrun would give them.  worker(args) runs in every rank and reads RANK / LOCAL_RANK / WORLD_SIZE."""
    import torch.multiprocessing as mp
    port = port or 29500 + os.getpid() % 2000
    mp.spawn(_spawned, nprocs=n, args=(n, port, worker, args), join=True)


def _spawned(rank, n, port, worker, args):
    os.environ.update({"RANK": str(rank), "LOCAL_RANK": str(rank), "WORLD_SIZE": str(n), "MASTER_ADDR": "127.0.0.1",
                       "MASTER_PORT": str(port)})
    worker(args)


def main(argv=None):
    args = parse_args(argv)
    if args.peaks:
        return run_peaks(args)
    if args.gpus > 1 and "WORLD_SIZE" not in os.environ:
        return spawn_ranks(args.gpus, rank_main, args)
    return rank_main(args)


def rank_main(args):
    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if args.impl == "reference":
        return run_reference(args, rank, world)

    import torch
    import torch.distributed as dist
    import paper_1809_01029_b200 as pj
    assert torch.cuda.is_available(), "bench.py needs a CUDA device (no CPU fallback)"
    torch.cuda.set_device(local)
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    c = args.config
    cfg = CONFIGS[c]
    mode = cfg["mode"] if args.mode is None else (mg.CONP if args.mode == "conp" else mg.CONV)
    what = "dense" if c in (1, 4) else "sparse"
    w_id = pj.WHAT_SPARSE if what == "sparse" else pj.WHAT_DENSE
    N = args.states or cfg["n_states"]
    mech = mg.config_mechanism(c)
    M = pj.Mechanism(mech, local, pj.PYJAC_PAIR_KERNEL if args.pair_kernel else 0)
    plan = pj.pyjac_plan_info(M.h)
    # the library's own launch policy (pyjac_launch_info): states per CTA for this batch; the benchmark layout is
    # tile = states per CTA of a large batch (a CTA's outputs are then one contiguous range)
    tile = args.tile or pj.pyjac_launch_info(M.h, w_id, N, 0)[0]
    S, threads, smem = pj.pyjac_launch_info(M.h, w_id, N, tile)
    ld = (N + tile - 1) // tile * tile
    n_e = M.nnz if what == "sparse" else M.nvar * M.nvar
    # weak scaling: every rank owns its own N states (independent problems, no collective on the data path)
    from paper_1809_01029_b200.sharding import weak_scaling_offset
    states = mg.config_states(c, N, start=weak_scaling_offset(N, rank))
    phi_h, par_h = pack_phi(states, mode, ld, tile)
    d_phi = torch.from_numpy(phi_h).cuda(); d_par = torch.from_numpy(par_h).cuda()
    d_out = torch.empty(n_e * ld, dtype=torch.float64, device="cuda")
    stream = torch.cuda.current_stream()
    flush = torch.empty(256 << 20, dtype=torch.uint8, device="cuda") if N * n_e * 8 < 512e6 else None

    def step():
        if what == "sparse":
            pj.pyjac_jacobian_sparse(M.h, mode, pj.PYJAC_CSR, N, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), d_out.data_ptr(), stream.cuda_stream)
        else:
            pj.pyjac_jacobian_dense(M.h, mode, "C", N, ld, tile, d_phi.data_ptr(), d_par.data_ptr(), d_out.data_ptr(), stream.cuda_stream)

    def barrier():
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize()

    warm = max(3, args.warmup)
    for _ in range(warm):
        step()
    barrier()
    evs = [(torch.cuda.Event(enable_timing=True), torch.cuda.Event(enable_timing=True)) for _ in range(args.steps)]
    with ClockSampler(local) as clk:
        barrier()
        t0 = torch.cuda.Event(enable_timing=True); t1 = torch.cuda.Event(enable_timing=True)
        t0.record(stream)
        for a, b in evs:
            if flush is not None:
                flush.zero_()
            a.record(stream); step(); b.record(stream)
        t1.record(stream)
        barrier()
    kern_ms = [a.elapsed_time(b) for a, b in evs]
    total_ms = sum(kern_ms) if flush is not None else t0.elapsed_time(t1)
    tt = torch.tensor([total_ms], dtype=torch.float64, device="cuda")
    if world > 1:
        dist.all_reduce(tt, op=dist.ReduceOp.MAX)
    total_ms = float(tt.item())
    value = world * N * args.steps / (total_ms * 1e-3)
    kavg_ms = float(np.mean(kern_ms))
    alg_bytes_state = 8 * n_e + 8 * (M.ns + 2)            # read phi+param once, write each output once
    peak, peak_src = measured_peaks()
    achieved = alg_bytes_state * N / (kavg_ms * 1e-3) / 1e9

    def timed(fn, reps, warm_=2):
        for _ in range(warm_):
            fn()
        torch.cuda.synchronize()
        a = torch.cuda.Event(enable_timing=True); b = torch.cuda.Event(enable_timing=True)
        a.record(stream)
        for _ in range(reps):
            fn()
        b.record(stream); torch.cuda.synchronize()
        return a.elapsed_time(b) / reps

    # source terms, timed separately (BASELINE.json configs[4]) in the layout that call prefers: its own states-per-CTA
    # (the source kernel keeps only q_i per reaction on chip, so more states fit a CTA than for the Jacobian)
    tile_s = args.tile or pj.pyjac_launch_info(M.h, pj.WHAT_SOURCE, N, 0)[0]
    ld_s = (N + tile_s - 1) // tile_s * tile_s
    d_phi_s = d_phi if tile_s == tile else torch.from_numpy(pack_phi(states, mode, ld_s, tile_s)[0]).cuda()
    d_par_s = torch.zeros(ld_s, dtype=torch.float64, device="cuda"); d_par_s[:N] = d_par[:N]
    d_src = torch.empty(M.nvar * ld_s, dtype=torch.float64, device="cuda")
    src_ms = timed(lambda: pj.pyjac_source_terms(M.h, mode, N, ld_s, tile_s, d_phi_s.data_ptr(), d_par_s.data_ptr(), d_src.data_ptr(),
                                                 stream.cuda_stream), 5, 3)

    # the paper's comparison (Fig. 12): first-order finite-difference Jacobian in the same output
    # format, same layout, on a bounded sample of the same states (it costs n_var + 1 source evaluations per state)
    fd = None
    if not args.no_fd:
        n_fd = min(N, (2048 + tile - 1) // tile * tile)      # one CTA per state: ~14 waves over the 148 SMs
        ffmt = pj.PYJAC_CSR if what == "sparse" else "C"
        fd_ms = timed(lambda: pj.pyjac_jacobian_fd(M.h, mode, ffmt, 2.0 ** -26, 1e-14, n_fd, ld, tile, d_phi.data_ptr(), d_par.data_ptr(),
                                                   d_out.data_ptr(), stream.cuda_stream), 3, 1)
        fd = {"states": n_fd, "ns_per_state": 1e6 * fd_ms / n_fd, "states_per_s": n_fd / (fd_ms * 1e-3),
              "columns_per_pass": pj.pyjac_launch_info(M.h, 3)[0], "rel_step": 2.0 ** -26, "abs_step": 1e-14,
              "analytical_speedup": (fd_ms / n_fd) / (kavg_ms / N)}

    # machine peaks measured here and now by the library's own microbenchmarks (rank 0 only; after the timed region)
    here = measure_peaks(pj, local, kinds=(0, 1), reps=3, tries=2) if rank == 0 else None

    # e2e: the C-ABI call on HOST buffers, H2D + kernel + D2H inside the timed region (pinned memory).  The pinned
    # buffers are capped per rank (28 GiB / world): with more ranks every rank times a prefix of its states.
    e2e = None
    if not args.no_e2e:
        cap = int((28 << 30) / world)
        n2 = min(N, max(tile, cap // (8 * n_e) // tile * tile))
        ld2 = (n2 + tile - 1) // tile * tile
        phi2, par2 = (phi_h, par_h) if n2 == N else pack_phi({k: (v[:n2] if v.ndim == 1 else v[:, :n2]) for k, v in states.items()}, mode, ld2, tile)
        pinned = True
        try:
            h_out = torch.empty(n_e * ld2, dtype=torch.float64).pin_memory()
            h_phi = torch.from_numpy(phi2).pin_memory(); h_par = torch.from_numpy(par2).pin_memory()
        except Exception:
            pinned = False
            h_out = torch.empty(n_e * ld2, dtype=torch.float64); h_phi = torch.from_numpy(phi2); h_par = torch.from_numpy(par2)
        f = pj.PYJAC_CSR if what == "sparse" else "C"
        e_steps = max(1, min(args.steps, 3))
        pj.pyjac_eval_host(M.h, w_id, mode, f, n2, ld2, tile, h_phi.numpy(), h_par.numpy(), h_out.numpy())     # warm-up: staging buffers
        barrier()
        t_0 = time.perf_counter()
        for _ in range(e_steps):
            pj.pyjac_eval_host(M.h, w_id, mode, f, n2, ld2, tile, h_phi.numpy(), h_par.numpy(), h_out.numpy())
        torch.cuda.synchronize()
        dt = time.perf_counter() - t_0
        tt = torch.tensor([dt], dtype=torch.float64, device="cuda")
        if world > 1:
            dist.all_reduce(tt, op=dist.ReduceOp.MAX)
        e2e = {"value": world * n2 * e_steps / float(tt.item()), "unit": UNIT,
               "h2d_bytes_per_step": int(8 * (M.nvar + 1) * n2), "d2h_bytes_per_step": int(8 * n_e * n2),
               "steps": e_steps, "states_per_gpu": n2, "pinned": pinned,
               "api": "pyjac_eval_host (chunked, double-buffered, host buffers; staging buffers owned by the handle)"}
        del h_out

    if rank == 0:
        cpu = None
        if not args.no_cpu:
            r, threads_cpu, n_s, dt = oracle_rate(c, mode, what)
            cpu = {"value": r, "unit": UNIT, "cores": threads_cpu, "kind": "oracle",
                   "sample": "%d states of the same workload in %.1f s (oracle/, OpenMP over states)" % (n_s, dt)}
        kernel = ("jacobian2_kernel<LS=%d>" % (S // 2)) if args.pair_kernel else ("jacobian_kernel<S=%d,%s>" % (S, "dense" if what == "dense" else "sparse"))
        ns_state = 1e6 * kavg_ms / N
        # two bounds (north_star: "the slower of FP64 ops at peak and bytes at peak bandwidth"):
        #   bytes: algorithmic bytes / the measured HBM peak of MEASURED_PEAKS.json;
        #   fp64:  a-priori DFMA-equivalent model count / the DFMA rate measured here by pyjac_measure_peak
        ops_j = fp64_model_ops(mech, what); ops_s = fp64_model_ops(mech, "source")
        t_hbm = alg_bytes_state / (peak * 1e9) * 1e9
        t_f64 = ops_j / here["dfma_per_s"] * 1e9
        bound = "hbm" if t_hbm >= t_f64 else "fp64"
        traffic = ncu_traffic(c, "pair" if args.pair_kernel else "tile")
        roofline = {"bound": "hbm", "achieved": achieved, "peak": peak, "unit": "GB/s", "frac": achieved / peak,
                    "traffic": None if traffic is None else traffic["dram_bytes"] * N / traffic["n_states"],
                    "traffic_source": None if traffic is None else traffic["source"] + " (a constant scaled to this run's states, not measured by this run)",
                    "peak_source": peak_src, "kernel": kernel, "algorithmic_bytes_per_state": alg_bytes_state,
                    "kernel_ms": kavg_ms, "ns_per_state": ns_state,
                    "binding_bound": bound, "frac_of_binding_bound": max(t_hbm, t_f64) / ns_state,
                    "hbm": {"bound_ns_per_state": t_hbm, "frac": t_hbm / ns_state,
                            "frac_of_write_stream_measured_here": alg_bytes_state * N / (kavg_ms * 1e-3) / here["hbm_write_Bps"]},
                    "fp64": {"model_dfma_per_state": ops_j, "peak_dfma_per_s_measured_here": here["dfma_per_s"],
                             "bound_ns_per_state": t_f64, "frac": t_f64 / ns_state}}
        src_ns = 1e6 * src_ms / N
        line = {"metric": METRIC, "value": value, "unit": UNIT, "n_gpus": world, "steps": args.steps, "warmup": warm,
                "ms_per_step": total_ms / args.steps, "higher_is_better": True, "scaling": "weak", "vs_baseline": None,
                "dtype": "f64", "data": "synthetic",
                "config": dict(workload_config(c, what, tile, S, N, mode),
                               l2="l2_flush_between_steps (256 MB written)" if flush is not None else "inputs+outputs larger than L2 (no flush needed)",
                               layout="tile = %d: %s" % (tile, "state-major values, one state per tile (not the pure SoA north_star names: pure SoA at this size "
                                                         "is 2x slower, profiles/r01_sweeps.md)" if tile == 1 else "chunked state-interleaved order (PAPER.md L106)")),
                "roofline": roofline, "cpu_baseline": cpu, "e2e": e2e, "gpu_launches": args.steps, "clocks": clk.summary(),
                "extra": {"source_terms_states_per_s": N / (src_ms * 1e-3), "source_terms_ms": src_ms, "source_terms_tile": tile_s,
                          "source_terms_fp64": {"model_dfma_per_state": ops_s, "bound_ns_per_state": ops_s / here["dfma_per_s"] * 1e9,
                                                "frac": ops_s / here["dfma_per_s"] * 1e9 / src_ns},
                          "nnz": M.nnz, "smem_bytes_per_cta": smem, "threads_per_cta": threads, "plan": plan,
                          "peaks_measured_here": {"dfma_per_s": here["dfma_per_s"], "hbm_write_gbs": here["hbm_write_Bps"] / 1e9},
                          "fd_jacobian": fd}}
        print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
