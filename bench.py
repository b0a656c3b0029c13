#!/usr/bin/env python
"""bench.py -- one JSON line: Y-drop GCUPS and kept alignments/s on 1 B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one batch: sfe_pack (target, query + reverse
complement) -> sfe_ydrop_batch (binning, persistent queue, systolic Y-drop DP with traceback,
CIGAR emission) -> sfe_resolve, on device-resident inputs (`value`), and the same through
sfe_extend_host with pinned HOST buffers (`e2e`).  Default workload = BASELINE.json configs[1]
(C2, divergent cross-species regime, 25,000 anchors); --workload c4 is the kernel
microbenchmark (configs[3]).  The path does not shard (BASELINE.json: one GPU, no collectives):
--gpus N runs N independent replicas ("replicas only"), value = sum over ranks.

--impl reference times the CPU oracle (oracle/) on a bounded sample of the same workload.
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

SCRATCH_GB = {"c1": 2, "c2": 16, "c4": 24, "c3": 32, "c3s": 24, "c5s": 32, "c5": 48}   # traceback arena (chunks are recycled)
# dram__bytes_read.sum + dram__bytes_write.sum of ONE ydrop_kernel<traceback> launch, from an `ncu --set full` capture of the
# default run (profiles/r1_04_final_round1.md, "full C2 launch"): 0.768 GB read + 15.376 GB written.  Algorithmic bytes of
# the same launch = the traceback records, `roofline.detail.tb_bytes_per_step` (15.8 GB): no wasted re-reads.
NCU_TRAFFIC_BYTES = {("c2", "cigar", 0, "auto"): 16_144_609_424}
DEFAULT_WINDOW = {"c3": 16384, "c3s": 16384, "c5s": 1024, "c5": 1024}   # Algorithm 3's K for the dense-anchor workloads; others: one batch


def make_workload(name):
    from paper_2606_06811_b200 import workloads as W
    if name == "c1":
        return W.config1(), "BASELINE.json configs[0]: tiny high-identity pair, 256 anchors"
    if name == "c2":
        return W.config2(), "BASELINE.json configs[1]: divergent cross-species regime, 2 Mbp, 25,000 anchors"
    if name == "c4":
        return W.config4(), "BASELINE.json configs[3]: 65,536 independent pairs, log-normal lengths"
    if name == "c3":
        return W.config3(), "BASELINE.json configs[2]: high-identity primate-like regime, 10 Mbp, 50,000 dense anchors"
    if name == "c5":
        return W.config5(), "BASELINE.json configs[4]: chromosome-scale pair, 100 Mbp, 1,000,000 anchors"
    if name == "c3s":
        return W.config3(t_len=1_000_000, n_anchors=5_000), "configs[2] scaled 1/10: 1 Mbp, 5,000 anchors (prefix-scale run)"
    if name == "c5s":
        return W.config5(t_len=10_000_000, n_anchors=100_000), "configs[4] scaled 1/10: 10 Mbp, 100,000 anchors"
    raise SystemExit(f"unknown workload {name}")


class ClockSampler:
    """nvidia-smi clocks / throttle reasons sampled DURING the timed region."""
    Q = ("clocks.sm,clocks.max.sm,power.draw,clocks_event_reasons.hw_slowdown,clocks_event_reasons.hw_thermal_slowdown,"
         "clocks_event_reasons.sw_thermal_slowdown,clocks_event_reasons.sw_power_cap")

    def __init__(self, index):
        self.f = tempfile.NamedTemporaryFile("w+", suffix=".csv", delete=False)
        try:
            self.p = subprocess.Popen(["nvidia-smi", f"--id={index}", f"--query-gpu={self.Q}", "--format=csv,noheader,nounits",
                                       "-lms", "100"], stdout=self.f, stderr=subprocess.DEVNULL)
        except OSError:
            self.p = None

    def stop(self):
        if self.p is None:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["nvidia-smi unavailable"]}
        self.p.terminate()
        try:
            self.p.wait(timeout=5)
        except Exception:
            self.p.kill()
        self.f.flush(); self.f.seek(0)
        sm, mx, reasons, pw = [], [], set(), []
        for ln in self.f:
            c = [x.strip() for x in ln.split(",")]
            if len(c) < 7:
                continue
            try:
                sm.append(float(c[0])); mx.append(float(c[1])); pw.append(float(c[2]))
            except ValueError:
                continue
            for name, v in zip(("hw_slowdown", "hw_thermal_slowdown", "sw_thermal_slowdown", "sw_power_cap"), c[3:7]):
                if v.lower().startswith("active"):
                    reasons.add(name)
        os.unlink(self.f.name)
        if not sm:
            return {"sm_mhz": None, "sm_max_mhz": None, "reasons": ["no samples"]}
        busy = sorted(sm)[len(sm) // 2:]                      # upper half = samples under load
        return {"sm_mhz": float(np.median(busy)), "sm_max_mhz": float(max(mx)), "power_w_max": float(max(pw)),
                "samples": len(sm), "reasons": sorted(reasons)}


def oracle_sample(w, budget_s):
    """The oracle as it stands, one thread, on a strided sample of the workload's anchors until
    ~budget_s seconds of CPU work are done.  Returns (cells, seconds, n_anchors_done)."""
    from oracle import sfe_oracle as O
    O.lib()
    sc = O.scoring()
    n = len(w.anchors)
    qrc = w.query_rc
    stride = max(1, n // 4096)
    order = [i for s in range(stride) for i in range(s, n, stride)]
    cells = 0; done = 0
    t0 = time.perf_counter()
    for i in order:
        a = w.anchors[i]; p = w.pairs[int(a[2])]
        qlim = (int(p[2]), int(p[3])) if a[3] > 0 else (len(w.query) - int(p[3]), len(w.query) - int(p[2]))
        r, _ = O.extend_anchor(w.target, w.query if a[3] > 0 else qrc, int(a[0]), int(a[1]), sc,
                               t_lim=(int(p[0]), int(p[1])), q_lim=qlim, want_ops=True)
        cells += r.cells; done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    return cells, time.perf_counter() - t0, done


def run_reference(args):
    rank = int(os.environ.get("RANK", "0"))
    if rank != 0:
        return
    w, desc = make_workload(args.workload)
    per_step = max(2.0, min(20.0, 100.0 / max(1, args.steps + args.warmup)))
    for _ in range(args.warmup):
        oracle_sample(w, per_step / 4)
    cells = 0; secs = 0.0; nd = 0
    for _ in range(args.steps):
        c, s, d = oracle_sample(w, per_step)
        cells += c; secs += s; nd += d
    v = cells / secs / 1e9
    sample = f"{nd // max(1, args.steps)} of {len(w.anchors)} anchors per step (strided), two-sided extension with CIGAR, 1 thread"
    print(json.dumps({"impl": "reference", "metric": "ydrop_gcups", "value": v, "unit": "GCUPS", "n_gpus": args.gpus,
                      "steps": args.steps, "warmup": args.warmup, "ms_per_step": 1e3 * secs / max(1, args.steps),
                      "higher_is_better": True, "scaling": "weak", "vs_baseline": None, "dtype": "int32", "data": "synthetic",
                      "config": {"workload": f"{args.workload}: {desc}"},
                      "cpu_baseline": {"value": v, "unit": "GCUPS", "cores": 1, "kind": "oracle", "sample": sample},
                      "e2e": {"value": v, "unit": "GCUPS", "h2d_bytes_per_step": 0, "d2h_bytes_per_step": 0}}))


def aggregate_replicas(ms, cells, world, device):
    """Replicas only: every rank runs the same single-GPU job; the job time is the MAX over ranks of the
    device-timed region, the work is the SUM of the cells the ranks computed.  No data-path collective exists; these two
    reductions of one float64 each are the whole multi-GPU path (tested with gloo, world size 2, in tests/test_replicas.py)."""
    if world <= 1:
        return float(ms), float(cells)
    import torch
    import torch.distributed as dist
    t = torch.tensor([float(ms)], dtype=torch.float64, device=device)
    c = torch.tensor([float(cells)], dtype=torch.float64, device=device)
    dist.all_reduce(t, op=dist.ReduceOp.MAX)
    dist.all_reduce(c, op=dist.ReduceOp.SUM)
    return float(t.item()), float(c.item())


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c2", choices=["c1", "c2", "c4", "c3", "c3s", "c5s", "c5"])
    ap.add_argument("--window", type=int, default=-1, help="Algorithm 3's K (sfe_speculate); 0 = one batch over all anchors; -1 = workload default")
    ap.add_argument("--kernel", default="auto", choices=["auto", "block", "systolic"],
                    help="block: the cooperative-warps kernel (one CTA per half) for every half; auto / systolic: one warp per half")
    ap.add_argument("--cigar-for", default="auto", choices=["auto", "all", "kept"],
                    help="windowed workloads: CIGARs for every extended anchor, or (SFE_CIGAR_KEPT_ONLY) score-only windows + one "
                         "traceback batch over the kept anchors; auto = kept for windowed workloads")
    ap.add_argument("--fidelity", action="store_true",
                    help="R4 fidelity report: one extra pass at prune_lag = 0 (serial-order pruning, block kernel) compared with the timed Lambda = 32 results")
    ap.add_argument("--sweep-k", default="", help="comma-separated K values: one extra timed pass each (PAPER.md:163, Fig. 3)")
    ap.add_argument("--flags", default="cigar", choices=["cigar", "score"])
    ap.add_argument("--cpu-seconds", type=float, default=12.0)
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--limit-anchors", type=int, default=0, help="profiling aid: keep every k-th anchor so that N remain")
    args = ap.parse_args()
    if args.impl == "reference":
        return run_reference(args)

    import torch
    import torch.distributed as dist
    import __graft_entry__ as entry
    from paper_2606_06811_b200 import binding as B, sassinfo

    rank = int(os.environ.get("RANK", "0")); world = int(os.environ.get("WORLD_SIZE", "1"))
    local = int(os.environ.get("LOCAL_RANK", "0"))
    if world > 1:
        dist.init_process_group("nccl", device_id=torch.device("cuda", local))
    torch.cuda.set_device(local)
    dev = torch.device("cuda", local)
    entry.build()

    w, desc = make_workload(args.workload)
    if args.limit_anchors and args.limit_anchors < len(w.anchors):
        w.anchors = w.anchors[:: len(w.anchors) // args.limit_anchors][: args.limit_anchors]
        desc += f" [profiling subset: {len(w.anchors)} anchors]"
    n = len(w.anchors)
    flags = B.WANT_CIGAR if args.flags == "cigar" else B.SCORE_ONLY
    flags |= {"auto": 0, "block": B.BLOCK_KERNEL, "systolic": B.NO_BLOCK_KERNEL}[args.kernel]
    free_b, _ = torch.cuda.mem_get_info(dev)
    scratch = min(SCRATCH_GB[args.workload] << 30, int(free_b * 0.6))
    sfe = B.Sfe(local, scratch)
    sc = B.scoring()

    # device-resident inputs
    t_ascii = torch.from_numpy(w.target_ascii().copy()).to(dev)
    q_ascii = torch.from_numpy(w.query_ascii().copy()).to(dev)
    anchors_np = B.make_anchors(w.anchors); pairs_np = B.make_pairs(w.pairs)
    anchors = B._dev(anchors_np, dev); pairs = B._dev(pairs_np, dev)
    acc = torch.zeros((n + 1) * B.BOX_DT.itemsize, dtype=torch.uint8, device=dev)
    nacc = torch.zeros(1, dtype=torch.int64, device=dev)
    stats = torch.zeros(B.STATS_DT.itemsize, dtype=torch.uint8, device=dev)
    cigar_cap = max(1 << 26 if DEFAULT_WINDOW.get(args.workload, 0) or args.window > 0 else 1 << 20, 96 * n)
    state = {}

    window = DEFAULT_WINDOW.get(args.workload, 0) if args.window < 0 else args.window
    kept_only = window > 0 and args.flags == "cigar" and args.cigar_for in ("auto", "kept")
    if kept_only:
        flags |= B.CIGAR_KEPT_ONLY

    def step(K=None):
        K = window if K is None else K
        nacc.zero_(); stats.zero_()
        tp = sfe.pack(t_ascii, with_rc=False)
        qp = sfe.pack(q_ascii, with_rc=True)
        if K > 0:
            o = sfe.speculate(tp[:2], len(w.target), qp, len(w.query), pairs, len(w.pairs), anchors, n, sc, K, flags, cigar_cap,
                              accepted_dev=acc, n_accepted_dev=nacc, stats_dev=stats)
            state.update(res=o["results"], keep=o["keep"])
        else:
            res, pool, used = sfe.ydrop_batch(tp[:2], len(w.target), qp, len(w.query), pairs, len(w.pairs), anchors, n, sc, flags,
                                              cigar_cap)
            keep = sfe.resolve(anchors, res, n, sc.min_score, acc, n + 1, nacc, stats)
            state.update(res=res, keep=keep)

    def launches_of(info, n_windows, K):
        # pack x3; per Y-drop pass: tickets x3, ydrop, select_wide, ydrop_wide, join, scan, emit (+ select_overflow on re-runs);
        # one batch: block_min + resolve; windows: prepare x3, scan + commit per window, finish
        return 3 + 9 * info["launches"] + (info["launches"] - max(1, n_windows)) + ((3 + 2 * n_windows + 1) if K > 0 else 2)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(max(3, args.warmup)):
        step()
    barrier()
    info0 = sfe.last_batch_info()
    st = stats.cpu().numpy().view(B.STATS_DT)[0]
    cells_step = int(st["cells_total"]); kept_step = int(st["n_kept"]); covered_step = int(st["n_covered"])
    cells_cov = int(st["cells_covered"]); ext_step = int(st["n_extended"]); below_step = int(st["n_below"]); windows_step = int(st["n_windows"])

    sampler = ClockSampler(local)
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    kernel_us = 0.0; launches = 0
    barrier()
    e0.record()
    for _ in range(args.steps):
        step()
        inf = sfe.last_batch_info()
        kernel_us += inf["ydrop_kernel_us"]
        launches += launches_of(inf, windows_step, window)
    e1.record()
    barrier()
    ms = e0.elapsed_time(e1)
    clocks = sampler.stop()
    ms, tot_cells = aggregate_replicas(ms, cells_step * args.steps, world, dev)
    gcups = tot_cells / (ms * 1e-3) / 1e9

    # e2e: host buffers through the C ABI, H2D/D2H inside the timed region
    e2e = None
    if not args.no_e2e:
        t_host = torch.from_numpy(w.target_ascii().copy()).pin_memory().numpy()
        q_host = torch.from_numpy(w.query_ascii().copy()).pin_memory().numpy()
        for _ in range(2):
            ho = sfe.extend_host(t_host, q_host, pairs_np, anchors_np, sc, flags, cigar_cap, window)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            ho = sfe.extend_host(t_host, q_host, pairs_np, anchors_np, sc, flags, cigar_cap, window)
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        h2d = len(t_host) + len(q_host) + anchors_np.nbytes + pairs_np.nbytes
        d2h = n * B.RESULT_DT.itemsize + n + 4 * int(ho["cigar_used"]) + B.STATS_DT.itemsize + 8
        e2e_cells = int(ho["stats"]["cells_total"]) * args.steps * world
        e2e = {"value": e2e_cells / dt / 1e9, "unit": "GCUPS", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": 1e3 * dt / args.steps, "kept_per_s": int(ho["stats"]["n_kept"]) * args.steps / dt}

    # f4: batch-size sweep (Fig. 3): one timed pass per K, same inputs
    sweep = []
    for K in [int(x) for x in args.sweep_k.split(",") if x.strip()]:
        step(K); torch.cuda.synchronize(dev)
        k0 = torch.cuda.Event(enable_timing=True); k1 = torch.cuda.Event(enable_timing=True)
        k0.record(); step(K); k1.record(); torch.cuda.synchronize(dev)
        s2 = stats.cpu().numpy().view(B.STATS_DT)[0]; kms = k0.elapsed_time(k1)
        sweep.append({"k": K, "ms": kms, "gcups": float(s2["cells_total"]) / (kms * 1e-3) / 1e9, "windows": int(s2["n_windows"]),
                      "extended": int(s2["n_extended"]), "kept": int(s2["n_kept"]),
                      "waste_ext": 1.0 - (int(s2["n_kept"]) + int(s2["n_below"])) / max(1, int(s2["n_extended"])),
                      "waste_cells": float(s2["cells_covered"]) / max(1.0, float(s2["cells_total"])),
                      "kept_per_s": int(s2["n_kept"]) / (kms * 1e-3)})

    # R4 fidelity: how often does the row-lagged threshold (Lambda = 32) change a result of Lambda = 0?
    fidelity = None
    if args.fidelity and window == 0:
        step(); torch.cuda.synchronize(dev)
        r32 = B.results_to_numpy(state["res"], n); k32 = state["keep"].cpu().numpy()[:n]
        sc0 = B.scoring(prune_lag=0)
        f0 = torch.cuda.Event(enable_timing=True); f1 = torch.cuda.Event(enable_timing=True)
        tp = sfe.pack(t_ascii, with_rc=False); qp = sfe.pack(q_ascii, with_rc=True)
        nacc.zero_(); stats.zero_()
        f0.record()
        res0, pool0, used0 = sfe.ydrop_batch(tp[:2], len(w.target), qp, len(w.query), pairs, len(w.pairs), anchors, n, sc0,
                                             B.WANT_CIGAR | B.BLOCK_KERNEL, cigar_cap)
        keep0 = sfe.resolve(anchors, res0, n, sc0.min_score, acc, n + 1, nacc, stats)
        f1.record(); torch.cuda.synchronize(dev)
        r0 = B.results_to_numpy(res0, n); k0 = keep0.cpu().numpy()[:n]
        box = lambda r: np.stack([r["tstart"], r["tend"], r["qstart"], r["qend"]], 1)
        fidelity = {"anchors": n, "ms_lag0_block_kernel": f0.elapsed_time(f1),
                    "score_differs": int((r0["score"] != r32["score"]).sum()), "box_differs": int((box(r0) != box(r32)).any(1).sum()),
                    "n_ops_differs": int((r0["n_ops"] != r32["n_ops"]).sum()), "keep_differs": int((k0 != k32).sum()),
                    "kept_lag0": int((k0 == 1).sum()), "kept_lag32": int((k32 == 1).sum()),
                    "cells_lag32_over_lag0": float(r32["cells"].sum()) / max(1.0, float(r0["cells"].sum()))}

    if rank != 0:
        if world > 1:
            dist.destroy_process_group()
        return

    # roofline of the dominant kernel (integer issue)
    tb_loop = bool(flags & B.WANT_CIGAR) and not kept_only       # kept-only windows run the score-only loop
    hl = sassinfo.hot_loop(traceback=tb_loop)
    r_alu, _ = sfe.probe_int_issue(1, 20000); r_dpx, _ = sfe.probe_int_issue(2, 20000)
    r_fma, _ = sfe.probe_int_issue(3, 20000); r_mix, _ = sfe.probe_int_issue(0, 20000)
    f_mhz = clocks.get("sm_mhz") or 1965.0
    fmax = clocks.get("sm_max_mhz") or 1965.0
    n_sm = torch.cuda.get_device_properties(dev).multi_processor_count
    # probe rates are per max-clock cycle.  ALU and FMA are separate 16-lane pipes (2 cycles per warp
    # instruction per SM sub-partition); DPX (VIADDMNMX/VIMNMX3) issues to the ALU pipe at the plain ALU rate.
    # Cycles per cell per SM = the slowest of the ALU pipe, the FMA pipe (IMAD) and instruction issue as a whole.
    r_alu_pipe = min(r_alu, r_dpx)
    cyc_per_cell = max(hl["alu"] / r_alu_pipe, hl["fma"] / r_fma, hl["per_cell"] / max(r_mix, r_alu, r_dpx))
    peak_gcups = n_sm * fmax * 1e6 / cyc_per_cell / 1e9
    k_gcups = cells_step * args.steps / (kernel_us * 1e-6) / 1e9 if kernel_us > 0 else None
    roof = {"bound": "alu", "achieved": k_gcups, "peak": peak_gcups, "unit": "GCUPS", "frac": (k_gcups / peak_gcups) if k_gcups else None,
            "traffic": NCU_TRAFFIC_BYTES.get((args.workload, args.flags, window, args.kernel)) if not args.limit_anchors else None, "kernel": "ydrop_kernel<%s>" % ("traceback" if tb_loop else "score-only"),
            "kernel_share_of_step": kernel_us * 1e-3 / ms,
            "detail": {"instr_per_cell_sass": hl["per_cell"], "alu_per_cell": hl["alu"], "dpx_per_cell": hl["dpx"], "fma_per_cell": hl["fma"],
                       "lsu_per_cell": hl["lsu"], "R_alu": r_alu, "R_dpx": r_dpx, "R_imad": r_fma, "R_mixed": r_mix,
                       "R_unit": "lane-instr/clk/SM at sm_max_mhz", "n_sm": n_sm, "f_mhz_used": fmax,
                       "f_mhz_sampled": f_mhz, "peak_source": "measured by sfe_probe_int_issue in this run",
                       "tb_bytes_per_step": info0["tb_bytes"], "tb_gbs": info0["tb_bytes"] * args.steps / (kernel_us * 1e-6) / 1e9 if kernel_us else None,
                       "lane_efficiency": cells_step / (32.0 * info0["steps"]) if info0["steps"] and window == 0 else None}}

    oc, osec, od = oracle_sample(w, args.cpu_seconds)
    cpu = {"value": oc / osec / 1e9, "unit": "GCUPS", "cores": 1, "kind": "oracle",
           "sample": f"{od} of {n} anchors (strided), two-sided extension with CIGAR, {osec:.1f} s"}

    line = {"metric": "ydrop_gcups", "value": gcups, "unit": "GCUPS", "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": f"{args.workload}: {desc}", "anchors": n, "flags": args.flags, "window_k": window, "kernel": args.kernel, "cigar_for": "kept" if kept_only else ("all" if args.flags == "cigar" else "none"),
                       "l2": "inputs+traceback per step exceed L2 (126 MB)",
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "scoring": "HOXD70/400/30/ydrop 9400/lag 32/tau 3000"},
            "kept_alignments_per_s": kept_step * args.steps * world / (ms * 1e-3),
            "kept": kept_step, "cells_per_step": cells_step,
            "extended": ext_step, "windows": windows_step,
            "speculation_waste": {"ext": 1.0 - (kept_step + below_step) / ext_step if ext_step else None,
                                  "cells": cells_cov / cells_step if cells_step else None},
            "gpu_launches": launches, "clocks": clocks, "e2e": e2e, "roofline": roof, "cpu_baseline": cpu,
            "batch_info": info0, "k_sweep": sweep or None, "lag0_fidelity": fidelity}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
