#!/usr/bin/env python
"""bench.py -- one JSON line: Y-drop GCUPS and kept alignments/s on 1 B200 (BASELINE.json metric).

A "step" is one pass of the whole hot path over one batch: sfe_pack (target, query + reverse
complement) -> sfe_ydrop_batch (binning, persistent queue, systolic Y-drop DP with traceback,
CIGAR emission) -> sfe_resolve, on device-resident inputs (`value`), and the same through
sfe_extend_host with pinned HOST buffers (`e2e`).  Default workload = BASELINE.json configs[3]
(C4: 65,536 independent pairs, the kernel microbenchmark SURVEY 8(d) names for "headline GCUPS and
roofline fraction"); the same line carries `c5_e2e`: Algorithm 3 end to end (sfe_speculate) on
configs[4] (C5, the chromosome-scale pair; see --c5).  --workload c1|c2|c3|c5|c3s|c5s select the others.
The path does not shard (BASELINE.json: one GPU, no collectives): --gpus N runs N independent
replicas ("replicas only"), value = sum over ranks.

--impl reference times the CPU oracle (oracle/) on a bounded sample of the same workload.
"""
import argparse
import glob
import hashlib
import json
import os
import subprocess
import sys
import tempfile
import time

import numpy as np

ROOT = os.path.dirname(os.path.abspath(__file__))
sys.path.insert(0, ROOT)

SCRATCH_GB = {"c1": 2, "c2": 16, "c4": 24, "c3": 32, "c3s": 24, "c5s": 32, "c5": 96, "filter": 2}   # traceback arena (chunks are recycled)
DEFAULT_WINDOW = {"c3": 16384, "c3s": 16384, "c5s": 1024, "c5": 1024}   # classic Algorithm 3: K for the dense-anchor workloads; others: one batch
LEADER_WINDOW = 262144                                                  # --spec leaders: most extensions per batch
TRAFFIC_FILE = os.path.join(ROOT, "profiles", "ncu_traffic.csv")      # written by hand from `ncu --set full` captures (see ncu_traffic.md)


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
        return W.config5(t_len=10_000_000, n_anchors=100_000), "configs[4] scaled 1/10: 10 Mbp, 100,000 anchors (the prefix-scale run SURVEY 8(d) allows)"
    if name == "filter":
        return W.filter_hits(), ("f3 (PAPER.md:213, 225-227): gapped Y-drop as the FILTER over 1,000,000 raw seed hits on a configs[1]-like pair, "
                                 "95 % of them false; score-only, ydrop 2000, +-1024-base budget per hit, pass = score >= 3000")
    raise SystemExit(f"unknown workload {name}")


def source_hash():
    """sha256 over the CUDA sources and the header: what an ncu capture was taken of (git is not on the GPU box)."""
    h = hashlib.sha256()
    for f in sorted(glob.glob(os.path.join(ROOT, "paper_2606_06811_b200", "csrc", "*.cu*")) + [os.path.join(ROOT, "include", "sfe.h")]):
        h.update(os.path.basename(f).encode()); h.update(open(f, "rb").read())
    return h.hexdigest()[:16]


def ncu_traffic(workload, flags, window, kernel):
    """roofline.traffic = dram__bytes_read.sum + dram__bytes_write.sum of ONE launch of the dominant kernel from an
    `ncu --set full` capture, recorded in profiles/ncu_traffic.csv together with the hash of the sources it was
    taken of.  A capture of other sources, or of another configuration, is not reported: null plus the reason."""
    import csv
    key = f"{workload}/{flags}/{window}/{kernel}"
    try:
        rows = [r for r in csv.DictReader(ln for ln in open(TRAFFIC_FILE) if not ln.startswith("#")) if r.get("key") == key]
    except OSError:
        return None, "no capture recorded (profiles/ncu_traffic.csv missing)"
    if not rows:
        return None, f"no capture for {key}"
    ent = rows[-1]
    if ent.get("source_hash") != source_hash():
        return None, f"capture is of sources {ent.get('source_hash')}, this run is {source_hash()} (stale: re-capture)"
    return int(ent["dram_bytes_read"]) + int(ent["dram_bytes_write"]), ent.get("profile")


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


# ---- CPU legs (the oracle as it stands; SURVEY 8(d) "Timing the oracle beside it") -------------------------------
def _oracle_one(w, qrc, sc, i):
    from oracle import sfe_oracle as O
    a = w.anchors[i]; p = w.pairs[int(a[2])]
    qlim = (int(p[2]), int(p[3])) if a[3] > 0 else (len(w.query) - int(p[3]), len(w.query) - int(p[2]))
    r, _ = O.extend_anchor(w.target, w.query if a[3] > 0 else qrc, int(a[0]), int(a[1]), sc,
                           t_lim=(int(p[0]), int(p[1])), q_lim=qlim, want_ops=True)
    return r.cells


def oracle_scoring(w):
    from oracle import sfe_oracle as O
    return O.scoring(ydrop=2000) if w.name == "filter" else O.scoring()


def strided_order(n):
    stride = max(1, n // 4096)
    return [i for s in range(stride) for i in range(s, n, stride)]


def oracle_sample(w, budget_s, indices=None):
    """The oracle, ONE thread, two-sided extension with CIGAR over a strided sample of the anchors (or `indices`) until
    ~budget_s seconds of CPU work are done.  Returns (cells, seconds, n_anchors_done)."""
    from oracle import sfe_oracle as O
    O.lib()
    sc = oracle_scoring(w)
    qrc = w.query_rc
    order = strided_order(len(w.anchors)) if indices is None else list(indices)
    cells = 0; done = 0
    t0 = time.perf_counter()
    for i in order:
        cells += _oracle_one(w, qrc, sc, i); done += 1
        if time.perf_counter() - t0 > budget_s:
            break
    return cells, time.perf_counter() - t0, done


def oracle_parallel(w, budget_s, indices=None):
    """The same extensions on ALL host cores: a thread pool over anchors (the ctypes call releases the GIL), the analogue
    of the paper's 32-core prototype.  Returns (cells, seconds, n_done, cores)."""
    from concurrent.futures import ThreadPoolExecutor
    from oracle import sfe_oracle as O
    O.lib()
    sc = oracle_scoring(w)
    qrc = w.query_rc
    cores = max(1, os.cpu_count() or 1)
    order = strided_order(len(w.anchors)) if indices is None else list(indices)
    cells = 0; done = 0; pos = 0
    t0 = time.perf_counter()
    with ThreadPoolExecutor(max_workers=cores) as ex:
        while pos < len(order) and time.perf_counter() - t0 < budget_s:
            chunk = order[pos:pos + 4 * cores]; pos += len(chunk)
            for c in ex.map(lambda i: _oracle_one(w, qrc, sc, i), chunk):
                cells += c; done += 1
    return cells, time.perf_counter() - t0, done, cores


def oracle_serial_prefix(w, budget_s):
    """Algorithm 1 as the oracle runs it, one thread, on growing PREFIXES of the anchor list until one
    call takes about budget_s.  Returns dict(anchors, extended, kept, cells, seconds)."""
    from oracle import sfe_oracle as O
    O.lib()
    sc = oracle_scoring(w)
    qrc = w.query_rc
    n = len(w.anchors)
    m = min(n, 16)
    best = None
    while True:
        t0 = time.perf_counter()
        r = O.serial_loop(w.target, w.query, qrc, w.pairs, w.anchors[:m], sc, want_results=False)
        dt = time.perf_counter() - t0
        best = dict(anchors=m, extended=int(r["n_extended"]), kept=int(r["n_kept"]), cells=int(r["cells"]), seconds=dt)
        if m >= n or dt > budget_s / 3:
            return best
        m = min(n, int(m * max(2.0, min(8.0, 0.6 * budget_s / max(dt, 1e-3)))))


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


class Job:
    """One workload resident on the device + the step that runs the hot path over it."""

    def __init__(self, sfe, w, dev, flags, window, cigar_cap):
        import torch
        from paper_2606_06811_b200 import binding as B
        self.B = B; self.sfe = sfe; self.w = w; self.dev = dev; self.flags = flags; self.window = window
        self.n = len(w.anchors)
        self.t_ascii = torch.from_numpy(w.target_ascii().copy()).to(dev)
        self.q_ascii = torch.from_numpy(w.query_ascii().copy()).to(dev)
        self.anchors_np = B.make_anchors(w.anchors); self.pairs_np = B.make_pairs(w.pairs)
        self.anchors = B._dev(self.anchors_np, dev); self.pairs = B._dev(self.pairs_np, dev)
        self.acc = torch.zeros((self.n + 1) * B.BOX_DT.itemsize, dtype=torch.uint8, device=dev)
        self.nacc = torch.zeros(1, dtype=torch.int64, device=dev)
        self.stats = torch.zeros(B.STATS_DT.itemsize, dtype=torch.uint8, device=dev)
        self.cigar_cap = cigar_cap
        self.filter = w.name == "filter"
        self.sc = B.scoring(ydrop=2000) if self.filter else B.scoring()
        self.state = {}

    def step(self, K=None, flags=None):
        B = self.B; w = self.w; sfe = self.sfe
        K = self.window if K is None else K
        flags = self.flags if flags is None else flags
        self.nacc.zero_(); self.stats.zero_()
        tp = sfe.pack(self.t_ascii, with_rc=False)
        qp = sfe.pack(self.q_ascii, with_rc=True)
        self.state.update(tp=tp, qp=qp)
        if self.filter:
            # the filter: one score-only batch; a hit passes iff its gapped score reaches tau.  No containment (nothing is
            # committed at this stage), so no resolve: the statistics below are filled from the results for the report.
            res, _, _ = sfe.ydrop_batch(tp[:2], len(w.target), qp, len(w.query), self.pairs, len(w.pairs), self.anchors, self.n,
                                        self.sc, flags & ~B.WANT_CIGAR, 0)
            self.state.update(res=res, keep=None)
        elif K > 0:
            o = sfe.speculate(tp[:2], len(w.target), qp, len(w.query), self.pairs, len(w.pairs), self.anchors, self.n, self.sc, K, flags,
                              self.cigar_cap, accepted_dev=self.acc, n_accepted_dev=self.nacc, stats_dev=self.stats)
            self.state.update(res=o["results"], keep=o["keep"])
        else:
            res, pool, used = sfe.ydrop_batch(tp[:2], len(w.target), qp, len(w.query), self.pairs, len(w.pairs), self.anchors, self.n,
                                              self.sc, flags, self.cigar_cap)
            keep = sfe.resolve(self.anchors, res, self.n, self.sc.min_score, self.acc, self.n + 1, self.nacc, self.stats)
            self.state.update(res=res, keep=keep)

    def stats_dict(self):
        if self.filter:
            r = self.B.results_to_numpy(self.state["res"], self.n)
            npass = int((r["score"] >= self.sc.min_score).sum())
            return {"n_anchors": self.n, "n_kept": npass, "n_covered": 0, "n_below": self.n - npass, "cells_total": int(r["cells"].sum()),
                    "cells_covered": 0, "n_extended": self.n, "n_windows": 1}
        st = self.stats.cpu().numpy().view(self.B.STATS_DT)[0]
        return {k: int(st[k]) for k in self.B.STATS_DT.names}


def summarize_pass(st, ms):
    ext = st["n_extended"]
    return {"ms": ms, "gcups": st["cells_total"] / (ms * 1e-3) / 1e9, "kept": st["n_kept"], "kept_per_s": st["n_kept"] / (ms * 1e-3),
            "extended": ext, "windows": st["n_windows"], "cells": st["cells_total"],
            "waste_ext": (1.0 - (st["n_kept"] + st["n_below"]) / ext) if ext else None,
            "waste_cells": (st["cells_covered"] / st["cells_total"]) if st["cells_total"] else None}


def main():
    ap = argparse.ArgumentParser()
    ap.add_argument("--gpus", type=int, default=1)
    ap.add_argument("--steps", type=int, default=5)
    ap.add_argument("--warmup", type=int, default=3)
    ap.add_argument("--impl", default="ours", choices=["ours", "reference"])
    ap.add_argument("--workload", default="c4", choices=["c1", "c2", "c4", "c3", "c3s", "c5s", "c5", "filter"])
    ap.add_argument("--window", type=int, default=-1, help="Algorithm 3's K (sfe_speculate); 0 = one batch over all anchors; -1 = workload default")
    ap.add_argument("--kernel", default="auto", choices=["auto", "block", "systolic"],
                    help="block: the cooperative-warps kernel (one CTA per half) for every half; auto / systolic: one warp per half")
    ap.add_argument("--cigar-for", default="auto", choices=["auto", "all", "kept"],
                    help="windowed workloads: CIGARs for every extended anchor, or (SFE_CIGAR_KEPT_ONLY) score-only windows + one "
                         "traceback batch over the kept anchors; auto = kept for windowed workloads")
    ap.add_argument("--fidelity", action="store_true",
                    help="R4 fidelity report: prune_lag = 0 (serial-order pruning, block kernel) against the Lambda = 32 results; "
                         "one-batch workloads in full, windowed ones on a seeded sample of their extended anchors")
    ap.add_argument("--sweep-k", default="", help="comma-separated K values: one extra timed pass each (PAPER.md:163, Fig. 3)")
    ap.add_argument("--spec", default="leaders", choices=["leaders", "classic"],
                    help="windowed workloads: leaders = SFE_SPEC_LEADERS (speculate on predicted leaders, results cached); "
                         "classic = Algorithm 3's 'next K uncovered anchors'")
    ap.add_argument("--flags", default="cigar", choices=["cigar", "score"])
    ap.add_argument("--cpu-seconds", type=float, default=10.0, help="budget of EACH CPU leg (1-core serial loop, all-core extensions)")
    ap.add_argument("--no-e2e", action="store_true")
    ap.add_argument("--c5", default="auto", choices=["auto", "full", "prefix", "off"],
                    help="the c5_e2e key of the default (c4) line: Algorithm 3 end to end on configs[4]; prefix = the 10 Mbp / "
                         "100,000-anchor prefix-scale run SURVEY 8(d) allows; auto = full")
    ap.add_argument("--opt", action="append", default=[], metavar="KEY=VALUE",
                    help="sfe_set_option, e.g. SPEC_SPAN=262144, SPARSE_WARPS=8, ROW_KERNEL_CAP=1048576 (binding.OPT_* names)")
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

    t_gen = time.perf_counter()
    w, desc = make_workload(args.workload)
    t_gen = time.perf_counter() - t_gen
    if args.limit_anchors and args.limit_anchors < len(w.anchors):
        w.anchors = w.anchors[:: len(w.anchors) // args.limit_anchors][: args.limit_anchors]
        desc += f" [profiling subset: {len(w.anchors)} anchors]"
    n = len(w.anchors)
    if args.workload == "filter":
        args.flags = "score"; args.no_e2e = True
    flags = B.WANT_CIGAR if args.flags == "cigar" else B.SCORE_ONLY
    flags |= {"auto": 0, "block": B.BLOCK_KERNEL, "systolic": B.NO_BLOCK_KERNEL}[args.kernel]
    free_b, _ = torch.cuda.mem_get_info(dev)
    scratch = min(SCRATCH_GB[args.workload] << 30, int(free_b * 0.6))
    sfe = B.Sfe(local, scratch)
    opts = {}
    for kv in args.opt:
        k, v = kv.split("=")
        sfe.set_option(getattr(B, "OPT_" + k.upper()), int(v)); opts[k.upper()] = int(v)

    window = DEFAULT_WINDOW.get(args.workload, 0) if args.window < 0 else args.window
    if args.window < 0 and window > 0 and args.spec == "leaders":
        window = LEADER_WINDOW
    # CIGARs for the kept anchors only (score-only speculation + one traceback batch) pays when most extensions are thrown
    # away (classic windows); with predicted leaders nearly every extension is kept or cheap: trace back while extending
    kept_only = window > 0 and args.flags == "cigar" and (args.cigar_for == "kept" or (args.cigar_for == "auto" and args.spec == "classic"))
    if kept_only:
        flags |= B.CIGAR_KEPT_ONLY
    if window > 0 and args.spec == "leaders":
        flags |= B.SPEC_LEADERS
    cigar_cap = max(1 << 26 if window > 0 else 1 << 20, 96 * n)
    job = Job(sfe, w, dev, flags, window, cigar_cap)

    def barrier():
        torch.cuda.synchronize(dev)
        if world > 1:
            dist.barrier()
        torch.cuda.synchronize(dev)

    for _ in range(max(3, args.warmup)):
        job.step()
    barrier()
    info0 = sfe.last_batch_info()
    st0 = job.stats_dict()
    cells_step = st0["cells_total"]; kept_step = st0["n_kept"]

    sampler = ClockSampler(local)
    e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
    kernel_us = 0.0
    barrier()
    launches0 = B.launch_counter()
    e0.record()
    for _ in range(args.steps):
        job.step()
        kernel_us += sfe.last_batch_info()["ydrop_kernel_us"]
    e1.record()
    barrier()
    launches = B.launch_counter() - launches0          # counted at the launch sites (sfe_launch_counter), not derived
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
            ho = sfe.extend_host(t_host, q_host, job.pairs_np, job.anchors_np, job.sc, flags, cigar_cap, window)
        barrier()
        t0 = time.perf_counter()
        for _ in range(args.steps):
            ho = sfe.extend_host(t_host, q_host, job.pairs_np, job.anchors_np, job.sc, flags, cigar_cap, window)
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        h2d = len(t_host) + len(q_host) + job.anchors_np.nbytes + job.pairs_np.nbytes
        d2h = n * B.RESULT_DT.itemsize + n + 4 * int(ho["cigar_used"]) + B.STATS_DT.itemsize + 8
        e2e_cells = int(ho["stats"]["cells_total"]) * args.steps * world
        e2e = {"value": e2e_cells / dt / 1e9, "unit": "GCUPS", "h2d_bytes_per_step": int(h2d), "d2h_bytes_per_step": int(d2h),
               "ms_per_step": 1e3 * dt / args.steps, "kept_per_s": int(ho["stats"]["n_kept"]) * args.steps / dt}
        del t_host, q_host

    # f4: batch-size sweep (Fig. 3): one timed pass per K, same inputs
    sweep = []
    for K in [int(x) for x in args.sweep_k.split(",") if x.strip()]:
        job.step(K); torch.cuda.synchronize(dev)
        k0 = torch.cuda.Event(enable_timing=True); k1 = torch.cuda.Event(enable_timing=True)
        k0.record(); job.step(K); k1.record(); torch.cuda.synchronize(dev)
        d = summarize_pass(job.stats_dict(), k0.elapsed_time(k1)); d["k"] = K
        sweep.append(d)

    # R4 fidelity: how often does the row-lagged threshold (Lambda = 32) change a result of Lambda = 0?
    fidelity = None
    if args.fidelity:
        job.step(); torch.cuda.synchronize(dev)
        r_all = B.results_to_numpy(job.state["res"], n); k_all = job.state["keep"].cpu().numpy()[:n]
        box = lambda r: np.stack([r["tstart"], r["tend"], r["qstart"], r["qend"]], 1)
        sc0 = B.scoring(prune_lag=0)
        tp, qp = job.state["tp"], job.state["qp"]
        f0 = torch.cuda.Event(enable_timing=True); f1 = torch.cuda.Event(enable_timing=True)
        if window == 0:
            job.nacc.zero_(); job.stats.zero_()
            f0.record()
            res0, _, _ = sfe.ydrop_batch(tp[:2], len(w.target), qp, len(w.query), job.pairs, len(w.pairs), job.anchors, n, sc0,
                                         B.WANT_CIGAR | B.BLOCK_KERNEL, cigar_cap)
            keep0 = sfe.resolve(job.anchors, res0, n, sc0.min_score, job.acc, n + 1, job.nacc, job.stats)
            f1.record(); torch.cuda.synchronize(dev)
            r0 = B.results_to_numpy(res0, n); k0 = keep0.cpu().numpy()[:n]; r32 = r_all
            extra = {"anchors": n, "keep_differs": int((k0 != k_all).sum()), "kept_lag0": int((k0 == 1).sum()), "kept_lag32": int((k_all == 1).sum()),
                     "n_ops_differs": int((r0["n_ops"] != r32["n_ops"]).sum())}
        else:
            # windowed workloads: a seeded sample of the anchors the speculative run extended (kept ones first), the same
            # anchors as ONE batch at Lambda = 0 on the block kernel; compared with their Lambda = 32 results of the timed path
            ext = np.nonzero((r_all["status"] & np.uint32(B.ST_SKIPPED)) == 0)[0]
            rng = np.random.default_rng(4)
            kept_i = ext[k_all[ext] == 1]; other = ext[k_all[ext] != 1]
            pick = np.sort(np.concatenate([rng.choice(kept_i, min(len(kept_i), 200), replace=False),
                                           rng.choice(other, min(len(other), 1800), replace=False)]))
            sub = B._dev(job.anchors_np[pick], dev)
            f0.record()
            res0, _, _ = sfe.ydrop_batch(tp[:2], len(w.target), qp, len(w.query), job.pairs, len(w.pairs), sub, len(pick), sc0,
                                         B.SCORE_ONLY | B.BLOCK_KERNEL, 0)
            f1.record(); torch.cuda.synchronize(dev)
            r0 = B.results_to_numpy(res0, len(pick)); r32 = r_all[pick]
            extra = {"anchors": int(len(pick)), "sample": f"{int(len(pick))} of {len(ext)} extended anchors (seeded; {min(len(kept_i), 200)} kept)",
                     "below_tau_flips": int(((r0["score"] >= job.sc.min_score) != (r32["score"] >= job.sc.min_score)).sum())}
        fidelity = {"ms_lag0_block_kernel": f0.elapsed_time(f1), "score_differs": int((r0["score"] != r32["score"]).sum()),
                    "box_differs": int((box(r0) != box(r32)).any(1).sum()),
                    "cells_lag32_over_lag0": float(r32["cells"].sum()) / max(1.0, float(r0["cells"].sum()))}
        fidelity.update(extra)

    # c5_e2e: Algorithm 3 end to end on the chromosome-scale config, in the same line (default run only)
    c5 = None
    if args.workload == "c4" and args.c5 != "off" and not args.limit_anchors:
        del job
        sfe.close(); torch.cuda.empty_cache()
        name5 = "c5s" if args.c5 == "prefix" else "c5"
        tg = time.perf_counter(); w5, desc5 = make_workload(name5); tg = time.perf_counter() - tg
        free_b, _ = torch.cuda.mem_get_info(dev)
        sfe5 = B.Sfe(local, min(SCRATCH_GB[name5] << 30, int(free_b * 0.6)))
        K5 = LEADER_WINDOW if args.spec == "leaders" else DEFAULT_WINDOW[name5]
        f5 = B.WANT_CIGAR | (B.SPEC_LEADERS if args.spec == "leaders" else B.CIGAR_KEPT_ONLY)
        cap5 = max(1 << 26, 96 * len(w5.anchors))
        job5 = Job(sfe5, w5, dev, f5, K5, cap5)
        job5.step(); torch.cuda.synchronize(dev)                       # warm-up pass
        a0 = torch.cuda.Event(enable_timing=True); a1 = torch.cuda.Event(enable_timing=True)
        a0.record(); job5.step(); a1.record(); torch.cuda.synchronize(dev)
        c5 = summarize_pass(job5.stats_dict(), a0.elapsed_time(a1))
        c5.update({"workload": f"{name5}: {desc5}", "anchors": len(w5.anchors), "window_k": K5, "spec": args.spec, "speculate_info": sfe5.last_speculate_info(),
                   "cigar_for": "all extended" if args.spec == "leaders" else "kept", "generation_s": tg,
                   "path": "sfe_pack x2 -> sfe_speculate (phase 1 scan, phase 2 Y-drop windows, phase 3 commit, all on the device) "
                           "-> one traceback batch over the kept anchors; device-resident inputs, CUDA events"})
        t_host = torch.from_numpy(w5.target_ascii().copy()).pin_memory().numpy()
        q_host = torch.from_numpy(w5.query_ascii().copy()).pin_memory().numpy()
        t0 = time.perf_counter()
        ho = sfe5.extend_host(t_host, q_host, job5.pairs_np, job5.anchors_np, job5.sc, f5, cap5, K5)
        torch.cuda.synchronize(dev)
        dt = time.perf_counter() - t0
        c5["host_e2e"] = {"ms": 1e3 * dt, "gcups": int(ho["stats"]["cells_total"]) / dt / 1e9, "kept_per_s": int(ho["stats"]["n_kept"]) / dt,
                          "h2d_bytes": int(len(t_host) + len(q_host) + job5.anchors_np.nbytes + job5.pairs_np.nbytes),
                          "d2h_bytes": int(len(w5.anchors) * (B.RESULT_DT.itemsize + 1) + 4 * int(ho["cigar_used"]))}
        # Algorithm 1 as the oracle runs it, one thread, on a prefix of the same anchor list ("LASTZ-like serial seconds")
        if rank == 0:
            sp = oracle_serial_prefix(w5, args.cpu_seconds)
            sp["gcups"] = sp["cells"] / sp["seconds"] / 1e9
            c5["cpu_serial_alg1"] = sp
        del t_host, q_host, job5
        sfe5.close()
        sfe = B.Sfe(local, 1 << 30)                                    # for the probes below

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
    # SURVEY 8(d)'s literal formula: N_SM x R x f / I with I = ALL SASS instructions per cell, R = the measured mixed issue rate
    peak_issue = n_sm * fmax * 1e6 * max(r_mix, r_alu, r_dpx) / hl["per_cell"] / 1e9
    k_gcups = cells_step * args.steps / (kernel_us * 1e-6) / 1e9 if kernel_us > 0 else None
    traffic, traffic_note = (None, "profiling subset") if args.limit_anchors else ncu_traffic(args.workload, args.flags, window, args.kernel)
    roof = {"bound": "alu", "achieved": k_gcups, "peak": peak_gcups, "unit": "GCUPS", "frac": (k_gcups / peak_gcups) if k_gcups else None,
            "frac_issue": (k_gcups / peak_issue) if k_gcups else None, "peak_issue": peak_issue,
            "traffic": traffic, "traffic_source": traffic_note, "kernel": "ydrop_kernel<%s>" % ("traceback" if tb_loop else "score-only"),
            "kernel_share_of_step": kernel_us * 1e-3 / ms,
            "detail": {"instr_per_cell_sass": hl["per_cell"], "alu_per_cell": hl["alu"], "dpx_per_cell": hl["dpx"], "fma_per_cell": hl["fma"],
                       "lsu_per_cell": hl["lsu"], "R_alu": r_alu, "R_dpx": r_dpx, "R_imad": r_fma, "R_mixed": r_mix,
                       "R_unit": "lane-instr/clk/SM at sm_max_mhz", "n_sm": n_sm, "f_mhz_used": fmax,
                       "f_mhz_sampled": f_mhz, "peak_source": "measured by sfe_probe_int_issue in this run",
                       "frac_is": "pipe-bound reading: the ALU pipe's instructions per cell over its measured rate",
                       "frac_issue_is": "SURVEY 8(d) literal: all SASS instructions per cell over the measured mixed issue rate",
                       "source_hash": source_hash(),
                       "algorithmic_bytes_per_step": 0.5 * cells_step, "tb_bytes_per_step": info0["tb_bytes"],
                       "tb_gbs": info0["tb_bytes"] * args.steps / (kernel_us * 1e-6) / 1e9 if kernel_us else None,
                       "lane_efficiency": cells_step / (32.0 * info0["steps"]) if info0["steps"] and window == 0 else None}}

    # CPU legs: (1) one thread; for a one-batch workload without coverage this IS Algorithm 1's serial work; (2) all cores
    oc, osec, od = oracle_sample(w, args.cpu_seconds)
    pc, psec, pd, cores = oracle_parallel(w, args.cpu_seconds)
    sp = oracle_serial_prefix(w, args.cpu_seconds)
    cpu = {"value": oc / osec / 1e9, "unit": "GCUPS", "cores": 1, "kind": "oracle",
           "sample": f"{od} of {n} anchors (strided), two-sided extension with CIGAR, {osec:.1f} s",
           "parallel": {"value": pc / psec / 1e9, "unit": "GCUPS", "cores": cores, "kind": "oracle",
                        "sample": f"{pd} of {n} anchors (strided; the extensions the GPU computed), thread pool over anchors, {psec:.1f} s"},
           "serial_alg1": {"seconds": sp["seconds"], "anchors": sp["anchors"], "extended": sp["extended"], "kept": sp["kept"], "cells": sp["cells"],
                           "gcups": sp["cells"] / sp["seconds"] / 1e9, "cores": 1,
                           "sample": f"Algorithm 1 on the first {sp['anchors']} of {n} anchors, 1 thread"}}

    line = {"metric": "ydrop_gcups", "value": gcups, "unit": "GCUPS", "n_gpus": world, "steps": args.steps,
            "warmup": max(3, args.warmup), "ms_per_step": ms / args.steps, "higher_is_better": True, "scaling": "weak",
            "vs_baseline": None, "dtype": "int32", "data": "synthetic",
            "config": {"workload": f"{args.workload}: {desc}", "anchors": n, "flags": args.flags, "window_k": window, "kernel": args.kernel, "spec": (args.spec if window > 0 else None), "options": opts or None, "cigar_for": "kept" if kept_only else ("all" if args.flags == "cigar" else "none"),
                       "l2": "inputs+traceback per step exceed L2 (126 MB)", "generation_s": t_gen,
                       "parallelism": "replicas only" if world > 1 else "1 GPU", "scoring": "HOXD70/400/30/ydrop 9400/lag 32/tau 3000"},
            "kept_alignments_per_s": kept_step * args.steps * world / (ms * 1e-3),
            "filter": ({"hits_per_s": n * args.steps * world / (ms * 1e-3), "pass_rate": kept_step / n, "passed": kept_step,
                        "true_hits": w.meta.get("n_true"), "tau": 3000, "ydrop": 2000, "budget_bases": w.meta.get("budget")}
                       if args.workload == "filter" else None),
            "kept": kept_step, "cells_per_step": cells_step,
            "extended": st0["n_extended"], "windows": st0["n_windows"],
            "speculation_waste": {"ext": 1.0 - (kept_step + st0["n_below"]) / st0["n_extended"] if st0["n_extended"] else None,
                                  "cells": st0["cells_covered"] / cells_step if cells_step else None},
            "gpu_launches": launches, "clocks": clocks, "e2e": e2e, "roofline": roof, "cpu_baseline": cpu, "c5_e2e": c5,
            "batch_info": info0, "speculate_info": (sfe.last_speculate_info() if window > 0 and args.workload != "c4" else None),
            "k_sweep": sweep or None, "lag0_fidelity": fidelity}
    print(json.dumps(line))
    if world > 1:
        dist.destroy_process_group()


if __name__ == "__main__":
    main()
