"""Per-half chain profile (Fig. 5: the spread of per-anchor extension runtimes).

    python -m paper_2606_06811_b200.halfprof c5s [--top 8] [--anchors 16]

Finds the kept alignments of a dense-anchor workload (sfe_speculate, predicted leaders, score-only), takes the `--anchors`
longest of them and extends those again as ONE sfe_ydrop_batch on each kernel (warp-systolic / cooperative row kernel) and in
each mode (score-only / traceback); prints, per run, the batch time and for the longest half its rows, SM cycles per row and
per wavefront step (sfe_last_half_profile), and checks that all four runs agree (scores, boxes, cells; CIGARs between the two
traceback runs).  One extension is a serial chain: these numbers are what bounds a pass once shadow work is gone.
"""
from __future__ import annotations

import argparse
import json

import numpy as np


def main():
    import torch
    from . import binding as B, workloads as W
    ap = argparse.ArgumentParser()
    ap.add_argument("workload", choices=["c3", "c3s", "c5s", "c5"])
    ap.add_argument("--anchors", type=int, default=16, help="how many of the longest kept alignments to re-extend")
    ap.add_argument("--top", type=int, default=3, help="halves reported per run")
    args = ap.parse_args()
    w = {"c3": W.config3, "c3s": lambda: W.config3(t_len=1_000_000, n_anchors=5_000),
         "c5s": lambda: W.config5(t_len=10_000_000, n_anchors=100_000), "c5": W.config5}[args.workload]()
    dev = torch.device("cuda", 0)
    free_b, _ = torch.cuda.mem_get_info(dev)
    sfe = B.Sfe(0, min(24 << 30, int(free_b * 0.5)))
    n = len(w.anchors)
    sc = B.scoring()
    tp = sfe.pack(torch.from_numpy(w.target_ascii().copy()).to(dev), with_rc=False)
    qp = sfe.pack(torch.from_numpy(w.query_ascii().copy()).to(dev), with_rc=True)
    pairs = B._dev(B.make_pairs(w.pairs), dev)
    o = sfe.speculate(tp[:2], len(w.target), qp, len(w.query), pairs, len(w.pairs), B._dev(B.make_anchors(w.anchors), dev), n, sc, 262144,
                      B.SCORE_ONLY | B.SPEC_LEADERS)
    torch.cuda.synchronize()
    keep = o["keep"].cpu().numpy()[:n]
    res0 = B.results_to_numpy(o["results"], n)
    kept = np.nonzero(keep == 1)[0]
    span = np.maximum(res0["tend"] - res0["tstart"], res0["qend"] - res0["qstart"])[kept]
    kept = np.sort(kept[np.argsort(-span)[: args.anchors]])
    A = B._dev(B.make_anchors(w.anchors[kept]), dev)
    ref = None; tb_ref = None
    for label, flags in (("systolic score-only", B.SCORE_ONLY | B.NO_BLOCK_KERNEL), ("row kernel score-only", B.SCORE_ONLY | B.BLOCK_KERNEL),
                         ("systolic traceback", B.WANT_CIGAR | B.NO_BLOCK_KERNEL), ("row kernel traceback", B.WANT_CIGAR | B.BLOCK_KERNEL)):
        for _ in range(2):
            e0 = torch.cuda.Event(enable_timing=True); e1 = torch.cuda.Event(enable_timing=True)
            e0.record()
            res, pool, used = sfe.ydrop_batch(tp[:2], len(w.target), qp, len(w.query), pairs, len(w.pairs), A, len(kept), sc, flags, 1 << 27)
            e1.record(); torch.cuda.synchronize()
        r = B.results_to_numpy(res, len(kept))
        prof = sfe.last_half_profile(2 * len(kept))
        out = {"run": label, "anchors": int(len(kept)), "batch_ms": round(e0.elapsed_time(e1), 1), "halves": []}
        for h in np.argsort(-prof["cells"])[: args.top]:
            p = prof[h]
            row_kernel = bool(int(p["status"]) & B.ST_BLOCK)
            rows = int(p["steps"]) if row_kernel else 32 * int(p["n_strips"])
            d = {"half": int(h), "rows": rows, "cells_per_row": round(int(p["cells"]) / max(1, rows)), "cycles_per_row": round(int(p["cycles"]) / max(1, rows), 1),
                 "ms": round(int(p["cycles"]) / 1.965e6, 1)}
            if not row_kernel:
                d.update(steps_per_strip=round(int(p["steps"]) / max(1, int(p["n_strips"])), 1), cycles_per_step=round(int(p["cycles"]) / max(1, int(p["steps"])), 1),
                         skew2=bool(int(p["status"]) & B.ST_SKEW2))
            out["halves"].append(d)
        if ref is None:
            ref = r
        out["same_as_first_run"] = all(bool((r[f] == ref[f]).all()) for f in ("score", "tstart", "tend", "qstart", "qend", "cells"))
        if flags & B.WANT_CIGAR:
            cig = pool.cpu().numpy().view(np.uint32)[: int(used.item())]
            if tb_ref is None:
                tb_ref = (r["n_ops"].copy(), cig.copy())
            else:
                out["cigars_equal_systolic"] = bool((r["n_ops"] == tb_ref[0]).all() and len(cig) == len(tb_ref[1]) and (cig == tb_ref[1]).all())
        print(json.dumps(out), flush=True)
    sfe.close()


if __name__ == "__main__":
    main()
