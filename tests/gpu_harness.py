"""Shared helpers of the -m gpu parity tests: run a workload through the C ABI (device-pointer
entry points) and through the oracle, and compare element by element."""
import numpy as np

from oracle import sfe_oracle as O
from paper_2606_06811_b200 import binding as B, workloads as W


def gpu_run(sfe, w, flags=B.WANT_CIGAR, window=None, **sc_kw):
    """pack -> ydrop_batch -> resolve through the device-pointer ABI.  Returns dict of numpy."""
    import torch
    dev = sfe.device
    sc = B.scoring(**sc_kw)
    t_ascii = torch.from_numpy(w.target_ascii().copy()).to(dev)
    q_ascii = torch.from_numpy(w.query_ascii().copy()).to(dev)
    tp = sfe.pack(t_ascii, with_rc=False)
    qp = sfe.pack(q_ascii, with_rc=True)
    n = len(w.anchors)
    anchors = B._dev(B.make_anchors(w.anchors), dev)
    pairs = B._dev(B.make_pairs(w.pairs), dev)
    res, pool, used = sfe.ydrop_batch(tp[:2], len(w.target), qp, len(w.query), pairs, len(w.pairs), anchors, n, sc, flags)
    acc = torch.zeros((n + 1) * B.BOX_DT.itemsize, dtype=torch.uint8, device=dev)
    nacc = torch.zeros(1, dtype=torch.int64, device=dev)
    stats = torch.zeros(B.STATS_DT.itemsize, dtype=torch.uint8, device=dev)
    keep = sfe.resolve(anchors, res, n, sc.min_score, acc, n + 1, nacc, stats)
    torch.cuda.synchronize()
    out = dict(results=B.results_to_numpy(res, n), keep=keep.cpu().numpy()[:n],
               stats=stats.cpu().numpy().view(B.STATS_DT)[0], n_accepted=int(nacc.item()),
               accepted=acc.cpu().numpy()[: int(nacc.item()) * B.BOX_DT.itemsize].view(B.BOX_DT),
               info=sfe.last_batch_info(), packs=(tp, qp))
    if flags & B.WANT_CIGAR:
        out["cigar"] = pool.cpu().numpy().view(np.uint32)
        out["cigar_used"] = int(used.item())
    return out


def oracle_anchor(w, i, **sc_kw):
    a = w.anchors[i]
    p = w.pairs[int(a[2])]
    Qs = w.query if a[3] > 0 else w.query_rc
    qlim = (int(p[2]), int(p[3])) if a[3] > 0 else (len(w.query) - int(p[3]), len(w.query) - int(p[2]))
    return O.extend_anchor(w.target, Qs, int(a[0]), int(a[1]), O.scoring(**sc_kw), t_lim=(int(p[0]), int(p[1])), q_lim=qlim)


def assert_anchor_equal(out, w, i, want_cigar=True, **sc_kw):
    r, ops = oracle_anchor(w, i, **sc_kw)
    g = out["results"][i]
    got = (int(g["score"]), int(g["score_fwd"]), int(g["score_bwd"]), int(g["tstart"]), int(g["tend"]), int(g["qstart"]),
           int(g["qend"]), int(g["cells"]))
    exp = (r.score, r.score_fwd, r.score_bwd, r.tstart, r.tend, r.qstart, r.qend, r.cells)
    assert got == exp, (i, tuple(w.anchors[i]), got, exp, int(g["status"]))
    if want_cigar:
        assert not (int(g["status"]) & (B.ST_TB_OVERFLOW | B.ST_CIGAR_OVERFLOW | B.ST_BAD_ANCHOR)), (i, int(g["status"]))
        assert (int(g["n_ops"]), int(g["n_ops_back"])) == (r.n_ops, r.n_ops_back), i
        assert B.ops_list(out["cigar"], int(g["cigar_off"]), int(g["n_ops"])) == ops, i
    return r


def oracle_many(w, indices, **sc_kw):
    """oracle_anchor for many anchors on all host cores (ctypes releases the GIL during the C call)."""
    import os
    from concurrent.futures import ThreadPoolExecutor
    O.lib()
    with ThreadPoolExecutor(max_workers=max(1, os.cpu_count() or 1)) as ex:
        return list(ex.map(lambda i: oracle_anchor(w, int(i), **sc_kw), indices))


def assert_anchors_equal(out, w, indices, want_cigar=True, **sc_kw):
    """assert_anchor_equal over many anchors, the oracle side run in parallel.  want_cigar: bool or a callable(i)."""
    indices = [int(i) for i in indices]
    for i, (r, ops) in zip(indices, oracle_many(w, indices, **sc_kw)):
        g = out["results"][i]
        got = (int(g["score"]), int(g["score_fwd"]), int(g["score_bwd"]), int(g["tstart"]), int(g["tend"]), int(g["qstart"]),
               int(g["qend"]), int(g["cells"]))
        exp = (r.score, r.score_fwd, r.score_bwd, r.tstart, r.tend, r.qstart, r.qend, r.cells)
        assert got == exp, (i, tuple(w.anchors[i]), got, exp, int(g["status"]))
        wc = want_cigar(i) if callable(want_cigar) else want_cigar
        if wc:
            assert not (int(g["status"]) & (B.ST_TB_OVERFLOW | B.ST_CIGAR_OVERFLOW | B.ST_BAD_ANCHOR)), (i, int(g["status"]))
            assert (int(g["n_ops"]), int(g["n_ops_back"])) == (r.n_ops, r.n_ops_back), i
            assert B.ops_list(out["cigar"], int(g["cigar_off"]), int(g["n_ops"])) == ops, i
    return len(indices)


def assert_resolve_equal(out, w, **sc_kw):
    """kept set / covered / below of the GPU resolver == Algorithm 1 run by the oracle."""
    ser = O.serial_loop(w.target, w.query, w.query_rc, w.pairs, w.anchors, O.scoring(**sc_kw), want_results=False)
    assert out["keep"].tolist() == ser["state"].tolist()
    assert out["n_accepted"] == ser["n_kept"] == int(out["stats"]["n_kept"])
    return ser
