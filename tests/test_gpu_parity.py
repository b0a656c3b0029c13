"""-m gpu parity tests: the CUDA path (through the C ABI) against the CPU oracle, bit-exact
(scores, boxes, cell counts, CIGARs, kept set): all arithmetic is integer."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2606_06811_b200 import binding as B, workloads as W  # noqa: E402

import gpu_harness as H  # noqa: E402


@pytest.fixture(scope="module")
def sfe():
    import __graft_entry__ as entry
    entry.build()
    s = B.Sfe(0, 2 << 30)
    yield s
    s.close()


def _wl(T, Q, anchors, pairs=None):
    T = np.asarray(T, np.uint8); Q = np.asarray(Q, np.uint8)
    pairs = np.array([[0, len(T), 0, len(Q)]] if pairs is None else pairs, np.int64)
    return W.Workload("t", T, Q, pairs, np.array(anchors, np.int64).reshape(-1, 4))


def test_pack_matches_definition(sfe, oracle):
    import torch
    rng = np.random.default_rng(5)
    for n in (1, 3, 31, 32, 33, 100, 4099, 65537):
        s = rng.choice(np.frombuffer(b"ACGTNacgtnXR", np.uint8), n)
        c2, nm, r2, rm = sfe.pack(torch.from_numpy(s.copy()).to(sfe.device))
        torch.cuda.synchronize()
        e = oracle.pack(s.tobytes())
        for got, exp in zip((c2, nm, r2, rm), e):
            assert got.cpu().numpy()[: len(exp)].tolist() == exp.tolist(), n


def test_appendix_a_examples(sfe, oracle):
    c = oracle.codes
    T = c("ACGTACGTTTGGCCAGTCAT"); Q = c("ACGTACGTGGCCAGTCAT")
    w = _wl(T, Q, [(0, 0, 0, 1), (14, 12, 0, 1), (10, 10, 0, 1), (9, 8, 0, 1), (3, 5, 0, 1), (20, 18, 0, 1), (0, 18, 0, 1)])
    out = H.gpu_run(sfe, w)
    for i in range(len(w.anchors)):
        H.assert_anchor_equal(out, w, i)
    for q, t in (("ACGTACGT", "ACGTACGT"), ("ACGNACGT", "ACGTACGT"), ("AAAA", "CCCC"), ("ACGTTA", "ACGTCA"), ("A", "A"),
                 ("A", "C"), ("ACGT", "A")):
        w = _wl(c(t), c(q), [(0, 0, 0, 1), (len(t), len(q), 0, 1)])
        out = H.gpu_run(sfe, w)
        H.assert_anchor_equal(out, w, 0); H.assert_anchor_equal(out, w, 1)


@pytest.mark.parametrize("ydrop", [120, 455, 1500, 9400])
def test_small_ydrops_and_ties(sfe, oracle, ydrop):
    """Y < O+X (gap-free), mid-range Y, default Y on related random pairs with N runs."""
    rng = np.random.default_rng(ydrop)
    T = rng.integers(0, 4, 900).astype(np.uint8)
    mu = W.mutate(T, 0.08, 0.02, W.Stream(ydrop))
    Q = mu.seq.copy()
    Q[100:104] = 4; T[300:302] = 4
    picks = rng.integers(0, len(mu.t_idx), 24)
    anchors = [(int(mu.t_idx[k]), int(mu.q_idx[k]), 0, 1) for k in picks] + [(0, 0, 0, 1), (len(T), len(Q), 0, 1), (5, 700, 0, 1)]
    w = _wl(T, Q, anchors)
    out = H.gpu_run(sfe, w, ydrop=ydrop)
    for i in range(len(anchors)):
        H.assert_anchor_equal(out, w, i, ydrop=ydrop)


def test_ydrop_inf_small(sfe, oracle):
    """R27: nothing is pruned; every cell of the rectangle is alive."""
    rng = np.random.default_rng(3)
    T = rng.integers(0, 4, 150).astype(np.uint8); Q = T.copy(); Q[40] = (Q[40] + 1) % 4
    Q = np.delete(Q, [70, 71])
    w = _wl(T, Q, [(0, 0, 0, 1), (60, 60, 0, 1), (150, 148, 0, 1)])
    out = H.gpu_run(sfe, w, ydrop=B.YDROP_INF)
    for i in range(3):
        r = H.assert_anchor_equal(out, w, i, ydrop=B.YDROP_INF)
    assert int(out["results"][0]["cells"]) == 151 * 149 + 1


def test_minus_strand_and_pairs(sfe, oracle):
    """- strand anchors use the reverse-complemented query; pair limits clip the DP."""
    w = W.config2(t_len=80_000, n_segments=40, per_seg=4, n_decoys=40, min_len=100, max_len=700)
    out = H.gpu_run(sfe, w)
    for i in range(len(w.anchors)):
        H.assert_anchor_equal(out, w, i)
    H.assert_resolve_equal(out, w)
    # sub-rectangle pairs: limits inside the sequences
    T = W.randseq(31, 3000); mu = W.mutate(T, 0.03, 0.005, W.Stream(32)); Q = mu.seq
    pairs = [[500, 2500, 480, 2480], [0, 3000, 0, len(Q)], [1000, 1200, 990, 1190]]
    k = np.searchsorted(mu.t_idx, [1100, 1500, 1100])
    anchors = [(int(mu.t_idx[k[0]]), int(mu.q_idx[k[0]]), 0, 1), (int(mu.t_idx[k[1]]), int(mu.q_idx[k[1]]), 1, 1),
               (int(mu.t_idx[k[2]]), int(mu.q_idx[k[2]]), 2, 1), (500, 480, 0, 1), (2500, 2480, 0, 1)]
    w = _wl(T, Q, anchors, pairs)
    out = H.gpu_run(sfe, w)
    for i in range(len(anchors)):
        H.assert_anchor_equal(out, w, i)


def test_config1_full(sfe, oracle):
    """BASELINE.json configs[0]: all 256 speculative extensions bit-exact; serial semantics keep 64."""
    w = W.config1()
    out = H.gpu_run(sfe, w)
    for i in range(len(w.anchors)):
        H.assert_anchor_equal(out, w, i)
    ser = H.assert_resolve_equal(out, w)
    assert ser["n_kept"] == 64 and int((out["keep"] == 1).sum()) == 64
    st = out["stats"]
    assert int(st["n_anchors"]) == 256 and int(st["n_covered"]) == 192 and int(st["n_below"]) == 0
    assert int(st["cells_total"]) == int(out["results"]["cells"].sum())
    # score-only mode gives the same scores / boxes / cells
    out2 = H.gpu_run(sfe, w, flags=B.SCORE_ONLY)
    for f in ("score", "tstart", "tend", "qstart", "qend", "cells"):
        assert (out2["results"][f] == out["results"][f]).all()
    assert out2["keep"].tolist() == out["keep"].tolist()


def test_host_api_equals_device_api(sfe, oracle):
    w = W.config1(n_segments=6, seg_len=500, slot=1200, per_seg=3)
    out = H.gpu_run(sfe, w)
    ho = sfe.extend_host(w.target_ascii(), w.query_ascii(), B.make_pairs(w.pairs), B.make_anchors(w.anchors), B.scoring())
    assert ho["keep"].tolist() == out["keep"].tolist()
    for f in ("score", "tstart", "tend", "qstart", "qend", "cells", "n_ops", "n_ops_back", "cigar_off"):
        assert (ho["results"][f] == out["results"][f]).all(), f
    assert ho["cigar_used"] == out["cigar_used"]
    assert (ho["cigar"][: ho["cigar_used"]] == out["cigar"][: out["cigar_used"]]).all()
    assert ho["stats"]["n_kept"] == int(out["stats"]["n_kept"])


def test_windowed_resolve_equals_serial(sfe, oracle):
    """Alg. 3 with windows of K through sfe_resolve (accepted list carried between calls, phase-1
    filter with results == NULL) keeps what Alg. 1 keeps (P7), for several K."""
    import torch
    w = W.config2(t_len=60_000, n_segments=30, per_seg=8, n_decoys=40, min_len=150, max_len=700)
    out = H.gpu_run(sfe, w)
    ser = H.assert_resolve_equal(out, w)
    n = len(w.anchors)
    dev = sfe.device
    A = B.make_anchors(w.anchors)
    res_all = out["results"]
    for K in (1, 5, 32, 33, n):
        acc = torch.zeros((n + 1) * B.BOX_DT.itemsize, dtype=torch.uint8, device=dev)
        nacc = torch.zeros(1, dtype=torch.int64, device=dev)
        state = np.zeros(n, np.uint8)
        j = 0
        while j < n:
            # phase 1: mask filter over the remaining anchors, take the first K unmasked
            rest = B._dev(A[j:], dev)
            m = sfe.resolve(rest, None, n - j, 0, acc, n + 1, nacc).cpu().numpy()[: n - j]
            idx = np.nonzero(m == 1)[0][:K] + j
            if len(idx) == 0:
                break
            nxt = (idx[-1] + 1) if len(idx) == K else n
            # phase 3 on the window (phase 2 results taken from the all-at-once batch: R20)
            kw = sfe.resolve(B._dev(A[idx], dev), B._dev(res_all[idx], dev), len(idx), 3000, acc, n + 1, nacc)
            state[idx] = kw.cpu().numpy()[: len(idx)]
            j = nxt
        assert (state == 1).tolist() == (ser["state"] == 1).tolist(), K
        assert int(nacc.item()) == ser["n_kept"]


def test_wide_band_path(sfe, oracle):
    """Bands wider than the 1024-column shared-memory window are re-run by the global-memory-ring
    kernel and stay bit-exact: huge ydrop, and ydrop = infinity on 1.6 kbp."""
    T = W.randseq(41, 2600); mu = W.mutate(T, 0.05, 0.01, W.Stream(42)); Q = mu.seq
    k = np.searchsorted(mu.t_idx, [1300, 100])
    anchors = [(int(mu.t_idx[k[0]]), int(mu.q_idx[k[0]]), 0, 1), (int(mu.t_idx[k[1]]), int(mu.q_idx[k[1]]), 0, 1)]
    w = _wl(T, Q, anchors)
    out = H.gpu_run(sfe, w, ydrop=40000)
    assert out["info"]["wide"] >= 2
    for i in range(2):
        H.assert_anchor_equal(out, w, i, ydrop=40000)
        assert int(out["results"][i]["status"]) & B.ST_WIDE
    w = _wl(T[:1600], Q[:1600], [(0, 0, 0, 1), (800, int(mu.q_idx[np.searchsorted(mu.t_idx, 800)]), 0, 1)])
    w.anchors[1, 0] = int(mu.t_idx[np.searchsorted(mu.t_idx, 800)])
    out = H.gpu_run(sfe, w, ydrop=B.YDROP_INF)
    assert out["info"]["wide"] >= 1
    for i in range(2):
        H.assert_anchor_equal(out, w, i, ydrop=B.YDROP_INF)
    # A17: 300-bp core + random tails, band up to ~700 columns: normal kernel, no wide path
    core = W.randseq(7, 300)
    w = _wl(np.concatenate([core, W.randseq(8, 1500)]), np.concatenate([core, W.randseq(9, 1500)]), [(0, 0, 0, 1), (150, 150, 0, 1)])
    out = H.gpu_run(sfe, w)
    assert out["info"]["wide"] == 0
    H.assert_anchor_equal(out, w, 0); H.assert_anchor_equal(out, w, 1)
    assert int(out["results"][0]["cells"]) == 598524 + 1 and int(out["results"][0]["score"]) == 28831


def test_tiny_arena_recycles_and_reruns(oracle):
    """A 6 MiB traceback arena (96 chunks) for a batch that writes ~8x more: chunks are recycled as soon as a
    half has been walked, halves that find no free chunk finish score-only and are re-run; results stay bit-exact."""
    import __graft_entry__ as entry
    entry.build()
    s = B.Sfe(0, 6 << 20)
    try:
        w = W.config1(n_segments=12, seg_len=1500, slot=2600, per_seg=4)
        out = H.gpu_run(s, w)
        assert out["info"]["tb_bytes"] > 6 * (6 << 20)
        for i in range(len(w.anchors)):
            H.assert_anchor_equal(out, w, i)
        H.assert_resolve_equal(out, w)
        # a second batch on the same context: the free ring is intact after the first one
        out2 = H.gpu_run(s, w)
        assert (out2["results"] == out["results"]).all() and (out2["cigar"][: out2["cigar_used"]] == out["cigar"][: out["cigar_used"]]).all()
    finally:
        s.close()


def _speculate(sfe, w, K, flags=B.WANT_CIGAR, **sc_kw):
    import torch
    dev = sfe.device
    sc = B.scoring(**sc_kw)
    tp = sfe.pack(torch.from_numpy(w.target_ascii().copy()).to(dev), with_rc=False)
    qp = sfe.pack(torch.from_numpy(w.query_ascii().copy()).to(dev), with_rc=True)
    n = len(w.anchors)
    o = sfe.speculate(tp[:2], len(w.target), qp, len(w.query), B._dev(B.make_pairs(w.pairs), dev), len(w.pairs),
                      B._dev(B.make_anchors(w.anchors), dev), n, sc, K, flags)
    torch.cuda.synchronize()
    out = dict(results=B.results_to_numpy(o["results"], n), keep=o["keep"].cpu().numpy()[:n],
               stats=o["stats"].cpu().numpy().view(B.STATS_DT)[0], n_accepted=int(o["n_accepted"].item()))
    if flags & B.WANT_CIGAR:
        out["cigar"] = o["pool"].cpu().numpy().view(np.uint32); out["cigar_used"] = int(o["used"].item())
    return out


@pytest.mark.parametrize("K", [1, 3, 32, 50, 10_000])
def test_speculate_equals_serial_loop(sfe, oracle, K):
    """sfe_speculate (Alg. 3: scan / extend / commit per window, all on the device) keeps exactly what Alg. 1
    keeps for every window size (P7); every anchor it extended is bit-exact against the oracle; anchors covered
    before their window are never extended; the waste counters add up."""
    w = W.config2(t_len=60_000, n_segments=30, per_seg=8, n_decoys=40, min_len=150, max_len=700)
    n = len(w.anchors)
    ser = oracle.serial_loop(w.target, w.query, w.query_rc, w.pairs, w.anchors, oracle.scoring(), want_results=False)
    out = _speculate(sfe, w, K)
    assert out["keep"].tolist() == ser["state"].tolist(), K
    st = out["stats"]
    skipped = (out["results"]["status"] & B.ST_SKIPPED) != 0
    assert int(st["n_anchors"]) == n and int(st["n_kept"]) == ser["n_kept"] == out["n_accepted"]
    assert int(st["n_extended"]) == int((~skipped).sum()) and int(st["n_kept"] + st["n_covered"] + st["n_below"]) == n
    assert (out["keep"][skipped] == 0).all()
    # serial semantics extend exactly the anchors that are not covered; speculation extends a superset
    serial_ext = ser["state"] != 0
    assert (~skipped)[serial_ext].all()
    if K == 1:
        assert int(st["n_extended"]) == int(serial_ext.sum())          # K = 1 is Algorithm 1: no shadow work
    else:
        assert int(st["n_extended"]) >= int(serial_ext.sum())
    assert int(st["cells_total"]) == int(out["results"]["cells"][~skipped].sum())
    for i in np.nonzero(~skipped)[0][:: max(1, int((~skipped).sum()) // 40)]:
        H.assert_anchor_equal(out, w, int(i))


def test_speculate_config1_windows(sfe, oracle):
    """configs[0] through the windowed path: 64 kept for every K; K = 256 computes all 256 (75 % shadow work),
    K = 1 only the 64 that the serial loop extends."""
    w = W.config1()
    for K, n_ext in ((256, 256), (1, 64)):
        out = _speculate(sfe, w, K, flags=B.SCORE_ONLY)
        assert int((out["keep"] == 1).sum()) == 64 and int(out["stats"]["n_extended"]) == n_ext, K
    full = H.gpu_run(sfe, w, flags=B.SCORE_ONLY)
    assert out["keep"].tolist() == full["keep"].tolist()


@pytest.mark.parametrize("seed,n,spread", [(1, 1000, 40), (2, 5000, 400), (3, 257, 5), (4, 4096, 3000), (5, 1500, 60)])
def test_resolve_random_boxes(sfe, oracle, seed, n, spread):
    """sfe_resolve alone on synthetic (score, box) records: dense chains of mutually covering boxes, below-tau
    anchors inside kept boxes (covered, not 'below': R17 is tested before R16), both strands, unsorted ties."""
    import torch
    rng = np.random.default_rng(seed)
    tpos = np.sort(rng.integers(0, n * spread // 8 + 50, n))
    if seed == 5:                                   # anchor order need not be position order: locally shuffled
        for a in range(0, n - 40, 40):
            rng.shuffle(tpos[a:a + 40])
    qpos = tpos + rng.integers(-30, 30, n)
    strand = np.where(rng.random(n) < 0.3, -1, 1)
    anchors = np.stack([tpos, qpos, np.zeros(n, np.int64), strand], 1).astype(np.int64)
    score = rng.integers(2000, 4500, n)
    lo_t = rng.integers(0, spread, n); hi_t = rng.integers(0, spread, n); lo_q = rng.integers(0, spread, n); hi_q = rng.integers(0, spread, n)
    boxes = np.stack([tpos - lo_t, tpos + hi_t, qpos - lo_q, qpos + hi_q], 1)
    state, acc = oracle.resolve(anchors, score, boxes, 3000)
    res = np.zeros(n, B.RESULT_DT)
    res["score"] = score; res["tstart"] = boxes[:, 0]; res["tend"] = boxes[:, 1]; res["qstart"] = boxes[:, 2]; res["qend"] = boxes[:, 3]
    res["cells"] = 7
    dev = sfe.device
    accd = torch.zeros((n + 1) * B.BOX_DT.itemsize, dtype=torch.uint8, device=dev)
    nacc = torch.zeros(1, dtype=torch.int64, device=dev)
    stats = torch.zeros(B.STATS_DT.itemsize, dtype=torch.uint8, device=dev)
    keep = sfe.resolve(B._dev(B.make_anchors(anchors), dev), B._dev(res, dev), n, 3000, accd, n + 1, nacc, stats).cpu().numpy()[:n]
    assert keep.tolist() == state.tolist()
    assert int(nacc.item()) == len(acc)
    got = accd.cpu().numpy()[: len(acc) * B.BOX_DT.itemsize].view(B.BOX_DT)
    assert [(int(b["tstart"]), int(b["tend"]), int(b["qstart"]), int(b["qend"]), int(b["strand"])) for b in got] == [tuple(int(x) for x in b) for b in acc]
    st = stats.cpu().numpy().view(B.STATS_DT)[0]
    assert (int(st["n_kept"]), int(st["n_covered"]), int(st["n_below"])) == (int((state == 1).sum()), int((state == 0).sum()), int((state == 2).sum()))
    assert int(st["cells_covered"]) == 7 * int((state == 0).sum())


def test_speculate_cigar_for_kept_only(sfe, oracle):
    """SFE_CIGAR_KEPT_ONLY: windows speculate score-only, the kept anchors get their CIGAR from one traceback batch at the
    end.  Same kept set and the same score / box / cells for every extended anchor as the all-CIGAR run; kept anchors are
    bit-exact against the oracle incl. the ops; everybody else carries no ops."""
    w = W.config2(t_len=60_000, n_segments=30, per_seg=8, n_decoys=40, min_len=150, max_len=700)
    full = _speculate(sfe, w, 32)
    ko = _speculate(sfe, w, 32, flags=B.WANT_CIGAR | B.CIGAR_KEPT_ONLY)
    assert ko["keep"].tolist() == full["keep"].tolist()
    for f in ("score", "score_fwd", "score_bwd", "tstart", "tend", "qstart", "qend", "cells", "status"):
        assert (ko["results"][f] == full["results"][f]).all(), f
    kept = ko["keep"] == 1
    assert (ko["results"]["n_ops"][~kept] == 0).all() and (ko["results"]["cigar_off"][~kept] == -1).all()
    assert (ko["results"]["n_ops"][kept] == full["results"]["n_ops"][kept]).all()
    assert ko["cigar_used"] == int(ko["results"]["n_ops"][kept].sum())
    for i in np.nonzero(kept)[0]:
        H.assert_anchor_equal(ko, w, int(i))


def test_degenerate_calls(sfe, oracle):
    """Boundary behaviour of the C ABI: zero anchors, anchors outside their pair / with an unknown pair / on the - strand
    without reverse-complement planes (SFE_ST_BAD_ANCHOR, nothing computed, no fault), invalid arguments (error codes)."""
    import ctypes as C
    import torch
    dev = sfe.device
    L = B.lib()
    T = W.randseq(3, 500); Q = T.copy()
    w = _wl(T, Q, [(10, 10, 0, 1)])
    tp = sfe.pack(torch.from_numpy(w.target_ascii().copy()).to(dev), with_rc=False)
    qp = sfe.pack(torch.from_numpy(w.query_ascii().copy()).to(dev), with_rc=True)
    pairs = B._dev(B.make_pairs(np.array([[0, 500, 0, 500], [100, 200, 100, 200]], np.int64)), dev)
    sc = B.scoring()
    # zero anchors: every entry point returns OK and touches nothing
    res, pool, used = sfe.ydrop_batch(tp[:2], 500, qp, 500, pairs, 2, None, 0, sc)
    keep = sfe.resolve(None, None, 0, 3000, None, 0, None)
    o = sfe.speculate(tp[:2], 500, qp, 500, pairs, 2, None, 0, sc, 8)
    torch.cuda.synchronize()
    assert int(used.item()) == 0
    # bad anchors next to a good one
    A = np.array([(10, 10, 0, 1), (600, 10, 0, 1), (10, 10, 7, 1), (50, 50, 1, 1), (150, 150, 1, 1), (-1, 5, 0, 1)], np.int64)
    res, pool, used = sfe.ydrop_batch(tp[:2], 500, qp, 500, pairs, 2, B._dev(B.make_anchors(A), dev), len(A), sc)
    torch.cuda.synchronize()
    r = B.results_to_numpy(res, len(A))
    bad = (r["status"] & B.ST_BAD_ANCHOR) != 0
    assert bad.tolist() == [False, True, True, True, False, True]
    assert (r["score"][bad] == 0).all() and (r["n_ops"][bad] == 0).all() and (r["cells"][bad] == 0).all()
    assert int(r["score"][0]) == oracle.extend_anchor(T, Q, 10, 10, oracle.scoring())[0].score
    assert int(r["score"][4]) == oracle.extend_anchor(T, Q, 150, 150, oracle.scoring(), t_lim=(100, 200), q_lim=(100, 200))[0].score
    # - strand anchors without reverse-complement planes
    Am = np.array([(10, 10, 0, -1)], np.int64)
    res, pool, used = sfe.ydrop_batch(tp[:2], 500, qp[:2], 500, pairs, 2, B._dev(B.make_anchors(Am), dev), 1, sc)
    torch.cuda.synchronize()
    assert int(B.results_to_numpy(res, 1)["status"][0]) & B.ST_BAD_ANCHOR
    # invalid arguments are refused with error codes, not faults
    assert L.sfe_ydrop_batch(sfe.h, None, None, 500, None, None, None, None, 500, None, 2, None, 5, C.byref(sc), 1, None, None, 0, None) == B.EINVAL
    bad_sc = B.scoring(prune_lag=7)
    with pytest.raises(B.SfeError):
        sfe.ydrop_batch(tp[:2], 500, qp, 500, pairs, 2, B._dev(B.make_anchors(A), dev), len(A), bad_sc)
    with pytest.raises(B.SfeError):
        sfe.ydrop_batch(tp[:2], 500, qp, 500, pairs, 2, B._dev(B.make_anchors(A), dev), len(A), B.scoring(gap_extend=0))
    with pytest.raises(B.SfeError):
        sfe.speculate(tp[:2], 500, qp, 500, pairs, 2, B._dev(B.make_anchors(A), dev), len(A), sc, 0)


@pytest.mark.parametrize("kernel", ["systolic", "block"])
def test_minus_strand_subrange_pairs(sfe, oracle, kernel):
    """R15 on the GPU (half_setup's mirrored branch): - strand anchors in pairs whose query interval is NOT the whole
    query, so the mirror [q_len - q_end, q_len - q_begin) differs from the interval itself.  First the closed form of
    tests/test_oracle_pins.py::test_r15_minus_strand_subrange_pair (Q = revcomp(T): pure matches up to the limits), then
    mutated sequences with random sub-range pairs on both strands against the oracle, element by element."""
    kflag = B.BLOCK_KERNEL if kernel == "block" else B.NO_BLOCK_KERNEL
    T = W.randseq(77, 40); Q = W.revcomp(T)
    diag = lambda lo, hi: sum(B.HOXD70[int(x)][int(x)] for x in T[lo:hi])
    cases = [((0, 40, 10, 26), (20, 20), (0, 40, 14, 30)), ((0, 40, 0, 9), (33, 33), (0, 40, 31, 40)),
             ((16, 27, 10, 26), (20, 20), (16, 27, 14, 30)), ((0, 40, 12, 13), (27, 27), (0, 40, 27, 28))]
    w = _wl(T, Q, [(tp, qp, k, -1) for k, (_, (tp, qp), _) in enumerate(cases)], [c[0] for c in cases])
    out = H.gpu_run(sfe, w, flags=B.WANT_CIGAR | kflag, min_score=0)
    for k, (_, (tp, qp), (tb, te, qb, qe)) in enumerate(cases):
        lo = max(tb - tp, qb - qp); hi = min(te - tp, qe - qp)
        g = out["results"][k]
        assert int(g["status"]) & 0xff == 0
        assert (int(g["score_bwd"]), int(g["score_fwd"])) == (diag(tp + lo, tp), diag(tp, tp + hi)), k
        assert (int(g["tstart"]), int(g["tend"]), int(g["qstart"]), int(g["qend"])) == (tp + lo, tp + hi, qp + lo, qp + hi), k
        exp_ops = ([(-lo, B.OP_M)] if lo else []) + ([(hi, B.OP_M)] if hi else [])
        assert B.ops_list(out["cigar"], int(g["cigar_off"]), int(g["n_ops"])) == exp_ops, k
        H.assert_anchor_equal(out, w, k, min_score=0)
    # mutated sequences, half the segments reverse-complemented, each anchor in its own random sub-range pair
    w2 = W.config2(t_len=50_000, n_segments=24, per_seg=5, n_decoys=20, min_len=200, max_len=700)
    rng = np.random.default_rng(15)
    qlen = len(w2.query)
    pairs, anchors = [], []
    for a in w2.anchors:
        tp, qp, strand = int(a[0]), int(a[1]), int(a[3])
        qf = qp if strand > 0 else qlen - qp                        # the anchor's corner in the forward query frame
        t0 = max(0, tp - int(rng.integers(0, 400))); t1 = min(len(w2.target), tp + int(rng.integers(0, 400)))
        q0 = max(0, qf - int(rng.integers(0, 400))); q1 = min(qlen, qf + int(rng.integers(0, 400)))
        anchors.append((tp, qp, len(pairs), strand)); pairs.append((t0, t1, q0, q1))
    w3 = W.Workload("subrange", w2.target, w2.query, np.array(pairs, np.int64), np.array(anchors, np.int64))
    assert int((w3.anchors[:, 3] < 0).sum()) > 20
    out = H.gpu_run(sfe, w3, flags=B.WANT_CIGAR | kflag)
    assert not (out["results"]["status"] & np.uint32(B.ST_BAD_ANCHOR)).any()
    assert H.assert_anchors_equal(out, w3, range(len(w3.anchors))) == len(anchors)
    H.assert_resolve_equal(out, w3)


def test_no_binning_equals_binned(sfe, oracle):
    """SFE_NO_BINNING (tickets in anchor order, no reserved longest-first segment): the same results as the binned
    queue, bit for bit, and equal to the oracle."""
    w = W.config2(t_len=80_000, n_segments=40, per_seg=4, n_decoys=40, min_len=100, max_len=700)
    a = H.gpu_run(sfe, w)
    b = H.gpu_run(sfe, w, flags=B.WANT_CIGAR | B.NO_BINNING)
    assert (a["results"] == b["results"]).all() and a["keep"].tolist() == b["keep"].tolist()
    assert a["cigar_used"] == b["cigar_used"] and (a["cigar"][: a["cigar_used"]] == b["cigar"][: b["cigar_used"]]).all()
    prof = sfe.last_half_profile(2 * len(w.anchors))
    assert not (prof["status"] & (B.ST_SKEW2 | B.ST_SKEW_RETRY)).any()          # no reserved tickets without binning
    H.assert_anchors_equal(b, w, range(len(w.anchors)))
    H.assert_resolve_equal(b, w)
    c = H.gpu_run(sfe, w, flags=B.SCORE_ONLY | B.NO_BINNING)
    for f in ("score", "tstart", "tend", "qstart", "qend", "cells"):
        assert (c["results"][f] == a["results"][f]).all()


@pytest.mark.parametrize("kernel", ["systolic", "block"])
def test_score_limit_is_flagged(sfe, oracle, kernel):
    """R25: a half whose running best reaches 2^29 - 2^22 is stopped and flagged SFE_ST_SCORE_LIMIT instead of running
    into the 2^29 sentinels.  An all-match C/G pair scores exactly 100 per row (closed form, pin P3), so the limit
    532,676,608 is crossed after 5,326,767 rows: a 5.2 Mbp pair stays below it (score = 100 * length, no flag), a
    5.6 Mbp pair trips it.  Score-only (the traceback of such a half would be > 1.5 GB)."""
    import torch
    LIMIT = (1 << 29) - (1 << 22)
    kflag = B.BLOCK_KERNEL if kernel == "block" else B.NO_BLOCK_KERNEL
    for n, tripped in ((5_200_000, False), (5_600_000, True)):
        T = np.tile(np.array([1, 2], np.uint8), n // 2)
        w = _wl(T, T.copy(), [(0, 0, 0, 1)])
        out = H.gpu_run(sfe, w, flags=B.SCORE_ONLY | kflag)
        g = out["results"][0]
        assert bool(int(g["status"]) & B.ST_SCORE_LIMIT) == tripped
        assert int(g["score_bwd"]) == 0 and int(g["score_fwd"]) == 100 * (int(g["qend"]) - int(g["qstart"]))
        assert int(g["tend"]) == int(g["qend"]) and int(g["tstart"]) == int(g["qstart"]) == 0
        if tripped:
            assert LIMIT <= int(g["score"]) < LIMIT + (1 << 22)
        else:
            assert int(g["score"]) == 100 * n and int(g["qend"]) == n
    # with traceback asked for, a flagged anchor carries no CIGAR (like SFE_ST_BAND_LIMIT)
    if kernel == "systolic":
        s2 = B.Sfe(0, 8 << 30)
        try:
            T = np.tile(np.array([1, 2], np.uint8), 2_800_000)
            out = H.gpu_run(s2, _wl(T, T.copy(), [(0, 0, 0, 1), (5_599_000, 5_599_000, 0, 1)]), flags=B.WANT_CIGAR | kflag)
            g = out["results"]
            assert int(g["status"][0]) & B.ST_SCORE_LIMIT and int(g["n_ops"][0]) == 0 and int(g["cigar_off"][0]) == -1
            assert int(g["status"][1]) & B.ST_SCORE_LIMIT and int(g["score_fwd"][1]) == 100_000
        finally:
            s2.close()
            torch.cuda.empty_cache()


def test_two_contexts_on_two_devices(oracle):
    """Function attributes (dynamic shared memory) are set per device in sfe_create: a context on a second GPU of the same
    process must run.  Skipped on a single-GPU box; there the same code path runs for a second context on device 0."""
    import torch
    w = W.config1(n_segments=3, seg_len=500, slot=1200, per_seg=2)
    devs = [0, 1] if torch.cuda.device_count() > 1 else [0, 0]
    ctxs = [B.Sfe(d, 256 << 20) for d in devs]
    try:
        outs = []
        for d, s in zip(devs, ctxs):
            with torch.cuda.device(d):
                outs.append(s.extend_host(w.target_ascii(), w.query_ascii(), B.make_pairs(w.pairs), B.make_anchors(w.anchors), B.scoring()))
        assert (outs[0]["results"] == outs[1]["results"]).all() and outs[0]["keep"].tolist() == outs[1]["keep"].tolist()
        r, _ = oracle.extend_anchor(w.target, w.query, int(w.anchors[0][0]), int(w.anchors[0][1]), oracle.scoring())
        assert int(outs[1]["results"]["score"][0]) == r.score
    finally:
        for s in ctxs:
            s.close()


def test_tiny_arena_many_short_halves(oracle):
    """Free-chunk ring under churn: 12 chunks (a half of this input needs up to 6) shared by thousands of halves -- every pop / push goes
    through the same few slots many laps over.  Results stay bit-exact, nothing is dropped (info ring_drops == 0)."""
    import __graft_entry__ as entry
    entry.build()
    s = B.Sfe(0, 12 * 65536)
    try:
        w = W.config2(t_len=120_000, n_segments=60, per_seg=10, n_decoys=600, min_len=100, max_len=300)
        out = H.gpu_run(s, w)
        assert out["info"]["ring_drops"] == 0
        bad = out["results"]["status"] & np.uint32(B.ST_TB_OVERFLOW | B.ST_INTERNAL)
        assert not bad.any()
        H.assert_anchors_equal(out, w, range(0, len(w.anchors), 3))
        H.assert_resolve_equal(out, w)
    finally:
        s.close()


def _dense_workload(seed=7, t_len=60_000, n_anchors=900):
    """A small configs[2]-like input: high identity, blocks, some inverted / moved, dense anchors on the true path --
    most anchors are followers of their block's first one."""
    return W.config3(t_len=t_len, n_anchors=n_anchors, blk_lo=1500, blk_hi=6000)


@pytest.mark.parametrize("force", [0, 1, 2, 3])
@pytest.mark.parametrize("K", [1, 7, 64, 4096])
def test_speculate_leaders_equals_serial_loop(sfe, oracle, K, force):
    """SFE_SPEC_LEADERS: Algorithm 3 with predicted leaders keeps exactly what Algorithm 1 keeps for ANY prediction --
    the classifier's (force 0), nobody leads (1: every uncovered anchor is reached by the commit and force-extended),
    everybody leads (2), the second half of the anchors never leads (3) -- and any batch size K.  Extended anchors are
    bit-exact against the oracle; anchors never extended are covered ones; the counters add up."""
    for w in (W.config2(t_len=60_000, n_segments=30, per_seg=8, n_decoys=40, min_len=150, max_len=700), _dense_workload()):
        n = len(w.anchors)
        ser = oracle.serial_loop(w.target, w.query, w.query_rc, w.pairs, w.anchors, oracle.scoring(), want_results=False)
        sfe.set_option(B.OPT_FORCE_CLASS, force)
        sfe.set_option(B.OPT_SPEC_SPAN, 256)
        try:
            out = _speculate(sfe, w, K, flags=B.WANT_CIGAR | B.SPEC_LEADERS)
            info = sfe.last_speculate_info()
        finally:
            sfe.set_option(B.OPT_FORCE_CLASS, 0); sfe.set_option(B.OPT_SPEC_SPAN, 1 << 20)
        assert out["keep"].tolist() == ser["state"].tolist(), (K, force)
        st = out["stats"]
        skipped = (out["results"]["status"] & B.ST_SKIPPED) != 0
        assert int(st["n_anchors"]) == n and int(st["n_kept"]) == ser["n_kept"] == out["n_accepted"]
        assert int(st["n_extended"]) == int((~skipped).sum()) and int(st["n_kept"] + st["n_covered"] + st["n_below"]) == n
        assert (out["keep"][skipped] == 0).all()
        serial_ext = ser["state"] != 0
        assert (~skipped)[serial_ext].all()                      # everything Algorithm 1 extends was extended
        assert int(st["cells_total"]) == int(out["results"]["cells"][~skipped].sum())
        assert info["batches"] == int(st["n_windows"]) >= 1
        H.assert_anchors_equal(out, w, np.nonzero(~skipped)[0][:: max(1, int((~skipped).sum()) // 60)])


def test_speculate_leaders_serial_when_nobody_leads(sfe, oracle):
    """With no predicted leader and no escalation the path degenerates to Algorithm 1 itself: one extension per commit
    stop, exactly the anchors the serial loop extends, no shadow work.  With the classifier on the dense input it extends
    far fewer anchors than classic windows of the same K."""
    w = _dense_workload()
    ser = oracle.serial_loop(w.target, w.query, w.query_rc, w.pairs, w.anchors, oracle.scoring(), want_results=False)
    n_serial = int((ser["state"] != 0).sum())
    sfe.set_option(B.OPT_FORCE_CLASS, 1); sfe.set_option(B.OPT_SPEC_ESC_MAX, 1)
    try:
        out = _speculate(sfe, w, 64, flags=B.SCORE_ONLY | B.SPEC_LEADERS)
        info = sfe.last_speculate_info()
    finally:
        sfe.set_option(B.OPT_FORCE_CLASS, 0); sfe.set_option(B.OPT_SPEC_ESC_MAX, 64)
    assert out["keep"].tolist() == ser["state"].tolist()
    assert int(out["stats"]["n_extended"]) == n_serial == info["stops"] == info["forced"]
    lead = _speculate(sfe, w, 64, flags=B.SCORE_ONLY | B.SPEC_LEADERS)
    classic = _speculate(sfe, w, 64, flags=B.SCORE_ONLY)
    assert lead["keep"].tolist() == classic["keep"].tolist() == ser["state"].tolist()
    assert n_serial <= int(lead["stats"]["n_extended"]) < int(classic["stats"]["n_extended"]) // 3
    for f in ("score", "tstart", "tend", "qstart", "qend", "cells"):
        both = ((lead["results"]["status"] | classic["results"]["status"]) & B.ST_SKIPPED) == 0
        assert (lead["results"][f][both] == classic["results"][f][both]).all()


def test_speculate_leaders_kept_only_and_carried_boxes(sfe, oracle):
    """SFE_SPEC_LEADERS with SFE_CIGAR_KEPT_ONLY (score-only batches + one traceback batch over the kept anchors) and with
    accepted boxes carried in from an earlier call (R26): the second half of the anchors resolved against the first half's."""
    import torch
    w = _dense_workload(n_anchors=700)
    n = len(w.anchors)
    ser = oracle.serial_loop(w.target, w.query, w.query_rc, w.pairs, w.anchors, oracle.scoring(), want_results=False)
    ko = _speculate(sfe, w, 128, flags=B.WANT_CIGAR | B.CIGAR_KEPT_ONLY | B.SPEC_LEADERS)
    assert ko["keep"].tolist() == ser["state"].tolist()
    kept = ko["keep"] == 1
    assert (ko["results"]["n_ops"][~kept] == 0).all() and ko["cigar_used"] == int(ko["results"]["n_ops"][kept].sum())
    H.assert_anchors_equal(ko, w, np.nonzero(kept)[0])
    # two calls, accepted list carried across
    dev = sfe.device
    tp = sfe.pack(torch.from_numpy(w.target_ascii().copy()).to(dev), with_rc=False)
    qp = sfe.pack(torch.from_numpy(w.query_ascii().copy()).to(dev), with_rc=True)
    acc = torch.zeros((n + 1) * B.BOX_DT.itemsize, dtype=torch.uint8, device=dev); nacc = torch.zeros(1, dtype=torch.int64, device=dev)
    pairs = B._dev(B.make_pairs(w.pairs), dev); A = B.make_anchors(w.anchors); h = n // 2
    keep = []
    for lo, hi in ((0, h), (h, n)):
        o = sfe.speculate(tp[:2], len(w.target), qp, len(w.query), pairs, len(w.pairs), B._dev(A[lo:hi], dev), hi - lo, B.scoring(), 64,
                          B.SCORE_ONLY | B.SPEC_LEADERS, accepted_dev=acc, n_accepted_dev=nacc)
        torch.cuda.synchronize()
        keep += o["keep"].cpu().numpy()[: hi - lo].tolist()
    assert keep == ser["state"].tolist() and int(nacc.item()) == ser["n_kept"]


@pytest.mark.parametrize("slots", [1, 64])
def test_long_half_handoff_equals_oracle(sfe, oracle, slots):
    """SFE_OPT_LONG_ROWS / SFE_OPT_LONG_ROWS_DENSE: systolic halves still alive at a check-point (here 64, 128, 256, 512 rows,
    so that most halves meet one) stop, queue themselves and are re-run from their start by row-kernel CTAs that serve the
    queue beside the systolic kernel.  Nothing may change: kept set = serial loop, every extended anchor bit-exact against
    the oracle (score, box, cells, CIGAR), with one serving CTA (almost every check-point finds it busy) and with 64."""
    w = W.config2(t_len=60_000, n_segments=30, per_seg=8, n_decoys=40, min_len=150, max_len=700)
    ser = oracle.serial_loop(w.target, w.query, w.query_rc, w.pairs, w.anchors, oracle.scoring(), want_results=False)
    sfe.set_option(B.OPT_LONG_ROWS, 64); sfe.set_option(B.OPT_LONG_ROWS_DENSE, 64); sfe.set_option(B.OPT_ROW_SLOTS, slots)
    cap0 = sfe.n_sm(); sfe.set_option(B.OPT_ROW_KERNEL_CAP, 0)      # (the priority split and the hand-off exclude each other)
    try:
        for flags in (B.WANT_CIGAR | B.SPEC_LEADERS, B.SCORE_ONLY | B.SPEC_LEADERS):
            out = _speculate(sfe, w, 64, flags=flags)
            if flags & B.WANT_CIGAR:
                assert sfe.last_batch_info()["block_halves"] > 0                   # halves were handed over
            assert out["keep"].tolist() == ser["state"].tolist()
            skipped = (out["results"]["status"] & B.ST_SKIPPED) != 0
            H.assert_anchors_equal(out, w, np.nonzero(~skipped)[0][:: max(1, int((~skipped).sum()) // 80)], want_cigar=bool(flags & B.WANT_CIGAR))
        # the dense launch of sfe_ydrop_batch + sfe_resolve
        full = H.gpu_run(sfe, w)
        assert sfe.last_batch_info()["block_halves"] > 0
        H.assert_resolve_equal(full, w)
        H.assert_anchors_equal(full, w, np.arange(0, len(w.anchors), max(1, len(w.anchors) // 80)))
        so = H.gpu_run(sfe, w, flags=B.SCORE_ONLY)
        for f in ("score", "tstart", "tend", "qstart", "qend", "cells"):
            assert (so["results"][f] == full["results"][f]).all(), f
    finally:
        sfe.set_option(B.OPT_LONG_ROWS, 0); sfe.set_option(B.OPT_LONG_ROWS_DENSE, 0); sfe.set_option(B.OPT_ROW_SLOTS, 64)
        sfe.set_option(B.OPT_ROW_KERNEL_CAP, cap0)


def test_filter_workload_equals_oracle(sfe, oracle):
    """f3: the gapped Y-drop extension as the filter over raw, mostly false seed hits -- score-only,
    ydrop 2000, one +-1024-base box per hit (a row / column budget), pass = score >= tau.  Every hit's score, box and cell
    count equal the oracle's; so does the pass set; about the planted fraction of the hits passes."""
    import torch
    w = W.filter_hits(n_hits=6000, true_frac=0.05, t_len=400_000, n_segments=400)
    n = len(w.anchors)
    dev = sfe.device
    sc = B.scoring(ydrop=2000)
    tp = sfe.pack(torch.from_numpy(w.target_ascii().copy()).to(dev), with_rc=False)
    qp = sfe.pack(torch.from_numpy(w.query_ascii().copy()).to(dev), with_rc=True)
    res, _, _ = sfe.ydrop_batch(tp[:2], len(w.target), qp, len(w.query), B._dev(B.make_pairs(w.pairs), dev), len(w.pairs),
                                B._dev(B.make_anchors(w.anchors), dev), n, sc, B.SCORE_ONLY)
    torch.cuda.synchronize()
    out = dict(results=B.results_to_numpy(res, n))
    assert not (out["results"]["status"] & np.uint32(B.ST_BAD_ANCHOR)).any()
    H.assert_anchors_equal(out, w, range(n), want_cigar=False, ydrop=2000)
    passed = out["results"]["score"] >= 3000
    assert 0.5 * w.meta["n_true"] < int(passed.sum()) <= w.meta["n_true"] + 5      # 70 %-identity segments: most true hits pass, false ones do not
    # the budget binds: no extension leaves its box
    r = out["results"]; P = w.pairs
    assert (r["tstart"] >= P[:, 0]).all() and (r["tend"] <= P[:, 1]).all()
