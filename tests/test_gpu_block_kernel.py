"""-m gpu parity tests of the cooperative-warps kernel (ydrop_block_kernel.cu: one CTA per anchor-half, rows in
order, F by a block-wide prefix maximum).  Same oracle, same bar as the systolic kernel: score,
halves, box, cell count and CIGAR bit-exact, on the same inputs, with SFE_BLOCK_KERNEL forcing every half onto it."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2606_06811_b200 import binding as B, workloads as W  # noqa: E402

import gpu_harness as H  # noqa: E402

BLK = B.WANT_CIGAR | B.BLOCK_KERNEL


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


def test_block_appendix_a_examples(sfe, oracle):
    c = oracle.codes
    T = c("ACGTACGTTTGGCCAGTCAT"); Q = c("ACGTACGTGGCCAGTCAT")
    w = _wl(T, Q, [(0, 0, 0, 1), (14, 12, 0, 1), (10, 10, 0, 1), (9, 8, 0, 1), (3, 5, 0, 1), (20, 18, 0, 1), (0, 18, 0, 1)])
    out = H.gpu_run(sfe, w, flags=BLK)
    assert out["info"]["block_halves"] == 2 * len(w.anchors)
    for i in range(len(w.anchors)):
        H.assert_anchor_equal(out, w, i)
    for q, t in (("ACGTACGT", "ACGTACGT"), ("ACGNACGT", "ACGTACGT"), ("AAAA", "CCCC"), ("ACGTTA", "ACGTCA"), ("A", "A"),
                 ("A", "C"), ("ACGT", "A")):
        w = _wl(c(t), c(q), [(0, 0, 0, 1), (len(t), len(q), 0, 1)])
        out = H.gpu_run(sfe, w, flags=BLK)
        H.assert_anchor_equal(out, w, 0); H.assert_anchor_equal(out, w, 1)


@pytest.mark.parametrize("ydrop", [120, 455, 1500, 9400])
def test_block_small_ydrops_and_ties(sfe, oracle, ydrop):
    rng = np.random.default_rng(ydrop)
    T = rng.integers(0, 4, 900).astype(np.uint8)
    mu = W.mutate(T, 0.08, 0.02, W.Stream(ydrop))
    Q = mu.seq.copy()
    Q[100:104] = 4; T[300:302] = 4
    picks = rng.integers(0, len(mu.t_idx), 24)
    anchors = [(int(mu.t_idx[k]), int(mu.q_idx[k]), 0, 1) for k in picks] + [(0, 0, 0, 1), (len(T), len(Q), 0, 1), (5, 700, 0, 1)]
    w = _wl(T, Q, anchors)
    out = H.gpu_run(sfe, w, flags=BLK, ydrop=ydrop)
    for i in range(len(anchors)):
        H.assert_anchor_equal(out, w, i, ydrop=ydrop)


def test_block_ydrop_inf_and_wide(sfe, oracle):
    """ydrop = infinity on a small rectangle; a band wider than the 1024-column window falls back to the wide kernel."""
    rng = np.random.default_rng(3)
    T = rng.integers(0, 4, 150).astype(np.uint8); Q = T.copy(); Q[40] = (Q[40] + 1) % 4
    Q = np.delete(Q, [70, 71])
    w = _wl(T, Q, [(0, 0, 0, 1), (60, 60, 0, 1), (150, 148, 0, 1)])
    out = H.gpu_run(sfe, w, flags=BLK, ydrop=B.YDROP_INF)
    for i in range(3):
        H.assert_anchor_equal(out, w, i, ydrop=B.YDROP_INF)
    T = W.randseq(41, 2600); mu = W.mutate(T, 0.05, 0.01, W.Stream(42)); Q = mu.seq
    k = np.searchsorted(mu.t_idx, [1300, 100])
    w = _wl(T, Q, [(int(mu.t_idx[k[0]]), int(mu.q_idx[k[0]]), 0, 1), (int(mu.t_idx[k[1]]), int(mu.q_idx[k[1]]), 0, 1)])
    out = H.gpu_run(sfe, w, flags=BLK, ydrop=40000)
    assert out["info"]["wide"] >= 2
    for i in range(2):
        H.assert_anchor_equal(out, w, i, ydrop=40000)


def test_block_minus_strand_pairs_and_resolve(sfe, oracle):
    w = W.config2(t_len=80_000, n_segments=40, per_seg=4, n_decoys=40, min_len=100, max_len=700)
    out = H.gpu_run(sfe, w, flags=BLK)
    for i in range(len(w.anchors)):
        H.assert_anchor_equal(out, w, i)
    H.assert_resolve_equal(out, w)
    T = W.randseq(31, 3000); mu = W.mutate(T, 0.03, 0.005, W.Stream(32)); Q = mu.seq
    pairs = [[500, 2500, 480, 2480], [0, 3000, 0, len(Q)], [1000, 1200, 990, 1190]]
    k = np.searchsorted(mu.t_idx, [1100, 1500, 1100])
    anchors = [(int(mu.t_idx[k[0]]), int(mu.q_idx[k[0]]), 0, 1), (int(mu.t_idx[k[1]]), int(mu.q_idx[k[1]]), 1, 1),
               (int(mu.t_idx[k[2]]), int(mu.q_idx[k[2]]), 2, 1), (500, 480, 0, 1), (2500, 2480, 0, 1)]
    w = _wl(T, Q, anchors, pairs)
    out = H.gpu_run(sfe, w, flags=BLK)
    for i in range(len(anchors)):
        H.assert_anchor_equal(out, w, i)


def test_block_config1_full_equals_systolic(sfe, oracle):
    """configs[0] on both kernels: identical results, CIGAR pools and kept sets; the oracle agrees on all 256."""
    w = W.config1()
    a = H.gpu_run(sfe, w, flags=BLK)
    b = H.gpu_run(sfe, w, flags=B.WANT_CIGAR | B.NO_BLOCK_KERNEL)
    assert a["info"]["block_halves"] == 512 and b["info"]["block_halves"] == 0
    assert (a["results"] == b["results"]).all() and a["keep"].tolist() == b["keep"].tolist()
    assert a["cigar_used"] == b["cigar_used"] and (a["cigar"][: a["cigar_used"]] == b["cigar"][: b["cigar_used"]]).all()
    for i in range(len(w.anchors)):
        H.assert_anchor_equal(a, w, i)
    assert int((a["keep"] == 1).sum()) == 64
    s = H.gpu_run(sfe, w, flags=B.SCORE_ONLY | B.BLOCK_KERNEL)
    for f in ("score", "tstart", "tend", "qstart", "qend", "cells"):
        assert (s["results"][f] == a["results"][f]).all()


# ---- f1: exact serial-order pruning (R4 with Lambda = 0) on the GPU ---------------------------------------------------
LAG0 = dict(prune_lag=0)


def test_lag0_order_matters_examples(sfe, oracle):
    """A10 / A11 and A4 / A5 give different alignments under different 'best so far' orders; the
    block kernel at prune_lag = 0 reproduces the serial (row-major) reading: A10 -> 191 (2,2) 2M, A4 -> 100 (1,1) 1M."""
    c = oracle.codes
    w = _wl(c("AGTACTAAAGA"), c("AGCTAAAGA"), [(0, 0, 0, 1)])
    out = H.gpu_run(sfe, w, flags=BLK, ydrop=455, **LAG0)
    g = out["results"][0]
    assert (int(g["score"]), int(g["tend"]), int(g["qend"]), int(g["cells"])) == (191, 2, 2, 19 + 1)   # + the empty backward half's origin cell
    assert B.ops_list(out["cigar"], int(g["cigar_off"]), int(g["n_ops"])) == [(2, 0)]
    H.assert_anchor_equal(out, w, 0, ydrop=455, **LAG0)
    w = _wl(c("CGCC"), c("CCCC"), [(0, 0, 0, 1)])
    out = H.gpu_run(sfe, w, flags=BLK, ydrop=120, **LAG0)
    assert int(out["results"][0]["score"]) == 100 and int(out["results"][0]["tend"]) == 1
    H.assert_anchor_equal(out, w, 0, ydrop=120, **LAG0)
    # and prune_lag = 0 is refused without the block kernel
    with pytest.raises(B.SfeError):
        H.gpu_run(sfe, w, flags=B.WANT_CIGAR, ydrop=120, **LAG0)


@pytest.mark.parametrize("ydrop", [120, 455, 1500, 9400])
def test_lag0_small_ydrops(sfe, oracle, ydrop):
    rng = np.random.default_rng(ydrop + 7)
    T = rng.integers(0, 4, 900).astype(np.uint8)
    mu = W.mutate(T, 0.08, 0.02, W.Stream(ydrop + 7))
    Q = mu.seq.copy()
    Q[100:104] = 4; T[300:302] = 4
    picks = rng.integers(0, len(mu.t_idx), 24)
    anchors = [(int(mu.t_idx[k]), int(mu.q_idx[k]), 0, 1) for k in picks] + [(0, 0, 0, 1), (len(T), len(Q), 0, 1), (5, 700, 0, 1)]
    w = _wl(T, Q, anchors)
    out = H.gpu_run(sfe, w, flags=BLK, ydrop=ydrop, **LAG0)
    for i in range(len(anchors)):
        H.assert_anchor_equal(out, w, i, ydrop=ydrop, **LAG0)


def test_lag0_config2_small_and_fidelity(sfe, oracle):
    """Divergent regime, both strands, at Lambda = 0: bit-exact vs the oracle at Lambda = 0, kept set == Algorithm 1 at
    Lambda = 0; and the R4 fidelity report: how often Lambda = 32 (the systolic kernel) differs from Lambda = 0."""
    w = W.config2(t_len=80_000, n_segments=40, per_seg=4, n_decoys=40, min_len=100, max_len=700)
    out0 = H.gpu_run(sfe, w, flags=BLK, **LAG0)
    for i in range(len(w.anchors)):
        H.assert_anchor_equal(out0, w, i, **LAG0)
    H.assert_resolve_equal(out0, w, **LAG0)
    out32 = H.gpu_run(sfe, w)
    same = sum(int(out0["results"][f][i]) == int(out32["results"][f][i]) for i in range(len(w.anchors)) for f in ("score", "tstart", "tend", "qstart", "qend"))
    assert same >= 0.95 * 5 * len(w.anchors)                      # the two readings rarely differ (SURVEY 8(c) "Why Lambda")
    assert int(out0["results"]["cells"].sum()) <= int(out32["results"]["cells"].sum())   # Lambda = 0 prunes earlier here
