"""-m gpu parity tests at BASELINE.json's full sizes, in the launch configuration bench.py times.

The oracle cannot run 10^10..10^12 cells, so at full size the CUDA path is checked
  (a) on sampled outputs the oracle computes one by one: a seeded sample of anchors plus the largest
      extensions (score, halves, box, cell count, CIGAR: bit-exact);
  (b) by properties that hold at any size and need neither side's code: every emitted CIGAR, rescored
      against the sequences with the R12 rule, reproduces the reported score and consumes exactly
      the box; the keep flags satisfy the in-order containment rule (R17/R18) given the reported
      boxes; the counters add up.
C1 is covered in full by test_gpu_parity.py.  C5 runs at 1/10 scale and at full size (100 Mbp, 1,000,000 anchors;
~90 s of GPU time per pass)."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2606_06811_b200 import binding as B, workloads as W  # noqa: E402

import gpu_harness as H  # noqa: E402

TAU = 3000
SUB = np.array(B.HOXD70, np.int64)


@pytest.fixture(scope="module")
def sfe_big():
    import __graft_entry__ as entry
    entry.build()
    s = B.Sfe(0, 24 << 30)
    yield s
    s.close()


def check_cigar(w, i, g, cigar):
    """The ops of anchor i rescore to its score and consume exactly its box; the first n_ops_back ops end at the anchor."""
    a = w.anchors[i]
    Q = w.query if a[3] > 0 else w.query_rc
    T = w.target
    n = int(g["n_ops"])
    if n == 0:                                         # both halves empty (R8): score 0, box = the anchor point
        assert int(g["score"]) == 0 and int(g["tstart"]) == int(g["tend"]) == int(a[0]) and int(g["qstart"]) == int(g["qend"]) == int(a[1])
        return
    assert int(g["cigar_off"]) >= 0, (i, int(g["status"]))
    words = cigar[int(g["cigar_off"]): int(g["cigar_off"]) + n].astype(np.int64)
    ln = words >> 4; op = words & 15
    assert ((op >= 0) & (op <= 2)).all() and (ln > 0).all()
    dq = np.where(op != 2, ln, 0); dt = np.where(op != 1, ln, 0)
    q0 = int(g["qstart"]) + np.concatenate([[0], np.cumsum(dq)[:-1]]) if n else np.zeros(0, np.int64)
    t0 = int(g["tstart"]) + np.concatenate([[0], np.cumsum(dt)[:-1]]) if n else np.zeros(0, np.int64)
    assert int(g["qstart"]) + int(dq.sum()) == int(g["qend"]) and int(g["tstart"]) + int(dt.sum()) == int(g["tend"]), i
    nb = int(g["n_ops_back"])
    assert int(g["qstart"]) + int(dq[:nb].sum()) == int(a[1]) and int(g["tstart"]) + int(dt[:nb].sum()) == int(a[0]), i
    score = -int((400 + 30 * ln[op != 0]).sum())
    m = op == 0
    if m.any():
        # expand the M runs into base index arrays
        lens = ln[m]; tot = int(lens.sum())
        starts = np.repeat(np.cumsum(lens) - lens, lens)
        off = np.arange(tot) - starts
        qi = np.repeat(q0[m], lens) + off; ti = np.repeat(t0[m], lens) + off
        qa = Q[qi].astype(np.int64); ta = T[ti].astype(np.int64)
        isn = (qa > 3) | (ta > 3)
        s = np.where(isn, -100, SUB[np.minimum(qa, 3), np.minimum(ta, 3)])
        score += int(s.sum())
    assert score == int(g["score"]), (i, score, int(g["score"]))
    # within a half no two adjacent runs share an op (R12); the junction may repeat one
    same = np.nonzero(op[1:] == op[:-1])[0] + 1
    assert all(int(k) == nb for k in same), (i, same[:4], nb)


def check_resolve_rule(w, res, keep, skipped=None):
    """keep flags vs the rule, from the reported boxes only: kept <=> score >= tau and not inside an earlier kept box
    of the same strand; covered <=> inside one; below <=> neither.  O(n log n + candidates) via the tpos order."""
    A = w.anchors
    n = len(A)
    tpos = A[:, 0]; qpos = A[:, 1]; strand = np.where(A[:, 3] >= 0, 1, -1)
    order = np.argsort(tpos, kind="stable"); ts = tpos[order]
    covered = np.zeros(n, bool)
    for j in np.nonzero(keep == 1)[0]:
        lo = np.searchsorted(ts, res["tstart"][j], "left"); hi = np.searchsorted(ts, res["tend"][j], "right")
        c = order[lo:hi]
        c = c[(c > j) & (strand[c] == strand[j]) & (qpos[c] >= res["qstart"][j]) & (qpos[c] <= res["qend"][j])]
        covered[c] = True
    assert ((keep == 0) == covered).all(), np.nonzero((keep == 0) != covered)[0][:8]
    ext = ~covered if skipped is None else ~skipped
    assert ((keep == 1) == (~covered & (res["score"] >= TAU) & ext)).all()
    assert ((keep == 2) == (~covered & (res["score"] < TAU))).all()
    if skipped is not None:
        assert covered[skipped].all()            # never-extended anchors are covered ones


def sample_indices(res, n, k, seed, mask=None, n_largest=6):
    rng = np.random.default_rng(seed)
    pool = np.arange(n) if mask is None else np.nonzero(mask)[0]
    pick = set(rng.choice(pool, min(k, len(pool)), replace=False).tolist())
    cells = res["cells"].astype(np.int64).copy()
    if mask is not None:
        cells[~mask] = -1
    pick.update(np.argsort(-cells)[:min(n_largest, len(pool))].tolist())     # the largest extensions
    pick.update(np.argsort(cells + (cells < 0) * (1 << 62))[:min(3, len(pool))].tolist())   # and the smallest
    return sorted(pick)


def profile_strata(sfe, n, k_each, seed):
    """Anchors whose halves went through the special schedules of the last batch (sfe_last_half_profile): a reserved
    longest-first ticket run with lane skew 2, a skew-2 attempt that outgrew its window and was re-run with skew 1,
    the wide-band path.  Returns {name: anchor indices} (up to k_each per stratum, seeded)."""
    prof = sfe.last_half_profile(2 * n)
    rng = np.random.default_rng(seed)
    out = {}
    for name, bit in (("skew2", B.ST_SKEW2), ("skew_retry", B.ST_SKEW_RETRY), ("wide", B.ST_WIDE)):
        a = np.unique(np.nonzero(prof["status"] & np.uint32(bit))[0] // 2)
        out[name] = sorted(rng.choice(a, min(k_each, len(a)), replace=False).tolist()) if len(a) else []
    return out


def test_config2_full(sfe_big, oracle):
    """configs[1], all 25,000 anchors in one speculative batch + resolve, as bench.py's default run."""
    w = W.config2()
    n = len(w.anchors)
    out = H.gpu_run(sfe_big, w)
    res = out["results"]
    assert not (res["status"] & ~np.uint32(B.ST_WIDE)).any()
    # >= 1 % of the anchors against the oracle (SURVEY 8(d) parity scope), plus every special schedule of this launch
    strata = profile_strata(sfe_big, n, 12, 22)
    assert len(strata["skew2"]) > 0                      # the reserved longest-first tickets ran with skew 2
    pick = sorted(set(sample_indices(res, n, 260, 2)) | {i for v in strata.values() for i in v})
    assert len(pick) >= n // 100
    H.assert_anchors_equal(out, w, pick)
    check_resolve_rule(w, res, out["keep"])
    st = out["stats"]
    assert out["info"]["ring_drops"] == 0
    assert int(st["n_anchors"]) == n and int(st["n_kept"]) == int((out["keep"] == 1).sum()) == out["n_accepted"]
    assert int(st["cells_total"]) == int(res["cells"].sum())
    assert int(st["cells_covered"]) == int(res["cells"][out["keep"] == 0].sum())
    for i in np.nonzero(out["keep"] == 1)[0]:
        check_cigar(w, int(i), res[i], out["cigar"])
    for i in np.nonzero(out["keep"] != 1)[0][::50]:
        check_cigar(w, int(i), res[i], out["cigar"])


def test_config4_full(sfe_big, oracle):
    """configs[3], 65,536 independent pairs (forward + backward for every anchor, no subsumption)."""
    w = W.config4()
    n = len(w.anchors)
    out = H.gpu_run(sfe_big, w)
    res = out["results"]
    assert not (res["status"] & ~np.uint32(B.ST_WIDE)).any()
    assert int(out["info"]["halves_rerun"]) == 0           # 24 GiB of recycled arena is enough for ~27 GB of pointers
    strata = profile_strata(sfe_big, n, 12, 44)
    assert len(strata["skew2"]) > 0
    pick = sorted(set(sample_indices(res, n, 660, 4)) | {i for v in strata.values() for i in v})
    assert len(pick) >= n // 100                          # >= 1 % of C4 against the oracle, incl. the 6 longest pairs
    H.assert_anchors_equal(out, w, pick)
    assert int((out["keep"] == 0).sum()) == 0 and ((out["keep"] == 1) == (res["score"] >= TAU)).all()
    check_resolve_rule(w, res, out["keep"])
    for i in range(0, n, 97):
        check_cigar(w, i, res[i], out["cigar"])


LEADERS = B.WANT_CIGAR | B.SPEC_LEADERS          # bench.py's configuration for the dense-anchor workloads (--spec leaders)


def _speculate_full(sfe, w, K, cigar_cap, flags=B.WANT_CIGAR | B.CIGAR_KEPT_ONLY):
    import torch
    dev = sfe.device
    tp = sfe.pack(torch.from_numpy(w.target_ascii().copy()).to(dev), with_rc=False)
    qp = sfe.pack(torch.from_numpy(w.query_ascii().copy()).to(dev), with_rc=True)
    n = len(w.anchors)
    o = sfe.speculate(tp[:2], len(w.target), qp, len(w.query), B._dev(B.make_pairs(w.pairs), dev), len(w.pairs),
                      B._dev(B.make_anchors(w.anchors), dev), n, B.scoring(), K, flags, cigar_cap)
    torch.cuda.synchronize()
    return dict(results=B.results_to_numpy(o["results"], n), keep=o["keep"].cpu().numpy()[:n],
                stats=o["stats"].cpu().numpy().view(B.STATS_DT)[0], n_accepted=int(o["n_accepted"].item()),
                cigar=o["pool"].cpu().numpy().view(np.uint32), cigar_used=int(o["used"].item()))


def _check_speculated(w, out, seed, n_sample, n_kept_sample=0, n_largest=6, kept_only=True):
    """n_sample extended anchors (mostly rejected ones) + n_kept_sample kept ones + the largest, against the oracle."""
    res = out["results"]; keep = out["keep"]; n = len(w.anchors)
    skipped = (res["status"] & B.ST_SKIPPED) != 0
    bad = res["status"] & np.uint32(B.ST_TB_OVERFLOW | B.ST_CIGAR_OVERFLOW | B.ST_INTERNAL | B.ST_BAND_LIMIT | B.ST_BAD_ANCHOR)
    assert not bad[keep == 1].any() and not (bad & np.uint32(B.ST_INTERNAL | B.ST_BAND_LIMIT | B.ST_BAD_ANCHOR)).any()
    check_resolve_rule(w, res, keep, skipped)
    st = out["stats"]
    assert int(st["n_anchors"]) == n and int(st["n_extended"]) == int((~skipped).sum())
    assert int(st["n_kept"]) == int((keep == 1).sum()) == out["n_accepted"]
    assert int(st["cells_total"]) == int(res["cells"][~skipped].sum())
    for i in np.nonzero(keep == 1)[0]:
        check_cigar(w, int(i), res[i], out["cigar"])
    ok = ~skipped & (bad == 0)
    pick = set(sample_indices(res, n, n_sample, seed, ok & (keep != 1), n_largest))
    if n_kept_sample:
        pick |= set(sample_indices(res, n, n_kept_sample, seed + 1, ok & (keep == 1), 2))
    # SFE_CIGAR_KEPT_ONLY: ops exist for the kept anchors only; otherwise for every extended one; score / box / cells always
    H.assert_anchors_equal(out, w, sorted(pick), want_cigar=(lambda i: bool(keep[i] == 1)) if kept_only else True)
    if kept_only:
        assert (res["n_ops"][keep != 1] == 0).all()
    return len(pick)


def test_config3_full_leaders(sfe_big, oracle):
    """configs[2] as bench.py runs it now: predicted leaders (SFE_SPEC_LEADERS), CIGARs while extending, the longest
    tickets on the cooperative row kernel.  Same kept set as the classic windows of the next test."""
    w = W.config3()
    out = _speculate_full(sfe_big, w, 262144, 1 << 26, flags=LEADERS)
    info = sfe_big.last_speculate_info()
    assert _check_speculated(w, out, 3, 2, n_kept_sample=40, n_largest=3, kept_only=False) >= 40
    assert int(out["stats"]["n_extended"]) < 2 * int((out["keep"] == 1).sum()) + 50      # hardly any shadow work
    assert info["batches"] <= 8
    classic = _speculate_full(sfe_big, w, 16384, 1 << 26)
    assert out["keep"].tolist() == classic["keep"].tolist()
    k = out["keep"] == 1
    for f in ("score", "tstart", "tend", "qstart", "qend", "cells", "n_ops", "n_ops_back"):
        assert (out["results"][f][k] == classic["results"][f][k]).all(), f


def test_config3_full_windowed(sfe_big, oracle):
    """configs[2] (10 Mbp, 50,000 dense anchors, extensions of 10^4..10^5 rows) through the classic Algorithm 3 windows:
    K = 16384, score-only windows, CIGARs for the kept anchors from one final traceback batch."""
    w = W.config3()
    out = _speculate_full(sfe_big, w, 16384, 1 << 26)
    assert _check_speculated(w, out, 3, 100, n_kept_sample=20, n_largest=3) >= 120      # >= 100 rejected + >= 20 kept
    assert int((out["keep"] == 0).sum()) > 0.9 * len(w.anchors)        # "most are subsumed under serial order"


def test_config5_scaled_windowed(sfe_big, oracle):
    """configs[4] at 1/10 scale (10 Mbp with N runs and segmental duplications, 100,000 anchors), K = 1024 as bench.py."""
    w = W.config5(t_len=10_000_000, n_anchors=100_000)
    out = _speculate_full(sfe_big, w, 1024, 1 << 26)
    n_ext = int(out["stats"]["n_extended"])
    assert _check_speculated(w, out, 5, max(60, n_ext // 1000), n_kept_sample=20) >= n_ext // 1000    # >= 0.1 % of the extended anchors


def test_config5_scaled_leaders_equals_classic(sfe_big, oracle):
    """configs[4] at 1/10 scale with predicted leaders: the same kept set, and for the kept anchors the same results, as
    the classic windows; here with every ticket on the systolic kernel (block_halves == 0; by default the cooperative row
    kernel takes the longest-predicted tickets, which test_config5_full_leaders and test_config3_full_leaders cover)."""
    w = W.config5(t_len=10_000_000, n_anchors=100_000)
    sfe_big.set_option(B.OPT_ROW_KERNEL_CAP, 0)
    try:
        out = _speculate_full(sfe_big, w, 262144, 1 << 26, flags=LEADERS)
        assert sfe_big.last_batch_info()["block_halves"] == 0
    finally:
        sfe_big.set_option(B.OPT_ROW_KERNEL_CAP, sfe_big.n_sm())
    n_ext = int(out["stats"]["n_extended"])
    assert _check_speculated(w, out, 5, max(40, n_ext // 1000), n_kept_sample=20, kept_only=False) >= n_ext // 1000
    classic = _speculate_full(sfe_big, w, 1024, 1 << 26)
    assert out["keep"].tolist() == classic["keep"].tolist()
    k = out["keep"] == 1
    for f in ("score", "tstart", "tend", "qstart", "qend", "cells", "n_ops", "n_ops_back"):
        assert (out["results"][f][k] == classic["results"][f][k]).all(), f
    assert n_ext < int(classic["stats"]["n_extended"])


def test_config5_full_leaders(sfe_big, oracle):
    """configs[4] at FULL size (100 Mbp, 1,000,000 anchors, N runs, segmental duplications, decoys) as bench.py runs it
    (predicted leaders, one batch of up to 262,144 extensions at a time, CIGARs while extending): resolve rule over all
    anchors, every kept CIGAR rescored, a sample + the largest extensions against the oracle."""
    w = W.config5()
    out = _speculate_full(sfe_big, w, 262144, 1 << 27, flags=LEADERS)
    info = sfe_big.last_speculate_info()
    _check_speculated(w, out, 55, 24, n_kept_sample=12, n_largest=2, kept_only=False)
    assert int((out["keep"] == 1).sum()) > 1000
    assert info["batches"] <= 16 and info["promoted"] > 0
