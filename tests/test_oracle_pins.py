"""Pins for the CPU oracle (oracle/sfe_oracle.c): SURVEY.md 8(c) P1..P7.

The paper prints no worked example, so the oracle is pinned to (P1) hand-worked examples
(stored under tests/golden with their citation), (P2) ydrop = infinity
against an independent brute-force Gotoh DP, (P3) closed forms, (P4) CIGAR rescoring and the
other invariants, (P5) upper bounds, (P6, P7) resolver order examples and Alg. 1 == Alg. 3.
None of these runs the CUDA path.
"""
import os

import numpy as np
import pytest

from paper_2606_06811_b200 import workloads as W

GOLD = os.path.join(os.path.dirname(__file__), "golden")
MM = ((10, -10, -10, -10), (-10, 10, -10, -10), (-10, -10, 10, -10), (-10, -10, -10, 10))


def _rows(name):
    with open(os.path.join(GOLD, name)) as f:
        return [ln.split() for ln in f if ln.strip() and not ln.startswith("#")]


@pytest.mark.parametrize("row", _rows("appendix_a_onesided.txt"), ids=lambda r: r[0])
def test_p1_onesided_examples(oracle, row):
    cid, q, t, ydrop, lag, score, ei, ej, cigar, cells = row
    kw = dict(ydrop=int(ydrop), prune_lag=int(lag))
    if cid == "A12":
        kw.update(sub=MM, gap_open=20, gap_extend=5)
    h = oracle.ext_onesided(oracle.codes(q), oracle.codes(t), oracle.scoring(**kw))
    assert (h.score, h.end_i, h.end_j) == (int(score), int(ei), int(ej))
    assert h.cigar == ("" if cigar == "-" else cigar)
    if int(cells) >= 0:
        assert h.cells == int(cells)


@pytest.mark.parametrize("row", _rows("appendix_a_twosided.txt"), ids=lambda r: r[0])
def test_p1_twosided_examples(oracle, row):
    cid, tpos, qpos, score, sb, sf, ops, nback, ts, te, qs, qe = row
    T = oracle.codes("ACGTACGTTTGGCCAGTCAT"); Q = oracle.codes("ACGTACGTGGCCAGTCAT")
    r, got = oracle.extend_anchor(T, Q, int(tpos), int(qpos), oracle.scoring(prune_lag=0))
    assert (r.score, r.score_bwd, r.score_fwd) == (int(score), int(sb), int(sf))
    assert (r.tstart, r.tend, r.qstart, r.qend) == (int(ts), int(te), int(qs), int(qe))
    back, fwd = ops.split("+")
    assert oracle.cigar_str(got[:r.n_ops_back]) == back and oracle.cigar_str(got[r.n_ops_back:]) == fwd
    assert r.n_ops_back == int(nback)


def _a15():
    """T = randseq(1, 600); Q = T with 200..202 deleted, p % 37 == 5
    replaced by the next letter, GATTACA inserted after index 400."""
    T = W.randseq(1, 600)
    out = []
    for p in range(600):
        if 200 <= p <= 202:
            continue
        b = int(T[p])
        out.append((b + 1) % 4 if p % 37 == 5 else b)
        if p == 400:
            out.extend([2, 0, 3, 3, 0, 1, 0])                 # GATTACA
    return T, np.array(out, dtype=np.uint8)


def test_p1_a15_medium(oracle):
    T, Q = _a15()
    assert len(Q) == 604
    for lag, ydrop, cf, cb in ((0, 9400, 142127, 9879), (32, 9400, 164238, 10200), (0, 1500, 22928, 3977)):
        sc = oracle.scoring(prune_lag=lag, ydrop=ydrop)
        r, ops = oracle.extend_anchor(T, Q, 100, 100, sc)
        assert (r.score_fwd, r.score_bwd, r.score) == (43349, 8917, 52266)
        assert oracle.cigar_str(ops[r.n_ops_back:]) == "98M3D200M7I199M"
        assert oracle.cigar_str(ops[:r.n_ops_back]) == "100M"
        assert (r.tstart, r.tend, r.qstart, r.qend) == (0, 600, 0, 604)
        assert (r.cells_fwd, r.cells_bwd) == (cf, cb)


def test_p1_a17_overrun(oracle):
    """A17: 300-bp identical core followed by unrelated random tails."""
    core = W.randseq(7, 300)
    T = np.concatenate([core, W.randseq(8, 1500)]); Q = np.concatenate([core, W.randseq(9, 1500)])
    for lag, cells in ((0, 562409), (1, 563345), (32, 598524)):
        h = oracle.ext_onesided(Q, T, oracle.scoring(prune_lag=lag))
        assert (h.score, h.end_i, h.end_j, h.cigar) == (28831, 301, 301, "301M")
        assert h.cells == cells
        if lag == 0:
            assert (h.rows, h.max_width) == (1186, 651)


def test_p2_ydrop_inf_equals_bruteforce(oracle):
    """R27: with pruning off, score and end cell equal the textbook Gotoh DP (first max)."""
    rng = np.random.default_rng(12345)
    for trial in range(3000):
        n, m = rng.integers(0, 13, 2)
        alpha = 5 if trial % 3 == 0 else 4          # include N sometimes
        q = rng.integers(0, alpha, n).astype(np.uint8); t = rng.integers(0, alpha, m).astype(np.uint8)
        if trial % 2:                                # make them related so gaps/matches matter
            t = np.resize(q, m).astype(np.uint8) if n else t
            if m:
                t[rng.integers(0, m)] = rng.integers(0, 4)
        go, ge = (400, 30) if trial % 4 else (int(rng.integers(0, 60)) + 1, int(rng.integers(1, 20)))
        for lag in (0, 32):
            sc = oracle.scoring(ydrop=oracle.YDROP_INF, prune_lag=lag, gap_open=go, gap_extend=ge)
            h = oracle.ext_onesided(q, t, sc, want_ops=False)
            assert (h.score, h.end_i, h.end_j) == oracle.gotoh_bruteforce(q, t, sc)
            assert h.cells == (n + 1) * (m + 1)


def test_p3_closed_forms(oracle):
    sc = oracle.scoring()
    for L in (1, 7, 100, 333):
        at = np.array([0, 3] * L, dtype=np.uint8)[:L]; cg = np.array([1, 2] * L, dtype=np.uint8)[:L]
        h = oracle.ext_onesided(at, at, sc); assert (h.score, h.cigar) == (91 * L, f"{L}M")
        h = oracle.ext_onesided(cg, cg, sc); assert (h.score, h.cigar) == (100 * L, f"{L}M")
    # one substitution: subtract s(x,x) - s(x,y)
    a = W.randseq(3, 200); b = a.copy(); b[77] = (b[77] + 1) % 4
    full = sum(oracle.HOXD70[int(x)][int(x)] for x in a)
    h = oracle.ext_onesided(a, b, sc)
    assert h.score == full - oracle.HOXD70[int(a[77])][int(a[77])] + oracle.HOXD70[int(a[77])][int(b[77])]
    # Y < O + X  => gap-free => 1-D X-drop scan along the main diagonal (lag 0 semantics)
    rng = np.random.default_rng(7)
    for _ in range(200):
        n = int(rng.integers(1, 60))
        q = rng.integers(0, 4, n).astype(np.uint8); t = q.copy()
        flips = rng.random(n) < 0.3
        t[flips] = (t[flips] + 1 + rng.integers(0, 3, flips.sum())) % 4
        Y = int(rng.integers(50, 430))
        h = oracle.ext_onesided(q, t, oracle.scoring(ydrop=Y, prune_lag=0))
        s = best = bi = 0
        for k in range(n):
            s += oracle.HOXD70[int(q[k])][int(t[k])]
            if s < best - Y:
                break
            if s > best:
                best, bi = s, k + 1
        assert (h.score, h.end_i, h.end_j) == (best, bi, bi)
        assert h.cigar == (f"{bi}M" if bi else "")
    # lag >= n: the threshold is the constant -Y, so lag n and lag 10 n agree
    q = W.randseq(11, 80); t = W.randseq(12, 90)
    h1 = oracle.ext_onesided(q, t, oracle.scoring(prune_lag=81, ydrop=2000))
    h2 = oracle.ext_onesided(q, t, oracle.scoring(prune_lag=800, ydrop=2000))
    assert (h1.score, h1.cells, h1.cigar) == (h2.score, h2.cells, h2.cigar)


def _mutated_pair(seed, n, p_sub, p_indel):
    src = W.randseq(seed, n)
    mu = W.mutate(src, p_sub, p_indel, W.Stream(seed + 1000))
    return src, mu.seq


@pytest.mark.parametrize("lag", [0, 1, 32])
def test_p4_invariants(oracle, lag):
    """Rescoring reproduces the score; score >= 0; first max; halves sum; ops consume the box."""
    for seed, (ps, pi), ydrop in ((21, (0.05, 0.01), 9400), (22, (0.3, 0.02), 9400), (23, (0.1, 0.05), 1500),
                                  (24, (0.02, 0.002), 600)):
        T, Qm = _mutated_pair(seed, 700, ps, pi)
        T = np.concatenate([W.randseq(seed + 50, 300), T, W.randseq(seed + 51, 300)])
        Q = np.concatenate([W.randseq(seed + 60, 250), Qm, W.randseq(seed + 61, 250)])
        if seed == 22:
            Q[400:403] = 4                       # a few N
        sc = oracle.scoring(prune_lag=lag, ydrop=ydrop)
        tpos, qpos = 300 + 350, 250 + 350
        r, ops = oracle.extend_anchor(T, Q, tpos, qpos, sc)
        assert r.score == r.score_fwd + r.score_bwd and r.score_fwd >= 0 and r.score_bwd >= 0
        fwd = ops[r.n_ops_back:]; back = ops[:r.n_ops_back]
        s, qu, tu = oracle.rescore(Q[qpos:], T[tpos:], fwd, sc)
        assert (s, qu, tu) == (r.score_fwd, r.qend - qpos, r.tend - tpos)
        # the backward half, in its own (reversed) frame, is the reversed op list
        s, qu, tu = oracle.rescore(Q[:qpos][::-1], T[:tpos][::-1], back[::-1], sc)
        assert (s, qu, tu) == (r.score_bwd, qpos - r.qstart, tpos - r.tstart)
        for half in (fwd, back[::-1]):
            if half:
                assert half[-1][1] == oracle.OP_M        # far end is an aligned pair
                assert all(a[1] != b[1] for a, b in zip(half, half[1:]))
        # one-sided call agrees with the two-sided one
        h = oracle.ext_onesided(Q[qpos:], T[tpos:], sc)
        assert (h.score, h.end_i, h.end_j, h.ops) == (r.score_fwd, r.qend - qpos, r.tend - tpos, fwd)


def test_p5_upper_bound(oracle):
    rng = np.random.default_rng(99)
    for _ in range(300):
        n, m = rng.integers(1, 40, 2)
        q = rng.integers(0, 4, n).astype(np.uint8)
        t = np.resize(q, m).astype(np.uint8)
        t[rng.random(m) < 0.2] = rng.integers(0, 4)
        bf = oracle.gotoh_bruteforce(q, t, oracle.scoring())[0]
        for lag in (0, 1, 32):
            for Y in (100, 500, 2000):
                h = oracle.ext_onesided(q, t, oracle.scoring(ydrop=Y, prune_lag=lag), want_ops=False)
                assert 0 <= h.score <= bf


def test_p6_resolver_order_examples(oracle):
    """A19 / A20: the kept set depends on anchor order by design."""
    T = oracle.codes("ACGTACGTTTGGCCAGTCAT"); Q = oracle.codes("ACGTACGTGGCCAGTCAT")
    sc = oracle.scoring(prune_lag=0, min_score=500)
    pairs = [(0, 20, 0, 18)]
    r = oracle.serial_loop(T, Q, W.revcomp(Q), pairs, [(14, 12, 0, 1), (10, 10, 0, 1), (3, 5, 0, 1)], sc)
    assert list(r["state"]) == [1, 0, 0] and r["n_extended"] == 1 and r["results"][0].score == 1268
    r = oracle.serial_loop(T, Q, W.revcomp(Q), pairs, [(10, 10, 0, 1), (14, 12, 0, 1)], sc)
    assert list(r["state"]) == [1, 0] and r["results"][0].score == 840
    # strand separates containment (R15, R17)
    r = oracle.serial_loop(T, Q, W.revcomp(Q), pairs, [(10, 10, 0, 1), (10, 10, 0, -1)], sc)
    assert r["state"][0] == 1 and r["state"][1] != 0


def test_p6_config1_keeps_64(oracle):
    w = W.config1()
    r = oracle.serial_loop(w.target, w.query, w.query_rc, w.pairs, w.anchors, oracle.scoring(), want_results=False)
    assert len(w.anchors) == 256 and r["n_kept"] == 64 and r["n_extended"] == 64


def test_p7_speculative_equals_serial(oracle):
    """Alg. 3 keeps exactly what Alg. 1 keeps, for every window K."""
    w = W.config1(n_segments=6, seg_len=400, slot=900, per_seg=5)
    w2 = W.config2(t_len=60_000, n_segments=40, per_seg=6, n_decoys=60, min_len=100, max_len=600)
    for wl in (w, w2):
        sc = oracle.scoring()
        ser = oracle.serial_loop(wl.target, wl.query, wl.query_rc, wl.pairs, wl.anchors, sc)
        assert ser["n_kept"] > 0
        for K in (1, 2, 7, 64, len(wl.anchors)):
            sp = oracle.speculative_loop(wl.target, wl.query, wl.query_rc, wl.pairs, wl.anchors, sc, K)
            assert (sp["state"] == 1).tolist() == (ser["state"] == 1).tolist()
            assert sp["n_extended"] >= ser["n_extended"]
            if K == 1:
                assert sp["n_extended"] == ser["n_extended"] and (sp["state"] == ser["state"]).all()
        # resolve-only on the all-at-once extensions gives the same kept set, and the covered /
        # below split of the serial loop
        scores, boxes = [], []
        for a in wl.anchors:
            Qs = wl.query if a[3] > 0 else wl.query_rc
            r, _ = oracle.extend_anchor(wl.target, Qs, int(a[0]), int(a[1]), sc, want_ops=False)
            scores.append(r.score); boxes.append((r.tstart, r.tend, r.qstart, r.qend))
        st, acc = oracle.resolve(wl.anchors, scores, boxes, sc.min_score)
        assert st.tolist() == ser["state"].tolist() and len(acc) == ser["n_kept"]


def test_pack_mapping(oracle):
    """R13: 2-bit plane + N mask + reverse-complement planes, checked against the definition."""
    s = "ACGTNacgtnXGGTCA"
    c2, nm, rc2, rnm = oracle.pack(s)
    code = {"A": 0, "C": 1, "G": 2, "T": 3}
    L = len(s)
    for k, ch in enumerate(s):
        isn = ch.upper() not in code
        assert ((nm[k // 8] >> (k % 8)) & 1) == int(isn)
        assert ((c2[k // 4] >> (2 * (k % 4))) & 3) == (0 if isn else code[ch.upper()])
        r = L - 1 - k
        assert ((rnm[r // 8] >> (r % 8)) & 1) == int(isn)
        assert ((rc2[r // 4] >> (2 * (r % 4))) & 3) == (0 if isn else 3 - code[ch.upper()])
    assert oracle.codes(s).tolist() == [0, 1, 2, 3, 4, 0, 1, 2, 3, 4, 4, 2, 2, 3, 1, 0]
    assert oracle.revcomp_codes(oracle.codes("AACGN")).tolist() == [4, 1, 2, 3, 3]
