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
    """R27: with pruning off, score and end cell equal the textbook Gotoh DP (first max).  SURVEY P2: random pairs
    <= 12 x 12, >= 10^5 trials (100,000 here; each at lag 0, every 8th also at lag 32)."""
    rng = np.random.default_rng(12345)
    N = 100_000
    nm = rng.integers(0, 13, (N, 2)); seqs = rng.integers(0, 5, (N, 2, 12)).astype(np.uint8); aux = rng.integers(0, 1 << 30, (N, 4))
    for trial in range(N):
        n, m = int(nm[trial, 0]), int(nm[trial, 1])
        q = seqs[trial, 0, :n].copy(); t = seqs[trial, 1, :m].copy()
        if trial % 3:                                # N only sometimes
            q[q == 4] = 0; t[t == 4] = 1
        if trial % 2:                                # make them related so gaps/matches matter
            t = np.resize(q, m).astype(np.uint8) if n else t
            if m:
                t[aux[trial, 0] % m] = aux[trial, 1] % 4
        go, ge = (400, 30) if trial % 4 else (int(aux[trial, 2] % 60), int(aux[trial, 3] % 19) + 1)
        bf = None
        for lag in ((0, 32) if trial % 8 == 0 else (0,)):
            sc = oracle.scoring(ydrop=oracle.YDROP_INF, prune_lag=lag, gap_open=go, gap_extend=ge)
            if bf is None:
                bf = oracle.gotoh_bruteforce(q, t, sc)
            h = oracle.ext_onesided(q, t, sc, want_ops=False)
            assert (h.score, h.end_i, h.end_j) == bf, (trial, q, t, go, ge)
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


def _gotoh_const_threshold(q, t, sub, n_score, O, X, thr):
    """Independent textbook Gotoh over the whole rectangle in which a cell is dead iff it has no alive predecessor
    or H < thr (a CONSTANT), dead cells feeding nothing.  Returns (best, end_i, end_j, cells, H, alive) with
    cells = sum over rows of (last alive - first alive + 1); thr = None disables the threshold."""
    NEG = -(1 << 40)
    n, m = len(q), len(t)
    H = np.full((n + 1, m + 1), NEG, np.int64); E = H.copy(); F = H.copy(); A = np.zeros((n + 1, m + 1), bool)
    H[0, 0] = 0; A[0, 0] = True
    best = (0, 0, 0)
    for i in range(n + 1):
        for j in range(m + 1):
            if i == 0 and j == 0:
                continue
            e = f = d = NEG
            if i and A[i - 1, j]:
                e = max(H[i - 1, j] - O - X, E[i - 1, j] - X)
            if j and A[i, j - 1]:
                f = max(H[i, j - 1] - O - X, F[i, j - 1] - X)
            if i and j and A[i - 1, j - 1]:
                a, b = int(q[i - 1]), int(t[j - 1])
                d = H[i - 1, j - 1] + (n_score if a > 3 or b > 3 else sub[a][b])
            h = max(d, e, f)
            E[i, j] = e; F[i, j] = f; H[i, j] = h
            if h > NEG // 2 and (thr is None or h >= thr):
                A[i, j] = True
                if h > best[0]:
                    best = (int(h), i, j)
    cells = 0
    for i in range(n + 1):
        c = np.nonzero(A[i])[0]
        if len(c):
            cells += int(c[-1] - c[0] + 1)
    return best + (cells, H, A)


def test_p3_lag_beyond_rows_is_constant_threshold(oracle):
    """R4 closed form: with lag > n no row ever sees a best, so T is the constant -Y: the result equals the plain
    Gotoh DP in which cells below -Y (and their descendants through dead-only routes) do not exist."""
    rng = np.random.default_rng(4242)
    for trial in range(150):
        n, m = (int(x) for x in rng.integers(1, 28, 2))
        q = rng.integers(0, 4, n).astype(np.uint8)
        t = np.resize(q, m).astype(np.uint8); t[rng.random(m) < 0.35] = rng.integers(0, 4)
        if trial % 3 == 0:
            t = rng.integers(0, 4, m).astype(np.uint8)
        Y = int(rng.choice([150, 450, 700, 1500]))
        ref = _gotoh_const_threshold(q, t, oracle.HOXD70, -100, 400, 30, -Y)
        for lag in (n + 1, 10 * n + 7):
            h = oracle.ext_onesided(q, t, oracle.scoring(prune_lag=lag, ydrop=Y), want_ops=False)
            assert (h.score, h.end_i, h.end_j, h.cells) == ref[:4], (trial, lag)


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


def test_p5_cellwise_bound_and_unpruned_equality(oracle):
    """SURVEY P5 on small inputs, cell by cell (through the oracle's inspection entry point): every ALIVE cell's H is
    <= its unpruned Gotoh value for any finite (Y, lag); with ydrop = infinity every cell equals it (R27) -- the
    unpruned table comes from the independent numpy DP above, not from the oracle."""
    rng = np.random.default_rng(31337)
    for trial in range(120):
        n, m = (int(x) for x in rng.integers(1, 22, 2))
        q = rng.integers(0, 5 if trial % 4 == 0 else 4, n).astype(np.uint8)
        t = np.resize(q, m).astype(np.uint8); t[rng.random(m) < 0.25] = rng.integers(0, 4)
        go, ge = ((400, 30), (0, 5), (37, 11))[trial % 3]
        sub = oracle.HOXD70 if trial % 2 else MM
        ref = _gotoh_const_threshold(q, t, sub, -100, go, ge, None)
        Href = ref[4]
        for lag in (0, 1, 32):
            sc = oracle.scoring(sub=sub, gap_open=go, gap_extend=ge, ydrop=oracle.YDROP_INF, prune_lag=lag)
            h, H, A = oracle.ext_onesided_cells(q, t, sc)
            assert A.all() and (H.astype(np.int64) == Href).all(), (trial, lag)
            assert (h.score, h.end_i, h.end_j) == ref[:3]
            for Y in (60, 300, 1200):
                sc = oracle.scoring(sub=sub, gap_open=go, gap_extend=ge, ydrop=Y, prune_lag=lag)
                h, H, A = oracle.ext_onesided_cells(q, t, sc)
                al = A.astype(bool)
                assert al[0, 0] and (H.astype(np.int64)[al] <= Href[al]).all(), (trial, lag, Y)
                assert h.score == int(H[al].max()) and 0 <= h.score <= ref[0]
                assert h.cells == sum(int(c[-1] - c[0] + 1) for c in (np.nonzero(r)[0] for r in al) if len(c))


@pytest.mark.parametrize("row", _rows("tiebreak_examples.txt"), ids=lambda r: r[0])
def test_p1_tiebreak_examples(oracle, row):
    """R11: E opens on ties, F opens on ties, H-source priority E over F (hand-worked)."""
    cid, q, t, score, ei, ej, cigar, wrong = row
    sc = oracle.scoring(sub=MM, gap_open=0, gap_extend=5, ydrop=1000, prune_lag=0)
    h = oracle.ext_onesided(oracle.codes(q), oracle.codes(t), sc)
    assert (h.score, h.end_i, h.end_j, h.cigar) == (int(score), int(ei), int(ej), cigar)
    assert cigar != wrong
    # both candidate CIGARs are optimal alignments (the rule picks among equals): rescoring gives the same score
    for c in (cigar, wrong):
        import re
        ops = [(int(a), "MID".index(b)) for a, b in re.findall(r"(\d+)([MID])", c)]
        assert oracle.rescore(oracle.codes(q), oracle.codes(t), ops, sc) == (int(score), len(q), len(t))


def test_r17_closed_box_edges(oracle):
    """R17: containment is a point-in-closed-box test on all four edges, same strand (tests/golden/resolver_edges.txt)."""
    with open(os.path.join(GOLD, "resolver_edges.txt")) as f:
        rows = [ln.split()[:4] for ln in f if ln.strip() and not ln.startswith("#")]
    anchors = [(10, 10, 0, 1)] + [(int(r[0]), int(r[1]), 0, int(r[2])) for r in rows]
    scores = [5000] + [100] * len(rows)
    boxes = [(5, 15, 6, 14)] + [(a[0], a[0], a[1], a[1]) for a in anchors[1:]]
    state, acc = oracle.resolve(anchors, scores, boxes, 3000)
    assert state[0] == 1 and acc == [(5, 15, 6, 14, 1)]
    assert state[1:].tolist() == [int(r[3]) for r in rows]
    # the same edges as boxes carried in from an earlier window (R26)
    state2, _ = oracle.resolve(anchors[1:], scores[1:], boxes[1:], 3000, accepted=[(5, 15, 6, 14, 1)])
    assert state2.tolist() == [int(r[3]) for r in rows]
    # through Algorithm 1 itself on the Appendix-A pair: the first anchor's alignment (1268) has box [0,20] x [0,18];
    # anchors exactly on its corners are covered and never extended (with an open interval they would be kept:
    # the whole alignment is reachable from either corner)
    T = oracle.codes("ACGTACGTTTGGCCAGTCAT"); Q = oracle.codes("ACGTACGTGGCCAGTCAT")
    sc = oracle.scoring(prune_lag=0, min_score=500)
    r = oracle.serial_loop(T, Q, W.revcomp(Q), [(0, 20, 0, 18)], [(14, 12, 0, 1), (20, 18, 0, 1), (0, 0, 0, 1), (20, 0, 0, 1)], sc)
    assert list(r["state"]) == [1, 0, 0, 0] and r["n_extended"] == 1
    for K in (1, 2, 4):
        sp = oracle.speculative_loop(T, Q, W.revcomp(Q), [(0, 20, 0, 18)], [(14, 12, 0, 1), (20, 18, 0, 1), (0, 0, 0, 1), (20, 0, 0, 1)], sc, K)
        assert list(sp["state"]) == [1, 0, 0, 0]


def test_r15_minus_strand_subrange_pair(oracle):
    """R15 / R9: for a - strand anchor the pair's query interval [q_begin, q_end) is mirrored into the reverse-
    complement frame, [q_len - q_end, q_len - q_begin); the target interval is not.  Qrc = T (Q = revcomp(T)), so an
    anchor on the main diagonal extends as pure matches until a LIMIT stops it: score = sum of s(x,x) over the bases
    inside the limits (closed form), CIGAR kM + kM, box = the limits.  A pair whose mirror is not the identity."""
    T = W.randseq(77, 40); Q = W.revcomp(T)
    assert (W.revcomp(Q) == T).all()
    diag = lambda lo, hi: sum(oracle.HOXD70[int(x)][int(x)] for x in T[lo:hi])
    sc = oracle.scoring(min_score=0)
    # (pair, anchor, limits that apply in the rc frame)
    cases = [((0, 40, 10, 26), (20, 20), (0, 40, 14, 30)),        # query interval mirrored: [40-26, 40-10) = [14, 30)
             ((0, 40, 0, 9), (33, 33), (0, 40, 31, 40)),          # [31, 40): touches the end of the rc frame
             ((16, 27, 10, 26), (20, 20), (16, 27, 14, 30)),      # target limits bite first (not mirrored)
             ((0, 40, 12, 12 + 1), (27, 27), (0, 40, 27, 28))]    # one-base interval [27, 28)
    for pair, (tp, qp), (tb, te, qb, qe) in cases:
        lo = max(tb - tp, qb - qp); hi = min(te - tp, qe - qp)           # diagonal run inside the limits, relative to the anchor
        r = oracle.serial_loop(T, Q, T.copy(), [pair], [(tp, qp, 0, -1)], sc)
        res = r["results"][0]
        assert r["state"][0] == 1
        assert (res.score_bwd, res.score_fwd) == (diag(tp + lo, tp), diag(tp, tp + hi)), (pair, res.score_bwd, res.score_fwd)
        assert (res.tstart, res.tend, res.qstart, res.qend) == (tp + lo, tp + hi, qp + lo, qp + hi)
        # the same through the two-sided entry point with explicit rc-frame limits, incl. the CIGAR
        r2, ops = oracle.extend_anchor(T, T, tp, qp, sc, t_lim=(tb, te), q_lim=(qb, qe))
        assert r2.score == res.score and oracle.cigar_str(ops) == (f"{-lo}M" if lo else "") + (f"{hi}M" if hi else "")
    # + strand control: the interval is used as given
    r = oracle.serial_loop(T, T.copy(), W.revcomp(T), [(0, 40, 10, 26)], [(20, 20, 0, 1)], sc)
    res = r["results"][0]
    assert (res.qstart, res.qend, res.score) == (10, 26, diag(10, 26))


def test_r3_substitution_matrix_orientation(oracle):
    """R3 / R13: sub[a][b] is indexed [query base][target base] (HOXD70 is symmetric, so only an asymmetric matrix can
    tell).  s(A over C) = +7, s(C over A) = -50, matches +10: q = A, t = C scores 7 with 1M; q = C, t = A scores nothing.
    q = AC vs t = CC: (1,1) = s(A,C) = 7, (2,2) = 7 + s(C,C) = 17 -> 2M, 17."""
    sub = [[10, 7, -50, -50], [-50, 10, -50, -50], [-50, -50, 10, -50], [-50, -50, -50, 10]]
    sc = oracle.scoring(sub=sub, gap_open=20, gap_extend=5, ydrop=1000, prune_lag=0)
    h = oracle.ext_onesided(oracle.codes("A"), oracle.codes("C"), sc); assert (h.score, h.cigar) == (7, "1M")
    h = oracle.ext_onesided(oracle.codes("C"), oracle.codes("A"), sc); assert (h.score, h.cigar) == (0, "")
    h = oracle.ext_onesided(oracle.codes("AC"), oracle.codes("CC"), sc); assert (h.score, h.end_i, h.end_j, h.cigar) == (17, 2, 2, "2M")
    ops = [(2, oracle.OP_M)]
    assert oracle.rescore(oracle.codes("AC"), oracle.codes("CC"), ops, sc)[0] == 17
    assert oracle.gotoh_bruteforce(oracle.codes("AC"), oracle.codes("CC"), oracle.scoring(sub=sub, gap_open=20, gap_extend=5))[0] == 17


def test_r16_tau_is_inclusive(oracle):
    """PAPER.md:62 / 143: Score(a) >= tau commits.  The Appendix-A alignment scores exactly 1268: tau = 1268 keeps it
    (and it masks the second anchor), tau = 1269 does not (state 2, masks nothing: R18), in Alg. 1, Alg. 3 and resolve."""
    T = oracle.codes("ACGTACGTTTGGCCAGTCAT"); Q = oracle.codes("ACGTACGTGGCCAGTCAT")
    A = [(14, 12, 0, 1), (10, 10, 0, 1)]
    for tau, exp in ((1268, [1, 0]), (1269, [2, 2])):
        sc = oracle.scoring(prune_lag=0, min_score=tau)
        assert list(oracle.serial_loop(T, Q, W.revcomp(Q), [(0, 20, 0, 18)], A, sc)["state"]) == exp
        for K in (1, 2):
            assert list(oracle.speculative_loop(T, Q, W.revcomp(Q), [(0, 20, 0, 18)], A, sc, K)["state"]) == exp
        st, _ = oracle.resolve(A, [1268, 840], [(0, 20, 0, 18), (0, 20, 0, 18)], tau)
        assert st.tolist() == exp


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
