"""-m gpu randomized parity: many small independent pairs per batch, random scoring (substitution matrix, N score, gap
open / extend incl. open = 0, ydrop from tiny to large), N-rich and degenerate sequences (length 0, 1), anchors at the
ends and in the middle -- the systolic kernel (Lambda = 32) and the block kernel (Lambda = 32 and Lambda = 0), each
bit-exact against the oracle run with the same parameters."""
import numpy as np
import pytest

pytestmark = pytest.mark.gpu

from paper_2606_06811_b200 import binding as B, workloads as W  # noqa: E402

import gpu_harness as H  # noqa: E402


@pytest.fixture(scope="module")
def sfe():
    import __graft_entry__ as entry
    entry.build()
    s = B.Sfe(0, 1 << 30)
    yield s
    s.close()


def _arena(seed, n_pairs, max_len):
    """Independent pairs concatenated in one arena (like config 4), related by substitutions / indels / N runs."""
    rng = np.random.default_rng(seed)
    T, Q, pairs, anchors = [], [], [], []
    tpos = qpos = 0
    for k in range(n_pairs):
        n = int(rng.choice([0, 1, 2, 5, 17, 33, 64, 100, max_len]))
        t = rng.integers(0, 4, n).astype(np.uint8)
        q = t.copy()
        if n:
            sub = rng.random(n) < rng.choice([0.0, 0.05, 0.3])
            q[sub] = (q[sub] + rng.integers(1, 4, int(sub.sum()))) % 4
            if rng.random() < 0.4:
                q[rng.integers(0, n): rng.integers(0, n) + 1] = 4          # N
            if rng.random() < 0.4 and n > 8:
                a = int(rng.integers(1, n - 4)); q = np.delete(q, slice(a, a + int(rng.integers(1, 4))))
            if rng.random() < 0.4 and n > 8:
                a = int(rng.integers(1, n - 4)); t = np.delete(t, slice(a, a + int(rng.integers(1, 4))))
            if rng.random() < 0.2:
                t[rng.integers(0, len(t))] = 4
        pairs.append([tpos, tpos + len(t), qpos, qpos + len(q)])
        lo = min(len(t), len(q))
        for a in {0, lo, lo // 2, int(rng.integers(0, lo + 1))}:
            anchors.append((tpos + a, qpos + min(a, len(q)), k, 1))
        anchors.append((tpos + len(t), qpos + len(q), k, 1))
        T.append(t); Q.append(q); tpos += len(t); qpos += len(q)
    T = np.concatenate(T + [np.zeros(1, np.uint8)]); Q = np.concatenate(Q + [np.zeros(1, np.uint8)])
    A = np.array(sorted(set(anchors)), np.int64)
    return W.Workload("fuzz", T, Q, np.array(pairs, np.int64), A)


def _scoring(seed):
    rng = np.random.default_rng(1000 + seed)
    if seed % 3 == 0:
        sub = B.HOXD70
    else:
        m = rng.integers(-127, 0, (4, 4)); m[np.arange(4), np.arange(4)] = rng.integers(1, 128, 4)
        sub = tuple(tuple(int(x) for x in r) for r in m)
    return dict(sub=sub, n_score=int(rng.integers(-128, 1)), gap_open=int(rng.choice([0, 1, 50, 400, 600])),
                gap_extend=int(rng.choice([1, 2, 30, 60])), ydrop=[1500, 100000, 100, 9400, 300, 0][seed % 6])


@pytest.mark.parametrize("seed", range(6))
def test_fuzz_small_pairs(sfe, oracle, seed):
    w = _arena(seed, 40, 260)
    kw = _scoring(seed)
    n = len(w.anchors)
    for flags, lag in ((B.WANT_CIGAR | B.NO_BLOCK_KERNEL, 32), (B.WANT_CIGAR | B.BLOCK_KERNEL, 32), (B.WANT_CIGAR | B.BLOCK_KERNEL, 0)):
        out = H.gpu_run(sfe, w, flags=flags, prune_lag=lag, **kw)
        for i in range(n):
            H.assert_anchor_equal(out, w, i, prune_lag=lag, **kw)
        H.assert_resolve_equal(out, w, prune_lag=lag, **kw)
