"""Seeded synthetic workload generators (the five BASELINE.json configs).

This module holds NONE of the method's arithmetic (no scoring, no DP, no containment): it
only draws sequences, mutates them and places anchors.  It is the one module both the CUDA
tests/bench and the oracle tests consume, so that both sides see identical bytes.

All randomness is SplitMix64 used as a counter-based generator:
output k of stream `seed` is mix(seed + (k+1) * GAMMA), which vectorises in numpy.
The inputs stand in for the paper's genome pairs (human/mouse, rat/mouse, primates, mm10
chr10 x rn6 chr20), which are not available; the recipes below take
their structure (identity regime, rearrangements, repeats, N runs, anchor density).
"""
from __future__ import annotations

from dataclasses import dataclass, field

import numpy as np

_GAMMA = np.uint64(0x9E3779B97F4A7C15)
_C1 = np.uint64(0xBF58476D1CE4E5B9)
_C2 = np.uint64(0x94D049BB133111EB)
_ASCII = np.frombuffer(b"ACGTN", dtype=np.uint8)
_COMP = np.array([3, 2, 1, 0, 4], dtype=np.uint8)


def splitmix64(seed: int, n: int, offset: int = 0) -> np.ndarray:
    """Outputs offset .. offset+n-1 of the SplitMix64 stream with initial state `seed`."""
    with np.errstate(over="ignore"):
        k = np.arange(offset + 1, offset + n + 1, dtype=np.uint64)
        z = np.uint64(seed & 0xFFFFFFFFFFFFFFFF) + k * _GAMMA
        z = (z ^ (z >> np.uint64(30))) * _C1
        z = (z ^ (z >> np.uint64(27))) * _C2
        return z ^ (z >> np.uint64(31))


class Stream:
    """A consumable SplitMix64 stream."""

    def __init__(self, seed: int):
        self.seed = int(seed)
        self.pos = 0

    def u64(self, n: int) -> np.ndarray:
        out = splitmix64(self.seed, n, self.pos)
        self.pos += n
        return out

    def uniform(self, n: int) -> np.ndarray:
        """float64 in [0, 1) from the top 53 bits."""
        return (self.u64(n) >> np.uint64(11)).astype(np.float64) * (1.0 / (1 << 53))

    def integers(self, lo: int, hi: int, n: int) -> np.ndarray:
        """int64 uniform in [lo, hi) (multiply-shift on the top 32 bits; bias < 2^-32 * range)."""
        r = (self.u64(n) >> np.uint64(32)).astype(np.uint64)
        return (lo + ((r * np.uint64(hi - lo)) >> np.uint64(32)).astype(np.int64))

    def bases(self, n: int) -> np.ndarray:
        """codes 0..3 = top 2 bits of successive outputs (randseq of SURVEY Appendix B)."""
        return (self.u64(n) >> np.uint64(62)).astype(np.uint8)

    def normal(self, n: int) -> np.ndarray:
        u1 = self.uniform(n); u2 = self.uniform(n)
        return np.sqrt(-2.0 * np.log(1.0 - u1)) * np.cos(2.0 * np.pi * u2)

    def permutation(self, n: int) -> np.ndarray:
        return np.argsort(self.u64(n), kind="stable")


def randseq(seed: int, n: int) -> np.ndarray:
    return Stream(seed).bases(n)


def to_ascii(codes: np.ndarray) -> np.ndarray:
    """code array (0..3, 4 = N) -> uint8 array of ASCII characters."""
    return _ASCII[codes]


def revcomp(codes: np.ndarray) -> np.ndarray:
    return _COMP[codes[::-1]]


def stream_seed(config: int, stream_id: int) -> int:
    return config * (1 << 32) + stream_id


@dataclass
class Mutated:
    seq: np.ndarray        # mutated copy (codes)
    t_idx: np.ndarray      # indices k of source bases that are aligned to a copy base
    q_idx: np.ndarray      # position of that base in `seq`


def mutate(src: np.ndarray, p_sub, p_indel, st: Stream, tstv: bool = False, no_indel=None) -> Mutated:
    """Mutation model of SURVEY 8(d): each source base is independently substituted with
    prob. p_sub (uniform over the 3 others, or transition with prob. 2/3 if tstv), or starts
    an indel with prob. p_indel (insertion / deletion with equal probability, length
    geometric p = 0.5, capped at 32).  A deletion of length L removes source bases k..k+L-1;
    an insertion puts L random bases after base k.  Events on deleted bases are ignored.
    p_sub / p_indel may be per-base arrays; no_indel (bool array) forbids indel starts."""
    n = len(src)
    u = st.uniform(n)
    alt = st.u64(n)
    geo = st.u64(n)
    ins_bases_stream = st
    is_sub = u < p_sub
    is_indel = (u >= p_sub) & (u < p_sub + p_indel)
    if no_indel is not None:
        is_indel &= ~no_indel
    is_ins = is_indel & ((alt & np.uint64(1)) == 0)
    is_del = is_indel & ~is_ins
    # geometric length: 1 + number of trailing one-bits of geo (p = 0.5), capped
    ln = np.ones(n, dtype=np.int64)
    run = np.ones(n, dtype=bool)
    for b in range(31):
        run &= ((geo >> np.uint64(b)) & np.uint64(1)) == 1
        if not run.any():
            break
        ln += run
    # substitutions
    out = src.copy()
    r = ((alt >> np.uint64(8)) % np.uint64(3)).astype(np.uint8)
    if tstv:
        # transition (A<->G, C<->T : code ^ 2) with prob 2/3, else one of the 2 transversions
        r6 = ((alt >> np.uint64(8)) % np.uint64(6)).astype(np.uint8)
        ts = r6 < 4
        tv = np.where(r6 == 4, src ^ np.uint8(1), src ^ np.uint8(3))
        sub_base = np.where(ts, src ^ np.uint8(2), tv).astype(np.uint8)
    else:
        sub_base = ((src.astype(np.int64) + 1 + r) % 4).astype(np.uint8)
    valid = src < 4
    out = np.where(is_sub & valid, sub_base, out).astype(np.uint8)
    # deletions: mark [k, k+len) as removed
    dk = np.nonzero(is_del)[0]
    diff = np.zeros(n + 34, dtype=np.int64)
    np.add.at(diff, dk, 1)
    np.add.at(diff, dk + ln[dk], -1)
    deleted = np.cumsum(diff)[:n] > 0
    keep = ~deleted
    ins_len = np.where(is_ins & keep, ln, 0)
    slots = keep.astype(np.int64) + ins_len                     # copy slots produced by source base k
    start = np.cumsum(slots) - slots                             # first slot of base k
    total = int(slots.sum())
    seq = ins_bases_stream.bases(total)                          # inserted bases; aligned ones overwritten
    t_idx = np.nonzero(keep)[0]
    q_idx = start[t_idx]
    seq[q_idx] = out[t_idx]
    return Mutated(seq=seq, t_idx=t_idx.astype(np.int64), q_idx=q_idx.astype(np.int64))


@dataclass
class Workload:
    """One config: code arrays (0..3, 4 = N), pair table, anchors in anchor order."""
    name: str
    target: np.ndarray
    query: np.ndarray
    pairs: np.ndarray                 # int64 [n_pairs, 4] : t_begin, t_end, q_begin, q_end
    anchors: np.ndarray               # int64 [n, 4]       : tpos, qpos (strand frame), pair, strand
    meta: dict = field(default_factory=dict)

    @property
    def query_rc(self) -> np.ndarray:
        return revcomp(self.query)

    def target_ascii(self) -> np.ndarray:
        return to_ascii(self.target)

    def query_ascii(self) -> np.ndarray:
        return to_ascii(self.query)


def _sort_anchors(a: np.ndarray) -> np.ndarray:
    """anchor order = sorted by (tpos, qpos, strand)."""
    order = np.lexsort((a[:, 3], a[:, 1], a[:, 0]))
    return a[order]


# ------------------------------------------------------------------------------------------
# Config 1: tiny high-identity pair (BASELINE.json configs[0])
# ------------------------------------------------------------------------------------------
def config1(n_segments: int = 64, seg_len: int = 2000, slot: int = 3125, per_seg: int = 4) -> Workload:
    """T = n_segments*slot random bases (seed 1); segment s sits at slot s of T; Q = fresh
    random background with the mutated copies (1% substitutions ts:tv 2:1, 0.1% indels) dropped
    into shuffled slots; per_seg anchors per segment on the true path, all + strand."""
    L = n_segments * slot
    T = randseq(1, L)                                           # "seed 1" (BASELINE.json)
    Q = Stream(stream_seed(1, 1)).bases(L)
    perm = Stream(stream_seed(1, 2)).permutation(n_segments)
    pos = Stream(stream_seed(1, 3))
    off = (slot - seg_len) // 2
    anchors = []
    mst = Stream(stream_seed(1, 4))
    for s in range(n_segments):
        t0 = s * slot + off
        mu = mutate(T[t0:t0 + seg_len], 0.01, 0.001, mst, tstv=True)
        q0 = int(perm[s]) * slot + off
        ln = min(len(mu.seq), slot - off)
        Q[q0:q0 + ln] = mu.seq[:ln]
        ok = mu.q_idx < ln
        picks = pos.integers(0, int(ok.sum()), per_seg)
        for k in picks:
            anchors.append((t0 + int(mu.t_idx[k]), q0 + int(mu.q_idx[k]), 0, 1))
    A = _sort_anchors(np.array(anchors, dtype=np.int64))
    pairs = np.array([[0, L, 0, L]], dtype=np.int64)
    return Workload("c1", T, Q, pairs, A, dict(n_segments=n_segments, expect_kept=n_segments))


# ------------------------------------------------------------------------------------------
# Config 2: divergent cross-species regime (configs[1]; C2)
# ------------------------------------------------------------------------------------------
def config2(t_len: int = 2_000_000, n_segments: int = 2000, per_seg: int = 10, n_decoys: int = 5000,
            min_len: int = 100, max_len: int = 800) -> Workload:
    """Segments of length U[min_len, max_len] at 70% identity (30% substitutions, 2% indels),
    one per equal slot of T, copies in shuffled slots of Q, every second segment (after the
    shuffle) reverse-complemented; per_seg anchors per segment with qpos jitter U{-3..3};
    n_decoys anchors at uniform random (tpos, qpos, strand).  - strand anchors are in the
    rc(Q) frame."""
    slot = t_len // n_segments
    assert slot >= max_len + 64
    T = Stream(stream_seed(2, 0)).bases(t_len)
    Q = Stream(stream_seed(2, 1)).bases(t_len)
    perm = Stream(stream_seed(2, 2)).permutation(n_segments)
    lens = Stream(stream_seed(2, 3)).integers(min_len, max_len + 1, n_segments)
    mst = Stream(stream_seed(2, 4))
    pos = Stream(stream_seed(2, 5))
    q_len = t_len
    anchors = []
    for s in range(n_segments):
        ln_t = int(lens[s])
        t0 = s * slot + 16
        mu = mutate(T[t0:t0 + ln_t], 0.30, 0.02, mst)
        q0 = int(perm[s]) * slot + 16
        ln = min(len(mu.seq), slot - 32)
        cp = mu.seq[:ln]
        minus = (s % 2 == 1)
        Q[q0:q0 + ln] = revcomp(cp) if minus else cp
        ok = np.nonzero(mu.q_idx < ln)[0]
        picks = pos.integers(0, len(ok), per_seg)
        jit = pos.integers(-3, 4, per_seg)
        for k, dj in zip(picks, jit):
            tp = t0 + int(mu.t_idx[ok[k]])
            qrel = int(mu.q_idx[ok[k]])
            qp = (q_len - q0 - ln + qrel) if minus else (q0 + qrel)
            qp = min(max(qp + int(dj), 0), q_len)
            anchors.append((tp, qp, 0, -1 if minus else 1))
    dst = Stream(stream_seed(2, 6))
    dt = dst.integers(0, t_len + 1, n_decoys); dq = dst.integers(0, q_len + 1, n_decoys)
    ds = dst.integers(0, 2, n_decoys)
    for a, b, c in zip(dt, dq, ds):
        anchors.append((int(a), int(b), 0, 1 if c else -1))
    A = _sort_anchors(np.array(anchors, dtype=np.int64))
    pairs = np.array([[0, t_len, 0, q_len]], dtype=np.int64)
    return Workload("c2", T, Q, pairs, A, dict(n_segments=n_segments, n_decoys=n_decoys))


def _pick_aligned(mu: Mutated, k: np.ndarray) -> np.ndarray:
    """index into mu.t_idx of the first aligned source base >= k (clipped)."""
    x = np.searchsorted(mu.t_idx, k)
    return np.minimum(x, len(mu.t_idx) - 1)


# ------------------------------------------------------------------------------------------
# Config 4: independent-extension kernel microbenchmark (configs[3]; C4)
# ------------------------------------------------------------------------------------------
def config4(n_pairs: int = 65536, median: int = 1000, sigma: float = 1.0, lo: int = 64, hi: int = 65536,
            chunk_bases: int = 8_000_000) -> Workload:
    """n_pairs independent pairs in one arena; length = clip(round(exp(ln median + sigma z)), lo, hi);
    identity u ~ U[0.75, 0.99] per pair: p_sub = 0.9 (1-u), p_indel = 0.1 (1-u); one anchor per
    pair on the true path at a uniform position in [10%, 90%] of the pair."""
    z = Stream(stream_seed(4, 0)).normal(n_pairs)
    lens = np.clip(np.rint(np.exp(np.log(median) + sigma * z)), lo, hi).astype(np.int64)
    ident = 0.75 + 0.24 * Stream(stream_seed(4, 1)).uniform(n_pairs)
    frac = 0.1 + 0.8 * Stream(stream_seed(4, 2)).uniform(n_pairs)
    t_off = np.concatenate([[0], np.cumsum(lens)])
    tst, mst = Stream(stream_seed(4, 3)), Stream(stream_seed(4, 4))
    T_parts, Q_parts, pairs, anchors = [], [], np.zeros((n_pairs, 4), np.int64), np.zeros((n_pairs, 4), np.int64)
    q_base = 0
    p0 = 0
    while p0 < n_pairs:
        p1 = p0 + 1
        while p1 < n_pairs and t_off[p1 + 1] - t_off[p0] <= chunk_bases:
            p1 += 1
        tb, te = int(t_off[p0]), int(t_off[p1])
        Tc = tst.bases(te - tb)
        pid = np.repeat(np.arange(p0, p1), lens[p0:p1])
        rate = 1.0 - ident[pid]
        rel_end = (t_off[pid + 1] - tb) - np.arange(te - tb)          # bases left in the pair (>= 1)
        mu = mutate(Tc, 0.9 * rate, 0.1 * rate, mst, no_indel=rel_end <= 34)
        # query offset of every pair start: slots before the first base of the pair
        starts = t_off[p0:p1] - tb
        # query start of a pair = first copy slot at or after the pair's first source base
        q_of_t = np.full(te - tb + 1, len(mu.seq), np.int64)
        q_of_t[mu.t_idx] = mu.q_idx
        # running minimum from the right gives "first slot at or after source base k"
        q_start = np.minimum.accumulate(q_of_t[::-1])[::-1]
        qs = q_start[starts]; qe = np.concatenate([qs[1:], [len(mu.seq)]])
        pairs[p0:p1, 0] = t_off[p0:p1]; pairs[p0:p1, 1] = t_off[p0 + 1:p1 + 1]
        pairs[p0:p1, 2] = q_base + qs; pairs[p0:p1, 3] = q_base + qe
        want = starts + (frac[p0:p1] * lens[p0:p1]).astype(np.int64)
        a = _pick_aligned(mu, want)
        anchors[p0:p1, 0] = tb + mu.t_idx[a]; anchors[p0:p1, 1] = q_base + mu.q_idx[a]
        anchors[p0:p1, 2] = np.arange(p0, p1); anchors[p0:p1, 3] = 1
        T_parts.append(Tc); Q_parts.append(mu.seq)
        q_base += len(mu.seq)
        p0 = p1
    T = np.concatenate(T_parts); Q = np.concatenate(Q_parts)
    # clip anchors that fell outside their pair (possible only at a pair's very end)
    anchors[:, 0] = np.clip(anchors[:, 0], pairs[:, 0], pairs[:, 1])
    anchors[:, 1] = np.clip(anchors[:, 1], pairs[:, 2], pairs[:, 3])
    return Workload("c4", T, Q, pairs, anchors, dict(n_pairs=n_pairs, mean_len=float(lens.mean())))


def _blocks_rearranged(Qm_len: int, n_t: int, mu: Mutated, bounds_t: np.ndarray, inverted: np.ndarray,
                       order: np.ndarray):
    """Cut the mutated copy at target coordinates bounds_t (increasing, first 0, last n_t), flip the
    blocks flagged `inverted`, and concatenate blocks in `order`.  Returns (block q start/end in the
    mutated copy, new start of each block in the rearranged query)."""
    q_of_t = np.full(n_t + 1, Qm_len, np.int64)
    q_of_t[mu.t_idx] = mu.q_idx
    q_start = np.minimum.accumulate(q_of_t[::-1])[::-1]
    qb = q_start[bounds_t]
    qb[0] = 0; qb[-1] = Qm_len
    blen = np.diff(qb)
    new_start = np.zeros(len(blen), np.int64)
    pos = 0
    for b in order:
        new_start[b] = pos
        pos += int(blen[b])
    return qb, new_start


def _assemble(Qm: np.ndarray, qb: np.ndarray, new_start: np.ndarray, inverted: np.ndarray) -> np.ndarray:
    Q = np.empty(len(Qm), np.uint8)
    for b in range(len(new_start)):
        blk = Qm[qb[b]:qb[b + 1]]
        Q[new_start[b]:new_start[b] + len(blk)] = revcomp(blk) if inverted[b] else blk
    return Q


def _true_path_anchors(mu: Mutated, picks: np.ndarray, bounds_t: np.ndarray, qb: np.ndarray, new_start: np.ndarray,
                       inverted: np.ndarray, q_len: int) -> np.ndarray:
    """anchors on the true path for aligned-pair indices `picks` (into mu.t_idx)."""
    t = mu.t_idx[picks]; qm = mu.q_idx[picks]
    b = np.searchsorted(bounds_t, t, side="right") - 1
    b = np.clip(b, 0, len(new_start) - 1)
    inside = (qm >= qb[b]) & (qm < qb[b + 1])
    rel = qm - qb[b]
    blen = qb[b + 1] - qb[b]
    q_plus = new_start[b] + rel
    # an inverted block appears, in the rc(Q) frame, in + orientation at q_len - (new_start + blen)
    q_minus = q_len - (new_start[b] + blen) + rel
    inv = inverted[b]
    a = np.stack([t, np.where(inv, q_minus, q_plus), np.zeros_like(t), np.where(inv, -1, 1)], axis=1)
    return a[inside]


# ------------------------------------------------------------------------------------------
# Config 3: high-identity primate-like regime (configs[2]; C3)
# ------------------------------------------------------------------------------------------
def config3(t_len: int = 10_000_000, n_anchors: int = 50_000, blk_lo: int = 5_000, blk_hi: int = 50_000) -> Workload:
    """T random with 5% of bases in tandem repeats (period U[2,50], tract U[50,500]); Q = T at
    98.5% identity (1.2% substitutions, 0.3% indels) cut into blocks of log-uniform length
    blk_lo..blk_hi, 10% inverted in place, 5% moved elsewhere; anchors uniform on the true path."""
    T = Stream(stream_seed(3, 0)).bases(t_len)
    rs = Stream(stream_seed(3, 1))
    n_tracts = int(0.05 * t_len / 275)
    starts = rs.integers(0, max(t_len - 600, 1), n_tracts); periods = rs.integers(2, 51, n_tracts)
    tl = rs.integers(50, 501, n_tracts)
    for s0, per, ln in zip(starts, periods, tl):
        unit = T[s0:s0 + per].copy()
        T[s0:s0 + ln] = np.resize(unit, ln)
    mu = mutate(T, 0.012, 0.003, Stream(stream_seed(3, 2)))
    bs = Stream(stream_seed(3, 3))
    bounds = [0]
    while bounds[-1] < t_len:
        u = float(bs.uniform(1)[0])
        bounds.append(bounds[-1] + int(round(np.exp(np.log(blk_lo) + u * (np.log(blk_hi) - np.log(blk_lo))))))
    bounds[-1] = t_len
    if len(bounds) > 2 and bounds[-1] - bounds[-2] < blk_lo // 2:
        bounds.pop(-2)
    bounds_t = np.array(bounds, np.int64)
    nb = len(bounds_t) - 1
    r = bs.uniform(nb)
    inverted = r < 0.10
    moved = (r >= 0.10) & (r < 0.15)
    order = [b for b in range(nb) if not moved[b]]
    for b in np.nonzero(moved)[0]:
        order.insert(int(bs.integers(0, len(order) + 1, 1)[0]), int(b))
    qb, new_start = _blocks_rearranged(len(mu.seq), t_len, mu, bounds_t, inverted, np.array(order))
    Q = _assemble(mu.seq, qb, new_start, inverted)
    picks = np.sort(Stream(stream_seed(3, 4)).integers(0, len(mu.t_idx), n_anchors))
    A = _sort_anchors(_true_path_anchors(mu, picks, bounds_t, qb, new_start, inverted, len(Q)))
    pairs = np.array([[0, t_len, 0, len(Q)]], dtype=np.int64)
    return Workload("c3", T, Q, pairs, A, dict(n_blocks=nb, n_inverted=int(inverted.sum()), n_moved=int(moved.sum())))


# ------------------------------------------------------------------------------------------
# Config 5: chromosome-scale pair (configs[4]; C5)
# ------------------------------------------------------------------------------------------
def config5(t_len: int = 100_000_000, n_anchors: int = 1_000_000) -> Workload:
    """T random with 3% N runs (length U[1,10] kbp) and segmental duplications (segments totalling
    2% of T, length U[5,50] kbp, each copied 2-5 more times elsewhere at 99% identity); Q = T at
    96% identity (3.5% substitutions, 0.5% indels) with 1% of bases in inverted segments
    (U[10,100] kbp); anchors: 70% on the true diagonal, 10% on duplicate-copy diagonals, 20%
    uniform random decoys, sorted by target position."""
    T = Stream(stream_seed(5, 0)).bases(t_len)
    rs = Stream(stream_seed(5, 1))
    scale = t_len / 100_000_000
    # segmental duplications first (so N runs may interrupt them, as in assemblies)
    dup_pairs = []                                   # (src start, copy start, length)
    n_dup = max(1, int(round(0.02 * t_len / 27_500)))
    dst = Stream(stream_seed(5, 2))
    for _ in range(n_dup):
        L = int(rs.integers(5_000, 50_001, 1)[0]); L = max(200, int(L * min(1.0, scale * 20))) if scale < 0.05 else L
        a = int(rs.integers(0, t_len - L, 1)[0])
        for _c in range(int(rs.integers(2, 6, 1)[0])):
            b = int(rs.integers(0, t_len - L - 64, 1)[0])
            cp = mutate(T[a:a + L], 0.008, 0.002, dst)
            ln = min(len(cp.seq), L)
            T[b:b + ln] = cp.seq[:ln]
            dup_pairs.append((a, b, ln, cp))
    n_runs = max(1, int(round(0.03 * t_len / 5_500)))
    for s0, ln in zip(rs.integers(0, t_len - 10_000, n_runs), rs.integers(1_000, 10_001, n_runs)):
        ln = int(ln if scale >= 0.05 else max(100, ln * scale * 20))
        T[s0:s0 + ln] = 4
    mu = mutate(T, 0.035, 0.005, Stream(stream_seed(5, 3)))
    # inverted segments: cut at their ends, flip in place
    n_inv = max(1, int(round(0.01 * t_len / 55_000)))
    inv_s = np.sort(rs.integers(0, t_len - 100_000 if t_len > 200_000 else t_len // 2, n_inv))
    inv_l = rs.integers(10_000, 100_001, n_inv)
    if scale < 0.05:
        inv_l = np.maximum(500, (inv_l * scale * 20).astype(np.int64))
    cuts = [0]; flags = []
    for s0, ln in zip(inv_s, inv_l):
        s0 = int(max(s0, cuts[-1] + 1)); e0 = int(min(s0 + ln, t_len - 1))
        if e0 <= s0:
            continue
        flags.append(False); cuts.append(s0); flags.append(True); cuts.append(e0)
    flags.append(False); cuts.append(t_len)
    bounds_t = np.array(cuts, np.int64); inverted = np.array(flags, bool)
    qb, new_start = _blocks_rearranged(len(mu.seq), t_len, mu, bounds_t, inverted, np.arange(len(inverted)))
    Q = _assemble(mu.seq, qb, new_start, inverted)
    q_len = len(Q)
    ast = Stream(stream_seed(5, 4))
    n_true = int(0.7 * n_anchors); n_dupa = int(0.1 * n_anchors); n_dec = n_anchors - n_true - n_dupa
    parts = [_true_path_anchors(mu, ast.integers(0, len(mu.t_idx), n_true), bounds_t, qb, new_start, inverted, q_len)]
    # duplicate diagonals: target position in the SOURCE segment, query position = image of the COPY
    q_of_t = np.full(t_len + 1, -1, np.int64); q_of_t[mu.t_idx] = mu.q_idx
    which = ast.integers(0, len(dup_pairs), n_dupa); frac = ast.uniform(n_dupa)
    da = []
    for w_, f_ in zip(which, frac):
        a, b, ln, cp = dup_pairs[int(w_)]
        k = int(f_ * (len(cp.t_idx) - 1))
        x, y = int(cp.t_idx[k]), int(cp.q_idx[k])
        if y >= ln:
            continue
        qm = q_of_t[b + y]
        if qm < 0:
            continue
        da.append((a + x, b + y, qm))
    if da:
        da = np.array(da, np.int64)
        bidx = np.clip(np.searchsorted(bounds_t, da[:, 1], side="right") - 1, 0, len(new_start) - 1)
        ok = (da[:, 2] >= qb[bidx]) & (da[:, 2] < qb[bidx + 1])
        rel = da[:, 2] - qb[bidx]; blen = qb[bidx + 1] - qb[bidx]
        inv = inverted[bidx]
        qq = np.where(inv, q_len - (new_start[bidx] + blen) + rel, new_start[bidx] + rel)
        parts.append(np.stack([da[:, 0], qq, np.zeros(len(da), np.int64), np.where(inv, -1, 1)], axis=1)[ok])
    dt = ast.integers(0, t_len + 1, n_dec); dq = ast.integers(0, q_len + 1, n_dec); ds = ast.integers(0, 2, n_dec)
    parts.append(np.stack([dt, dq, np.zeros(n_dec, np.int64), np.where(ds > 0, 1, -1)], axis=1))
    A = _sort_anchors(np.concatenate(parts).astype(np.int64))
    pairs = np.array([[0, t_len, 0, q_len]], dtype=np.int64)
    return Workload("c5", T, Q, pairs, A, dict(n_dup_copies=len(dup_pairs), n_inverted=int(inverted.sum())))


CONFIGS = {"c1": config1, "c2": config2, "c3": config3, "c4": config4, "c5": config5}


# ------------------------------------------------------------------------------------------
# Filter workload (gapped Y-drop as the FILTER over raw seed hits)
# ------------------------------------------------------------------------------------------
def filter_hits(n_hits: int = 1_000_000, true_frac: float = 0.05, t_len: int = 2_000_000, n_segments: int = 2000,
                budget: int = 1024) -> Workload:
    """Raw, mostly false seed hits on a configs[1]-like pair: the sequences of config2 (segments U[100, 800] at 70 %
    identity, every second one reverse-complemented); `true_frac` of the hits lie on a segment's true path (qpos jitter
    U{-3..3}), the rest are uniform random (tpos, qpos, strand) -- what a seeding stage hands to the filter before anything
    has been verified.  Every hit gets its own pair: the box of +-`budget` bases around it (clipped to the sequences),
    i.e. a fixed row / column budget per one-sided extension.  Hits are sorted by target position."""
    base = config2(t_len=t_len, n_segments=n_segments, per_seg=1, n_decoys=0)
    T, Q = base.target, base.query
    q_len = len(Q)
    slot = t_len // n_segments
    st = Stream(stream_seed(6, 0))
    n_true = int(true_frac * n_hits)
    # true hits: re-derive each segment's placement exactly as config2 does (same streams), then pick aligned pairs
    perm = Stream(stream_seed(2, 2)).permutation(n_segments)
    lens = Stream(stream_seed(2, 3)).integers(100, 801, n_segments)
    mst = Stream(stream_seed(2, 4))
    per = np.bincount(st.integers(0, n_segments, n_true), minlength=n_segments)
    hits = []
    for s in range(n_segments):
        ln_t = int(lens[s]); t0 = s * slot + 16
        mu = mutate(T[t0:t0 + ln_t], 0.30, 0.02, mst)
        if per[s] == 0:
            continue
        q0 = int(perm[s]) * slot + 16
        ln = min(len(mu.seq), slot - 32)
        ok = np.nonzero(mu.q_idx < ln)[0]
        k = ok[st.integers(0, len(ok), int(per[s]))]
        jit = st.integers(-3, 4, int(per[s]))
        minus = (s % 2 == 1)
        tp = t0 + mu.t_idx[k]
        qrel = mu.q_idx[k]
        qp = (q_len - q0 - ln + qrel) if minus else (q0 + qrel)
        qp = np.clip(qp + jit, 0, q_len)
        hits.append(np.stack([tp, qp, np.zeros_like(tp), np.full_like(tp, -1 if minus else 1)], 1))
    n_false = n_hits - sum(len(h) for h in hits)
    ft = st.integers(0, t_len + 1, n_false); fq = st.integers(0, q_len + 1, n_false); fs = st.integers(0, 2, n_false)
    hits.append(np.stack([ft, fq, np.zeros_like(ft), np.where(fs > 0, 1, -1)], 1))
    A = _sort_anchors(np.concatenate(hits).astype(np.int64))
    n = len(A)
    A[:, 2] = np.arange(n)
    # per-hit pair in the FORWARD query frame (sfe_pair): a - strand hit at rc-frame qpos sits at q_len - qpos forward
    qf = np.where(A[:, 3] > 0, A[:, 1], q_len - A[:, 1])
    pairs = np.stack([np.maximum(A[:, 0] - budget, 0), np.minimum(A[:, 0] + budget, t_len),
                      np.maximum(qf - budget, 0), np.minimum(qf + budget, q_len)], 1).astype(np.int64)
    return Workload("filter", T, Q, pairs, A, dict(n_true=int(n - n_false), n_false=int(n_false), budget=budget))
