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


def mutate(src: np.ndarray, p_sub: float, p_indel: float, st: Stream, tstv: bool = False) -> Mutated:
    """Mutation model of SURVEY 8(d): each source base is independently substituted with
    prob. p_sub (uniform over the 3 others, or transition with prob. 2/3 if tstv), or starts
    an indel with prob. p_indel (insertion / deletion with equal probability, length
    geometric p = 0.5, capped at 32).  A deletion of length L removes source bases k..k+L-1;
    an insertion puts L random bases after base k.  Events on deleted bases are ignored."""
    n = len(src)
    u = st.uniform(n)
    alt = st.u64(n)
    geo = st.u64(n)
    ins_bases_stream = st
    is_sub = u < p_sub
    is_indel = (u >= p_sub) & (u < p_sub + p_indel)
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
