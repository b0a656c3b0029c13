"""ctypes binding of oracle/sfe_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.

Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / ``--impl reference`` legs
may import this module.  It imports nothing from ``paper_2606_06811_b200`` and shares no
code with the CUDA path; the struct layouts below mirror the oracle's own C structs
(checked against ``osfe_sizeof`` at load time).
"""
from __future__ import annotations

import ctypes as C
import os
import subprocess
from dataclasses import dataclass

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
_SRC = os.path.join(_HERE, "sfe_oracle.c")
_LIB = os.path.join(_HERE, "libsfe_oracle.so")

YDROP_INF = 0x7FFFFFFF
OP_M, OP_I, OP_D = 0, 1, 2

# LASTZ default scoring (BASELINE.json config 1): HOXD70, N = -100, gaps 400 + 30k, ydrop 9400
HOXD70 = ((91, -114, -31, -123), (-114, 100, -125, -31), (-31, -125, 100, -114), (-123, -31, -114, 91))


def build(force: bool = False) -> str:
    """Compile the oracle with gcc (plain C99, no CUDA)."""
    if force or not os.path.exists(_LIB) or os.path.getmtime(_LIB) < os.path.getmtime(_SRC):
        subprocess.check_call(["gcc", "-O2", "-std=c99", "-Wall", "-shared", "-fPIC", "-o", _LIB, _SRC])
    return _LIB


class Scoring(C.Structure):
    _fields_ = [("sub", (C.c_int32 * 4) * 4), ("n_score", C.c_int32), ("gap_open", C.c_int32),
                ("gap_extend", C.c_int32), ("ydrop", C.c_int32), ("prune_lag", C.c_int32),
                ("min_score", C.c_int32)]


class Half(C.Structure):
    _fields_ = [("score", C.c_int32), ("end_i", C.c_int64), ("end_j", C.c_int64), ("cells", C.c_int64),
                ("rows", C.c_int64), ("max_width", C.c_int64), ("n_ops", C.c_int64)]


class Result(C.Structure):
    _fields_ = [("score", C.c_int32), ("score_fwd", C.c_int32), ("score_bwd", C.c_int32),
                ("tstart", C.c_int64), ("tend", C.c_int64), ("qstart", C.c_int64), ("qend", C.c_int64),
                ("n_ops", C.c_int64), ("n_ops_back", C.c_int64),
                ("cells", C.c_int64), ("cells_fwd", C.c_int64), ("cells_bwd", C.c_int64),
                ("rows_fwd", C.c_int64), ("rows_bwd", C.c_int64), ("max_width", C.c_int64)]


class Box(C.Structure):
    _fields_ = [("tstart", C.c_int64), ("tend", C.c_int64), ("qstart", C.c_int64), ("qend", C.c_int64),
                ("strand", C.c_int32)]


class Anchor(C.Structure):
    _fields_ = [("tpos", C.c_int64), ("qpos", C.c_int64), ("pair", C.c_int32), ("strand", C.c_int32)]


class Pair(C.Structure):
    _fields_ = [("t_begin", C.c_int64), ("t_end", C.c_int64), ("q_begin", C.c_int64), ("q_end", C.c_int64)]


_lib = None


def lib():
    global _lib
    if _lib is None:
        _lib = C.CDLL(build())
        _lib.osfe_sizeof.restype = C.c_int64
        for k, t in enumerate((Scoring, Half, Result, Box, Anchor, Pair)):
            assert _lib.osfe_sizeof(k) == C.sizeof(t), (k, _lib.osfe_sizeof(k), C.sizeof(t))
        _lib.osfe_rescore.restype = C.c_int64
        _lib.osfe_serial_loop.restype = C.c_int64
        _lib.osfe_speculative_loop.restype = C.c_int64
        _lib.osfe_resolve.restype = C.c_int64
    return _lib


def scoring(sub=HOXD70, n_score=-100, gap_open=400, gap_extend=30, ydrop=9400, prune_lag=32,
            min_score=3000) -> Scoring:
    s = Scoring()
    for a in range(4):
        for b in range(4):
            s.sub[a][b] = sub[a][b]
    s.n_score, s.gap_open, s.gap_extend = n_score, gap_open, gap_extend
    s.ydrop, s.prune_lag, s.min_score = ydrop, prune_lag, min_score
    return s


def _u8(a) -> np.ndarray:
    return np.ascontiguousarray(a, dtype=np.uint8)


def _p(a: np.ndarray, t=C.c_uint8):
    return a.ctypes.data_as(C.POINTER(t))


def codes(seq) -> np.ndarray:
    """ASCII (str / bytes / uint8 array of characters) -> code array 0..3, 4 = N (R13, R14)."""
    if isinstance(seq, str):
        seq = seq.encode()
    a = np.frombuffer(seq, dtype=np.uint8) if isinstance(seq, (bytes, bytearray)) else _u8(seq)
    out = np.empty(len(a), dtype=np.uint8)
    lib().osfe_codes(a.ctypes.data_as(C.c_char_p), C.c_int64(len(a)), _p(out))
    return out


def revcomp_codes(c: np.ndarray) -> np.ndarray:
    c = _u8(c)
    out = np.empty(len(c), dtype=np.uint8)
    lib().osfe_revcomp_codes(_p(c), C.c_int64(len(c)), _p(out))
    return out


def pack(ascii_seq, with_rc: bool = True):
    """R13 packing, byte by byte: returns (codes2, nmask, rc_codes2, rc_nmask) uint8 arrays."""
    if isinstance(ascii_seq, str):
        ascii_seq = ascii_seq.encode()
    a = np.frombuffer(ascii_seq, dtype=np.uint8) if isinstance(ascii_seq, (bytes, bytearray)) else _u8(ascii_seq)
    n = len(a)
    c2 = np.zeros((n + 3) // 4, np.uint8); nm = np.zeros((n + 7) // 8, np.uint8)
    rc2 = np.zeros((n + 3) // 4, np.uint8); rnm = np.zeros((n + 7) // 8, np.uint8)
    lib().osfe_pack(a.ctypes.data_as(C.c_char_p), C.c_int64(n), _p(c2), _p(nm),
                    _p(rc2) if with_rc else None, _p(rnm) if with_rc else None)
    return c2, nm, rc2, rnm


@dataclass
class HalfOut:
    score: int
    end_i: int
    end_j: int
    cells: int
    rows: int
    max_width: int
    ops: list  # [(len, op)], origin -> end

    @property
    def cigar(self) -> str:
        return cigar_str(self.ops)


def cigar_str(ops) -> str:
    return "".join(f"{ln}{'MID'[op]}" for ln, op in ops)


def _ops_list(arr, n):
    return [(int(arr[k]) >> 4, int(arr[k]) & 15) for k in range(n)]


def ext_onesided(q, t, sc: Scoring, want_ops: bool = True) -> HalfOut:
    """One-sided extension of code arrays q (rows) and t (columns)."""
    q = _u8(q); t = _u8(t)
    h = Half()
    rc = lib().osfe_ext_onesided(_p(q), C.c_int64(len(q)), _p(t), C.c_int64(len(t)), C.byref(sc),
                                 C.byref(h), None, C.c_int64(0))
    assert rc == 0
    ops = []
    if want_ops and h.n_ops:
        buf = np.zeros(h.n_ops, np.uint32)
        h2 = Half()
        lib().osfe_ext_onesided(_p(q), C.c_int64(len(q)), _p(t), C.c_int64(len(t)), C.byref(sc),
                                C.byref(h2), _p(buf, C.c_uint32), C.c_int64(h.n_ops))
        ops = _ops_list(buf, h.n_ops)
    return HalfOut(h.score, h.end_i, h.end_j, h.cells, h.rows, h.max_width, ops)


def ext_onesided_cells(q, t, sc: Scoring):
    """One-sided extension that also returns dense (n+1) x (m+1) arrays with every visited cell's H and alive flag
    (cells never visited: H = -2**31, alive 0).  Inspection only (pin P5)."""
    q = _u8(q); t = _u8(t)
    h = Half()
    H = np.full((len(q) + 1, len(t) + 1), -2**31, np.int32); A = np.zeros((len(q) + 1, len(t) + 1), np.uint8)
    rc = lib().osfe_ext_onesided_cells(_p(q), C.c_int64(len(q)), _p(t), C.c_int64(len(t)), C.byref(sc), C.byref(h),
                                       _p(H, C.c_int32), _p(A))
    assert rc == 0
    return HalfOut(h.score, h.end_i, h.end_j, h.cells, h.rows, h.max_width, []), H, A


def gotoh_bruteforce(q, t, sc: Scoring):
    q = _u8(q); t = _u8(t)
    s = C.c_int32(); ei = C.c_int64(); ej = C.c_int64()
    rc = lib().osfe_gotoh_bruteforce(_p(q), C.c_int64(len(q)), _p(t), C.c_int64(len(t)), C.byref(sc),
                                     C.byref(s), C.byref(ei), C.byref(ej))
    assert rc == 0
    return s.value, ei.value, ej.value


def rescore(q, t, ops, sc: Scoring):
    """R12 rescoring of [(len, op)] over code arrays starting at index 0: (score, q_used, t_used)."""
    q = _u8(q); t = _u8(t)
    arr = np.array([(ln << 4) | op for ln, op in ops], dtype=np.uint32) if ops else np.zeros(1, np.uint32)
    qu = C.c_int64(); tu = C.c_int64()
    s = lib().osfe_rescore(_p(q), _p(t), _p(arr, C.c_uint32), C.c_int64(len(ops)), C.byref(sc),
                           C.byref(qu), C.byref(tu))
    return int(s), qu.value, tu.value


def extend_anchor(T, Q, tpos, qpos, sc: Scoring, t_lim=None, q_lim=None, want_ops=True):
    """Two-sided extension; Q in the anchor's strand frame.  Returns (Result, [(len, op)])."""
    T = _u8(T); Q = _u8(Q)
    tb, te = t_lim if t_lim else (0, len(T))
    qb, qe = q_lim if q_lim else (0, len(Q))
    r = Result()
    rc = lib().osfe_extend_anchor(_p(T), C.c_int64(tb), C.c_int64(te), _p(Q), C.c_int64(qb), C.c_int64(qe),
                                  C.c_int64(tpos), C.c_int64(qpos), C.byref(sc), C.byref(r), None, C.c_int64(0))
    assert rc == 0, rc
    ops = []
    if want_ops and r.n_ops:
        buf = np.zeros(r.n_ops, np.uint32)
        r2 = Result()
        lib().osfe_extend_anchor(_p(T), C.c_int64(tb), C.c_int64(te), _p(Q), C.c_int64(qb), C.c_int64(qe),
                                 C.c_int64(tpos), C.c_int64(qpos), C.byref(sc), C.byref(r2),
                                 _p(buf, C.c_uint32), C.c_int64(r.n_ops))
        ops = _ops_list(buf, r.n_ops)
    return r, ops


def _anchor_array(anchors):
    """anchors: structured/2-D array-like of (tpos, qpos, pair, strand)."""
    n = len(anchors)
    arr = (Anchor * max(n, 1))()
    for k in range(n):
        arr[k].tpos, arr[k].qpos, arr[k].pair, arr[k].strand = (int(x) for x in anchors[k])
    return arr


def _pair_array(pairs):
    n = len(pairs)
    arr = (Pair * max(n, 1))()
    for k in range(n):
        arr[k].t_begin, arr[k].t_end, arr[k].q_begin, arr[k].q_end = (int(x) for x in pairs[k])
    return arr


def serial_loop(T, Q, Qrc, pairs, anchors, sc: Scoring, want_results=True):
    """Algorithm 1.  Returns dict(state, results, n_kept, n_extended, cells)."""
    T = _u8(T); Q = _u8(Q); Qrc = _u8(Qrc)
    n = len(anchors)
    A = _anchor_array(anchors); P = _pair_array(pairs)
    state = np.zeros(max(n, 1), np.uint8)
    res = (Result * max(n, 1))()
    ne = C.c_int64(); ce = C.c_int64()
    k = lib().osfe_serial_loop(_p(T), _p(Q), _p(Qrc), C.c_int64(len(Q)), P, A, C.c_int64(n), C.byref(sc),
                               _p(state), res if want_results else None, C.byref(ne), C.byref(ce))
    assert k >= 0
    return dict(state=state[:n], results=res, n_kept=int(k), n_extended=ne.value, cells=ce.value)


def speculative_loop(T, Q, Qrc, pairs, anchors, sc: Scoring, K: int):
    """Algorithm 3 with window K.  Returns dict(state, spec_extended, n_kept, n_extended, cells)."""
    T = _u8(T); Q = _u8(Q); Qrc = _u8(Qrc)
    n = len(anchors)
    A = _anchor_array(anchors); P = _pair_array(pairs)
    state = np.zeros(max(n, 1), np.uint8); spec = np.zeros(max(n, 1), np.uint8)
    ne = C.c_int64(); ce = C.c_int64()
    k = lib().osfe_speculative_loop(_p(T), _p(Q), _p(Qrc), C.c_int64(len(Q)), P, A, C.c_int64(n),
                                    C.byref(sc), C.c_int64(K), _p(state), _p(spec), C.byref(ne), C.byref(ce))
    assert k >= 0
    return dict(state=state[:n], spec_extended=spec[:n], n_kept=int(k), n_extended=ne.value, cells=ce.value)


def resolve(anchors, scores, boxes, min_score, accepted=()):
    """Phase 3 alone.  boxes[i] = (tstart, tend, qstart, qend); accepted = [(tstart,tend,qstart,qend,strand)].
    Returns (state, accepted_out)."""
    n = len(anchors)
    A = _anchor_array(anchors)
    res = (Result * max(n, 1))()
    for k in range(n):
        res[k].score = int(scores[k])
        res[k].tstart, res[k].tend, res[k].qstart, res[k].qend = (int(x) for x in boxes[k])
    cap = len(accepted) + n + 1
    acc = (Box * cap)()
    for k, b in enumerate(accepted):
        acc[k].tstart, acc[k].tend, acc[k].qstart, acc[k].qend, acc[k].strand = (int(x) for x in b)
    state = np.zeros(max(n, 1), np.uint8)
    na = lib().osfe_resolve(A, res, C.c_int64(n), C.c_int32(min_score), acc, C.c_int64(len(accepted)),
                            C.c_int64(cap), _p(state))
    assert na >= 0
    out = [(acc[k].tstart, acc[k].tend, acc[k].qstart, acc[k].qend, acc[k].strand) for k in range(na)]
    return state[:n], out
