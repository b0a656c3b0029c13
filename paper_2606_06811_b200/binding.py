"""Thin ctypes binding of libsfe (include/sfe.h).  Argument marshalling only: every step of
the path runs in the CUDA kernels of csrc/.  PyTorch is used for device memory and streams.

There is no CPU fallback: importing works without a GPU (so the ABI can be checked), but
every compute entry point needs the compiled library and a CUDA device and fails loudly
otherwise.
"""
from __future__ import annotations

import ctypes as C
import os

import numpy as np

_HERE = os.path.dirname(os.path.abspath(__file__))
LIB_PATH = os.environ.get("SFE_LIB_PATH") or os.path.join(_HERE, "libsfe.so")      # (override: A/B builds of the same sources)

OK, EINVAL, ENOMEM, ECUDA, ELIMIT = 0, -1, -2, -3, -4
YDROP_INF = 0x7FFFFFFF
PRUNE_LAG = 32
WANT_CIGAR, SCORE_ONLY, NO_BINNING, BLOCK_KERNEL, NO_BLOCK_KERNEL, CIGAR_KEPT_ONLY, SPEC_LEADERS = 1, 0, 2, 4, 8, 16, 32
(OPT_LEADER_DIAG_TOL, OPT_LEADER_GAP, OPT_LEADER_LOOKBACK, OPT_LEADER_NBREAK, OPT_SPEC_SPAN, OPT_SPEC_ESC_MAX, OPT_SPARSE_WARPS,
 OPT_FORCE_CLASS, OPT_PROMOTE_REACH, OPT_ROW_KERNEL_CAP, OPT_ROW_KERNEL_SCORE_ONLY, OPT_LONG_ROWS, OPT_LONG_ROWS_DENSE, OPT_ROW_SLOTS) = range(14)
ST_TB_OVERFLOW, ST_CIGAR_OVERFLOW, ST_WIDE, ST_SCORE_LIMIT, ST_BAD_ANCHOR, ST_BAND_LIMIT, ST_INTERNAL, ST_SKIPPED = 1, 2, 4, 8, 16, 32, 64, 128
OP_M, OP_I, OP_D = 0, 1, 2
INFO_N = 12
ST_SKEW2, ST_SKEW_RETRY, ST_BLOCK = 0x1000, 0x2000, 0x800      # profile-only bits of sfe_half_profile.status (internal)

EXPORTS = ("sfe_create", "sfe_destroy", "sfe_strerror", "sfe_last_error_detail", "sfe_pack", "sfe_ydrop_batch", "sfe_resolve",
           "sfe_speculate", "sfe_extend_host", "sfe_speculate_host", "sfe_probe_int_issue", "sfe_last_batch_info", "sfe_last_half_profile",
           "sfe_launch_counter", "sfe_set_option", "sfe_last_speculate_info", "sfe_resolve_static", "sfe_resolve_static_limits")


class Scoring(C.Structure):
    _fields_ = [("sub", (C.c_int32 * 4) * 4), ("n_score", C.c_int32), ("gap_open", C.c_int32),
                ("gap_extend", C.c_int32), ("ydrop", C.c_int32), ("prune_lag", C.c_int32), ("min_score", C.c_int32)]


class Stats(C.Structure):
    _fields_ = [("n_anchors", C.c_int64), ("n_kept", C.c_int64), ("n_covered", C.c_int64), ("n_below", C.c_int64),
                ("cells_total", C.c_uint64), ("cells_covered", C.c_uint64), ("n_extended", C.c_int64), ("n_windows", C.c_int64)]


# numpy mirrors of the POD structs (layout = the C structs of sfe.h)
ANCHOR_DT = np.dtype([("tpos", "<i8"), ("qpos", "<i8"), ("pair", "<i4"), ("strand", "<i4")])
PAIR_DT = np.dtype([("t_begin", "<i8"), ("t_end", "<i8"), ("q_begin", "<i8"), ("q_end", "<i8")])
RESULT_DT = np.dtype([("score", "<i4"), ("score_fwd", "<i4"), ("score_bwd", "<i4"), ("status", "<u4"),
                      ("tstart", "<i8"), ("tend", "<i8"), ("qstart", "<i8"), ("qend", "<i8"),
                      ("cigar_off", "<i8"), ("n_ops", "<i4"), ("n_ops_back", "<i4"), ("cells", "<u8")])
BOX_DT = np.dtype([("tstart", "<i8"), ("tend", "<i8"), ("qstart", "<i8"), ("qend", "<i8"),
                   ("strand", "<i4"), ("reserved", "<i4")])
STATS_DT = np.dtype([("n_anchors", "<i8"), ("n_kept", "<i8"), ("n_covered", "<i8"), ("n_below", "<i8"),
                     ("cells_total", "<u8"), ("cells_covered", "<u8"), ("n_extended", "<i8"), ("n_windows", "<i8")])
HALF_PROFILE_DT = np.dtype([("cells", "<i8"), ("cycles", "<i8"), ("steps", "<i4"), ("n_strips", "<i4"), ("max_steps", "<i4"),
                            ("n_ops", "<i4"), ("smid", "<u4"), ("wslot", "<u4"), ("status", "<u4"), ("reserved", "<u4")])
assert ANCHOR_DT.itemsize == 24 and PAIR_DT.itemsize == 32 and RESULT_DT.itemsize == 72 and BOX_DT.itemsize == 40

HOXD70 = ((91, -114, -31, -123), (-114, 100, -125, -31), (-31, -125, 100, -114), (-123, -31, -114, 91))

_lib = None


class SfeError(RuntimeError):
    pass


def lib():
    """Load libsfe.so (built in-tree by __graft_entry__.build()); raises if it is missing."""
    global _lib
    if _lib is None:
        if not os.path.exists(LIB_PATH):
            raise SfeError(f"{LIB_PATH} is missing: run `python -c 'import __graft_entry__ as g; g.build()'` "
                           "(there is no CPU fallback)")
        _lib = C.CDLL(LIB_PATH)
        _lib.sfe_strerror.restype = C.c_char_p
        _lib.sfe_strerror.argtypes = [C.c_int]
        _lib.sfe_last_error_detail.restype = C.c_char_p
        _lib.sfe_launch_counter.restype = C.c_int64
        vp, i64, i32, u32 = C.c_void_p, C.c_int64, C.c_int32, C.c_uint32
        _lib.sfe_create.argtypes = [C.POINTER(vp), C.c_int, vp, C.c_size_t]
        _lib.sfe_destroy.argtypes = [vp]
        _lib.sfe_pack.argtypes = [vp, vp, i64, vp, vp, vp, vp]
        _lib.sfe_ydrop_batch.argtypes = [vp, vp, vp, i64, vp, vp, vp, vp, i64, vp, i32, vp, i64,
                                         C.POINTER(Scoring), u32, vp, vp, i64, vp]
        _lib.sfe_speculate.argtypes = [vp, vp, vp, i64, vp, vp, vp, vp, i64, vp, i32, vp, i64, C.POINTER(Scoring), u32, i64,
                                       vp, vp, vp, i64, vp, vp, i64, vp, vp]
        _lib.sfe_resolve.argtypes = [vp, vp, vp, i64, i32, vp, i64, vp, vp, vp]
        _lib.sfe_extend_host.argtypes = [vp, vp, i64, vp, i64, vp, i32, vp, i64, C.POINTER(Scoring), u32,
                                         vp, vp, vp, i64, C.POINTER(i64), C.POINTER(Stats)]
        _lib.sfe_last_half_profile.argtypes = [vp, i64, vp]
        _lib.sfe_speculate_host.argtypes = [vp, vp, i64, vp, i64, vp, i32, vp, i64, C.POINTER(Scoring), u32, i64,
                                            vp, vp, vp, i64, C.POINTER(i64), C.POINTER(Stats)]
        _lib.sfe_probe_int_issue.argtypes = [vp, C.c_int, C.c_int, C.POINTER(C.c_double), C.POINTER(C.c_double)]
        _lib.sfe_last_batch_info.argtypes = [vp, C.POINTER(i64)]
        _lib.sfe_set_option.argtypes = [vp, C.c_int, i64]
        _lib.sfe_last_speculate_info.argtypes = [vp, C.POINTER(i64)]
        _lib.sfe_resolve_static.argtypes = [C.c_int, vp, vp, vp, i64, i32, vp, i64, vp, vp, vp]
        _lib.sfe_resolve_static_limits.argtypes = [C.POINTER(i64), C.POINTER(i64), C.POINTER(i64)]
    return _lib


def _check(rc: int, what: str):
    if rc != OK:
        raise SfeError(f"{what}: {lib().sfe_strerror(rc).decode()} ({rc}) {lib().sfe_last_error_detail().decode()}")


def scoring(sub=HOXD70, n_score=-100, gap_open=400, gap_extend=30, ydrop=9400, prune_lag=PRUNE_LAG,
            min_score=3000) -> Scoring:
    s = Scoring()
    for a in range(4):
        for b in range(4):
            s.sub[a][b] = sub[a][b]
    s.n_score, s.gap_open, s.gap_extend = n_score, gap_open, gap_extend
    s.ydrop, s.prune_lag, s.min_score = ydrop, prune_lag, min_score
    return s


def make_anchors(a) -> np.ndarray:
    """int array [n, 4] (tpos, qpos, pair, strand) -> structured sfe_anchor array."""
    a = np.asarray(a, dtype=np.int64).reshape(-1, 4)
    out = np.zeros(len(a), dtype=ANCHOR_DT)
    out["tpos"], out["qpos"], out["pair"], out["strand"] = a[:, 0], a[:, 1], a[:, 2], a[:, 3]
    return out


def make_pairs(p) -> np.ndarray:
    p = np.asarray(p, dtype=np.int64).reshape(-1, 4)
    out = np.zeros(len(p), dtype=PAIR_DT)
    out["t_begin"], out["t_end"], out["q_begin"], out["q_end"] = p[:, 0], p[:, 1], p[:, 2], p[:, 3]
    return out


def _torch():
    import torch
    if not torch.cuda.is_available():
        raise SfeError("no CUDA device: libsfe has no CPU fallback")
    return torch


def _dev(arr: np.ndarray, device):
    """numpy (any POD dtype) -> uint8 CUDA tensor holding the same bytes."""
    torch = _torch()
    b = np.ascontiguousarray(arr).view(np.uint8).reshape(-1)
    if b.size == 0:
        return torch.zeros(16, dtype=torch.uint8, device=device)
    return torch.from_numpy(b.copy()).to(device)


def _ptr(t):
    return C.c_void_p(t.data_ptr()) if t is not None else C.c_void_p(0)


class Sfe:
    """One sfe_ctx bound to torch's current CUDA stream on `device`."""

    def __init__(self, device: int = 0, scratch_bytes: int = 1 << 30):
        torch = _torch()
        self.device = torch.device("cuda", device)
        self.stream = torch.cuda.current_stream(self.device)
        h = C.c_void_p()
        _check(lib().sfe_create(C.byref(h), device, C.c_void_p(self.stream.cuda_stream), scratch_bytes), "sfe_create")
        self.h = h

    def close(self):
        if getattr(self, "h", None):
            lib().sfe_destroy(self.h)
            self.h = None

    def __del__(self):
        try:
            self.close()
        except Exception:
            pass

    # ---- sfe_pack -------------------------------------------------------------------------------
    def pack(self, ascii_dev, with_rc: bool = True):
        """ascii_dev: uint8 CUDA tensor of characters.  Returns (codes2, nmask, rc_codes2, rc_nmask)."""
        torch = _torch()
        n = int(ascii_dev.numel())
        nb2 = ((n + 3) // 4 + 15) // 16 * 16 + 16
        nbm = ((n + 7) // 8 + 15) // 16 * 16 + 16
        mk = lambda k: torch.zeros(k, dtype=torch.uint8, device=self.device)
        c2, nm = mk(nb2), mk(nbm)
        r2, rm = (mk(nb2), mk(nbm)) if with_rc else (None, None)
        _check(lib().sfe_pack(self.h, _ptr(ascii_dev), n, _ptr(c2), _ptr(nm), _ptr(r2), _ptr(rm)), "sfe_pack")
        return c2, nm, r2, rm

    # ---- sfe_ydrop_batch --------------------------------------------------------------------------
    def ydrop_batch(self, t_pack, t_len, q_pack, q_len, pairs_dev, n_pairs, anchors_dev, n_anchors, sc: Scoring,
                    flags: int = WANT_CIGAR, cigar_cap: int = 0):
        """t_pack = (codes2, nmask); q_pack = (codes2, nmask, rc_codes2, rc_nmask) CUDA tensors.
        Returns (results_dev [uint8 view of sfe_result], cigar_pool_dev, cigar_used_dev)."""
        torch = _torch()
        res = torch.zeros(max(n_anchors, 1) * RESULT_DT.itemsize, dtype=torch.uint8, device=self.device)
        want = bool(flags & WANT_CIGAR)
        if want and cigar_cap <= 0:
            cigar_cap = max(1024, 64 * n_anchors)
        pool = torch.zeros(max(cigar_cap, 1), dtype=torch.int32, device=self.device) if want else None
        used = torch.zeros(1, dtype=torch.int64, device=self.device)
        rc2 = q_pack[2] if len(q_pack) > 2 else None
        rcm = q_pack[3] if len(q_pack) > 3 else None
        _check(lib().sfe_ydrop_batch(self.h, _ptr(t_pack[0]), _ptr(t_pack[1]), t_len, _ptr(q_pack[0]), _ptr(q_pack[1]),
                                     _ptr(rc2), _ptr(rcm), q_len, _ptr(pairs_dev), n_pairs, _ptr(anchors_dev), n_anchors,
                                     C.byref(sc), flags, _ptr(res), _ptr(pool), cigar_cap if want else 0,
                                     _ptr(used) if want else C.c_void_p(0)), "sfe_ydrop_batch")
        return res, pool, used

    # ---- sfe_speculate ------------------------------------------------------------------------------
    def speculate(self, t_pack, t_len, q_pack, q_len, pairs_dev, n_pairs, anchors_dev, n_anchors, sc: Scoring, window_k: int,
                  flags: int = WANT_CIGAR, cigar_cap: int = 0, accepted_dev=None, n_accepted_dev=None, stats_dev=None):
        """Algorithm 3 on device buffers.  Returns dict(results, keep, pool, used, accepted, n_accepted, stats) of CUDA tensors."""
        torch = _torch()
        n = max(n_anchors, 1)
        res = torch.zeros(n * RESULT_DT.itemsize, dtype=torch.uint8, device=self.device)
        keep = torch.zeros(n, dtype=torch.uint8, device=self.device)
        want = bool(flags & WANT_CIGAR)
        if want and cigar_cap <= 0:
            cigar_cap = max(1024, 64 * n_anchors)
        pool = torch.zeros(max(cigar_cap, 1), dtype=torch.int32, device=self.device) if want else None
        used = torch.zeros(1, dtype=torch.int64, device=self.device)
        if accepted_dev is None:
            accepted_dev = torch.zeros((n + 1) * BOX_DT.itemsize, dtype=torch.uint8, device=self.device)
            n_accepted_dev = torch.zeros(1, dtype=torch.int64, device=self.device)
        if stats_dev is None:
            stats_dev = torch.zeros(STATS_DT.itemsize, dtype=torch.uint8, device=self.device)
        cap = accepted_dev.numel() // BOX_DT.itemsize
        rc2 = q_pack[2] if len(q_pack) > 2 else None
        rcm = q_pack[3] if len(q_pack) > 3 else None
        _check(lib().sfe_speculate(self.h, _ptr(t_pack[0]), _ptr(t_pack[1]), t_len, _ptr(q_pack[0]), _ptr(q_pack[1]), _ptr(rc2),
                                   _ptr(rcm), q_len, _ptr(pairs_dev), n_pairs, _ptr(anchors_dev), n_anchors, C.byref(sc), flags,
                                   window_k, _ptr(res), _ptr(keep), _ptr(pool), cigar_cap if want else 0,
                                   _ptr(used) if want else C.c_void_p(0), _ptr(accepted_dev), cap, _ptr(n_accepted_dev),
                                   _ptr(stats_dev)), "sfe_speculate")
        return dict(results=res, keep=keep, pool=pool, used=used, accepted=accepted_dev, n_accepted=n_accepted_dev, stats=stats_dev)

    # ---- sfe_resolve --------------------------------------------------------------------------------
    def resolve(self, anchors_dev, results_dev, n, min_score, accepted_dev, accepted_cap, n_accepted_dev, stats_dev=None):
        torch = _torch()
        keep = torch.zeros(max(n, 1), dtype=torch.uint8, device=self.device)
        _check(lib().sfe_resolve(self.h, _ptr(anchors_dev), _ptr(results_dev), n, min_score, _ptr(accepted_dev),
                                 accepted_cap, _ptr(n_accepted_dev), _ptr(keep), _ptr(stats_dev)), "sfe_resolve")
        return keep

    # ---- sfe_extend_host ------------------------------------------------------------------------------
    def extend_host(self, t_ascii: np.ndarray, q_ascii: np.ndarray, pairs: np.ndarray, anchors: np.ndarray, sc: Scoring,
                    flags: int = WANT_CIGAR, cigar_cap: int = 0, window_k: int = 0):
        """Host buffers in, host buffers out (numpy).  window_k >= 1 selects sfe_speculate_host (Algorithm 3's windows).
        Returns dict(results, keep, cigar, cigar_used, stats)."""
        n = len(anchors)
        t_ascii = np.ascontiguousarray(t_ascii, dtype=np.uint8); q_ascii = np.ascontiguousarray(q_ascii, dtype=np.uint8)
        pairs = np.ascontiguousarray(pairs); anchors = np.ascontiguousarray(anchors)
        assert pairs.dtype == PAIR_DT and anchors.dtype == ANCHOR_DT
        res = np.zeros(n, dtype=RESULT_DT); keep = np.zeros(n, dtype=np.uint8)
        want = bool(flags & WANT_CIGAR)
        if want and cigar_cap <= 0:
            cigar_cap = max(1024, 64 * n)
        cig = np.zeros(max(cigar_cap, 1), dtype=np.uint32)
        used = C.c_int64(0); st = Stats()
        vp = lambda a: C.c_void_p(a.ctypes.data)
        tail = (vp(res), vp(keep), vp(cig) if want else C.c_void_p(0), cigar_cap if want else 0, C.byref(used), C.byref(st))
        head = (self.h, vp(t_ascii), len(t_ascii), vp(q_ascii), len(q_ascii), vp(pairs), len(pairs), vp(anchors), n, C.byref(sc), flags)
        if window_k >= 1:
            _check(lib().sfe_speculate_host(*head, window_k, *tail), "sfe_speculate_host")
        else:
            _check(lib().sfe_extend_host(*head, *tail), "sfe_extend_host")
        return dict(results=res, keep=keep, cigar=cig, cigar_used=used.value,
                    stats={k: getattr(st, k) for k, _ in Stats._fields_})

    # ---- measurement helpers ----------------------------------------------------------------------------
    def probe_int_issue(self, mix: int = 0, iters: int = 20000):
        r = C.c_double(); ms = C.c_double()
        _check(lib().sfe_probe_int_issue(self.h, mix, iters, C.byref(r), C.byref(ms)), "sfe_probe_int_issue")
        return r.value, ms.value

    def last_half_profile(self, n_halves: int) -> np.ndarray:
        """Per-half (cells, cycles, steps, SM, warp slot, ...) of the most recent ydrop_batch (entry 2a / 2a+1 = fwd / bwd of anchor a)."""
        out = np.zeros(max(n_halves, 1), dtype=HALF_PROFILE_DT)
        _check(lib().sfe_last_half_profile(self.h, n_halves, C.c_void_p(out.ctypes.data)), "sfe_last_half_profile")
        return out[:n_halves]

    def n_sm(self) -> int:
        """SM count of the context's device (the default of OPT_ROW_KERNEL_CAP)"""
        return int(_torch().cuda.get_device_properties(self.device).multi_processor_count)

    def set_option(self, key: int, value: int):
        _check(lib().sfe_set_option(self.h, key, value), "sfe_set_option")

    def last_speculate_info(self):
        a = (C.c_int64 * 8)()
        _check(lib().sfe_last_speculate_info(self.h, a), "sfe_last_speculate_info")
        return dict(batches=a[0], stops=a[1], forced=a[2], cold_stops=a[3], promoted=a[4])

    def last_batch_info(self):
        a = (C.c_int64 * INFO_N)()
        _check(lib().sfe_last_batch_info(self.h, a), "sfe_last_batch_info")
        keys = ("launches", "halves", "halves_rerun", "tb_bytes", "steps", "wide", "ydrop_kernel_us", "block_halves", "ring_drops")
        return dict(zip(keys, list(a)))


def resolve_static(device: int, stream, anchors_dev, results_dev, n, min_score, accepted_dev, accepted_cap, n_accepted_dev,
                   keep_dev, stats_dev=None):
    """sfe_resolve_static: the resolve rule with no context and no allocation (the scratch is a static device array in
    libsfe.so).  `stream` is a raw cudaStream_t value (0 / None = default stream); keep_dev is the caller's."""
    _check(lib().sfe_resolve_static(device, C.c_void_p(stream or 0), _ptr(anchors_dev), _ptr(results_dev), n, min_score,
                                    _ptr(accepted_dev), accepted_cap, _ptr(n_accepted_dev), _ptr(keep_dev), _ptr(stats_dev)),
           "sfe_resolve_static")


def resolve_static_limits():
    """(max anchors per call, max accepted_cap, bytes of the static scratch array)"""
    a, b, c = C.c_int64(0), C.c_int64(0), C.c_int64(0)
    _check(lib().sfe_resolve_static_limits(C.byref(a), C.byref(b), C.byref(c)), "sfe_resolve_static_limits")
    return int(a.value), int(b.value), int(c.value)


def launch_counter() -> int:
    """Kernel launches enqueued so far by this thread through libsfe (sfe_launch_counter)."""
    return int(lib().sfe_launch_counter())


def results_to_numpy(results_dev, n) -> np.ndarray:
    return results_dev.cpu().numpy()[: n * RESULT_DT.itemsize].view(RESULT_DT).copy()


def ops_list(cigar: np.ndarray, off: int, n: int):
    return [(int(w) >> 4, int(w) & 15) for w in cigar[off:off + n]]
