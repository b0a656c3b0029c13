"""CPU-only checks of the boundary: the C-ABI library loads and exports every symbol that
include/sfe.h declares; struct layouts of the binding match the header; the product path fails
loudly without a GPU (no CPU fallback)."""
import ctypes as C
import os
import re

import numpy as np
import pytest

import __graft_entry__ as entry
from paper_2606_06811_b200 import binding as B

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))


@pytest.fixture(scope="module")
def built():
    entry.build()
    return B.lib()


def _declared():
    src = open(os.path.join(ROOT, "include", "sfe.h")).read()
    src = re.sub(r"/\*.*?\*/", "", src, flags=re.S)
    return sorted(set(re.findall(r"\b(sfe_[a-z_0-9]+)\s*\(", src)))


def test_exports_every_declared_symbol(built):
    names = _declared()
    assert set(B.EXPORTS) == set(names), (names, B.EXPORTS)
    for n in names:
        assert hasattr(built, n), n


def test_struct_layouts_match_header():
    assert C.sizeof(B.Scoring) == 22 * 4
    assert B.ANCHOR_DT.itemsize == 24 and B.PAIR_DT.itemsize == 32
    assert B.RESULT_DT.itemsize == 72 and B.RESULT_DT.fields["cells"][1] == 64
    assert B.BOX_DT.itemsize == 40 and B.STATS_DT.itemsize == C.sizeof(B.Stats) == 64 and B.HALF_PROFILE_DT.itemsize == 48


def test_strerror_and_null_args(built):
    assert built.sfe_strerror(0) == b"ok" and built.sfe_strerror(-4).startswith(b"value")
    assert built.sfe_destroy(None) == B.EINVAL
    assert built.sfe_pack(None, None, 0, None, None, None, None) == B.EINVAL


def test_no_cpu_fallback():
    import torch
    if torch.cuda.is_available():
        pytest.skip("GPU present")
    with pytest.raises(B.SfeError):
        B.Sfe(0)
    h = C.c_void_p()
    assert B.lib().sfe_create(C.byref(h), 0, None, 1 << 20) != B.OK and not h.value


def test_product_does_not_import_oracle():
    """The package never imports / includes anything under oracle/, and the oracle never
    imports the package or its header (they share no code)."""
    pkg = os.path.join(ROOT, "paper_2606_06811_b200")
    pat = re.compile(r"^\s*(from\s+oracle|import\s+oracle|#\s*include\s*[\"<][^\">]*oracle)", re.M)
    for dp, _, fs in os.walk(pkg):
        for f in fs:
            if f.endswith((".py", ".cu", ".cuh", ".h")):
                assert not pat.search(open(os.path.join(dp, f)).read()), f
    assert not pat.search(open(os.path.join(ROOT, "include", "sfe.h")).read())
    for f in os.listdir(os.path.join(ROOT, "oracle")):
        if f.endswith((".py", ".c")):
            txt = open(os.path.join(ROOT, "oracle", f)).read()
            assert not re.search(r"^\s*(from|import)\s+paper_2606_06811_b200", txt, re.M), f
            assert not re.search(r"#\s*include\s*\"[^\"]*sfe[^\"]*\.(h|cuh)\"", txt), f


def test_workload_generators():
    from paper_2606_06811_b200 import workloads as W
    assert int(W.splitmix64(0, 2)[0]) == 0xE220A8397B1DCDAF and int(W.splitmix64(0, 2)[1]) == 0x6E789E6AA1B965F4
    assert W.to_ascii(W.randseq(1, 16)).tobytes() == b"GGTCCTTGCTCGCGCA"
    assert W.to_ascii(W.randseq(2, 16)).tobytes() == b"GGGTCCGGCGCCGCTA"
    w = W.config1()
    assert len(w.anchors) == 256 and len(w.target) == 200_000 and (w.anchors[:, 3] == 1).all()
    assert (np.diff(w.anchors[:, 0]) >= 0).all()
    src = W.randseq(5, 5000)
    mu = W.mutate(src, 0.1, 0.02, W.Stream(6))
    # aligned positions are a strictly increasing map and substitutions ~10%
    assert (np.diff(mu.t_idx) > 0).all() and (np.diff(mu.q_idx) > 0).all()
    ident = (src[mu.t_idx] == mu.seq[mu.q_idx]).mean()
    assert 0.86 < ident < 0.94


def test_binding_constants_match_header():
    """Flags, status bits, op codes and error codes of the Python binding are the header's #defines / enum values."""
    src = open(os.path.join(ROOT, "include", "sfe.h")).read()
    defs = {m.group(1): int(m.group(2), 0) for m in re.finditer(r"#define\s+(SFE_[A-Z_0-9]+)\s+(0x[0-9a-fA-F]+|\d+)u?\b", src)}
    enum = {m.group(1): int(m.group(2)) for m in re.finditer(r"\b(SFE_E?[A-Z]+)\s*=\s*(-?\d+)", src)}
    pairs = {"SFE_WANT_CIGAR": B.WANT_CIGAR, "SFE_SCORE_ONLY": B.SCORE_ONLY, "SFE_NO_BINNING": B.NO_BINNING,
             "SFE_BLOCK_KERNEL": B.BLOCK_KERNEL, "SFE_NO_BLOCK_KERNEL": B.NO_BLOCK_KERNEL, "SFE_CIGAR_KEPT_ONLY": B.CIGAR_KEPT_ONLY, "SFE_SPEC_LEADERS": B.SPEC_LEADERS,
             "SFE_ST_TB_OVERFLOW": B.ST_TB_OVERFLOW, "SFE_ST_CIGAR_OVERFLOW": B.ST_CIGAR_OVERFLOW, "SFE_ST_WIDE": B.ST_WIDE,
             "SFE_ST_SCORE_LIMIT": B.ST_SCORE_LIMIT, "SFE_ST_BAD_ANCHOR": B.ST_BAD_ANCHOR, "SFE_ST_BAND_LIMIT": B.ST_BAND_LIMIT,
             "SFE_ST_INTERNAL": B.ST_INTERNAL, "SFE_ST_SKIPPED": B.ST_SKIPPED, "SFE_OP_M": B.OP_M, "SFE_OP_I": B.OP_I,
             "SFE_OP_D": B.OP_D, "SFE_YDROP_INF": B.YDROP_INF, "SFE_PRUNE_LAG": B.PRUNE_LAG}
    for name, val in pairs.items():
        assert defs[name] == val, name
    for name, val in {"SFE_OK": B.OK, "SFE_EINVAL": B.EINVAL, "SFE_ENOMEM": B.ENOMEM, "SFE_ECUDA": B.ECUDA, "SFE_ELIMIT": B.ELIMIT}.items():
        assert enum[name] == val, name
    # status bits are distinct single bits
    st = [v for k, v in defs.items() if k.startswith("SFE_ST_")]
    assert len(set(st)) == len(st) and all(v & (v - 1) == 0 for v in st)


def test_hot_loop_codegen_guard(built):
    """The Y-drop kernel's steady-state loop is sensitive to register pressure: an innocent edit elsewhere in the kernel
    once turned 16 VIADD into IMAD, added spills and cost 16 % ("Codegen notes").  Guard the static
    instruction mix of the 16-step group (what the roofline denominator is computed from) and the absence of spills."""
    import subprocess
    from paper_2606_06811_b200 import sassinfo
    tb = sassinfo.hot_loop(True); so = sassinfo.hot_loop(False)
    assert tb["per_cell"] <= 22.7 and tb["alu"] <= 14.2 and tb["fma"] <= 4.2 and tb["lsu"] <= 3.2, tb
    assert so["per_cell"] <= 14.6 and so["alu"] <= 10.1, so
    assert tb["hist"].get("VIADDMNMX") == 32 and tb["hist"].get("VIMNMX3") == 24          # DPX: E, F and H / best
    out = subprocess.run(["cuobjdump", "-res-usage", B.LIB_PATH], capture_output=True, text=True).stdout
    blocks = out.split("Function ")
    for b in blocks:
        if b.startswith("_Z12ydrop_kernelILb"):
            assert "STACK:0" in b.replace(" ", ""), b[:300]


def test_resolve_static_limits_and_argument_checks(built):
    """sfe_resolve_static's host logic needs no GPU: the limits are reported, sizes beyond them are refused with a message
    that names the limit before any CUDA call, n == 0 is a no-op, negative sizes / a device ordinal out of range are invalid."""
    import ctypes as C
    L = B.lib()
    max_n, max_acc, nbytes = B.resolve_static_limits()
    assert (max_n, max_acc) == (1 << 20, 1 << 16) and nbytes == 262400 + ((65537 * 40 + 255) // 256) * 256
    one = C.c_void_p(64)                                    # never dereferenced: the checks come first
    assert L.sfe_resolve_static(0, None, one, None, max_n + 1, 0, one, 1, one, one, None) == B.ELIMIT
    assert b"SFE_STATIC_MAX_ANCHORS" in L.sfe_last_error_detail()
    assert L.sfe_resolve_static(0, None, one, None, 1, 0, one, max_acc + 1, one, one, None) == B.ELIMIT
    assert b"SFE_STATIC_MAX_ACCEPTED" in L.sfe_last_error_detail()
    assert L.sfe_resolve_static(0, None, None, None, 0, 0, None, 0, None, None, None) == B.OK
    assert L.sfe_resolve_static(0, None, one, None, -1, 0, one, 1, one, one, None) == B.EINVAL
    assert L.sfe_resolve_static(-1, None, one, None, 1, 0, one, 1, one, one, None) == B.EINVAL
    assert L.sfe_resolve_static(64, None, one, None, 1, 0, one, 1, one, one, None) == B.EINVAL

