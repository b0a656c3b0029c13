"""sfe_resolve_static: the allocation-free entry point (its scratch is a static __device__ array in libsfe.so) against
sfe_resolve, byte for byte, on two calls in a row.  Collected last on purpose (the suite runs with pytest -x).
Passes alone in a fresh process and after the other GPU tests: it shares nothing with them but the library."""
import numpy as np
import pytest

from paper_2606_06811_b200 import binding as B

pytestmark = pytest.mark.gpu


def _records(seed, n, spread):
    """synthetic (anchor, score, box) records as in test_resolve_random_boxes: chains of mutually covering boxes, below-tau
    anchors, both strands"""
    rng = np.random.default_rng(seed)
    tpos = np.sort(rng.integers(0, n * spread // 8 + 50, n))
    qpos = tpos + rng.integers(-30, 30, n)
    strand = np.where(rng.random(n) < 0.3, -1, 1)
    anchors = np.stack([tpos, qpos, np.zeros(n, np.int64), strand], 1).astype(np.int64)
    res = np.zeros(n, B.RESULT_DT)
    res["score"] = rng.integers(2000, 4500, n)
    res["tstart"] = tpos - rng.integers(0, spread, n); res["tend"] = tpos + rng.integers(0, spread, n)
    res["qstart"] = qpos - rng.integers(0, spread, n); res["qend"] = qpos + rng.integers(0, spread, n)
    res["cells"] = rng.integers(1, 1000, n)
    return B.make_anchors(anchors), res


def _run(call, dev, A, res, n, cap, carried=None):
    """one resolve through `call`; returns (keep, n_accepted, accepted bytes, stats bytes)"""
    import torch
    accd = torch.zeros((cap + 1) * B.BOX_DT.itemsize, dtype=torch.uint8, device=dev)
    nacc = torch.zeros(1, dtype=torch.int64, device=dev)
    if carried is not None:
        accd[: len(carried)] = torch.from_numpy(carried).to(dev)
        nacc[0] = len(carried) // B.BOX_DT.itemsize
    stats = torch.zeros(B.STATS_DT.itemsize, dtype=torch.uint8, device=dev)
    keep = call(B._dev(A, dev), None if res is None else B._dev(res, dev), n, 3000, accd, cap, nacc, stats)
    torch.cuda.synchronize()
    na = int(nacc.item())
    return keep.cpu().numpy()[:n].copy(), na, accd.cpu().numpy()[: max(na, 0) * B.BOX_DT.itemsize].copy(), stats.cpu().numpy().copy()


def test_resolve_static_equals_resolve_twice_in_a_row():
    import torch
    dev = torch.device("cuda", 0)
    max_n, max_acc, nbytes = B.resolve_static_limits()
    assert max_n == 1 << 20 and max_acc == 1 << 16 and 0 < nbytes <= 4 << 20

    def static_call(A, R, n, tau, accd, cap, nacc, stats):
        keep = torch.full((max(n, 1),), 9, dtype=torch.uint8, device=dev)          # the caller's buffer
        B.resolve_static(0, torch.cuda.current_stream(dev).cuda_stream, A, R, n, tau, accd, cap, nacc, keep, stats)
        return keep

    # the existing path (it owns a context; the new one needs none)
    sfe = B.Sfe(0, 64 << 20)
    try:
        # two DIFFERENT problems back to back, the larger first: the second call finds the first one's leftovers in the
        # shared scratch (more block minima, a longer active list) and must not read them
        cases = [(11, 6000, 400), (12, 700, 20)]
        want = [_run(sfe.resolve, dev, *_records(*c), c[1], c[1] + 1) for c in cases]
        got = [_run(static_call, dev, *_records(*c), c[1], c[1] + 1) for c in cases]
        for c, w, g in zip(cases, want, got):
            assert g[0].tolist() == w[0].tolist(), c
            assert g[1] == w[1] and g[1] > 0, c
            assert g[2].tobytes() == w[2].tobytes(), c
            assert g[3].tobytes() == w[3].tobytes(), c
        assert set(got[0][0].tolist()) == {0, 1, 2}                                 # covered, kept and below-tau all occur
        # the same problem twice in a row: identical outputs
        again = [_run(static_call, dev, *_records(*cases[0]), cases[0][1], cases[0][1] + 1) for _ in range(2)]
        for g in again:
            assert all(np.array_equal(x, y) if isinstance(x, np.ndarray) else x == y for x, y in zip(g, want[0]))
        # accepted boxes carried in (R26) and the phase-1 "is covered" filter (results == NULL)
        A, res = _records(13, 3000, 200)
        first = _run(sfe.resolve, dev, A[:1500], res[:1500], 1500, 3001)
        for R in (res[1500:], None):
            w = _run(sfe.resolve, dev, A[1500:], R, 1500, 3001, carried=first[2])
            g = _run(static_call, dev, A[1500:], R, 1500, 3001, carried=first[2])
            assert g[0].tolist() == w[0].tolist() and g[1] == w[1] and g[2].tobytes() == w[2].tobytes() and g[3].tobytes() == w[3].tobytes()
        # accepted_cap too small: the same negative count as sfe_resolve reports
        w = _run(sfe.resolve, dev, A, res, 3000, 10)
        g = _run(static_call, dev, A, res, 3000, 10)
        assert w[1] < 0 and g[1] == w[1] and g[0].tolist() == w[0].tolist()
    finally:
        sfe.close()

    # beyond the limits: refused before anything is launched, with a message that says which limit
    L = B.lib()
    one = torch.zeros(64, dtype=torch.uint8, device=dev)
    launches = B.launch_counter()
    assert L.sfe_resolve_static(0, None, B._ptr(one), None, max_n + 1, 0, B._ptr(one), 1, B._ptr(one), B._ptr(one), None) == B.ELIMIT
    assert b"SFE_STATIC_MAX_ANCHORS" in L.sfe_last_error_detail()
    assert L.sfe_resolve_static(0, None, B._ptr(one), None, 32, 0, B._ptr(one), max_acc + 1, B._ptr(one), B._ptr(one), None) == B.ELIMIT
    assert b"SFE_STATIC_MAX_ACCEPTED" in L.sfe_last_error_detail()
    assert L.sfe_resolve_static(0, None, None, None, 32, 0, B._ptr(one), 1, B._ptr(one), B._ptr(one), None) == B.EINVAL
    assert L.sfe_resolve_static(0, None, None, None, 0, 0, None, 0, None, None, None) == B.OK
    assert B.launch_counter() == launches
    # at the limits it runs (n = max anchors on one diagonal chain: every anchor after the first is covered)
    n = max_n
    A = np.zeros(n, B.ANCHOR_DT); A["tpos"] = np.arange(n); A["qpos"] = np.arange(n); A["strand"] = 1
    res = np.zeros(n, B.RESULT_DT); res["score"] = 5000
    res["tstart"] = A["tpos"]; res["tend"] = n; res["qstart"] = A["qpos"]; res["qend"] = n
    g = _run(static_call, dev, A, res, n, max_acc)
    assert g[1] == 1 and g[0][0] == 1 and not g[0][1:].any()
    torch.cuda.synchronize()
