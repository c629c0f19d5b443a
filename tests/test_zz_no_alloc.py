"""-m gpu test of tpcclus_select_static, the entry point that allocates nothing (include/tpcclus.h: the D13 selection
with its look-back scratch in a fixed `static __device__` array inside the library, for callers that cannot call
cudaMalloc).  Its output must be byte-identical to the existing path's (tpcclus_select on a context) — the tolerance
the other selection tests use — on calls IN A ROW, which share the array: the second call runs over whatever the first
left there, also when it uses fewer or more tiles than the one before.

Collected last on purpose (the suite runs with pytest -x; `pytest --collect-only -q tests` shows the order).  Needs
nothing from the tests before it: passes alone in a fresh process and after the rest of the suite.
"""
import ctypes

import numpy as np
import pytest

import gen
import oracle
from gpu_util import GpuClusterizer

pytestmark = pytest.mark.gpu


def _records():
    """A cluster list from the existing path: the stress generator's fragment (ties, splits, saturation, pad edges)."""
    cfg = gen.config("c4mini")
    d, offs, _ = gen.generate_fragment(cfg, 0, device="cuda")
    g = GpuClusterizer(cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins, max_digits=int(d.shape[0]))
    rec, _ = g.run(d, offs, 0, cfg.tf_time_bins)
    return g, rec


def _existing(T, ctx, d_in, n, cap, stream, **cuts):
    import torch

    out = torch.zeros((max(cap, 1), 32), dtype=torch.uint8, device="cuda")
    T.tpcclus_select(ctx, d_in.data_ptr(), n, out.data_ptr(), cap, stream, **cuts)
    kept = T.tpcclus_select_result(ctx, check=False)
    return out[: min(kept, cap)].cpu().numpy().tobytes(), kept


def test_select_static_matches_the_existing_path_on_calls_in_a_row():
    import torch
    import paper_2412_13755_b200 as T

    g, rec = _records()
    try:
        n = len(rec)
        assert 3e5 < n <= T.TPCCLUS_SELECT_STATIC_MAX_RECORDS and n % 1024 != 0
        stream = torch.cuda.current_stream().cuda_stream
        d_in = torch.from_numpy(rec.view(np.uint8).reshape(-1, 32).copy()).cuda()
        # (n, capacity, cuts) in the order they are issued: full list twice with different cuts, a short prefix (fewer
        # tiles than the call before: the array still holds that call's words beyond them), the full list again,
        # an empty call, the same cuts twice, and a capacity smaller than the kept count
        calls = [(n, n, dict(min_qtot=20.0)),
                 (n, n, dict(min_ncells=4, reject_single_pad=True)),
                 (1025, 1025, dict(min_qtot=15.0)),
                 (n, n, dict(reject_single_time=True, reject_flags=4)),
                 (0, 0, dict()),
                 (n, n, dict(min_qtot=20.0)),
                 (n, n, dict(min_qtot=20.0)),
                 (n, 1000, dict(min_ncells=4)),
                 (n, n, dict())]
        want = [_existing(T, g.ctx, d_in, m, cap, stream, **cuts) for m, cap, cuts in calls]
        assert want[0][1] not in (0, n) and want[8][1] == n and want[7][1] > 1000

        # everything the new path touches is allocated BEFORE the calls; one empty call does the once-per-device set-up
        outs = [torch.zeros((max(cap, 1), 32), dtype=torch.uint8, device="cuda") for _, cap, _ in calls]
        kept = torch.full((len(calls),), -1, dtype=torch.int64, device="cuda")
        T.tpcclus_select_static(0, 0, 0, 0, kept.data_ptr(), stream)
        torch.cuda.synchronize()
        assert int(kept[0].item()) == 0
        kept.fill_(-1)
        torch.cuda.synchronize()
        free_before, _ = torch.cuda.mem_get_info()
        # all calls back to back on one stream, no synchronisation in between: each runs over the previous one's leftovers
        for i, (m, cap, cuts) in enumerate(calls):
            T.tpcclus_select_static(d_in.data_ptr(), m, outs[i].data_ptr(), cap, kept.data_ptr() + 8 * i, stream, **cuts)
        torch.cuda.synchronize()
        free_after, _ = torch.cuda.mem_get_info()
        assert free_after == free_before                       # the device's free memory did not move: nothing was allocated
        kept_h = kept.cpu().numpy()
        for i, (m, cap, cuts) in enumerate(calls):
            assert int(kept_h[i]) == want[i][1], (i, cuts)
            got = outs[i][: min(int(kept_h[i]), cap)].cpu().numpy().tobytes()
            assert got == want[i][0], (i, cuts)
        # and against the oracle's definition of D13 for one of them
        ref, k_o = oracle.select(rec, min_ncells=4, reject_single_pad=True)
        assert k_o == int(kept_h[1]) and ref.tobytes() == want[1][0]
    finally:
        g.close()


def test_select_static_rejects_what_it_cannot_hold():
    """Sizes beyond the fixed array are refused with their own error before anything is enqueued; so are bad pointers."""
    import torch
    import paper_2412_13755_b200 as T

    word = torch.full((2,), 7, dtype=torch.int64, device="cuda")
    buf = torch.zeros((64, 32), dtype=torch.uint8, device="cuda")
    stream = torch.cuda.current_stream().cuda_stream
    with pytest.raises(T.TpcclusError) as ei:
        T.tpcclus_select_static(buf.data_ptr(), T.TPCCLUS_SELECT_STATIC_MAX_RECORDS + 1, buf.data_ptr(), 64, word.data_ptr(), stream)
    assert ei.value.code == T.TPCCLUS_ERR_TOO_LARGE
    assert "TPCCLUS_SELECT_STATIC_MAX_RECORDS" in T.tpcclus_strerror(T.TPCCLUS_ERR_TOO_LARGE)
    for args in [(buf.data_ptr(), 64, buf.data_ptr() + 32 * 32, 32, 0),                    # no place for the count
                 (buf.data_ptr() + 8, 16, buf.data_ptr() + 32 * 32, 16, word.data_ptr()),  # misaligned input
                 (buf.data_ptr(), 16, buf.data_ptr() + 32 * 32, 16, word.data_ptr() + 4),  # misaligned count
                 (0, 16, buf.data_ptr(), 16, word.data_ptr())]:                            # records but no input
        with pytest.raises(T.TpcclusError) as ei:
            T.tpcclus_select_static(*args, stream)
        assert ei.value.code == T.TPCCLUS_ERR_INVALID
    with pytest.raises(T.TpcclusError) as ei:
        T.tpcclus_select_static(buf.data_ptr(), 16, buf.data_ptr() + 32 * 32, 16, word.data_ptr(), stream, min_qtot=float("nan"))
    assert ei.value.code == T.TPCCLUS_ERR_INVALID
    torch.cuda.synchronize()
    assert word.tolist() == [7, 7]                             # a refused call wrote nothing
    # the largest size it accepts is the stated maximum (checked on the argument path only: a 16-record list, n = 16)
    T.tpcclus_select_static(buf.data_ptr(), 16, buf.data_ptr() + 32 * 32, 16, word.data_ptr(), stream)
    torch.cuda.synchronize()
    assert word.tolist() == [16, 7]                            # all-zero records pass the default cuts
    assert ctypes.sizeof(T.tpcclus_cuts) == 12


def test_select_static_is_capturable_in_a_cuda_graph():
    """include/tpcclus.h says the call enqueues two memsets and one kernel, "all capturable": capture it once (after the
    set-up call), replay the graph twice with different inputs in the same buffers, compare with the existing path."""
    import torch
    import paper_2412_13755_b200 as T

    g, rec = _records()
    try:
        n = len(rec) // 2                                      # two different inputs of the same length
        assert n > 1e5
        a = torch.from_numpy(rec[:n].view(np.uint8).reshape(-1, 32).copy()).cuda()
        b = torch.from_numpy(rec[n: 2 * n].view(np.uint8).reshape(-1, 32).copy()).cuda()
        cuts = dict(min_qtot=18.0, reject_single_time=True)
        cur = torch.cuda.current_stream().cuda_stream
        want = [_existing(T, g.ctx, x, n, n, cur, **cuts) for x in (a, b)]
        assert want[0][0] != want[1][0] and 0 < want[0][1] < n

        d_in = torch.zeros_like(a)
        d_out = torch.zeros((n, 32), dtype=torch.uint8, device="cuda")
        kept = torch.full((1,), -1, dtype=torch.int64, device="cuda")
        T.tpcclus_select_static(0, 0, 0, 0, kept.data_ptr(), cur)      # once-per-device set-up, outside the capture
        torch.cuda.synchronize()
        graph = torch.cuda.CUDAGraph()
        with torch.cuda.graph(graph):
            T.tpcclus_select_static(d_in.data_ptr(), n, d_out.data_ptr(), n, kept.data_ptr(),
                                    torch.cuda.current_stream().cuda_stream, **cuts)
        for x, (w_bytes, w_kept) in zip((a, b), want):
            d_in.copy_(x)
            d_out.zero_()
            graph.replay()
            torch.cuda.synchronize()
            k = int(kept.item())
            assert k == w_kept
            assert d_out[:k].cpu().numpy().tobytes() == w_bytes
    finally:
        g.close()
