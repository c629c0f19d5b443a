"""-m gpu parity of tpcclus_select (D13, the order-preserving quality selection) against
tpc_oracle_select: same kept records, same bytes, same order, for every cut alone and combined, on the cluster
list of the stress generator (ties, splits, saturation, pad edges) and on edge cases."""
import numpy as np
import pytest

import gen
import oracle
from gpu_util import GpuClusterizer

pytestmark = pytest.mark.gpu


def _select(T, ctx, d_in, n, cap, **cuts):
    import torch

    out = torch.zeros((max(cap, 1), 32), dtype=torch.uint8, device="cuda")
    T.tpcclus_select(ctx, d_in.data_ptr(), n, out.data_ptr(), cap, torch.cuda.current_stream().cuda_stream, **cuts)
    kept = T.tpcclus_select_result(ctx, check=False)
    return out[: min(kept, cap)].cpu().numpy().view(T.CLUSTER_DTYPE).reshape(-1), kept


CUTS = [dict(), dict(min_qtot=20.0), dict(min_qtot=1e9), dict(min_qmax_q16=160), dict(min_ncells=4),
        dict(reject_single_pad=True), dict(reject_single_time=True), dict(reject_flags=8), dict(reject_flags=1 | 2 | 4),
        dict(min_qtot=12.5, min_ncells=3, reject_single_pad=True, reject_single_time=True, reject_flags=4)]


def test_select_matches_the_oracle_on_the_stress_list():
    import torch
    import paper_2412_13755_b200 as T

    cfg = gen.config("c4mini")
    d, offs, _ = gen.generate_fragment(cfg, 0, device="cuda")
    with GpuClusterizer(cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins,
                        max_digits=int(d.shape[0])) as g:
        rec, _ = g.run(d, offs, 0, cfg.tf_time_bins)
        n = len(rec)
        assert n > 3e5 and n % 1024 != 0
        d_in = torch.from_numpy(rec.view(np.uint8).reshape(-1, 32).copy()).cuda()
        for cuts in CUTS:
            want, kept_o = oracle.select(rec, **cuts)
            got, kept = _select(T, g.ctx, d_in, n, n, **cuts)
            assert kept == kept_o, cuts
            assert got.tobytes() == want.tobytes(), cuts
        assert 0 < oracle.select(rec, reject_single_time=True)[1] < n
        # capacity: the first `cap` kept records, the count is the number required
        want, kept_o = oracle.select(rec, min_ncells=4)
        got, kept = _select(T, g.ctx, d_in, n, 1000, min_ncells=4)
        assert kept == kept_o > 1000 and got.tobytes() == want[:1000].tobytes()
        # prefixes of every length class: empty, one record, one short of / exactly / one past a 1024-record tile
        for m in (0, 1, 1023, 1024, 1025, 5000):
            want, kept_o = oracle.select(rec[:m], min_qtot=15.0)
            got, kept = _select(T, g.ctx, d_in, m, m, min_qtot=15.0)
            assert kept == kept_o and got.tobytes() == want.tobytes(), m
        # repeat: the look-back scratch is reused from call to call
        a, _ = _select(T, g.ctx, d_in, n, n, min_qtot=20.0)
        b, _ = _select(T, g.ctx, d_in, n, n, min_qtot=20.0)
        assert a.tobytes() == b.tobytes()


def test_select_argument_errors():
    import torch
    import paper_2412_13755_b200 as T

    ctx = T.tpcclus_create([10], n_sectors=1, tf_time_bins=100, max_digits=10)
    try:
        buf = torch.zeros((64, 32), dtype=torch.uint8, device="cuda")
        with pytest.raises(T.TpcclusError) as ei:
            T.tpcclus_select(ctx, buf.data_ptr() + 8, 2, buf.data_ptr(), 2)          # misaligned
        assert ei.value.code == T.TPCCLUS_ERR_INVALID
        with pytest.raises(T.TpcclusError) as ei:
            T.tpcclus_select(ctx, buf.data_ptr(), 2, buf.data_ptr() + 1024, 2, min_qtot=float("nan"))
        assert ei.value.code == T.TPCCLUS_ERR_INVALID
        with pytest.raises(T.TpcclusError) as ei:
            T.tpcclus_select_result(ctx)                                              # nothing pending
        assert ei.value.code == T.TPCCLUS_ERR_INVALID
        T.tpcclus_select(ctx, buf.data_ptr(), 0, buf.data_ptr() + 1024, 0)
        assert T.tpcclus_select_result(ctx) == 0
    finally:
        T.tpcclus_destroy(ctx)
