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


@pytest.mark.parametrize("in_off,out_off", [(0, 0), (16, 0), (0, 16), (16, 16)])
def test_select_alignment_classes(in_off, out_off):
    """Buffers aligned to 32 bytes move records as single 256-bit accesses, buffers aligned to 16 bytes only as two
    halves (include/tpcclus.h asks for 16): both paths, and their mixes, give the oracle's bytes."""
    import torch
    import paper_2412_13755_b200 as T

    rng = np.random.default_rng(7 + in_off + 2 * out_off)
    n = 5000
    rec = np.zeros(n, dtype=T.CLUSTER_DTYPE)
    rec["sector"], rec["row"], rec["pad"] = 0, rng.integers(0, 4, n), rng.integers(0, 100, n)
    rec["time"] = np.arange(n)
    rec["flags"] = rng.integers(0, 16, n)
    rec["qmax_q16"], rec["ncells"] = rng.integers(64, 16368, n), rng.integers(1, 25, n)
    rec["qtot"] = rng.integers(64, 40000, n) / 16.0
    rec["sigma_pad"] = np.where(rng.random(n) < 0.2, 0.0, rng.random(n)).astype(np.float32)
    rec["sigma_time"] = np.where(rng.random(n) < 0.2, 0.0, rng.random(n)).astype(np.float32)
    cuts = dict(min_qtot=300.0, min_ncells=3, reject_single_pad=True, reject_flags=2)
    want, kept_o = oracle.select(rec.view(oracle.CLUSTER_DTYPE), **cuts)
    assert 0 < kept_o < n
    raw = torch.zeros(n * 32 + 64, dtype=torch.uint8, device="cuda")
    out = torch.zeros(n * 32 + 64, dtype=torch.uint8, device="cuda")
    base_in = raw.data_ptr() + (-raw.data_ptr()) % 32 + in_off
    base_out = out.data_ptr() + (-out.data_ptr()) % 32 + out_off
    o_in, o_out = base_in - raw.data_ptr(), base_out - out.data_ptr()
    raw[o_in: o_in + n * 32] = torch.from_numpy(rec.view(np.uint8).copy()).cuda()
    ctx = T.tpcclus_create([100], n_sectors=1, tf_time_bins=100, max_digits=10)
    try:
        T.tpcclus_select(ctx, base_in, n, base_out, n, torch.cuda.current_stream().cuda_stream, **cuts)
        kept = T.tpcclus_select_result(ctx)
        assert kept == kept_o
        assert out[o_out: o_out + kept * 32].cpu().numpy().tobytes() == want.tobytes()
        word = torch.zeros(1, dtype=torch.int64, device="cuda")
        out.zero_()
        T.tpcclus_select_static(base_in, n, base_out, n, word.data_ptr(), torch.cuda.current_stream().cuda_stream, **cuts)
        torch.cuda.synchronize()
        assert int(word.item()) == kept_o
        assert out[o_out: o_out + kept * 32].cpu().numpy().tobytes() == want.tobytes()
    finally:
        T.tpcclus_destroy(ctx)
