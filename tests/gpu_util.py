"""Helpers for the -m gpu parity tests: run the CUDA path through the C-ABI binding."""
import numpy as np

import oracle


def to_device_digits(digits):
    """numpy structured digits or a uint8 [n,8] tensor -> uint8 [n,8] CUDA tensor."""
    import torch

    if isinstance(digits, np.ndarray):
        raw = np.ascontiguousarray(digits).view(np.uint8).reshape(-1, 8)
        return torch.from_numpy(raw.copy()).cuda()
    return digits.cuda()


class GpuClusterizer:
    """One context; run(...) returns the records as a numpy structured array."""

    def __init__(self, npads, *, n_sectors, tf_time_bins, max_core_bins=None, halo_bins=0, peak_min_q16=64,
                 max_digits, options=0, max_clusters=0, bin_occupancy_pct=0):
        import paper_2412_13755_b200 as T

        self.T = T
        self.ctx = T.tpcclus_create(npads, n_sectors=n_sectors, tf_time_bins=tf_time_bins,
                                    max_core_bins=max_core_bins, halo_bins=halo_bins,
                                    peak_min_q16=peak_min_q16, options=options,
                                    max_digits=max(int(max_digits), 1), max_clusters=max_clusters,
                                    bin_occupancy_pct=bin_occupancy_pct)

    def close(self):
        if self.ctx:
            self.T.tpcclus_destroy(self.ctx)
            self.ctx = None

    def __enter__(self):
        return self

    def __exit__(self, *a):
        self.close()

    def run(self, d_digits, offs, b, e, capacity=None, check=True, t_time_base=0):
        """d_digits: uint8 [n,8] CUDA tensor.  capacity None: count first (capacity 0), then
        run again with exactly the required capacity."""
        import torch

        T = self.T
        n = int(d_digits.shape[0])
        stream = torch.cuda.current_stream().cuda_stream
        if capacity is None:
            T.tpcclus_run_based(self.ctx, d_digits.data_ptr(), n, offs, t_time_base, b, e, 0, 0, stream)
            st = T.tpcclus_result(self.ctx, check=False)
            assert st["status"] in (T.TPCCLUS_OK, T.TPCCLUS_ERR_CAPACITY), st
            capacity = int(st["n_clusters"])
        out = torch.zeros((max(capacity, 1), 32), dtype=torch.uint8, device="cuda")
        T.tpcclus_run_based(self.ctx, d_digits.data_ptr(), n, offs, t_time_base, b, e, out.data_ptr(), capacity, stream)
        st = T.tpcclus_result(self.ctx, check=check)
        k = min(int(st["n_clusters"]), capacity)
        rec = out[:k].cpu().numpy().view(T.CLUSTER_DTYPE).reshape(-1)
        return rec, st


def gpu_clusters(digits, offs, npads, *, n_sectors, tf_time_bins, t_core_begin=0, t_core_end=None, halo_bins=0,
                 peak_min_q16=64, options=0, bin_occupancy_pct=0):
    if t_core_end is None:
        t_core_end = tf_time_bins
    d = to_device_digits(digits)
    with GpuClusterizer(npads, n_sectors=n_sectors, tf_time_bins=tf_time_bins,
                        max_core_bins=t_core_end - t_core_begin, halo_bins=halo_bins,
                        peak_min_q16=peak_min_q16, max_digits=d.shape[0], options=options,
                        bin_occupancy_pct=bin_occupancy_pct) as g:
        return g.run(d, offs, t_core_begin, t_core_end)


def oracle_clusters(digits, offs, npads, **kw):
    if not isinstance(digits, np.ndarray):
        digits = digits.cpu().numpy().view(oracle.DIGIT_DTYPE).reshape(-1)
    return oracle.run(digits, offs, npads, **kw)
