"""-m gpu parity at BASELINE.json's FULL sizes (BJ:north_star: "bit-exact ... clusters versus the oracle on all
5 configs"): C2 and C4 whole (36 sectors x 4096 bins), and fragments 0, 6 and 13 of the C3 time frame with all 36
sectors — the first fragment (TF start, no lower halo), a middle one (halos on both sides) and the ragged last one
(3776 bins, true TF end).  C0 and C1 at full size are in test_gpu_parity.py.

The CUDA path runs once over the whole fragment, in the launch configuration bench.py times (one context, one
run, all sectors); the oracle runs sector by sector on the host cores (sectors are independent, D-rules are per
sector and row), and the two record lists are compared byte for byte per sector — which implies D12's rule
(integer fields, count and order bit-exact; floats within 1e-6 relative / 1e-4 absolute)."""
import os
from concurrent.futures import ThreadPoolExecutor

import numpy as np
import pytest

import gen
import oracle
from gpu_util import GpuClusterizer
from util import assert_clusters_match

pytestmark = pytest.mark.gpu
THETA = 64


def _oracle_by_sector(cfg, dn, offs, b, e, theta=THETA):
    npads = cfg.npads_array()

    def one(s):
        a, z = int(offs[s]), int(offs[s + 1])
        rec, st = oracle.run(dn[a:z], np.array([0, z - a], dtype=np.uint64), npads, n_sectors=1,
                             tf_time_bins=cfg.tf_time_bins, t_core_begin=b, t_core_end=e,
                             halo_bins=cfg.halo_bins, peak_min_q16=theta)
        assert st["n_duplicates"] == 0 and st["n_digits_dropped"] == 0
        return rec

    with ThreadPoolExecutor(max_workers=os.cpu_count() or 1) as ex:
        return list(ex.map(one, range(cfg.n_sectors)))


def _check_fragment(cfg, f, g, min_records):
    b, e = cfg.fragments()[f]
    d, offs, info = gen.generate_fragment(cfg, f, device="cuda", row_chunk=64)
    got, st = g.run(d, offs, b, e)
    assert st["n_digits_dropped"] == 0
    dn = gen.as_numpy_digits(d)
    del d
    refs = _oracle_by_sector(cfg, dn, offs, b, e)
    assert sum(len(r) for r in refs) == st["n_clusters"] == len(got) > min_records
    bounds = np.searchsorted(got["sector"], np.arange(cfg.n_sectors + 1))
    for s, ref in enumerate(refs):
        part = got[bounds[s]: bounds[s + 1]].copy()
        assert np.all(part["sector"] == s)
        part["sector"] = 0                                    # the oracle ran this sector as sector 0
        if part.tobytes() != ref.tobytes():
            assert_clusters_match(part, ref, f"{cfg.name} fragment {f} sector {s}")   # says which field differs
            raise AssertionError(f"{cfg.name} fragment {f} sector {s}: records within tolerance but not bit-identical")
    return len(got), len(dn)


@pytest.mark.parametrize("index,min_records", [(2, 1.0e7), (4, 4.0e7)])
def test_full_size_fragment_configs(index, min_records):
    """BASELINE.json:configs[2] and configs[4], all 36 sectors."""
    cfg = gen.config(index)
    with GpuClusterizer(cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins,
                        max_core_bins=cfg.core_bins, halo_bins=cfg.halo_bins, peak_min_q16=THETA,
                        max_digits=1 << 30) as g:
        _check_fragment(cfg, 0, g, min_records)


def test_full_size_tf_fragments_first_middle_last():
    """BASELINE.json:configs[3]: fragments 0, 6 and 13 (of 14) of the 57024-bin time frame, 36 sectors each,
    through ONE context (the digit bins are reused from fragment to fragment, as in bench.py)."""
    cfg = gen.config(3)
    frs = cfg.fragments()
    assert len(frs) == 14 and frs[13] == (53248, 57024)
    with GpuClusterizer(cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins,
                        max_core_bins=cfg.core_bins, halo_bins=cfg.halo_bins, peak_min_q16=THETA,
                        max_digits=1 << 30) as g:
        for f in (0, 6, 13):
            _check_fragment(cfg, f, g, 9.0e6)
