"""-m gpu parity on RANDOM GEOMETRIES (seeded): the fixed configs of BASELINE.json all have 152 rows of 66..138 pads and
4096-bin fragments; this fuzz draws what they never exercise together — rows of 1, 2, 7..9, 31..33, 255, 256 pads, time
frames of 1 to 2600 bins, cores of 1 / 255 / 256 / 257 / ... bins with halos of 5..13, thresholds from 1/16 ADC to
18.75 ADC, occupancies from 2 % to 60 %, tie-heavy charges, invalid digits (dropped and counted), both binning kernels —
and compares every fragment's records BYTE FOR BYTE with the oracle's (which implies D12's tolerances).

Inputs are built here with numpy (no method arithmetic: random cells, charges from a small alphabet of 1/16-ADC values).
"""
import numpy as np
import pytest

import oracle
from gpu_util import GpuClusterizer, to_device_digits

pytestmark = pytest.mark.gpu

PADS = [1, 2, 3, 7, 8, 9, 15, 16, 17, 31, 32, 33, 63, 64, 65, 100, 138, 140, 255, 256]
TFS = [1, 6, 255, 256, 257, 511, 700, 1500, 2600]
CORES = [1, 100, 255, 256, 257, 300, 512, 1 << 20]
Q16 = np.array([7, 16, 17, 32, 48, 64, 65, 80, 96, 200, 1000, 4800, 16368, 16500], dtype=np.float64)   # 16500 clamps to 16368


def _case(seed):
    rng = np.random.default_rng(424242 + seed)
    n_sectors, n_rows = int(rng.integers(1, 5)), int(rng.integers(1, 33))
    npads = rng.choice(PADS, size=n_rows).astype(np.int64)
    tf = int(rng.choice(TFS))
    occ = float(rng.choice([0.02, 0.1, 0.3, 0.6]))
    occ = min(occ, 2.5e5 / float(n_sectors * int(npads.sum()) * tf))          # at most ~250 000 digits per case
    parts, offs = [], [0]
    for _ in range(n_sectors):
        rows, pads, times = [], [], []
        for r in range(n_rows):
            cells = int(npads[r]) * tf
            k = int(rng.binomial(cells, occ))
            idx = rng.choice(cells, size=k, replace=False)                     # distinct cells: no duplicate digits (A11)
            rows.append(np.full(k, r)), pads.append(idx % npads[r]), times.append(idx // npads[r])
        row, pad, time = (np.concatenate(x) if x else np.zeros(0, dtype=np.int64) for x in (rows, pads, times))
        n = len(row)
        d = np.zeros(n, dtype=oracle.DIGIT_DTYPE)
        d["row"], d["pad"], d["time"] = row, pad, time
        d["charge"] = (rng.choice(Q16, size=n) / 16.0).astype(np.float32)
        bad = rng.random(n) < 0.01                                             # dropped and counted (D1), in three ways
        kind = rng.integers(0, 3, size=n)
        d["charge"][bad & (kind == 0)] = 0.0
        d["row"][bad & (kind == 1)] = min(255, n_rows)                         # a row beyond the geometry (255: may exist)
        wide = npads[row] < 256                                                # (a 256-pad row has no pad beyond it in 8 bits)
        m2 = bad & (kind == 2) & wide
        d["pad"][m2] = npads[row][m2]                                          # the first pad beyond the row
        parts.append(d[rng.permutation(n)])
        offs.append(offs[-1] + n)
    core = min(int(rng.choice(CORES)), tf)
    return dict(npads=[int(x) for x in npads], n_sectors=n_sectors, tf=tf, theta=int(rng.choice([1, 16, 64, 300])),
                halo=int(rng.choice([5, 6, 8, 13])), core=core, direct=bool(seed % 3 == 0),
                digits=np.concatenate(parts) if parts else np.zeros(0, dtype=oracle.DIGIT_DTYPE),
                offs=np.array(offs, dtype=np.uint64), rng=rng)


@pytest.mark.parametrize("seed", range(40))
def test_random_geometry_matches_the_oracle(seed):
    import paper_2412_13755_b200 as T

    c = _case(seed)
    dn, offs, tf, core = c["digits"], c["offs"], c["tf"], c["core"]
    starts = list(range(0, tf, core))
    if len(starts) > 6:                                                        # first, last and four random fragments
        mid = sorted(int(x) for x in c["rng"].choice(starts[1:-1], size=4, replace=False))
        starts = [starts[0]] + mid + [starts[-1]]
    dd = to_device_digits(dn)
    total = 0
    with GpuClusterizer(c["npads"], n_sectors=c["n_sectors"], tf_time_bins=tf, max_core_bins=core, halo_bins=c["halo"],
                        peak_min_q16=c["theta"], max_digits=max(len(dn), 1), bin_occupancy_pct=100,
                        options=T.TPCCLUS_OPT_BIN_DIRECT if c["direct"] else 0) as g:
        for b in starts:
            e = min(tf, b + core)
            got, st = g.run(dd, offs, b, e)
            ref, ost = oracle.run(dn, offs, c["npads"], n_sectors=c["n_sectors"], tf_time_bins=tf, t_core_begin=b,
                                  t_core_end=e, halo_bins=c["halo"], peak_min_q16=c["theta"])
            what = f"seed {seed}: {c['n_sectors']} sectors, pads {c['npads']}, tf {tf}, core [{b},{e}), halo {c['halo']}, theta {c['theta']}"
            assert ost["n_duplicates"] == 0, what
            assert st["n_digits_dropped"] == ost["n_digits_dropped"], what
            assert st["n_clusters"] == ost["n_clusters"] == len(ref), what
            assert got.tobytes() == ref.tobytes(), what
            total += len(ref)
    assert total > 0 or len(dn) < 50, (seed, len(dn))
