"""Pins of the oracle's time base (reading A19): a time frame longer than 65536 bins keeps the
8-byte digit of BASELINE.json:configs[0] — its u16 time field counts from a per-run base, global time =
t_time_base + digit.time ("256 orbits needs a 32-bit digit time"; §4: TFs of
up to 256 orbits = 114048 bins were tested).  Nothing here calls the CUDA path.

What fixes the arithmetic without another implementation:
* translation (I4): the same charge pattern placed at global times around 70000 / 100000 (base 69000 / 99000) and
  around 1000 (base 0, which the P1..P9 pins and the brute-force checker cover) gives the same records, times
  shifted by the difference;
* base independence: the same set of global digits expressed against two different bases gives the same bytes;
* I7 across the 16-bit boundary: fragments whose seam lies at bin 65536, each with its own base, concatenate to
  the monolithic run;
* the TF-end flag and the loaded range use GLOBAL time: EDGE_TIME at bin 114047 of a 114048-bin TF, digits
  outside [b - halo, e + halo) are dropped whatever the base.
"""
import numpy as np
import pytest

import oracle
from util import digits_from_cells

NP = [40, 17]


def _pattern(rng, n_blobs, t_lo, t_hi):
    """cells {(row, pad, t_global): charge}: blobs with ties, some saturated."""
    cells = {}
    for _ in range(n_blobs):
        r = int(rng.integers(len(NP)))
        pc, tc = int(rng.integers(NP[r])), int(rng.integers(t_lo, t_hi))
        for _ in range(10):
            p, t = pc + int(rng.integers(-2, 3)), tc + int(rng.integers(-3, 4))
            if 0 <= p < NP[r] and t_lo <= t < t_hi:
                q = float(rng.integers(32, 3000)) / 16.0
                if rng.random() < 0.2:
                    q = 12.5
                if rng.random() < 0.03:
                    q = 1023.0
                cells[(r, p, t)] = q
    return cells


def _digits(cells, base):
    return digits_from_cells([(0, r, p, t - base, q) for (r, p, t), q in cells.items()])


@pytest.mark.parametrize("shift,base", [(69000, 69000), (69000, 68500), (99000, 65536), (112000, 111999)])
def test_translation_to_times_beyond_16_bits(shift, base):
    rng = np.random.default_rng(shift + base)
    cells = _pattern(rng, 120, 20, 1400)
    d0, offs = _digits(cells, 0)
    ref, st0 = oracle.run(d0, offs, NP, n_sectors=1, tf_time_bins=114048, t_core_begin=10, t_core_end=1450, halo_bins=8)
    moved = {(r, p, t + shift): q for (r, p, t), q in cells.items()}
    d1, _ = _digits(moved, base)
    got, st1 = oracle.run(d1, offs, NP, n_sectors=1, tf_time_bins=114048, t_core_begin=10 + shift,
                          t_core_end=1450 + shift, halo_bins=8, t_time_base=base)
    assert len(ref) > 100 and st0["n_digits_dropped"] == st1["n_digits_dropped"] == 0
    want = ref.copy()
    want["time"] += shift
    assert got.tobytes() == want.tobytes()


def test_records_do_not_depend_on_the_base():
    rng = np.random.default_rng(5)
    cells = _pattern(rng, 150, 66000, 67000)
    outs = []
    for base in (66000 - 40, 65000, 3000):                    # 67000 - 3000 = 64000 still fits the u16 field
        d, offs = _digits(cells, base)
        rec, st = oracle.run(d, offs, NP, n_sectors=1, tf_time_bins=114048, t_core_begin=66000, t_core_end=67000,
                             halo_bins=8, t_time_base=base)
        assert st["n_digits_dropped"] == 0
        outs.append(rec.tobytes())
    assert outs[0] == outs[1] == outs[2] and len(outs[0]) > 100 * 32


def test_fragments_with_their_own_bases_concatenate_across_bin_65536():
    """I7 with the seam exactly at the 16-bit boundary."""
    rng = np.random.default_rng(9)
    cells = _pattern(rng, 400, 65000, 66100)
    d, offs = _digits(cells, 64990)
    mono, _ = oracle.run(d, offs, NP, n_sectors=1, tf_time_bins=114048, t_core_begin=65000, t_core_end=66100,
                         halo_bins=0, t_time_base=64990)
    parts = []
    for (b, e) in [(65000, 65536), (65536, 65537), (65537, 66100)]:
        base = max(0, b - 8)                                   # every cell time (>= 65000) fits the u16 field from here
        df, _ = _digits(cells, base)
        rec, st = oracle.run(df, offs, NP, n_sectors=1, tf_time_bins=114048, t_core_begin=b, t_core_end=e,
                             halo_bins=8, t_time_base=base)
        parts.append(rec)
    got = np.concatenate(parts)
    k = np.lexsort((got["pad"], got["time"], got["row"]))
    assert len(mono) > 300 and got[k].tobytes() == mono.tobytes()
    assert (mono["time"] >= 65536).any() and (mono["time"] < 65536).any()


def test_tf_end_flag_and_loaded_range_use_global_time():
    tf = 114048
    base = tf - 300
    cells = [(0, 0, 10, tf - 1 - base, 30.0), (0, 0, 11, tf - 1 - base, 10.0),      # at the true TF end: EDGE_TIME
             (0, 0, 20, tf - 40 - base, 30.0),                                      # well inside
             (0, 1, 5, tf - 120 - base, 50.0),                                      # below b - halo: dropped
             (0, 1, 6, tf - 108 - base, 9.0)]                                       # in the halo: loaded, not emitted
    d, offs = digits_from_cells(cells)
    rec, st = oracle.run(d, offs, NP, n_sectors=1, tf_time_bins=tf, t_core_begin=tf - 100, t_core_end=tf,
                         halo_bins=8, t_time_base=base)
    assert st["n_digits_dropped"] == 1 and len(rec) == 2
    assert rec["time"].tolist() == [tf - 40, tf - 1]
    assert rec["flags"].tolist() == [0, oracle.FLAG_EDGE_TIME]
    assert rec["qtot"].tolist() == [30.0, 40.0]
    # the same digits read against base 0 would sit at times < 300: all outside the loaded range
    rec0, st0 = oracle.run(d, offs, NP, n_sectors=1, tf_time_bins=tf, t_core_begin=tf - 100, t_core_end=tf, halo_bins=8)
    assert len(rec0) == 0 and st0["n_digits_dropped"] == 5
