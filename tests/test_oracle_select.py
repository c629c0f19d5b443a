"""Pins of the oracle's selection D13 (reading A20: SURVEY.md §8(f) f-4, cluster-quality cuts as parameters).  The
records come from hand-built maps whose cluster values are worked out by hand in SURVEY.md §8(c) (pins P2, P3, P6,
P7), so what each cut must do to them is known without running anything:

  P7   a single digit of 10 ADC                -> qtot 10, ncells 1, sigma_pad = sigma_time = 0
  P2   pads 10,11,12 = 50,2,3 in one time bin  -> qtot 52, ncells 2, sigma_pad = 5/26, sigma_time = 0
  P3   pads 10..14 = 60,20,10,20,60            -> two clusters, qtot 85 each, ncells 3, SPLIT, sigma_time = 0
  P6   pad 0 = 30, pad 1 = 10 at time 0        -> qtot 40, EDGE_PAD | EDGE_TIME
  2x2  block of 20s (pin P4)                   -> qtot 80, ncells 4, sigma_pad = sigma_time = 0.5
"""
import numpy as np

import oracle
from util import digits_from_cells

NP = [40]


def _records():
    cells = [(0, 0, 20, 100, 10.0),                                                  # P7-like, far from anything else
             (0, 0, 10, 200, 50.0), (0, 0, 11, 200, 2.0), (0, 0, 12, 200, 3.0),      # P2
             (0, 0, 10, 300, 60.0), (0, 0, 11, 300, 20.0), (0, 0, 12, 300, 10.0), (0, 0, 13, 300, 20.0), (0, 0, 14, 300, 60.0),  # P3
             (0, 0, 0, 0, 30.0), (0, 0, 1, 0, 10.0),                                 # P6
             (0, 0, 5, 400, 20.0), (0, 0, 6, 400, 20.0), (0, 0, 5, 401, 20.0), (0, 0, 6, 401, 20.0)]  # P4
    d, offs = digits_from_cells(cells)
    rec, _ = oracle.run(d, offs, NP, n_sectors=1, tf_time_bins=500)
    assert [int(t) for t in rec["time"]] == [0, 100, 200, 300, 300, 400]
    assert rec["qtot"].tolist() == [40.0, 10.0, 52.0, 85.0, 85.0, 80.0]
    return rec


def _times(rec):
    return [(int(t), int(p)) for t, p in zip(rec["time"], rec["pad"])]


def test_no_cut_keeps_everything_in_order():
    rec = _records()
    out, kept = oracle.select(rec)
    assert kept == 6 and out.tobytes() == rec.tobytes()


def test_each_cut_on_hand_worked_records():
    rec = _records()
    out, kept = oracle.select(rec, min_qtot=52.0)                       # >= is inclusive: P2's 52 stays
    assert _times(out) == [(200, 10), (300, 10), (300, 14), (400, 5)] and kept == 4
    out, _ = oracle.select(rec, min_qtot=52.000004)
    assert _times(out) == [(300, 10), (300, 14), (400, 5)]
    out, _ = oracle.select(rec, min_qmax_q16=480)                        # qmax: 30, 10, 50, 60, 60, 20 ADC -> keep >= 30 ADC
    assert _times(out) == [(0, 0), (200, 10), (300, 10), (300, 14)]
    out, _ = oracle.select(rec, min_ncells=3)                            # ncells: 2, 1, 2, 3, 3, 4
    assert _times(out) == [(300, 10), (300, 14), (400, 5)]
    out, _ = oracle.select(rec, reject_single_pad=True)                  # only the lone digit has all weight in one pad
    assert _times(out) == [(0, 0), (200, 10), (300, 10), (300, 14), (400, 5)]
    out, _ = oracle.select(rec, reject_single_time=True)                 # everything in one time bin goes; the 2x2 block stays
    assert _times(out) == [(400, 5)]
    out, _ = oracle.select(rec, reject_flags=oracle.FLAG_SPLIT)
    assert _times(out) == [(0, 0), (100, 20), (200, 10), (400, 5)]
    out, _ = oracle.select(rec, reject_flags=oracle.FLAG_EDGE_PAD | oracle.FLAG_SPLIT)
    assert _times(out) == [(100, 20), (200, 10), (400, 5)]
    out, _ = oracle.select(rec, min_qtot=40.0, reject_single_time=True, min_ncells=4)
    assert _times(out) == [(400, 5)]


def test_capacity_is_an_ordered_prefix_and_kept_is_the_required_count():
    rec = _records()
    out, kept = oracle.select(rec, min_ncells=2, capacity=3)
    assert kept == 5 and _times(out) == [(0, 0), (200, 10), (300, 10)]
    out, kept = oracle.select(rec[:0])
    assert kept == 0 and len(out) == 0


def test_kept_records_are_unchanged_bytes():
    rec = _records()
    out, _ = oracle.select(rec, min_qtot=50.0)
    want = rec[rec["qtot"] >= 50.0]
    assert out.tobytes() == want.tobytes()
