"""Pins for the two oracle functions that tests/test_oracle_pins.py does not reach directly:

* ``tpc_oracle_peak_flags`` (D4 flag map of one row; BASELINE.json:north_star "peak flags ... must be
  bit-exact against the oracle") — against a separately written, vectorised numpy form of D4 on
  C0 rows 0 / 77 / 151 and against the hand-worked peak cells of the tie maps P4, P4', P5, P9
  (tests/golden/oracle_pins.json; SURVEY.md §8(c) pin table);
* ``tpc_oracle_quantise`` (D1) — against exact rational arithmetic (``fractions.Fraction``,
  round-half-to-even written out by hand) on half-way cases, the clamp, signs, infinities, NaN and
  subnormals.
"""
import json
import math
import os
from fractions import Fraction

import numpy as np
import pytest

import gen
import oracle
from util import digits_from_cells

HERE = os.path.dirname(os.path.abspath(__file__))
PINS = {p["name"]: p for p in json.load(open(os.path.join(HERE, "golden", "oracle_pins.json")))["pins"]}


def numpy_d4(Q, theta):
    """D4 on a zero-padded integer map Q[time, pad]: >= theta, strictly greater than the four
    neighbours earlier in (time, pad) order, >= the four later ones.  Returns a bool map."""
    Z = np.zeros((Q.shape[0] + 2, Q.shape[1] + 2), dtype=np.int64)
    Z[1:-1, 1:-1] = Q
    c = Z[1:-1, 1:-1]
    pk = c >= theta
    for dt, dp, strict in [(-1, -1, 1), (-1, 0, 1), (-1, 1, 1), (0, -1, 1), (0, 1, 0), (1, -1, 0), (1, 0, 0), (1, 1, 0)]:
        nb = Z[1 + dt:Z.shape[0] - 1 + dt, 1 + dp:Z.shape[1] - 1 + dp]
        pk &= (c > nb) if strict else (c >= nb)
    return pk


def test_peak_flags_c0_rows_against_numpy_d4():
    cfg = gen.config(0)
    d, offs, _ = gen.generate_fragment(cfg, 0)
    d = gen.as_numpy_digits(d)
    npads = cfg.npads_array()
    for theta in (64, 32):
        out, _ = oracle.run(d, offs, npads, n_sectors=1, tf_time_bins=cfg.tf_time_bins, peak_min_q16=theta)
        for r in (0, 77, 151):
            flags, q = oracle.peak_flags(d, offs, npads, n_sectors=1, tf_time_bins=cfg.tf_time_bins,
                                         sector=0, row=r, peak_min_q16=theta)
            m = d["row"] == r
            Q = np.zeros((cfg.tf_time_bins, int(npads[r])), dtype=np.int64)
            Q[d["time"][m].astype(int), d["pad"][m].astype(int)] = np.round(d["charge"][m] * 16)
            assert np.array_equal(q.astype(np.int64), Q)
            ref = numpy_d4(Q, theta)
            assert np.array_equal(flags.astype(bool), ref), (theta, r)
            assert ref.sum() > 10
            # and the flag map is exactly the peak set of the cluster list (one record per peak, D10)
            pk = out[out["row"] == r]
            from_records = np.zeros_like(ref)
            from_records[pk["time"].astype(int), pk["pad"].astype(int)] = True
            assert np.array_equal(from_records, ref)


@pytest.mark.parametrize("name", ["P4", "P4prime", "P5", "P5four", "P9", "P3", "P2prime"])
def test_peak_flags_on_tie_pins(name):
    """The hand-worked peak cells of the tie maps: the flag map has exactly those cells set."""
    pin = PINS[name]
    d, offs = digits_from_cells([(0, 0, p, t, q) for p, t, q in pin["cells"]])
    flags, q = oracle.peak_flags(d, offs, [pin["npads"]], n_sectors=1, tf_time_bins=pin["tf_time_bins"],
                                 sector=0, row=0, peak_min_q16=int(round(pin["theta_adc"] * 16)))
    want = {(e["time"], e["pad"]) for e in pin["expect"]}
    got = {(int(t), int(p)) for t, p in zip(*np.nonzero(flags))}
    assert got == want
    for p, t, adc in pin["cells"]:
        assert q[t, p] == int(round(adc * 16))


def test_peak_flags_fragment_window_and_halo():
    """Flags over the loaded range [b-h, e+h): the array starts at b-h and a peak in the halo is flagged
    (flags are a property of the map; ownership D9 is applied to the records, not to the flags)."""
    cells = [(0, 0, 5, 95, 30.0), (0, 0, 5, 100, 40.0), (0, 0, 6, 100, 10.0), (0, 0, 9, 116, 25.0)]
    d, offs = digits_from_cells(cells)
    flags, q = oracle.peak_flags(d, offs, [16], n_sectors=1, tf_time_bins=400, sector=0, row=0,
                                 t_core_begin=100, t_core_end=110, halo_bins=5)
    assert flags.shape == (20, 16)
    assert {(int(t), int(p)) for t, p in zip(*np.nonzero(flags))} == {(0, 5), (5, 5)}   # t = 95, 100; 116 is not loaded
    out, st = oracle.run(d, offs, [16], n_sectors=1, tf_time_bins=400, t_core_begin=100, t_core_end=110, halo_bins=5)
    assert [(int(c["time"]), int(c["pad"])) for c in out] == [(100, 5)] and st["n_digits_dropped"] == 1


# ---------------------------------------------------------------------------------------------
def exact_d1(x: float) -> int:
    """D1 in exact arithmetic: clamp(round_half_even(16 x), 0, 16368); NaN -> 0.  x is a float32
    value (so 16 x is exact in float32 unless it overflows to inf, which clamps anyway)."""
    if math.isnan(x):
        return 0
    if math.isinf(x):
        return 16368 if x > 0 else 0
    v = Fraction(x) * 16
    fl = v.numerator // v.denominator
    rem = v - fl
    if rem > Fraction(1, 2) or (rem == Fraction(1, 2) and fl % 2 == 1):
        fl += 1
    return max(0, min(16368, fl))


def d1_special_values():
    f32 = np.float32
    vals = [0.0, -0.0, 1.0 / 32, 1.0 / 16, 3.0 / 32, 5.0 / 32, 7.0 / 32, 2.0, 2.03125, 2.09375, 1022.96875, 1023.0,
            1023.03125, 1023.5, 1024.0, 5000.0, 3.4e38, float("inf"), float("-inf"), float("nan"), -1.0, -0.03, -1e-30,
            1e-45, 1.1754942e-38, 1e-39, 0.01, 0.03, 0.031, 0.0313, 0.09374999, 0.0937501]
    vals += [float(np.nextafter(f32(1.0 / 32), f32(0))), float(np.nextafter(f32(1.0 / 32), f32(1)))]
    vals += [float(np.nextafter(f32(1023.0), f32(0))), float(np.nextafter(f32(1023.0), f32(2000)))]
    vals += [k / 32.0 for k in range(0, 200)]                       # every half-way case up to 6.2 ADC
    vals += [1000.0 + k / 32.0 for k in range(0, 800, 7)]           # around and beyond the clamp
    return [float(f32(v)) for v in vals]


def test_d1_quantise_against_exact_rationals():
    for v in d1_special_values():
        assert oracle.quantise(v) == exact_d1(v), v
    rng = np.random.default_rng(12)
    bits = rng.integers(0, 2 ** 32, size=20000, dtype=np.uint64).astype(np.uint32)
    for v in bits.view(np.float32)[:20000]:
        assert oracle.quantise(float(v)) == exact_d1(float(v)), v
    for v in rng.uniform(0, 1100, size=20000).astype(np.float32):
        assert oracle.quantise(float(v)) == exact_d1(float(v)), v


def test_d1_through_run_counts_dropped():
    """The run applies D1 before D2: q16 == 0 digits are dropped and counted, the rest fill the map."""
    vals = d1_special_values()
    cells = [(0, 0, i % 200, i // 200, v) for i, v in enumerate(vals)]
    d, offs = digits_from_cells(cells)
    d["charge"] = np.array(vals, dtype=np.float32)                 # digits_from_cells goes through float64
    ntime = len(vals) // 200 + 1
    flags, q = oracle.peak_flags(d, offs, [200], n_sectors=1, tf_time_bins=ntime, sector=0, row=0, peak_min_q16=1)
    want = np.array([exact_d1(v) for v in vals])
    got = np.array([q[i // 200, i % 200] for i in range(len(vals))])
    assert np.array_equal(got, want)
    _, st = oracle.run(d, offs, [200], n_sectors=1, tf_time_bins=ntime, peak_min_q16=1)
    assert st["n_digits_dropped"] == int((want == 0).sum())
