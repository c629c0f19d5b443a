"""Pins P1..P9 of SURVEY.md §8(c): the oracle against hand-built maps whose clusters were
worked out by hand (tests/golden/oracle_pins.json), and against closed forms (P8)."""
import json
import math
import os

import numpy as np
import pytest

import oracle
from util import digits_from_cells

HERE = os.path.dirname(os.path.abspath(__file__))
PINS = json.load(open(os.path.join(HERE, "golden", "oracle_pins.json")))["pins"]


def run_pin(pin, order=None):
    cells = [(0, 0, p, t, q) for p, t, q in pin["cells"]]
    if order is not None:
        cells = [cells[i] for i in order]
    d, offs = digits_from_cells(cells)
    return oracle.run(d, offs, [pin["npads"]], n_sectors=1, tf_time_bins=pin["tf_time_bins"],
                      peak_min_q16=int(round(pin["theta_adc"] * 16)))


@pytest.mark.parametrize("pin", PINS, ids=[p["name"] for p in PINS])
def test_pin(pin):
    out, st = run_pin(pin)
    exp = pin["expect"]
    assert st["n_duplicates"] == 0 and st["n_digits_dropped"] == 0
    assert len(out) == len(exp), (pin["name"], out)
    for c, e in zip(out, exp):
        assert (c["pad"], c["time"]) == (e["pad"], e["time"])
        assert c["flags"] == e["flags"]
        assert c["qmax_q16"] == e["qmax_adc"] * 16
        assert c["ncells"] == e["ncells"]
        assert abs(float(c["qtot"]) - e["qtot"]) <= 1e-6 * e["qtot"]
        for f in ("dpad", "dtime", "sigma_pad", "sigma_time"):
            if f in e:
                assert abs(float(c[f]) - e[f]) <= 1e-6, (pin["name"], f, c[f], e[f])
    # reversed digit order gives the same bytes (I3 on the pins)
    out2, _ = run_pin(pin, order=list(range(len(pin["cells"])))[::-1])
    assert out.tobytes() == out2.tobytes()


def test_p9_plateau_moments():
    pin = next(p for p in PINS if p["name"] == "P9")
    out, _ = run_pin(pin)
    s = math.sqrt(2.0 / 3.0)  # three equally weighted positions 0,1,2 -> variance 2/3
    assert abs(float(out[0]["sigma_pad"]) - s) < 1e-6 and abs(float(out[0]["sigma_time"]) - s) < 1e-6


@pytest.mark.parametrize("sp,st_", [(0.8, 1.2), (0.6, 0.9), (1.2, 1.8)])
def test_p8_gaussian_closed_form(sp, st_):
    """P8: noise-free centred Gaussian sampled at cell centres.  By symmetry dpad = dtime = 0
    exactly; by separability sigma_pad = sqrt(sum k^2 g(k) / sum g(k)), k=-2..2, g the 1-D
    Gaussian with the pad width (same for time).  Quantisation to 1/16 ADC moves it by
    < 1e-3.  qtot equals the sum of the quantised 5x5 samples."""
    A = 1000.0
    cells, q55, n55 = [], 0.0, 0
    for dt in range(-6, 7):
        for dp in range(-4, 5):
            v = A * math.exp(-dp * dp / (2 * sp * sp) - dt * dt / (2 * st_ * st_))
            q = round(v * 16) / 16
            if q > 0.0:      # no zero suppression here: the closed form is for the full 5x5
                cells.append((0, 0, 12 + dp, 100 + dt, q))
                if abs(dp) <= 2 and abs(dt) <= 2:
                    q55 += q
                    n55 += 1
    d, offs = digits_from_cells(cells)
    out, _ = oracle.run(d, offs, [24], n_sectors=1, tf_time_bins=200, peak_min_q16=64)
    assert len(out) == 1
    c = out[0]
    assert (c["pad"], c["time"], c["ncells"]) == (12, 100, n55)
    assert c["dpad"] == 0.0 and c["dtime"] == 0.0

    def closed(sig):
        g = [math.exp(-k * k / (2 * sig * sig)) for k in range(-2, 3)]
        return math.sqrt(sum(k * k * gk for k, gk in zip(range(-2, 3), g)) / sum(g))

    assert abs(float(c["sigma_pad"]) - closed(sp)) < 1e-3
    assert abs(float(c["sigma_time"]) - closed(st_)) < 1e-3
    assert abs(float(c["qtot"]) - q55) <= 1e-6 * q55


def test_p8_printed_values():
    """The closed-form numbers SURVEY.md §8(c) P8 prints: 0.795274 (sigma 0.8), 1.081836 (1.2),
    0.592941 (0.6), 0.883815 (0.9), 1.260815 (1.8); qtot 5834.25 for (0.8, 1.2), A = 1000."""
    def closed(sig):
        g = [math.exp(-k * k / (2 * sig * sig)) for k in range(-2, 3)]
        return math.sqrt(sum(k * k * gk for k, gk in zip(range(-2, 3), g)) / sum(g))
    for sig, val in [(0.8, 0.795274), (1.2, 1.081836), (0.6, 0.592941), (0.9, 0.883815), (1.8, 1.260815)]:
        assert abs(closed(sig) - val) < 1e-6
    cells = []
    for dt in range(-2, 3):
        for dp in range(-2, 3):
            v = 1000.0 * math.exp(-dp * dp / (2 * 0.64) - dt * dt / (2 * 1.44))
            cells.append((0, 0, 12 + dp, 100 + dt, round(v * 16) / 16))
    d, offs = digits_from_cells(cells)
    out, _ = oracle.run(d, offs, [24], n_sectors=1, tf_time_bins=200)
    assert abs(float(out[0]["qtot"]) - 5834.25) < 0.07       # printed to 2 decimals
    assert abs(float(out[0]["sigma_pad"]) - 0.795268) < 2e-6  # quantised values printed in P8
    assert abs(float(out[0]["sigma_time"]) - 1.081858) < 2e-6


def test_quantise_d1():
    """D1: rint half-to-even on charge*16, clamp to [0, 16368], NaN and non-positive dropped."""
    assert oracle.quantise(2.0) == 32
    assert oracle.quantise(1023.0) == 16368
    assert oracle.quantise(5000.0) == 16368
    assert oracle.quantise(float("inf")) == 16368
    assert oracle.quantise(float("nan")) == 0
    assert oracle.quantise(-3.0) == 0
    assert oracle.quantise(0.03125) == 0      # 0.5 -> 0 (half to even)
    assert oracle.quantise(0.09375) == 2      # 1.5 -> 2
    assert oracle.quantise(0.15625) == 2      # 2.5 -> 2
    assert oracle.quantise(7.4375) == 119


def test_dropped_and_duplicates_counted():
    cells = [(0, 0, 3, 5, 10.0), (0, 0, 3, 5, 12.0),      # duplicate cell
             (0, 0, 30, 5, 10.0),                          # pad out of range
             (0, 1, 3, 5, 10.0),                           # row out of range
             (0, 0, 3, 300, 10.0),                         # time out of range
             (0, 0, 4, 9, float("nan")), (0, 0, 5, 9, 0.0)]
    d, offs = digits_from_cells(cells)
    out, st = oracle.run(d, offs, [24], n_sectors=1, tf_time_bins=200)
    assert st["n_duplicates"] == 1
    assert st["n_digits_dropped"] == 5
    assert len(out) == 1


def test_capacity_truncates_in_order():
    cells = [(0, 0, 3 + 4 * k, 10 + k, 20.0) for k in range(5)]
    d, offs = digits_from_cells(cells)
    full, st = oracle.run(d, offs, [24], n_sectors=1, tf_time_bins=200)
    part, st2 = oracle.run(d, offs, [24], n_sectors=1, tf_time_bins=200, capacity=3)
    assert st2["n_clusters"] == 5 and len(part) == 3
    assert part.tobytes() == full[:3].tobytes()


def test_order_sector_row_time_pad():
    """D10: records ascend strictly in (sector,row,time,pad)."""
    rng = np.random.default_rng(0)
    cells = []
    for s in range(3):
        for r in range(4):
            for _ in range(20):
                cells.append((s, r, int(rng.integers(0, 20)), int(rng.integers(0, 100)), float(rng.integers(4, 50))))
    # drop duplicate cells
    seen, uniq = set(), []
    for c in cells:
        if c[:4] not in seen:
            seen.add(c[:4]); uniq.append(c)
    d, offs = digits_from_cells(uniq, n_sectors=3)
    out, st = oracle.run(d, offs, [20, 22, 24, 26], n_sectors=3, tf_time_bins=100)
    key = (out["sector"].astype(np.int64) << 40) | (out["row"].astype(np.int64) << 32) | \
          (out["time"].astype(np.int64) << 8) | out["pad"].astype(np.int64)
    assert len(out) > 50 and np.all(np.diff(key) > 0)
