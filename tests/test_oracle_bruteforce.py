"""Pins B1/B2 of SURVEY.md §8(c): the oracle against the independently written set/path-form
checker (tests/bruteforce.py, exact Fractions) on exhaustive 3x3 and 4x4 maps and on random
8x8 maps with forced ties (BASELINE.json:north_star (4): "brute-force enumeration on 8x8
maps").  Many tiny maps are packed as the (sector,row) grid of ONE oracle call, which also
pins I8 (rows and sectors do not couple)."""
import itertools

import numpy as np
import pytest

import bruteforce
import oracle


def pack_maps(maps, side):
    """maps: list of {(pad,time): q16}.  Map m goes to sector m // 256, row m % 256."""
    n_sectors = (len(maps) + 255) // 256
    recs, offs = [], [0]
    for s in range(n_sectors):
        for r in range(256):
            m = s * 256 + r
            if m >= len(maps):
                break
            for (p, t), q in maps[m].items():
                recs.append((r, p, t, q / 16.0))
        offs.append(len(recs))
    d = np.zeros(len(recs), dtype=oracle.DIGIT_DTYPE)
    a = np.array(recs, dtype=np.float64).reshape(-1, 4)
    d["row"], d["pad"], d["time"], d["charge"] = a[:, 0], a[:, 1], a[:, 2], a[:, 3]
    return d, np.array(offs, dtype=np.uint64), n_sectors


def check_maps(maps, side, theta, chunk=4096):
    """Split over worker processes (the Fraction checker is the slow side)."""
    import multiprocessing as mp
    import os
    jobs = [(maps[i:i + chunk], side, theta) for i in range(0, len(maps), chunk)]
    nproc = max(1, min(len(jobs), os.cpu_count() or 1))
    if nproc == 1:
        return sum(_check_chunk(j) for j in jobs)
    with mp.get_context("fork").Pool(nproc) as pool:
        return sum(pool.map(_check_chunk, jobs))


def _check_chunk(job):
    maps, side, theta = job
    d, offs, n_sectors = pack_maps(maps, side)
    out, st = oracle.run(d, offs, [side] * 256, n_sectors=n_sectors, tf_time_bins=side,
                         peak_min_q16=theta)
    assert st["n_duplicates"] == 0 and st["n_digits_dropped"] == 0
    mid = out["sector"].astype(np.int64) * 256 + out["row"]
    bounds = np.searchsorted(mid, np.arange(len(maps) + 1))
    n_checked = 0
    for m, Q in enumerate(maps):
        exp = bruteforce.clusters(Q, theta, side, side)
        got = out[bounds[m]:bounds[m + 1]]
        assert len(got) == len(exp), (m, Q, got, exp)
        for g, e in zip(got, exp):
            assert (g["pad"], g["time"], g["flags"], g["qmax_q16"], g["ncells"]) == \
                   (e["pad"], e["time"], e["flags"], e["qmax_q16"], e["ncells"]), (m, Q, g, e)
            assert abs(float(g["qtot"]) - e["qtot"]) <= 2e-7 * e["qtot"], (m, Q, g, e)
            for f in ("dpad", "dtime", "sigma_pad", "sigma_time"):
                assert abs(float(g[f]) - e[f]) <= 3e-7, (m, Q, f, g, e)
            n_checked += 1
    return n_checked


def test_b1_exhaustive_3x3():
    """All 3^9 = 19683 maps on a 3x3 geometry with charges {0, 5, 9} ADC."""
    cells = [(p, t) for t in range(3) for p in range(3)]
    maps = []
    for combo in itertools.product((0, 80, 144), repeat=9):
        maps.append({c: q for c, q in zip(cells, combo) if q})
    assert len(maps) == 19683
    assert check_maps(maps, 3, 64) > 19000


def test_b1_exhaustive_4x4():
    """All 2^16 maps on 4x4 with charges {0, 7} ADC: every tie pattern on a small board."""
    cells = [(p, t) for t in range(4) for p in range(4)]
    maps = []
    for bits in range(1 << 16):
        maps.append({cells[i]: 112 for i in range(16) if bits >> i & 1})
    assert check_maps(maps, 4, 64) > 60000


@pytest.mark.parametrize("theta", [1, 32, 64])
def test_b2_random_8x8(theta):
    """Random 8x8 maps, charges from a small alphabet so that ties are everywhere; three
    thresholds (1/16, 2 and 4 ADC).  3 x 34000 > 1e5 maps in total."""
    rng = np.random.default_rng(1000 + theta)
    cells = [(p, t) for t in range(8) for p in range(8)]
    alphabet = np.array([0, 0, 0, 16, 32, 48, 64, 80, 96, 200, 16368], dtype=np.int64)
    maps = []
    for m in range(34000):
        fill = rng.choice([0.15, 0.3, 0.5, 0.8])
        q = rng.choice(alphabet[3:], size=64) * (rng.random(64) < fill)
        maps.append({cells[i]: int(q[i]) for i in range(64) if q[i]})
    assert check_maps(maps, 8, theta) > 34000
