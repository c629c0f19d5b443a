"""Shared test helpers: building digit arrays and comparing cluster lists (D12)."""
import numpy as np

import oracle

INT_FIELDS = ("sector", "row", "pad", "flags", "time", "qmax_q16", "ncells")
POS_FIELDS = ("dpad", "dtime", "sigma_pad", "sigma_time")

QTOT_RTOL = 1e-6   # BASELINE.json:north_star "qTot must match to relative 1e-6"
POS_ATOL = 1e-4    # "Centroids and sigmas must match to absolute 1e-4 pad/time-bin in float32"


def digits_from_cells(cells, n_sectors=1):
    """cells: iterable of (sector, row, pad, time, charge_adc).  Returns (digits, offsets)
    grouped per sector, in the order given inside each sector."""
    per = [[] for _ in range(n_sectors)]
    for s, r, p, t, q in cells:
        per[s].append((r, p, t, q))
    offs = np.zeros(n_sectors + 1, dtype=np.uint64)
    out = []
    for s in range(n_sectors):
        out.extend(per[s])
        offs[s + 1] = len(out)
    d = np.zeros(len(out), dtype=oracle.DIGIT_DTYPE)
    if out:
        a = np.array(out, dtype=np.float64)
        d["row"] = a[:, 0].astype(np.uint8)
        d["pad"] = a[:, 1].astype(np.uint8)
        d["time"] = a[:, 2].astype(np.uint16)
        d["charge"] = a[:, 3].astype(np.float32)
    return d, offs


def permute_within_sectors(digits, offs, rng):
    out = digits.copy()
    for s in range(len(offs) - 1):
        a, b = int(offs[s]), int(offs[s + 1])
        out[a:b] = digits[a:b][rng.permutation(b - a)]
    return out


def assert_clusters_match(got, ref, what=""):
    """D12 comparison rule: integer fields, count and order bit-exact; qtot relative 1e-6;
    dpad, dtime, sigma_pad, sigma_time absolute 1e-4.  `got`/`ref` are structured arrays with
    the cluster fields (any dtype object exposing them by name)."""
    assert len(got) == len(ref), f"{what}: cluster count {len(got)} != {len(ref)}"
    for f in INT_FIELDS:
        g, r = np.asarray(got[f]), np.asarray(ref[f])
        if not np.array_equal(g, r):
            k = int(np.flatnonzero(g != r)[0])
            raise AssertionError(f"{what}: field {f} differs first at record {k}: {g[k]} != {r[k]}"
                                 f" (ref record: {ref[k]})")
    g, r = np.asarray(got["qtot"], dtype=np.float64), np.asarray(ref["qtot"], dtype=np.float64)
    bad = np.abs(g - r) > QTOT_RTOL * np.abs(r)
    assert not bad.any(), f"{what}: qtot off at {np.flatnonzero(bad)[:5]}: {g[bad][:5]} vs {r[bad][:5]}"
    for f in POS_FIELDS:
        g, r = np.asarray(got[f], dtype=np.float64), np.asarray(ref[f], dtype=np.float64)
        bad = ~(np.abs(g - r) <= POS_ATOL)
        assert not bad.any(), f"{what}: {f} off at {np.flatnonzero(bad)[:5]}: {g[bad][:5]} vs {r[bad][:5]}"


def count_bit_mismatches(got, ref):
    """How many records differ in any byte (the tolerance is the gate; this is reported)."""
    a = np.frombuffer(np.ascontiguousarray(got).tobytes(), dtype=np.uint8).reshape(-1, 32)
    b = np.frombuffer(np.ascontiguousarray(ref).tobytes(), dtype=np.uint8).reshape(-1, 32)
    return int((a != b).any(axis=1).sum())
