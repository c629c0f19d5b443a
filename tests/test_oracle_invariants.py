"""Invariants I1..I9 of SURVEY.md §8(c) on generated workloads (BASELINE.json:north_star (4):
"total clustered charge never exceeds total digit charge, peaks are local maxima, and results
do not change when the input digits are permuted")."""
import numpy as np
import pytest

import gen
import oracle
from util import digits_from_cells, permute_within_sectors


@pytest.fixture(scope="module")
def c0():
    cfg = gen.config(0)
    d, offs, info = gen.generate_fragment(cfg, 0)
    return cfg, gen.as_numpy_digits(d), offs, info


def run_cfg(cfg, d, offs, **kw):
    return oracle.run(d, offs, cfg.npads_array(), n_sectors=cfg.n_sectors,
                      tf_time_bins=cfg.tf_time_bins, **kw)


def test_c0_shape(c0):
    """BASELINE.json:configs[0]: ~3e5 digits, charges multiples of 1/16 in [2,1023]."""
    cfg, d, offs, info = c0
    assert 2.5e5 < len(d) < 3.5e5
    assert d["charge"].min() >= 2.0 and d["charge"].max() <= 1023.0
    assert np.all(d["charge"] * 16 == np.round(d["charge"] * 16))
    cell = (d["row"].astype(np.int64) << 32) | (d["time"].astype(np.int64) << 8) | d["pad"]
    assert len(np.unique(cell)) == len(d)          # one digit per cell (D2 precondition)


def test_i1_charge_conservation(c0):
    """I1: sum_W <= 2520 * sum q16, exactly, for several thresholds; in floats sum qtot <= sum charge."""
    cfg, d, offs, _ = c0
    for theta in (32, 64, 160):
        out, st = run_cfg(cfg, d, offs, peak_min_q16=theta)
        assert st["n_duplicates"] == 0 and st["n_digits_dropped"] == 0
        assert st["sum_W"] <= 2520 * st["sum_q16_loaded"]
        assert out["qtot"].astype(np.float64).sum() <= d["charge"].astype(np.float64).sum() * (1 + 1e-6)
    # with theta = ZS threshold every digit is a peak or adjacent to a larger cell; still <=
    assert st["sum_W"] > 0


def test_i2_peaks_are_local_maxima(c0):
    """I2: every emitted peak re-checked against a freshly built numpy map; no two peaks adjacent."""
    cfg, d, offs, _ = c0
    out, _ = run_cfg(cfg, d, offs)
    npads = cfg.npads_array()
    for r in (0, 77, 151):
        Q = np.zeros((cfg.tf_time_bins + 2, int(npads[r]) + 2), dtype=np.int64)
        m = d["row"] == r
        Q[d["time"][m].astype(int) + 1, d["pad"][m].astype(int) + 1] = np.round(d["charge"][m] * 16)
        pk = out[out["row"] == r]
        assert len(pk) > 10
        pos = set()
        for c in pk:
            t, p = int(c["time"]) + 1, int(c["pad"]) + 1
            q = Q[t, p]
            assert q == c["qmax_q16"] and q >= 64
            # strictly greater than the 4 earlier neighbours, >= the 4 later ones (D4)
            assert q > Q[t - 1, p - 1] and q > Q[t - 1, p] and q > Q[t - 1, p + 1] and q > Q[t, p - 1]
            assert q >= Q[t, p + 1] and q >= Q[t + 1, p - 1] and q >= Q[t + 1, p] and q >= Q[t + 1, p + 1]
            pos.add((t, p))
        for t, p in pos:
            assert not any((t + a, p + b) in pos for a in (-1, 0, 1) for b in (-1, 0, 1) if (a, b) != (0, 0))
        # and the count: every cell that satisfies D4 is in the list
        inner = Q[1:-1, 1:-1]
        is_pk = inner >= 64
        for a, b, strict in [(-1, -1, 1), (-1, 0, 1), (-1, 1, 1), (0, -1, 1), (0, 1, 0), (1, -1, 0), (1, 0, 0), (1, 1, 0)]:
            nb = Q[1 + a:Q.shape[0] - 1 + a, 1 + b:Q.shape[1] - 1 + b]
            is_pk &= (inner > nb) if strict else (inner >= nb)
        assert int(is_pk.sum()) == len(pk)


def test_i3_permutation_invariance(c0):
    cfg, d, offs, _ = c0
    ref, _ = run_cfg(cfg, d, offs)
    rng = np.random.default_rng(7)
    out, _ = run_cfg(cfg, permute_within_sectors(d, offs, rng), offs)
    assert out.tobytes() == ref.tobytes()


def test_i4_translation():
    """I4: translating all digits away from the edges translates the clusters, rest identical."""
    cfg = gen.config(0, n_rows=4, tf_time_bins=256, core_bins=256, clusters_per_row=15)
    d, offs, _ = gen.generate_fragment(cfg, 0)
    d = gen.as_numpy_digits(d)
    npads = cfg.npads_array()
    keep = (d["pad"] >= 8) & (d["pad"] < npads[d["row"]] - 14) & (d["time"] >= 8) & (d["time"] < 200)
    d = d[keep]
    offs = np.array([0, len(d)], dtype=np.uint64)
    a, _ = run_cfg(cfg, d, offs)
    d2 = d.copy()
    d2["pad"] += 5
    d2["time"] += 17
    b, _ = run_cfg(cfg, d2, offs)
    assert len(a) == len(b) > 20
    b2 = b.copy()
    b2["pad"] -= 5
    b2["time"] -= 17
    assert a.tobytes() == b2.tobytes()


def test_i5_scaling():
    """I5: charges x2 (no saturation, theta x2): same peaks/members, qmax and qtot double,
    offsets and sigmas bit-identical."""
    cfg = gen.config(0, n_rows=4, tf_time_bins=256, core_bins=256, clusters_per_row=15)
    d, offs, _ = gen.generate_fragment(cfg, 0)
    d = gen.as_numpy_digits(d)
    d = d[d["charge"] < 500.0]
    offs = np.array([0, len(d)], dtype=np.uint64)
    a, _ = run_cfg(cfg, d, offs, peak_min_q16=64)
    d2 = d.copy()
    d2["charge"] *= 2
    b, _ = run_cfg(cfg, d2, offs, peak_min_q16=128)
    assert len(a) == len(b) > 20
    for f in ("sector", "row", "pad", "time", "ncells", "dpad", "dtime", "sigma_pad", "sigma_time"):
        assert np.array_equal(a[f], b[f]), f
    assert np.array_equal(a["qmax_q16"].astype(int) * 2, b["qmax_q16"])
    assert np.array_equal(a["qtot"] * 2, b["qtot"])


def test_i6_mirror_tie_free():
    """I6: mirroring the pad axis on a tie-free map: dpad -> -dpad, everything else identical."""
    rng = np.random.default_rng(3)
    npad, T = 30, 60
    vals = rng.permutation(np.arange(40, 40 + npad * T))           # all charges distinct: no ties
    occ = rng.random(npad * T) < 0.3
    cells = [(0, 0, i % npad, i // npad, vals[i] / 16.0) for i in range(npad * T) if occ[i]]
    d, offs = digits_from_cells(cells)
    a, _ = oracle.run(d, offs, [npad], n_sectors=1, tf_time_bins=T)
    d2 = d.copy()
    d2["pad"] = npad - 1 - d["pad"]
    b, _ = oracle.run(d2, offs, [npad], n_sectors=1, tf_time_bins=T)
    assert len(a) == len(b) > 10
    ka = {(int(c["time"]), int(c["pad"])): c for c in a}
    for c in b:
        m = ka[(int(c["time"]), npad - 1 - int(c["pad"]))]
        assert (m["qmax_q16"], m["ncells"], m["flags"]) == (c["qmax_q16"], c["ncells"], c["flags"])
        assert m["qtot"] == c["qtot"] and m["dtime"] == c["dtime"] and m["dpad"] == -c["dpad"]
        assert m["sigma_pad"] == c["sigma_pad"] and m["sigma_time"] == c["sigma_time"]


@pytest.mark.parametrize("name", ["c3mini"])
def test_i7_fragmented_equals_monolithic(name):
    """I7 / D9: fragmented run (core 512, halo 8; ragged last core) == monolithic run."""
    cfg = gen.config(name, n_sectors=1)
    mono_cfg = gen.config(name, n_sectors=1, core_bins=cfg.tf_time_bins, halo_bins=0)
    d, offs, _ = gen.generate_fragment(mono_cfg, 0)
    ref, _ = run_cfg(mono_cfg, gen.as_numpy_digits(d), offs)
    parts = []
    for f, (b, e) in enumerate(cfg.fragments()):
        df, of, info = gen.generate_fragment(cfg, f)
        out, st = run_cfg(cfg, gen.as_numpy_digits(df), of, t_core_begin=b, t_core_end=e,
                          halo_bins=cfg.halo_bins)
        assert st["n_digits_dropped"] == 0
        parts.append(out)
    got = np.concatenate(parts)
    # a TF's canonical list is the fragments' lists concatenated (D10): same SET as the
    # monolithic list; compare after sorting both by (sector,row,time,pad)
    def key(x):
        return np.lexsort((x["pad"], x["time"], x["row"], x["sector"]))
    assert len(got) == len(ref)
    assert got[key(got)].tobytes() == ref[key(ref)].tobytes()


def test_i7_core_sizes_and_halo5():
    """I7: any core size >= 1 with halo >= 5 reproduces the monolithic result."""
    cfg = gen.config(0, n_rows=3, tf_time_bins=200, core_bins=200, clusters_per_row=25)
    d, offs, _ = gen.generate_fragment(cfg, 0)
    d = gen.as_numpy_digits(d)
    ref, _ = run_cfg(cfg, d, offs)
    for core, halo in [(1, 5), (7, 5), (64, 8), (199, 6)]:
        parts = []
        for b in range(0, 200, core):
            e = min(200, b + core)
            out, _ = run_cfg(cfg, d, offs, t_core_begin=b, t_core_end=e, halo_bins=halo)
            parts.append(out)
        got = np.concatenate(parts)
        k = np.lexsort((got["pad"], got["time"], got["row"], got["sector"]))
        assert got[k].tobytes() == ref.tobytes(), (core, halo)


def test_i7_halo4_is_not_enough():
    """The bound of D9 is tight: peak at core time e-1, member at e+1, a would-be peak at e+3
    that a larger cell at e+4 disqualifies.  With halo 4 the cell at e+4 is not loaded, e+3
    looks like a peak, the member at e+1 is shared (S=2) and qtot changes; halo 5 is exact."""
    e = 50
    cells = [(0, 0, 10, e - 1, 40.0), (0, 0, 10, e, 20.0), (0, 0, 10, e + 1, 10.0),
             (0, 0, 10, e + 3, 30.0), (0, 0, 10, e + 4, 35.0)]
    d, offs = digits_from_cells(cells)
    mono, _ = oracle.run(d, offs, [24], n_sectors=1, tf_time_bins=200)
    c_ref = mono[mono["time"] == e - 1][0]
    h5, _ = oracle.run(d, offs, [24], n_sectors=1, tf_time_bins=200, t_core_begin=0, t_core_end=e, halo_bins=5)
    h4, _ = oracle.run(d, offs, [24], n_sectors=1, tf_time_bins=200, t_core_begin=0, t_core_end=e, halo_bins=4)
    assert h5[h5["time"] == e - 1][0].tobytes() == c_ref.tobytes()
    assert c_ref["qtot"] == 70.0
    assert h4[h4["time"] == e - 1][0]["qtot"] == 65.0          # member at e+1 halved


def test_i8_rows_and_sectors_do_not_couple():
    cfg = gen.config("c2mini", tf_time_bins=128, core_bins=128)
    d, offs, _ = gen.generate_fragment(cfg, 0)
    d = gen.as_numpy_digits(d)
    ref, _ = run_cfg(cfg, d, offs)
    s, r = 1, 100
    sl = d[int(offs[1]):int(offs[2])]
    only = sl[sl["row"] == r]
    o2 = np.array([0, 0, len(only)], dtype=np.uint64)
    out, _ = run_cfg(cfg, only, o2)
    want = ref[(ref["sector"] == s) & (ref["row"] == r)]
    assert len(want) > 5 and out.tobytes() == want.tobytes()


def test_i9_field_ranges(c0):
    cfg, d, offs, _ = c0
    out, _ = run_cfg(cfg, d, offs)
    key = (out["row"].astype(np.int64) << 32) | (out["time"].astype(np.int64) << 8) | out["pad"]
    assert np.all(np.diff(key) > 0)
    assert out["ncells"].min() >= 1 and out["ncells"].max() <= 25
    qmax = out["qmax_q16"] / 16.0
    assert np.all(qmax <= out["qtot"] * (1 + 1e-6)) and np.all(out["qtot"] <= 25 * qmax * (1 + 1e-6))
    assert np.all(np.abs(out["dpad"]) < 2) and np.all(np.abs(out["dtime"]) < 2)
    assert np.all(out["sigma_pad"] <= 2) and np.all(out["sigma_time"] <= 2)
    single = out[out["ncells"] == 1]
    for f in ("dpad", "dtime", "sigma_pad", "sigma_time"):
        assert np.all(single[f] == 0)


def test_i10_physics_soft(c0):
    """I10 (soft, reported): clusters found ~ clusters generated (40 per row x 152 rows) plus
    noise peaks; at theta = 4 ADC the count is within a factor of the generated number."""
    cfg, d, offs, _ = c0
    out, _ = run_cfg(cfg, d, offs)
    assert 0.5 * 40 * 152 < len(out) < 2.0 * 40 * 152
