"""-m gpu parity tests: the CUDA path (through the C-ABI binding) against the oracle, element by
element on the same seeded inputs, under the comparison rule D12 of SURVEY.md §8(c):
integer fields, count and order bit-exact; qtot relative 1e-6; offsets and sigmas absolute 1e-4
(BASELINE.json:north_star)."""
import json
import os

import numpy as np
import pytest

import gen
import oracle
from gpu_util import GpuClusterizer, gpu_clusters, oracle_clusters, to_device_digits
from util import assert_clusters_match, count_bit_mismatches, digits_from_cells, permute_within_sectors

pytestmark = pytest.mark.gpu
HERE = os.path.dirname(os.path.abspath(__file__))


def both(digits, offs, npads, **kw):
    got, st = gpu_clusters(digits, offs, npads, **kw)
    ref, ost = oracle_clusters(digits, offs, npads, **kw)
    assert st["n_clusters"] == ost["n_clusters"]
    assert st["n_digits_dropped"] == ost["n_digits_dropped"]
    return got, ref, st


PINS = json.load(open(os.path.join(HERE, "golden", "oracle_pins.json")))["pins"]


@pytest.mark.parametrize("pin", PINS, ids=[p["name"] for p in PINS])
def test_pins_on_gpu(pin):
    """The hand-built maps P1..P9 through the CUDA path: same records as the oracle, bit for bit."""
    d, offs = digits_from_cells([(0, 0, p, t, q) for p, t, q in pin["cells"]])
    got, ref, _ = both(d, offs, [pin["npads"]], n_sectors=1, tf_time_bins=pin["tf_time_bins"],
                       peak_min_q16=int(round(pin["theta_adc"] * 16)))
    assert len(got) == len(pin["expect"])
    assert_clusters_match(got, ref, pin["name"])
    assert got.tobytes() == ref.tobytes()


@pytest.mark.parametrize("theta", [1, 32, 64])
def test_random_8x8_maps(theta):
    """60000 random 8x8 maps with forced ties (the B2 family), packed as a 235 x 256 (sector,row)
    grid of one run: tiny geometry, pad edges and time edges everywhere."""
    rng = np.random.default_rng(2000 + theta)
    n_maps, side = 60000, 8
    alphabet = np.array([16, 32, 48, 64, 80, 96, 200, 16368], dtype=np.int64)
    n_sectors = (n_maps + 255) // 256
    q = rng.choice(alphabet, size=(n_maps, side, side))
    fill = rng.choice([0.15, 0.3, 0.5, 0.8], size=n_maps)
    keep = rng.random((n_maps, side, side)) < fill[:, None, None]
    m, t, p = np.nonzero(keep)
    d = np.zeros(len(m), dtype=oracle.DIGIT_DTYPE)
    d["row"], d["pad"], d["time"] = m % 256, p, t
    d["charge"] = q[m, t, p] / 16.0
    offs = np.searchsorted(m // 256, np.arange(n_sectors + 1)).astype(np.uint64)
    got, ref, _ = both(d, offs, [side] * 256, n_sectors=n_sectors, tf_time_bins=side, peak_min_q16=theta)
    assert len(ref) > n_maps
    assert_clusters_match(got, ref, "8x8")
    assert count_bit_mismatches(got, ref) == 0


def run_config(name, theta=64, **over):
    cfg = gen.config(name, **over)
    parts_g, parts_o = [], []
    with GpuClusterizer(cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins,
                        max_core_bins=cfg.core_bins, halo_bins=cfg.halo_bins, peak_min_q16=theta,
                        max_digits=1 << 28) as g:
        for f, (b, e) in enumerate(cfg.fragments()):
            d, offs, info = gen.generate_fragment(cfg, f, device="cuda")
            got, st = g.run(d, offs, b, e)
            ref, ost = oracle_clusters(d, offs, cfg.npads_array(), n_sectors=cfg.n_sectors,
                                       tf_time_bins=cfg.tf_time_bins, t_core_begin=b, t_core_end=e,
                                       halo_bins=cfg.halo_bins, peak_min_q16=theta)
            assert ost["n_duplicates"] == 0
            assert st["n_clusters"] == ost["n_clusters"] and st["n_digits_dropped"] == ost["n_digits_dropped"] == 0
            assert_clusters_match(got, ref, f"{cfg.name} fragment {f}")
            parts_g.append(got)
            parts_o.append(ref)
    return cfg, np.concatenate(parts_g), np.concatenate(parts_o)


@pytest.mark.parametrize("theta", [64, 32])
def test_c0_tiny(theta):
    """BASELINE.json:configs[0], full size, theta = 4 ADC and theta = ZS threshold (D11)."""
    cfg, got, ref = run_config(0, theta)
    assert len(ref) > 3000
    assert count_bit_mismatches(got, ref) == 0


def test_c1_pp_sector():
    """BASELINE.json:configs[1], full size (1 sector x 4096 bins, ~2.2e6 digits)."""
    cfg, got, ref = run_config(1)
    assert len(ref) > 30000
    assert count_bit_mismatches(got, ref) == 0


@pytest.mark.parametrize("name,theta", [("c2mini", 64), ("c4mini", 64), ("c4mini", 32)])
def test_pbpb_and_stress_minis(name, theta):
    """The C2 and C4 generators on 2 sectors (several tiles per row, ragged last tile)."""
    cfg, got, ref = run_config(name, theta)
    assert len(ref) > 1e5
    assert count_bit_mismatches(got, ref) == 0
    if name == "c4mini":
        assert (ref["flags"] & 8).any() and (ref["flags"] & 4).any() and (ref["flags"] & 1).any()


def test_c3mini_fragmented_tf():
    """configs[3] in small: 3 fragments (512,512,476 bins) with an 8-bin halo; the concatenated
    fragment lists equal the monolithic oracle run (D9/D10, invariant I7)."""
    cfg, got, ref = run_config("c3mini")
    mono = gen.config("c3mini", core_bins=cfg.tf_time_bins, halo_bins=0)
    d, offs, _ = gen.generate_fragment(mono, 0, device="cuda")
    full, _ = oracle_clusters(d, offs, mono.npads_array(), n_sectors=mono.n_sectors, tf_time_bins=mono.tf_time_bins)
    k = np.lexsort((got["pad"], got["time"], got["row"], got["sector"]))
    assert_clusters_match(got[k], full, "fragmented vs monolithic")


def test_determinism_and_permutation():
    """I3 + the determinism guarantee: two runs and a permuted-input run are byte-identical."""
    cfg = gen.config("c4mini", tf_time_bins=300, core_bins=300)
    d, offs, _ = gen.generate_fragment(cfg, 0, device="cuda")
    dn = gen.as_numpy_digits(d)
    a, _ = gpu_clusters(dn, offs, cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins)
    b, _ = gpu_clusters(dn, offs, cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins)
    p = permute_within_sectors(dn, offs, np.random.default_rng(5))
    c, _ = gpu_clusters(p, offs, cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins)
    assert len(a) > 1e4 and a.tobytes() == b.tobytes() == c.tobytes()
    key = (a["sector"].astype(np.int64) << 48) | (a["row"].astype(np.int64) << 40) | \
          (a["time"].astype(np.int64) << 8) | a["pad"]
    assert np.all(np.diff(key) > 0)


def test_odd_core_sizes_and_halo():
    """Any core size with halo >= 5 (ragged tiles, core of 1 bin, core not a multiple of the tile)."""
    cfg = gen.config(0, n_rows=5, tf_time_bins=700, core_bins=700, clusters_per_row=120)
    d, offs, _ = gen.generate_fragment(cfg, 0)
    dn = gen.as_numpy_digits(d)
    dd = to_device_digits(dn)
    npads = cfg.npads_array()
    for core, halo in [(1, 5), (129, 5), (257, 8), (700, 0)]:
        with GpuClusterizer(npads, n_sectors=1, tf_time_bins=700, max_core_bins=core, halo_bins=halo,
                            max_digits=len(dn)) as g:
            for b in ([0, 313, 699] if core == 1 else range(0, 700, core)):
                e = min(700, b + core)
                got, st = g.run(dd, offs, b, e)
                ref, ost = oracle.run(dn, offs, npads, n_sectors=1, tf_time_bins=700, t_core_begin=b,
                                      t_core_end=e, halo_bins=halo)
                assert st["n_digits_dropped"] == ost["n_digits_dropped"]
                assert_clusters_match(got, ref, f"core {core} halo {halo} b {b}")
                assert got.tobytes() == ref.tobytes()


def test_empty_and_degenerate_inputs():
    import paper_2412_13755_b200 as T

    npads = [10, 1, 246]
    empty = np.zeros(0, dtype=oracle.DIGIT_DTYPE)
    got, st = gpu_clusters(empty, np.zeros(3, dtype=np.uint64), npads, n_sectors=2, tf_time_bins=40)
    assert len(got) == 0 and st["n_clusters"] == 0
    # single digit in the widest row's last pad, last time bin; a 1-pad row; dropped digits
    cells = [(1, 2, 245, 39, 9.0), (0, 1, 0, 0, 5.0), (0, 1, 0, 1, 5.0), (0, 0, 10, 3, 50.0),
             (0, 3, 1, 1, 50.0), (1, 0, 2, 40, 50.0), (1, 0, 3, 3, float("nan")), (1, 0, 4, 3, 0.01)]
    d, offs = digits_from_cells(cells, n_sectors=2)
    got, ref, st = both(d, offs, npads, n_sectors=2, tf_time_bins=40)
    assert st["n_digits_dropped"] == 5 and len(ref) == 2
    assert got.tobytes() == ref.tobytes()
    # strict mode turns dropped digits into an error
    with GpuClusterizer(npads, n_sectors=2, tf_time_bins=40, max_digits=16,
                        options=T.TPCCLUS_OPT_STRICT_DIGITS) as g:
        _, st = g.run(to_device_digits(d), offs, 0, 40, capacity=8, check=False)
        assert st["status"] == T.TPCCLUS_ERR_DIGIT


def test_capacity_overflow_is_ordered_prefix():
    """ERR_CAPACITY: the first out_capacity records are valid and ordered, n_clusters = required."""
    import paper_2412_13755_b200 as T

    cfg = gen.config(0, n_rows=6, tf_time_bins=256, core_bins=256, clusters_per_row=60)
    d, offs, _ = gen.generate_fragment(cfg, 0)
    dn = gen.as_numpy_digits(d)
    ref, _ = oracle.run(dn, offs, cfg.npads_array(), n_sectors=1, tf_time_bins=256)
    with GpuClusterizer(cfg.npads_array(), n_sectors=1, tf_time_bins=256, max_digits=len(dn)) as g:
        got, st = g.run(to_device_digits(dn), offs, 0, 256, capacity=100, check=False)
    assert st["status"] == T.TPCCLUS_ERR_CAPACITY and st["n_clusters"] == len(ref) > 100
    assert got.tobytes() == ref[:100].tobytes()


def test_invalid_arguments():
    import torch
    import paper_2412_13755_b200 as T

    with pytest.raises(T.TpcclusError) as ei:
        T.tpcclus_create([10, 300], n_sectors=1, tf_time_bins=100, max_digits=10)
    assert ei.value.code == T.TPCCLUS_ERR_GEOMETRY
    with pytest.raises(T.TpcclusError) as ei:
        T.tpcclus_create([10], n_sectors=1, tf_time_bins=100, halo_bins=3, max_digits=10)
    assert ei.value.code == T.TPCCLUS_ERR_GEOMETRY
    ctx = T.tpcclus_create([10], n_sectors=1, tf_time_bins=100, max_core_bins=50, max_digits=10)
    try:
        buf = torch.zeros(64, dtype=torch.uint8, device="cuda")
        offs = np.array([0, 2], dtype=np.uint64)
        for args in [(buf.data_ptr(), 2, offs, 0, 60, 0, 0),             # core larger than max_core_bins
                     (buf.data_ptr(), 2, offs, 90, 120, 0, 0),           # core outside the TF
                     (buf.data_ptr(), 2, np.array([0, 1], dtype=np.uint64), 0, 50, 0, 0),  # off[n] != n
                     (buf.data_ptr() + 4, 2, offs, 0, 50, 0, 0),         # misaligned digits
                     (buf.data_ptr(), 11, np.array([0, 11], dtype=np.uint64), 0, 50, 0, 0)]:  # n > max_digits
            with pytest.raises(T.TpcclusError) as ei:
                T.tpcclus_run(ctx, *args)
            assert ei.value.code == T.TPCCLUS_ERR_INVALID
    finally:
        T.tpcclus_destroy(ctx)


def test_host_api_single_and_tf():
    """tpcclus_run_host / tpcclus_run_tf_host: host buffers in, host records out, fragments
    concatenated in order (D10)."""
    import paper_2412_13755_b200 as T

    cfg = gen.config("c3mini", n_sectors=2)
    frs, keep, refs = [], [], []
    for f, (b, e) in enumerate(cfg.fragments()):
        d, offs, _ = gen.generate_fragment(cfg, f)
        dn = gen.as_numpy_digits(d)
        keep.append(dn)
        frs.append((dn.ctypes.data, len(dn), offs, b, e))
        ref, _ = oracle.run(dn, offs, cfg.npads_array(), n_sectors=2, tf_time_bins=cfg.tf_time_bins,
                            t_core_begin=b, t_core_end=e, halo_bins=8)
        refs.append(ref)
    total = sum(len(r) for r in refs)
    ctx = T.tpcclus_create(cfg.npads_array(), n_sectors=2, tf_time_bins=cfg.tf_time_bins, max_core_bins=512,
                           halo_bins=8, options=T.TPCCLUS_OPT_HOST_STAGING,
                           max_digits=max(len(k) for k in keep), max_clusters=max(len(r) for r in refs) + 10)
    try:
        out = np.zeros(total, dtype=T.CLUSTER_DTYPE)
        stats = T.tpcclus_run_tf_host(ctx, frs, out.ctypes.data, total)
        assert [s["n_clusters"] for s in stats] == [len(r) for r in refs]
        assert out.tobytes() == np.concatenate(refs).tobytes()
        one = np.zeros(len(refs[1]), dtype=T.CLUSTER_DTYPE)
        st = T.tpcclus_run_host(ctx, keep[1], frs[1][2], frs[1][3], frs[1][4], one)
        assert st["n_clusters"] == len(refs[1]) and one.tobytes() == refs[1].tobytes()
        assert T.tpcclus_launch_count(ctx) == 3 * 4 and T.tpcclus_device_bytes(ctx) > 0
    finally:
        T.tpcclus_destroy(ctx)


def _sorted_within_sectors(dn, offs, keys):
    out = dn.copy()
    for s in range(len(offs) - 1):
        a, b = int(offs[s]), int(offs[s + 1])
        seg = dn[a:b]
        out[a:b] = seg[np.lexsort(tuple(seg[k] for k in reversed(keys)))]
    return out


@pytest.mark.parametrize("order", ["row_time_pad", "time_row_pad", "reverse"])
def test_sorted_digit_orders(order):
    """Digit order inside a sector slice is arbitrary.  Sorted input is the worst
    case for the write-combining binning kernel: a whole chunk of consecutive digits falls into one
    or two bins (ranks far beyond a buffer, several sectors reserved at once, time-major order puts
    every digit of a chunk next to a bin seam).  Output must be byte-identical to the shuffled run
    and to the oracle."""
    cfg = gen.config("c2mini", tf_time_bins=600, core_bins=600)
    d, offs, _ = gen.generate_fragment(cfg, 0, device="cuda")
    dn = gen.as_numpy_digits(d)
    if order == "row_time_pad":
        sn = _sorted_within_sectors(dn, offs, ["row", "time", "pad"])
    elif order == "time_row_pad":
        sn = _sorted_within_sectors(dn, offs, ["time", "row", "pad"])
    else:
        sn = _sorted_within_sectors(dn, offs, ["row", "time", "pad"])
        for s in range(len(offs) - 1):
            a, b = int(offs[s]), int(offs[s + 1])
            sn[a:b] = sn[a:b][::-1]
    kw = dict(n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins)
    shuffled, _ = gpu_clusters(dn, offs, cfg.npads_array(), **kw)
    got, st = gpu_clusters(sn, offs, cfg.npads_array(), **kw)
    ref, ost = oracle.run(dn, offs, cfg.npads_array(), **kw)
    assert len(ref) > 1e4 and st["n_digits_dropped"] == ost["n_digits_dropped"] == 0
    assert got.tobytes() == shuffled.tobytes()
    assert_clusters_match(got, ref, order)


def test_unaligned_digit_buffer_and_sector_seams():
    """The digit buffer only has to be 8-byte aligned; sector slices may start on odd digits, so the
    16-byte pairs at slice seams hold digits of two sectors (k_bin's slot_lo / slot_hi logic)."""
    import torch

    cfg = gen.config("c2mini", tf_time_bins=300, core_bins=300)
    d, offs, _ = gen.generate_fragment(cfg, 0, device="cuda")
    dn = gen.as_numpy_digits(d)
    # drop one digit of sector 0 so that sector 1 starts on an odd index; then shift the buffer by 8 bytes
    dn2 = np.concatenate([dn[:1], dn[2:]])
    offs2 = np.array(offs, dtype=np.uint64).copy()
    offs2[1:] -= 1
    ref, _ = oracle.run(dn2, offs2, cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins)
    for shift in (0, 1):
        raw = torch.zeros((len(dn2) + shift + 1, 8), dtype=torch.uint8, device="cuda")
        view = raw[shift: shift + len(dn2)]
        view.copy_(to_device_digits(dn2))
        assert view.data_ptr() % 8 == 0 and (view.data_ptr() - raw.data_ptr()) == 8 * shift
        with GpuClusterizer(cfg.npads_array(), n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins,
                            max_digits=len(dn2)) as g:
            got, st = g.run(view, offs2, 0, cfg.tf_time_bins)
        assert st["n_digits_dropped"] == 0
        assert got.tobytes() == ref.tobytes(), shift


def test_direct_binning_fallback_matches():
    """k_bin_direct (taken when a geometry's bins do not fit the write-combining kernel's shared
    memory; forced here with TPCCLUS_OPT_BIN_DIRECT) gives the same bytes."""
    import paper_2412_13755_b200 as T

    cfg = gen.config("c4mini", tf_time_bins=300, core_bins=300)
    d, offs, _ = gen.generate_fragment(cfg, 0, device="cuda")
    dn = gen.as_numpy_digits(d)
    kw = dict(n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins)
    a, _ = gpu_clusters(dn, offs, cfg.npads_array(), **kw)
    b, _ = gpu_clusters(dn, offs, cfg.npads_array(), options=T.TPCCLUS_OPT_BIN_DIRECT, **kw)
    ref, _ = oracle.run(dn, offs, cfg.npads_array(), **kw)
    assert len(a) > 1e4 and a.tobytes() == b.tobytes() == ref.tobytes()


def test_bin_occupancy_sizing_and_overflow_error():
    """The digit bins are sized from geometry.bin_occupancy_pct (scratch is sized ahead with a
    safety margin).  100 % can never overflow; the default (50 %) holds the 35 % stress config; a context sized
    for 2 % reports TPCCLUS_ERR_OCCUPANCY on it — a defined error, not a fault — and works again on sparse input."""
    import paper_2412_13755_b200 as T

    cfg = gen.config("c4mini", tf_time_bins=600, core_bins=600)
    d, offs, _ = gen.generate_fragment(cfg, 0, device="cuda")
    dn = gen.as_numpy_digits(d)
    npads = cfg.npads_array()
    kw = dict(n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins)
    ref, _ = oracle.run(dn, offs, npads, **kw)
    sizes = {}
    for pct in (0, 100, 40):
        with GpuClusterizer(npads, max_digits=len(dn), bin_occupancy_pct=pct, **kw) as g:
            got, st = g.run(d, offs, 0, cfg.tf_time_bins)
            sizes[pct] = T.tpcclus_device_bytes(g.ctx)
        assert st["status"] == 0 and got.tobytes() == ref.tobytes(), pct
    assert sizes[40] < sizes[0] < sizes[100]
    sparse, so = digits_from_cells([(0, 3, 5, 17, 30.0), (1, 9, 2, 400, 9.0)], n_sectors=2)
    with GpuClusterizer(npads, max_digits=len(dn), bin_occupancy_pct=2, **kw) as g:
        _, st = g.run(d, offs, 0, cfg.tf_time_bins, capacity=len(ref), check=False)
        assert st["status"] == T.TPCCLUS_ERR_OCCUPANCY and st["cuda_error"] == 0
        got, st = g.run(to_device_digits(sparse), so, 0, cfg.tf_time_bins)
        want, _ = oracle.run(sparse, so, npads, **kw)
        assert st["status"] == 0 and len(want) == 2 and got.tobytes() == want.tobytes()
    with pytest.raises(T.TpcclusError) as ei:
        T.tpcclus_create(npads, max_digits=10, bin_occupancy_pct=101, **kw)
    assert ei.value.code == T.TPCCLUS_ERR_GEOMETRY


@pytest.mark.parametrize("name,rows", [(0, [0, 77, 151]), ("c4mini", [0, 40, 151]), ("c3mini", [3, 100])])
def test_peak_flags_cell_by_cell(name, rows):
    """BJ:north_star: "peak flags ... must be bit-exact against the oracle".  The library emits exactly one record
    per peak of the core (D10), so its D4 flag map is the set of its records' (time, pad): rebuilt per
    (sector,row) and fragment and compared cell by cell with tpc_oracle_peak_flags (the oracle's steps 1-2)."""
    cfg = gen.config(name)
    npads = cfg.npads_array()
    with GpuClusterizer(npads, n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins, max_core_bins=cfg.core_bins,
                        halo_bins=cfg.halo_bins, max_digits=1 << 28) as g:
        for f, (b, e) in enumerate(cfg.fragments()):
            d, offs, _ = gen.generate_fragment(cfg, f, device="cuda")
            got, _ = g.run(d, offs, b, e)
            dn = gen.as_numpy_digits(d)
            lo = max(0, b - cfg.halo_bins)
            n_flags = 0
            for s in range(cfg.n_sectors):
                for r in rows:
                    want, _q = oracle.peak_flags(dn, offs, npads, n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins,
                                                 sector=s, row=r, t_core_begin=b, t_core_end=e, halo_bins=cfg.halo_bins)
                    want = want[b - lo: e - lo]                          # D9: only the core's peaks emit
                    mine = np.zeros_like(want)
                    k = got[(got["sector"] == s) & (got["row"] == r)]
                    assert np.all((k["time"] >= b) & (k["time"] < e))
                    mine[k["time"].astype(np.int64) - b, k["pad"]] = 1
                    assert int(mine.sum()) == len(k)                      # no two records on one cell
                    assert np.array_equal(mine, want != 0), (f, s, r)
                    n_flags += int(mine.sum())
            assert n_flags > 50


def _d1_fuzz_charges(rng, n):
    """float32 charges that exercise every branch of D1: half-way cases of the 1/16 grid (round-half-even), values
    one ulp either side of them, the ZS / zero boundary 1/32, the clamp at 1023, negatives, -0.0, tiny and
    subnormal values, infinities, NaN and huge values."""
    f32 = np.float32
    k = rng.integers(0, 16400, size=n)                                     # 16 * half = k + 0.5, up to just past the clamp
    half = ((2 * k + 1) / 32.0).astype(f32)                                # exactly between two grid points
    kind = rng.integers(0, 12, size=n)
    out = np.empty(n, dtype=f32)
    special = np.array([1e-30, -1e-30, -0.0, 0.0, -3.5, np.inf, -np.inf, np.nan, 1e-40, -1e-40, 5000.0, 3e38,
                        1022.96875, 1023.0, 1023.03125, 16367.5 / 16, 16368.5 / 16, 1.0 / 32, 3.0 / 32, 0.5 / 16],
                       dtype=f32)
    near = np.array([1.0 / 32, 1023.0, 16367.5 / 16, 1022.96875, 0.09375, 2.0], dtype=f32)
    for i in range(12):
        m = kind == i
        c = int(m.sum())
        if i < 3:
            out[m] = half[m]
        elif i == 3:
            out[m] = np.nextafter(half[m], f32(np.inf))
        elif i == 4:
            out[m] = np.nextafter(half[m], f32(-np.inf))
        elif i == 5:
            out[m] = rng.choice(special, size=c)
        elif i == 6:
            b = rng.choice(near, size=c)
            steps = rng.integers(-3, 4, size=c)
            v = b.copy()
            for _ in range(3):
                up = steps > 0
                dn = steps < 0
                v[up] = np.nextafter(v[up], f32(np.inf))
                v[dn] = np.nextafter(v[dn], f32(-np.inf))
                steps = steps - np.sign(steps)
            out[m] = v
        elif i == 7:
            out[m] = rng.uniform(0.0, 40.0, size=c).astype(f32)            # off-grid ordinary values
        elif i == 8:
            out[m] = rng.uniform(1000.0, 1050.0, size=c).astype(f32)       # around the clamp
        elif i == 9:
            out[m] = rng.uniform(0.0, 0.2, size=c).astype(f32)             # around the zero boundary
        elif i == 10:
            out[m] = -rng.uniform(0.0, 10.0, size=c).astype(f32)
        else:
            out[m] = (rng.integers(32, 16368, size=c) / 16.0).astype(f32)  # on the grid
    return out


def test_d1_quantisation_fuzz_through_the_cuda_path():
    """D1 on the CUDA path beyond the 1/16 grid: 1.3e6 digits on distinct cells whose charges hit the half-way
    cases, both clamps, signs, infinities, NaN and subnormals; records and n_digits_dropped equal the oracle's
    (whose quantiser is pinned against exact rationals in test_oracle_peakflags_d1.py).  The same input in
    STRICT mode is the error TPCCLUS_ERR_DIGIT."""
    import paper_2412_13755_b200 as T

    rng = np.random.default_rng(77)
    n_sectors, n_rows, w, nt, n = 2, 64, 128, 300, 1_300_000
    cell = rng.choice(n_sectors * n_rows * w * nt, size=n, replace=False)
    cell.sort()
    d = np.zeros(n, dtype=oracle.DIGIT_DTYPE)
    d["pad"] = cell % w
    d["time"] = (cell // w) % nt
    d["row"] = (cell // (w * nt)) % n_rows
    sec = cell // (w * nt * n_rows)
    d["charge"] = _d1_fuzz_charges(rng, n)
    offs = np.searchsorted(sec, np.arange(n_sectors + 1)).astype(np.uint64)
    d = permute_within_sectors(d, offs, rng)
    npads = [w] * n_rows
    for theta in (1, 64):
        got, ref, st = both(d, offs, npads, n_sectors=n_sectors, tf_time_bins=nt, peak_min_q16=theta)
        assert st["n_digits_dropped"] > 0.1 * n and len(ref) > 1e4
        assert (ref["flags"] & 4).any()
        assert got.tobytes() == ref.tobytes()
    with GpuClusterizer(npads, n_sectors=n_sectors, tf_time_bins=nt, max_digits=n,
                        options=T.TPCCLUS_OPT_STRICT_DIGITS) as g:
        _, st = g.run(to_device_digits(d), offs, 0, nt, capacity=8, check=False)
        assert st["status"] == T.TPCCLUS_ERR_DIGIT


def _random_cells(rng, n_sectors, npads, t_lo, t_hi, n, max_q=400.0):
    """n random distinct cells with charges on the 1/16 ADC grid (some saturated, some tied)."""
    cells = {}
    rows = len(npads)
    while len(cells) < n:
        s = int(rng.integers(n_sectors)); r = int(rng.integers(rows))
        p = int(rng.integers(npads[r])); t = int(rng.integers(t_lo, t_hi))
        q = float(rng.integers(32, int(max_q * 16))) / 16.0
        if rng.random() < 0.05:
            q = 1023.0
        if rng.random() < 0.2:
            q = 20.0                               # exact ties
        cells[(s, r, p, t)] = q
    return [(s, r, p, t, q) for (s, r, p, t), q in cells.items()]


def test_maximum_geometry():
    """Largest geometry the ABI accepts: 256 rows of up to 256 pads (a 1-pad row too), a 65536-bin time
    frame, fragments at its very end and with the largest halo-free core (one CTA per SM: the 266 x 264
    charge map takes most of the shared memory).  Dense random blobs so that peaks touch, split and saturate."""
    rng = np.random.default_rng(11)
    npads = [256] * 256
    npads[3] = 1
    npads[200] = 17
    # blobs of cells around random centres (clusters of touching cells)
    cells = {}
    for _ in range(900):
        s = int(rng.integers(2)); r = int(rng.choice([0, 3, 77, 200, 255]))
        pc = int(rng.integers(npads[r])); tc = int(rng.integers(65536 - 700, 65536))
        for _ in range(12):
            p = pc + int(rng.integers(-2, 3)); t = tc + int(rng.integers(-3, 4))
            if 0 <= p < npads[r] and 65536 - 700 <= t < 65536:
                q = 1023.0 if rng.random() < 0.03 else float(rng.integers(32, 4000)) / 16.0
                cells[(s, r, p, t)] = q
    d, offs = digits_from_cells([(s, r, p, t, q) for (s, r, p, t), q in cells.items()], n_sectors=2)
    dd = to_device_digits(d)
    for core, halo, spans in [(300, 8, [(65236, 65536), (64936, 65236)]), (700, 0, [(64836, 65536)])]:
        with GpuClusterizer(npads, n_sectors=2, tf_time_bins=65536, max_core_bins=core, halo_bins=halo,
                            max_digits=len(d)) as g:
            for b, e in spans:
                got, st = g.run(dd, offs, b, e)
                ref, ost = oracle.run(d, offs, npads, n_sectors=2, tf_time_bins=65536, t_core_begin=b,
                                      t_core_end=e, halo_bins=halo)
                assert st["n_digits_dropped"] == ost["n_digits_dropped"]
                assert len(ref) > 100
                assert_clusters_match(got, ref, f"max geometry core {core} [{b},{e})")
                assert got.tobytes() == ref.tobytes()


def test_duplicate_cells_are_memory_safe_and_context_survives():
    """D2's precondition (one digit per cell) violated massively: the result is unspecified, but the
    library must neither fault nor leave the context unusable (bins are bounded; overfull bins drop)."""
    npads = [8, 8]
    n = 200_000
    d = np.zeros(n, dtype=oracle.DIGIT_DTYPE)
    d["row"] = 1
    d["pad"] = 3
    d["time"] = 7
    d["charge"] = 10.0
    offs = np.array([0, n], dtype=np.uint64)
    good_cells = [(0, 0, 2, 5, 9.0), (0, 0, 3, 5, 30.0), (0, 1, 4, 20, 12.0)]
    dg, og = digits_from_cells(good_cells, n_sectors=1)
    with GpuClusterizer(npads, n_sectors=1, tf_time_bins=64, max_digits=n) as g:
        _, st = g.run(to_device_digits(d), offs, 0, 64, capacity=16, check=False)
        assert st["cuda_error"] == 0
        got, st = g.run(to_device_digits(dg), og, 0, 64)
        ref, _ = oracle.run(dg, og, npads, n_sectors=1, tf_time_bins=64)
        assert st["status"] == 0 and got.tobytes() == ref.tobytes() and len(ref) == 2


def test_many_small_sectors():
    """200 sectors (more than k_bin has CTAs) of uneven, partly empty digit slices: CTAs cross sector
    boundaries between chunks (buffer flush + re-reservation per sector), 16-byte pairs straddle slices."""
    rng = np.random.default_rng(23)
    npads = [20, 33, 7]
    n_sectors = 200
    cells = {}
    for s in range(n_sectors):
        if s % 7 == 3:
            continue                                     # empty slice
        for _ in range(int(rng.integers(1, 60))):
            r = int(rng.integers(3)); pc = int(rng.integers(npads[r])); tc = int(rng.integers(0, 300))
            for _ in range(6):
                p = pc + int(rng.integers(-1, 2)); t = tc + int(rng.integers(-2, 3))
                if 0 <= p < npads[r] and 0 <= t < 300:
                    cells[(s, r, p, t)] = float(rng.integers(32, 3000)) / 16.0
    d, offs = digits_from_cells([(s, r, p, t, q) for (s, r, p, t), q in cells.items()], n_sectors=n_sectors)
    got, ref, st = both(d, offs, npads, n_sectors=n_sectors, tf_time_bins=300)
    assert len(ref) > 2000 and st["n_digits_dropped"] == 0
    assert got.tobytes() == ref.tobytes()


def test_two_contexts_with_different_geometries_coexist():
    """Shared-memory limits are per kernel function, not per context: a small context created after a
    large one must not break the large one (and vice versa)."""
    rng = np.random.default_rng(3)
    big_np, small_np = [256, 200], [12]
    cb = _random_cells(rng, 1, big_np, 0, 120, 1500)
    cs = _random_cells(rng, 1, small_np, 0, 50, 200)
    db, ob = digits_from_cells(cb, n_sectors=1)
    ds, os_ = digits_from_cells(cs, n_sectors=1)
    with GpuClusterizer(big_np, n_sectors=1, tf_time_bins=120, max_digits=len(db)) as gb:
        with GpuClusterizer(small_np, n_sectors=1, tf_time_bins=50, max_digits=len(ds)) as gs:
            got_b, _ = gb.run(to_device_digits(db), ob, 0, 120)
            got_s, _ = gs.run(to_device_digits(ds), os_, 0, 50)
            got_b2, _ = gb.run(to_device_digits(db), ob, 0, 120)
    ref_b, _ = oracle.run(db, ob, big_np, n_sectors=1, tf_time_bins=120)
    ref_s, _ = oracle.run(ds, os_, small_np, n_sectors=1, tf_time_bins=50)
    assert got_b.tobytes() == ref_b.tobytes() == got_b2.tobytes() and len(ref_b) > 50
    assert got_s.tobytes() == ref_s.tobytes() and len(ref_s) > 5


def test_checked_build_runs_clean():
    """The -DTPCCLUS_CHECKED build (device asserts on every shared-memory / list index of k_bin and k_tile; the
    repo's stand-in for compute-sanitizer memcheck, which is closed on this GPU pool) runs the sanitizer cases —
    smoke, C0, dense C4, time-sorted input, the direct binning kernel, a fragmented TF — without tripping an
    assert and with records identical to the oracle's."""
    import subprocess
    import sys

    p = subprocess.run([sys.executable, os.path.join(HERE, "sanitizer_cases.py"), "--checked"], capture_output=True,
                       text=True, timeout=900)
    assert p.returncode == 0, (p.stdout[-1500:], p.stderr[-1500:])
    assert "sanitizer cases done" in p.stdout


def test_peak_lattice_denser_than_a_list_segment():
    """The densest peak pattern D4 allows — a digit on every second pad of every second time bin, all of them
    peaks — gives k_tile thousands of peaks per tile: many hand-over items per tile, and more peaks per 32 core
    rows than a count warp's peak-list segment holds (the per-item list path)."""
    rng = np.random.default_rng(41)
    npads = [128, 21, 256]
    cells = []
    for r, w in enumerate(npads):
        for t in range(0, 300, 2):
            for p in range(r % 2, w, 2):
                cells.append((0, r, p, t, float(rng.integers(64, 16000)) / 16.0))
    # a second sector: the same lattice thinned out at random, plus neighbours that make some peaks share cells
    for (s, r, p, t, q) in list(cells):
        if rng.random() < 0.5:
            cells.append((1, r, p, t, q))
            if rng.random() < 0.3 and p + 1 < npads[r]:
                cells.append((1, r, p + 1, t, 2.5))
    d, offs = digits_from_cells(cells, n_sectors=2)
    for theta in (64, 1):
        got, ref, st = both(d, offs, npads, n_sectors=2, tf_time_bins=300, peak_min_q16=theta)
        assert len(ref) > 40000 and st["n_digits_dropped"] == 0
        assert got.tobytes() == ref.tobytes()


def test_time_frame_longer_than_the_u16_time_field():
    """DESIGN.md §3 A19 / SURVEY.md §8(f) f-3: a 66560-bin time frame (the C3 generator, 2 sectors, 512-bin fragments
    with an 8-bin halo); the fragments around bin 65536 and the last one, each with its own time base, through
    tpcclus_run_based and through tpcclus_run_tf_host, against the oracle; the concatenation against a monolithic
    oracle run across the 16-bit boundary (I7)."""
    import paper_2412_13755_b200 as T

    cfg = gen.config("longmini")
    npads = cfg.npads_array()
    frs = cfg.fragments()
    assert len(frs) == 130 and frs[128] == (65536, 66048)
    pick = [126, 127, 128, 129]
    kw = dict(n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins, halo_bins=cfg.halo_bins)
    got_all, host_frs, keep = [], [], []
    with GpuClusterizer(npads, max_core_bins=cfg.core_bins, max_digits=1 << 24, **kw) as g:
        for f in pick:
            b, e = frs[f]
            base = cfg.time_base(f)
            assert base == b - 8 and base + 65536 > e + 8
            d, offs, info = gen.generate_fragment(cfg, f, device="cuda")
            dn = gen.as_numpy_digits(d)
            got, st = g.run(d, offs, b, e, t_time_base=base)
            ref, ost = oracle.run(dn, offs, npads, t_core_begin=b, t_core_end=e, t_time_base=base, **kw)
            assert st["n_digits_dropped"] == ost["n_digits_dropped"] == 0 and len(ref) > 1e4
            assert got.tobytes() == ref.tobytes(), f
            got_all.append(got)
            keep.append(dn)
            host_frs.append((dn.ctypes.data, len(dn), offs, b, e, base))
    cat = np.concatenate(got_all)
    assert (cat["time"] < 65536).any() and (cat["time"] >= 65536).any() and cat["time"].max() >= 66500
    assert (cat[cat["time"] >= 66558]["flags"] & 2).all()                  # EDGE_TIME at the true TF end only
    assert not (cat[(cat["time"] < 66558)]["flags"] & 2).any()
    # the host-staging pipeline with a base per fragment
    ctx = T.tpcclus_create(npads, max_core_bins=cfg.core_bins, options=T.TPCCLUS_OPT_HOST_STAGING,
                           max_digits=max(len(k) for k in keep), max_clusters=max(len(x) for x in got_all) + 1, **kw)
    try:
        out = np.zeros(len(cat), dtype=T.CLUSTER_DTYPE)
        T.tpcclus_run_tf_host(ctx, host_frs, out.ctypes.data, len(cat))
        assert out.tobytes() == cat.tobytes()
    finally:
        T.tpcclus_destroy(ctx)
    # I7 across bin 65536: one monolithic oracle run over the four cores, digits re-based to the first fragment
    b0, e1 = frs[pick[0]][0], frs[pick[-1]][1]
    base0 = cfg.time_base(pick[0])
    parts = []
    for dn, fr in zip(keep, host_frs):
        offs_f, base_f = fr[2], fr[5]
        sec = np.repeat(np.arange(cfg.n_sectors), np.diff(offs_f).astype(np.int64))
        key = ((sec.astype(np.int64) * 256 + dn["row"]) * 256 + dn["pad"]) * (1 << 20) + dn["time"].astype(np.int64) + base_f
        parts.append((key, dn["charge"]))
    key = np.concatenate([k_ for k_, _ in parts])
    chg = np.concatenate([c_ for _, c_ in parts])
    key, first = np.unique(key, return_index=True)                      # halo bins are shared by neighbouring fragments
    chg = chg[first]
    dm = np.zeros(len(key), dtype=oracle.DIGIT_DTYPE)
    dm["time"] = (key % (1 << 20)) - base0
    dm["pad"] = (key >> 20) % 256
    dm["row"] = (key >> 28) % 256
    dm["charge"] = chg
    om = np.searchsorted(key >> 36, np.arange(cfg.n_sectors + 1)).astype(np.uint64)
    full, _ = oracle.run(dm, om, npads, n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins, t_core_begin=b0,
                         t_core_end=e1, halo_bins=8, t_time_base=base0)
    k = np.lexsort((cat["pad"], cat["time"], cat["row"], cat["sector"]))
    assert cat[k].tobytes() == full.tobytes()


@pytest.mark.parametrize("n_cells", [4095, 4096, 4097, 4100])
def test_tile_at_the_sparse_dense_boundary(n_cells):
    """k_tile tests a tile digit by digit when its list has at most 4096 entries (every thread keeps its share in
    registers) and sweeps the map otherwise.  One tile with exactly 4095 / 4096 / 4097 / 4100 digits through the
    direct binning kernel (lists of exact length, also lengths that are not a multiple of 4), blobs with ties and
    saturation so that neighbouring peaks, shared cells and plateaus occur on both paths."""
    import paper_2412_13755_b200 as T

    rng = np.random.default_rng(n_cells)
    npads, nt = 100, 256
    cells = {}
    while len(cells) < n_cells:
        pc, tc = int(rng.integers(npads)), int(rng.integers(nt))
        for _ in range(9):
            p, t = pc + int(rng.integers(-2, 3)), tc + int(rng.integers(-2, 3))
            if 0 <= p < npads and 0 <= t < nt and len(cells) < n_cells:
                q = float(rng.integers(32, 2000)) / 16.0
                if rng.random() < 0.25:
                    q = 9.0
                if rng.random() < 0.03:
                    q = 1023.0
                cells[(p, t)] = q
    d, offs = digits_from_cells([(0, 0, p, t, q) for (p, t), q in cells.items()])
    assert len(d) == n_cells
    for opt in (T.TPCCLUS_OPT_BIN_DIRECT, 0):
        got, st = gpu_clusters(d, offs, [npads], n_sectors=1, tf_time_bins=nt, options=opt)
        ref, _ = oracle.run(d, offs, [npads], n_sectors=1, tf_time_bins=nt)
        assert len(ref) > 300 and got.tobytes() == ref.tobytes(), opt


def test_sparse_and_dense_tiles_with_direct_lists():
    """The C2 generator has both kinds of tile (dense low pad rows, sparse upper ones); through k_bin_direct the
    lists have arbitrary lengths (tail entries outside the 16-byte loads) on both paths."""
    import paper_2412_13755_b200 as T

    cfg = gen.config("c2mini", tf_time_bins=700, core_bins=700)
    d, offs, _ = gen.generate_fragment(cfg, 0, device="cuda")
    dn = gen.as_numpy_digits(d)
    kw = dict(n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins)
    got, _ = gpu_clusters(dn, offs, cfg.npads_array(), options=T.TPCCLUS_OPT_BIN_DIRECT, **kw)
    ref, _ = oracle.run(dn, offs, cfg.npads_array(), **kw)
    assert len(ref) > 1e4 and got.tobytes() == ref.tobytes()
