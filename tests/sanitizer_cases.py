"""Workloads for compute-sanitizer: small cases that still reach every kernel path.

    compute-sanitizer --tool memcheck|racecheck|initcheck|synccheck python tests/sanitizer_cases.py
    python tests/sanitizer_cases.py --checked        # the -DTPCCLUS_CHECKED build: device asserts on every index

(one tool per gpurun call; the results are summarised in profiles/r2_sanitizer.md).  Inputs are generated on the
CPU so that only this repository's kernels run instrumented.  Every case is also compared with the oracle, so a
sanitizer run doubles as a parity run of the instrumented build.

  smoke      __graft_entry__.smoke()'s configuration (C0 geometry, 8 rows)
  c0         BASELINE.json:configs[0] at full size
  c4         the stress generator (pile-up pairs, bursts, saturation, pad-edge clusters): dense tiles, several
             hand-over items per tile, a ragged last tile (600 bins)
  sorted     C2 generator, digits sorted by (time,row,pad): k_bin's overflow paths (ranks beyond a bin buffer,
             several sectors reserved at once, second entries beyond the per-chunk list -> single-entry appends)
  direct     the same through k_bin_direct (TPCCLUS_OPT_BIN_DIRECT)
  frag       three fragments with an 8-bin halo through one context (bins and look-back state reused)
"""
import os
import sys

import numpy as np

ROOT = os.path.dirname(os.path.dirname(os.path.abspath(__file__)))
sys.path.insert(0, ROOT)
sys.path.insert(0, os.path.join(ROOT, "tests"))

import gen  # noqa: E402
import oracle  # noqa: E402
import paper_2412_13755_b200 as T  # noqa: E402
from gpu_util import GpuClusterizer, to_device_digits  # noqa: E402


def check(name, cfg, dn_by_fragment, options=0):
    npads = cfg.npads_array()
    with GpuClusterizer(npads, n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins, max_core_bins=cfg.core_bins,
                        halo_bins=cfg.halo_bins, max_digits=max(len(d) for d, _ in dn_by_fragment),
                        options=options) as g:
        for (dn, offs), (b, e) in zip(dn_by_fragment, cfg.fragments()):
            got, st = g.run(to_device_digits(dn), offs, b, e)
            ref, ost = oracle.run(dn, offs, npads, n_sectors=cfg.n_sectors, tf_time_bins=cfg.tf_time_bins,
                                  t_core_begin=b, t_core_end=e, halo_bins=cfg.halo_bins)
            assert st["n_digits_dropped"] == ost["n_digits_dropped"]
            assert got.tobytes() == ref.tobytes(), name
            print(f"{name}: [{b},{e}) {len(dn)} digits -> {len(ref)} clusters, identical to the oracle", flush=True)


def cpu_fragments(cfg):
    out = []
    for f in range(len(cfg.fragments())):
        d, offs, _ = gen.generate_fragment(cfg, f, device="cpu")
        out.append((gen.as_numpy_digits(d), offs))
    return out


def main():
    if "--checked" in sys.argv:
        T.use_checked_build()
    oracle.build()
    cfg = gen.config(0, n_rows=8, clusters_per_row=40)
    check("smoke", cfg, cpu_fragments(cfg))
    cfg = gen.config(0)
    check("c0", cfg, cpu_fragments(cfg))
    cfg = gen.config("c4mini", n_sectors=1, n_rows=24, tf_time_bins=600, core_bins=600)
    check("c4", cfg, cpu_fragments(cfg))
    cfg = gen.config("c2mini", n_sectors=2, n_rows=24, tf_time_bins=600, core_bins=600)
    fr = cpu_fragments(cfg)
    dn, offs = fr[0]
    sn = dn.copy()
    for s in range(cfg.n_sectors):
        a, b = int(offs[s]), int(offs[s + 1])
        seg = dn[a:b]
        sn[a:b] = seg[np.lexsort((seg["pad"], seg["row"], seg["time"]))]
    check("sorted", cfg, [(sn, offs)])
    check("direct", cfg, [(dn, offs)], options=T.TPCCLUS_OPT_BIN_DIRECT)
    cfg = gen.config("c3mini", n_sectors=1, n_rows=16)
    check("frag", cfg, cpu_fragments(cfg))
    print("sanitizer cases done", flush=True)


if __name__ == "__main__":
    main()
