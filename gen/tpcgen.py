"""Seeded synthetic TPC digit generator for BASELINE.json:configs C0..C4 (+ small variants).

This module is the ONE thing the oracle side and the CUDA side share: it makes inputs.  It
holds none of the method's arithmetic (no quantisation rule of the clusterizer, no peak,
member, moment or ordering logic) and imports neither ``oracle`` nor the product package.

Recipe (SURVEY.md §8(d) "Generator specification G"; readings G1..G9 are listed in DESIGN.md):
every random draw is a pure function ``hash(seed, tag, index)`` (SplitMix64 finaliser), so a
cell's value depends only on (seed, sector, row, pad, GLOBAL time) and on the cluster list —
fragments of one time frame therefore agree on their shared halo bins, and nothing depends
on iteration order.  Runs on CPU or CUDA tensors (same code; libm differences in the last
ulp of exp/log/cos may flip a rare cell between devices, so one run's digits are generated
ONCE and fed to both sides).

The paper's own inputs are real ALICE data that is not available; these
synthetic time frames take the detector's shape (36 sectors x 152 rows, 66..138 pads,
128-orbit TF = 57024 bins, zero suppression at the front end) and stand
in for them.
"""
from __future__ import annotations

import math
from dataclasses import dataclass, field, replace

import numpy as np
import torch

_M64 = (1 << 64) - 1


def _s64(x: int) -> int:
    x &= _M64
    return x - (1 << 64) if x >= (1 << 63) else x


_C1 = _s64(0x9E3779B97F4A7C15)
_C2 = _s64(0xBF58476D1CE4E5B9)
_C3 = _s64(0x94D049BB133111EB)

TAG_NOISE_A, TAG_NOISE_B, TAG_ORDER, TAG_SAT = 1, 2, 3, 4
TAG_CL_P, TAG_CL_T, TAG_CL_A, TAG_CL_SP, TAG_CL_ST, TAG_CL_A2 = 10, 11, 12, 13, 14, 15
TAG_PAIR_D, TAG_PAIR_DP, TAG_PAIR_DT, TAG_PAIR_SIDE, TAG_PAIR_EQ = 20, 21, 22, 23, 24
TAG_BURST_P, TAG_BURST_T = 30, 31

ZS_THRESHOLD_ADC = 2.0       # BASELINE.json:configs[0] "Zero suppression at 2 ADC"
CHARGE_CLAMP_ADC = 1023.0    # "clamped to 1023"
NOISE_SIGMA_ADC = 1.0        # "Per-cell Gaussian noise sigma=1 ADC"
WIN_P, WIN_T = 6, 9          # evaluation window half-sizes (>= 5 sigma at the largest sigma)


def _lsr(x: torch.Tensor, s: int) -> torch.Tensor:
    return (x >> s) & ((1 << (64 - s)) - 1)


def _mix(z: torch.Tensor) -> torch.Tensor:
    z = (z ^ _lsr(z, 30)) * _C2
    z = (z ^ _lsr(z, 27)) * _C3
    return z ^ _lsr(z, 31)


def hash64(seed: int, tag: int, idx: torch.Tensor) -> torch.Tensor:
    """SplitMix64-style counter hash of an int64 index tensor (wrapping int64 arithmetic)."""
    k = _s64(seed * 0xD1B54A32D192ED03 + tag * 0x8CB92BA72F3D8DD7 + 0x2545F4914F6CDD1D)
    return _mix(_mix(idx * _C1 + k))


def u01(h: torch.Tensor) -> torch.Tensor:
    """Top 24 bits -> float32 in (0,1)."""
    return (_lsr(h, 40).to(torch.float32) + 0.5) * (1.0 / 16777216.0)


def normal(seed: int, tag_a: int, tag_b: int, idx: torch.Tensor) -> torch.Tensor:
    """Box-Muller on two counter draws."""
    u1 = u01(hash64(seed, tag_a, idx))
    u2 = u01(hash64(seed, tag_b, idx))
    return torch.sqrt(-2.0 * torch.log(u1)) * torch.cos((2.0 * math.pi) * u2)


def geometry_npads(n_rows: int = 152) -> np.ndarray:
    """BASELINE.json:configs[0]: pads per row rise linearly from 66 (row 0) to 138 (row 151),
    rounded to (the nearest) even: npads(r) = 2*floor((66*151 + 72*r + 151) / 302) (G1)."""
    r = np.arange(n_rows, dtype=np.int64)
    if n_rows == 152:
        return (2 * ((66 * 151 + 72 * r + 151) // 302)).astype(np.uint16)
    # small test geometries: same line, scaled to n_rows
    den = max(n_rows - 1, 1)
    return (2 * ((66 * den + 72 * r + den) // (2 * den))).astype(np.uint16)


@dataclass(frozen=True)
class Config:
    name: str
    seed: int
    n_sectors: int
    tf_time_bins: int
    core_bins: int                 # fragment core length; == tf_time_bins for single-fragment configs
    halo_bins: int                 # 0 for single-fragment configs, 8 for the fragmented TF
    n_rows: int = 152
    model: str = "c0"              # "c0" (fixed sigma, Exp(60) amplitudes) | "c2" (Pb-Pb like) | "c4" (stress)
    clusters_per_row: int = 0      # c0: exact count per row over the TF
    signal_occ: float = 0.0        # c0-model alternative: target SIGNAL occupancy (C1, reading G3-A)
    occ_row0: float = 0.0          # c2/c4: target total occupancy at row 0 ...
    occ_rowN: float = 0.0          # ... and at the last row (linear in between)
    npads: tuple = field(default=None)

    def npads_array(self) -> np.ndarray:
        return geometry_npads(self.n_rows) if self.npads is None else np.asarray(self.npads, dtype=np.uint16)

    def time_base(self, frag: int) -> int:
        """Global time bin that the u16 time field of fragment `frag`'s digits counts from (DESIGN.md §3 A19):
        0 for time frames of up to 65536 bins, else the first loaded bin of the fragment."""
        if self.tf_time_bins <= 65536:
            return 0
        b, _ = self.fragments()[frag]
        return max(0, b - self.halo_bins)

    def fragments(self):
        """Cores [b,e): consecutive chunks of core_bins over the TF (C3: 13 x 4096 + 3776)."""
        out, b = [], 0
        while b < self.tf_time_bins:
            e = min(b + self.core_bins, self.tf_time_bins)
            out.append((b, e))
            b = e
        return out


def config(i: int | str, **over) -> Config:
    """The five BASELINE.json configs (0..4) and small variants for element-wise parity."""
    table = {
        0: Config("C0-tiny", 1, 1, 512, 512, 0, model="c0", clusters_per_row=40),
        1: Config("C1-pp-sector", 2, 1, 4096, 4096, 0, model="c0", signal_occ=0.01),
        2: Config("C2-PbPb-fragment", 3, 36, 4096, 4096, 0, model="c2", occ_row0=0.25, occ_rowN=0.05),
        3: Config("C3-PbPb-TF", 4, 36, 57024, 4096, 8, model="c2", occ_row0=0.25, occ_rowN=0.05),
        4: Config("C4-stress", 5, 36, 4096, 4096, 0, model="c4", occ_row0=0.35, occ_rowN=0.35),
        # small variants (same generator, fewer sectors / bins) for tests the oracle finishes in seconds
        "c2mini": Config("C2-mini", 3, 2, 1024, 1024, 0, model="c2", occ_row0=0.25, occ_rowN=0.05),
        "c3mini": Config("C3-mini", 4, 2, 1500, 512, 8, model="c2", occ_row0=0.25, occ_rowN=0.05),
        "c4mini": Config("C4-mini", 5, 2, 768, 768, 0, model="c4", occ_row0=0.35, occ_rowN=0.35),
        # TF-length sweep (§4: 32 / 128 / 256 orbits): the C3 generator over
        # 14256 / 57024 / 114048 time bins (3564 bunch crossings per orbit / 8 per bin), 4096-bin fragments, 8-bin halo
        "tf32": Config("TF-32-orbits", 4, 36, 14256, 4096, 8, model="c2", occ_row0=0.25, occ_rowN=0.05),
        "tf128": Config("TF-128-orbits", 4, 36, 57024, 4096, 8, model="c2", occ_row0=0.25, occ_rowN=0.05),
        "tf256": Config("TF-256-orbits", 4, 36, 114048, 4096, 8, model="c2", occ_row0=0.25, occ_rowN=0.05),
        # pp-like occupancy on the full detector (the C1 model on 36 sectors): the low-occupancy case of SURVEY.md §8(f) f-4
        "ppfrag": Config("PP-fragment", 2, 36, 4096, 4096, 0, model="c0", signal_occ=0.01),
        # a time frame longer than the u16 time field in small: 130 fragments of 512 bins, the 16-bit boundary at a seam
        "longmini": Config("TF-long-mini", 4, 2, 66560, 512, 8, model="c2", occ_row0=0.25, occ_rowN=0.05),
    }
    return replace(table[i], **over)


# mean number of cells >= ZS that one cluster adds, calibrated once against realised occupancy
_FOOTPRINT_C0 = 17.3     # sigma (0.8, 1.2), A ~ Exp(60)
_FOOTPRINT_C2 = 23.0     # sigma_p U(0.6,1.2), sigma_t U(0.9,1.8), log-normal A
_FOOTPRINT_C4 = 18.8    # c2 shapes, but the two halves of a pile-up pair overlap
_NOISE_FLOOR = 0.0245    # P[N(0,1) >= 2 - 1/32]: noise-only cells surviving ZS


def clusters_per_row(cfg: Config) -> np.ndarray:
    """K(r): clusters per (sector,row) over the WHOLE time frame."""
    npads = cfg.npads_array().astype(np.float64)
    N = npads * cfg.tf_time_bins
    if cfg.model == "c0":
        if cfg.clusters_per_row:
            return np.full(cfg.n_rows, cfg.clusters_per_row, dtype=np.int64)
        # C1: 1 - exp(-K a / N) = signal_occ
        return np.rint(-N / _FOOTPRINT_C0 * math.log(1.0 - cfg.signal_occ)).astype(np.int64)
    r = np.arange(cfg.n_rows, dtype=np.float64)
    occ = cfg.occ_row0 + (cfg.occ_rowN - cfg.occ_row0) * r / max(cfg.n_rows - 1, 1)
    # 1 - (1 - f_n) exp(-K a / N) = occ(r)
    a = _FOOTPRINT_C4 if cfg.model == "c4" else _FOOTPRINT_C2
    K = -N / a * np.log((1.0 - occ) / (1.0 - _NOISE_FLOOR))
    K = np.rint(K).astype(np.int64)
    if cfg.model == "c4":
        K = (K // 2) * 2          # generated in pairs
    return K


def _cluster_params(cfg: Config, sector: int, K: np.ndarray, dev):
    """All clusters of one sector over the whole TF: row, centre (p_c,t_c), A, sigma_p, sigma_t."""
    seed = cfg.seed
    Kt = torch.as_tensor(K, device=dev)
    row = torch.repeat_interleave(torch.arange(cfg.n_rows, device=dev), Kt)
    start = torch.cumsum(Kt, 0) - Kt
    k = torch.arange(row.numel(), device=dev) - start[row]
    npads = torch.as_tensor(cfg.npads_array().astype(np.int64), device=dev)[row]
    if cfg.model == "c4":
        pair, second = k // 2, (k % 2) == 1
        cid = ((sector * cfg.n_rows + row) << 32) | pair        # both halves draw the pair's numbers
    else:
        cid = ((sector * cfg.n_rows + row) << 32) | k
    pc = u01(hash64(seed, TAG_CL_P, cid)) * npads.to(torch.float32) - 0.5
    tc = u01(hash64(seed, TAG_CL_T, cid)).to(torch.float64) * float(cfg.tf_time_bins) - 0.5
    if cfg.model == "c0":
        A = -60.0 * torch.log(u01(hash64(seed, TAG_CL_A, cid)))
        sp = torch.full_like(A, 0.8)
        st = torch.full_like(A, 1.2)
    else:
        A = torch.exp(math.log(40.0) + 0.8 * normal(seed, TAG_CL_A, TAG_CL_A2, cid))
        sp = 0.6 + 0.6 * u01(hash64(seed, TAG_CL_SP, cid))
        st = 0.9 + 0.9 * u01(hash64(seed, TAG_CL_ST, cid))
    if cfg.model == "c4":
        # pile-up pairs (G8): second centre = first + integer offset, Chebyshev distance 1..3;
        # 20 % of the pairs sit on exact cell centres and share (A, sigma): equal-amplitude ties
        d = 1 + (_lsr(hash64(seed, TAG_PAIR_D, cid), 33) % 3)
        dp = (_lsr(hash64(seed, TAG_PAIR_DP, cid), 33) % (2 * d + 1)) - d
        dt = (_lsr(hash64(seed, TAG_PAIR_DT, cid), 33) % (2 * d + 1)) - d
        side = torch.where(_lsr(hash64(seed, TAG_PAIR_SIDE, cid), 63) == 1, d, -d)
        dt = torch.where(torch.maximum(dp.abs(), dt.abs()) < d, side, dt)
        eq = u01(hash64(seed, TAG_PAIR_EQ, cid)) < 0.2
        pc = torch.where(eq, torch.round(pc), pc)
        tc = torch.where(eq, torch.round(tc), tc)
        cid2 = cid | (1 << 31)
        A2 = torch.exp(math.log(40.0) + 0.8 * normal(seed, TAG_CL_A, TAG_CL_A2, cid2))
        sp2 = 0.6 + 0.6 * u01(hash64(seed, TAG_CL_SP, cid2))
        st2 = 0.9 + 0.9 * u01(hash64(seed, TAG_CL_ST, cid2))
        pc = torch.where(second, pc + dp.to(pc.dtype), pc)
        tc = torch.where(second, tc + dt.to(tc.dtype), tc)
        A = torch.where(second & ~eq, A2, A)
        sp = torch.where(second & ~eq, sp2, sp)
        st = torch.where(second & ~eq, st2, st)
        # pad-edge clusters: per row and per 512 time bins one centred on pad 0, one on the last pad
        nblk = (cfg.tf_time_bins + 511) // 512
        er = torch.arange(cfg.n_rows, device=dev).repeat_interleave(2 * nblk)
        eb = torch.arange(2 * nblk, device=dev).repeat(cfg.n_rows)
        eid = ((sector * cfg.n_rows + er) << 32) | (1 << 30) | eb
        enp = torch.as_tensor(cfg.npads_array().astype(np.int64), device=dev)[er]
        epc = torch.where(eb % 2 == 0, torch.zeros_like(enp), enp - 1).to(torch.float32)
        etc = ((eb // 2) * 512).to(torch.float64) + torch.floor(
            u01(hash64(seed, TAG_CL_T, eid)).to(torch.float64) * min(512, cfg.tf_time_bins))
        eA = torch.exp(math.log(40.0) + 0.8 * normal(seed, TAG_CL_A, TAG_CL_A2, eid))
        esp = 0.6 + 0.6 * u01(hash64(seed, TAG_CL_SP, eid))
        est = 0.9 + 0.9 * u01(hash64(seed, TAG_CL_ST, eid))
        row, pc, tc = torch.cat([row, er]), torch.cat([pc, epc]), torch.cat([tc, etc])
        A, sp, st = torch.cat([A, eA]), torch.cat([sp, esp]), torch.cat([st, est])
    return row, pc, tc, A, sp, st


def _add_signal(sig: torch.Tensor, row, pc, tc, A, sp, st, lo: int, npads_t: torch.Tensor, chunk: int):
    """Accumulate point-sampled 2-D Gaussians (G5) in fixed point, 1/256 ADC, integer adds."""
    n_rows, Tl, P = sig.shape
    dev = sig.device
    dpp = torch.arange(-WIN_P, WIN_P + 1, device=dev)
    dtt = torch.arange(-WIN_T, WIN_T + 1, device=dev)
    flat = sig.view(-1)
    for a in range(0, row.numel(), chunk):
        sl = slice(a, a + chunk)
        r = row[sl]
        p0 = torch.round(pc[sl]).to(torch.int64)
        t0 = torch.round(tc[sl]).to(torch.int64)
        p = p0[:, None, None] + dpp[None, None, :]                  # [n,1,13]
        t = t0[:, None, None] + dtt[None, :, None]                  # [n,19,1]
        gx = torch.exp(-((p.to(torch.float32) - pc[sl][:, None, None]) ** 2) / (2.0 * sp[sl][:, None, None] ** 2))
        gt = torch.exp(-((t.to(torch.float64) - tc[sl][:, None, None]).to(torch.float32) ** 2)
                       / (2.0 * st[sl][:, None, None] ** 2))
        val = torch.round(A[sl][:, None, None] * gx * gt * 256.0).to(torch.int32)   # [n,19,13]
        tl = t - lo
        ok = (p >= 0) & (p < npads_t[r][:, None, None]) & (tl >= 0) & (tl < Tl) & (val > 0)
        idx = (r[:, None, None] * Tl + tl) * P + p
        flat.index_add_(0, idx[ok], val[ok])


def generate_fragment(cfg: Config, frag: int = 0, device="cpu", sectors=None, row_chunk: int = 16,
                      cluster_chunk: int = 100_000):
    """Digits of fragment `frag` of the config's time frame.

    Returns (digits, offsets, info): digits is a uint8 tensor [n, 8] on `device` holding
    (u8 row, u8 pad, u16 time, f32 charge) records grouped per sector, in hash-random order
    inside each sector slice; offsets is a numpy uint64 [n_sectors+1]; info has the core
    range, the time base the u16 time field counts from (cfg.time_base(frag); 0 unless the TF
    is longer than 65536 bins) and the realised occupancy.
    `sectors` restricts generation to a subset (the other slices are empty).
    """
    dev = torch.device(device)
    b, e = cfg.fragments()[frag]
    lo, hi = max(0, b - cfg.halo_bins), min(cfg.tf_time_bins, e + cfg.halo_bins)
    Tl = hi - lo
    t_base = cfg.time_base(frag)
    assert 0 <= lo - t_base and hi - t_base <= 65536
    npads = cfg.npads_array()
    P = int(npads.max())
    npads_t = torch.as_tensor(npads.astype(np.int64), device=dev)
    K = clusters_per_row(cfg)
    seed = cfg.seed
    parts, offs = [], [0]
    n_cells = int(npads.astype(np.int64).sum()) * Tl
    want = set(range(cfg.n_sectors)) if sectors is None else set(sectors)
    for s in range(cfg.n_sectors):
        if s not in want:
            offs.append(offs[-1])
            continue
        row, pc, tc, A, sp, st = _cluster_params(cfg, s, K, dev)
        sel = (tc >= lo - WIN_T - 1) & (tc < hi + WIN_T + 1)
        sig = torch.zeros((cfg.n_rows, Tl, P), dtype=torch.int32, device=dev)
        _add_signal(sig, row[sel], pc[sel], tc[sel], A[sel], sp[sel], st[sel], lo, npads_t, cluster_chunk)
        recs = []
        for r0 in range(0, cfg.n_rows, row_chunk):
            r1 = min(cfg.n_rows, r0 + row_chunk)
            rr = torch.arange(r0, r1, device=dev)[:, None, None]
            tt = torch.arange(lo, hi, device=dev)[None, :, None]
            pp = torch.arange(P, device=dev)[None, None, :]
            cell = ((s * cfg.n_rows + rr) * cfg.tf_time_bins + tt) * 256 + pp      # global cell index
            v = sig[r0:r1].to(torch.float32) * (1.0 / 256.0) + NOISE_SIGMA_ADC * normal(seed, TAG_NOISE_A, TAG_NOISE_B, cell)
            if cfg.model == "c4":
                # correlated noise bursts (G6): 2 per (sector,row) per 4096 bins, 3 pads x 50 bins, v := max(v, 8)
                nb = 2 * ((cfg.tf_time_bins + 4095) // 4096)
                for kb in range(nb):
                    bid = ((s * cfg.n_rows + rr) << 8) | kb
                    bp = (u01(hash64(seed, TAG_BURST_P, bid)) * (npads_t[r0:r1, None, None] - 2).to(torch.float32)).to(torch.int64)
                    bt = (u01(hash64(seed, TAG_BURST_T, bid)) * float(max(cfg.tf_time_bins - 50, 1))).to(torch.int64)
                    inb = (pp >= bp) & (pp < bp + 3) & (tt >= bt) & (tt < bt + 50)
                    v = torch.where(inb, torch.clamp(v, min=8.0), v)
            v = torch.clamp(v, max=CHARGE_CLAMP_ADC)
            q = torch.round(v * 16.0) * (1.0 / 16.0)                 # G2: clamp, round to 1/16, then ZS
            keep = (q >= ZS_THRESHOLD_ADC) & (pp < npads_t[r0:r1, None, None])
            ri, ti, pi = torch.nonzero(keep, as_tuple=True)
            qk = q[ri, ti, pi]
            ck = cell.expand(r1 - r0, Tl, P)[ri, ti, pi]
            if cfg.model == "c4":
                # G7: 5 % of the digits (hash-selected) saturate at 1023
                sat = u01(hash64(seed, TAG_SAT, ck)) < 0.05
                qk = torch.where(sat, torch.full_like(qk, CHARGE_CLAMP_ADC), qk)
            word = (ri + r0) | (pi << 8) | ((ti + (lo - t_base)) << 16) | (qk.view(torch.int32).to(torch.int64) << 32)
            recs.append((word, hash64(seed, TAG_ORDER, ck)))
        word = torch.cat([w for w, _ in recs])
        key = torch.cat([k_ for _, k_ in recs])
        del recs, sig
        order = torch.argsort(key)                                   # "random order", reproducible
        parts.append(word[order])
        offs.append(offs[-1] + int(word.numel()))
    words = torch.cat(parts) if parts else torch.zeros(0, dtype=torch.int64, device=dev)
    digits = words.view(torch.uint8).view(-1, 8)
    n = int(words.numel())
    info = dict(config=cfg.name, fragment=frag, t_core_begin=b, t_core_end=e, t_loaded=(lo, hi), t_time_base=t_base,
                n_digits=n, n_cells=n_cells * len(want),
                occupancy=(n / (n_cells * len(want))) if n_cells and want else 0.0)
    return digits, np.asarray(offs, dtype=np.uint64), info


def fnv1a64(buf: np.ndarray) -> int:
    """FNV-1a over a byte buffer (logged next to digit counts)."""
    h = 0xCBF29CE484222325
    for x in np.ascontiguousarray(buf).view(np.uint8).ravel()[: 1 << 16].tolist():
        h = ((h ^ x) * 0x100000001B3) & _M64
    return h


def as_numpy_digits(digits: torch.Tensor) -> np.ndarray:
    """uint8 [n,8] tensor -> numpy structured array (row,pad,time,charge)."""
    dt = np.dtype([("row", "u1"), ("pad", "u1"), ("time", "<u2"), ("charge", "<f4")])
    return digits.detach().cpu().contiguous().numpy().view(dt).reshape(-1)
