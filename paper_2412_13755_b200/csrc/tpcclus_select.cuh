// tpcclus_select.cuh — D13: order-preserving quality selection over a finished cluster list (device side).
//
// SURVEY.md §8(f) f-4 ("cluster-quality cuts ... as parameters"; the same code runs online and offline
// "with appropriate selections and parameters").  D10 rejects nothing — one record per peak — so the cuts are a pass
// of their own over the 32-byte records: a single-pass ordered stream compaction (per-tile popc ranks + the same
// decoupled look-back across tiles as k_tile), bound by HBM: 32 B read per record, 32 B written per kept record.
// A tile is 1024 records; a warp instruction reads or writes 32 consecutive records.
// No code here is shared with oracle/.
#pragma once

namespace tpcclus {

struct SelectParams {
  const uint4* in;                     // n records, two 16-byte halves each
  uint4* out;
  unsigned long long* tile_state;      // [n_tiles] decoupled look-back words, epoch-tagged
  unsigned long long* n_kept;          // device: records kept (the number REQUIRED; may exceed out_capacity)
  unsigned int* ticket;
  uint64_t n, out_capacity;
  uint32_t n_tiles, epoch;
  float min_qtot;
  uint32_t min_qmax_q16, min_ncells, reject_flags, reject_single_pad, reject_single_time;
  uint32_t wide;                       // in and out are 32-byte aligned: records move as single 256-bit accesses
};

constexpr int kSelThreads = 256;
constexpr int kSelPer = 4;                                   // records per thread
constexpr int kSelTile = kSelThreads * kSelPer;              // 1024 records = 32 KB
constexpr int kSelWarps = kSelThreads / 32;

// A 32-byte record as ONE 256-bit access (sm_100: LDG / STG .256): a warp instruction then touches every 128-byte line
// once, where two 16-byte halves touch it twice — the LSU's line rate, not bytes, is what bounds this kernel.
__device__ __forceinline__ void ld_rec(const uint4* p, uint4& lo, uint4& hi) {
  asm volatile("ld.global.nc.v8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
               : "=r"(lo.x), "=r"(lo.y), "=r"(lo.z), "=r"(lo.w), "=r"(hi.x), "=r"(hi.y), "=r"(hi.z), "=r"(hi.w)
               : "l"(p));
}
__device__ __forceinline__ void st_rec(uint4* p, const uint4& lo, const uint4& hi) {
  asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "r"(lo.x), "r"(lo.y), "r"(lo.z), "r"(lo.w),
               "r"(hi.x), "r"(hi.y), "r"(hi.z), "r"(hi.w)
               : "memory");
}

__device__ __forceinline__ bool select_keep(const SelectParams& P, const uint4& lo, const uint4& hi) {
  // ClusterRec: lo = {sector | row << 8 | pad << 16 | flags << 24, time, qmax_q16 | ncells << 16, qtot}, hi = {dpad, dtime, sigma_pad, sigma_time}
  bool keep = __uint_as_float(lo.w) >= P.min_qtot;
  keep = keep && (lo.z & 0xFFFFu) >= P.min_qmax_q16;
  keep = keep && (lo.z >> 16) >= P.min_ncells;
  keep = keep && ((lo.x >> 24) & P.reject_flags) == 0u;
  keep = keep && !(P.reject_single_pad && __uint_as_float(hi.z) == 0.0f);
  keep = keep && !(P.reject_single_time && __uint_as_float(hi.w) == 0.0f);
  return keep;
}

// Record k * 256 + tid of the tile belongs to thread tid (k = 0..3): a warp instruction reads or writes 32 consecutive
// records.  The in-tile rank of a kept record is the kept count of the (k, warp) groups before its own — 32 counts,
// scanned by warp 0 — plus its rank inside the warp's ballot.
__global__ void __launch_bounds__(kSelThreads) k_select(const __grid_constant__ SelectParams P) {
  __shared__ uint32_t s_tile, s_cnt[kSelPer * kSelWarps], s_off[kSelPer * kSelWarps], s_base_lo, s_base_hi;
  static_assert(kSelPer * kSelWarps == 32, "one lane of warp 0 per (k, warp) group");
  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  for (;;) {
    if (tid == 0) s_tile = atomicAdd(P.ticket, 1u);          // tiles in list order (the look-back needs earlier tiles running)
    __syncthreads();
    const uint32_t t = s_tile;
    if (t >= P.n_tiles) break;
    const uint64_t first = uint64_t(t) * kSelTile + tid;
    uint4 lo[kSelPer], hi[kSelPer];
    uint32_t rank[kSelPer], keepm = 0;
#pragma unroll
    for (int k = 0; k < kSelPer; ++k) {
      const uint64_t i = first + uint64_t(k) * kSelThreads;
      bool keep = false;
      if (i < P.n) {
        if (P.wide) {
          ld_rec(P.in + 2 * i, lo[k], hi[k]);
        } else {                                             // buffers aligned to 16 but not to 32 bytes
          lo[k] = __ldg(P.in + 2 * i);
          hi[k] = __ldg(P.in + 2 * i + 1);
        }
        keep = select_keep(P, lo[k], hi[k]);
      }
      const uint32_t bal = __ballot_sync(0xffffffffu, keep);
      rank[k] = __popc(bal & ((1u << lane) - 1u));
      keepm |= keep ? 1u << k : 0u;
      if (lane == 0) s_cnt[k * kSelWarps + warp] = __popc(bal);
    }
    __syncthreads();
    if (warp == 0) {                                         // S6-style: scan of the 32 group counts, then the decoupled look-back
      const uint32_t c = s_cnt[lane];
      uint32_t incl = c;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
        if (lane >= uint32_t(o)) incl += v;
      }
      s_off[lane] = incl - c;
      const uint32_t total = __shfl_sync(0xffffffffu, incl, 31);
      if (lane == 0 && t != 0u) st_release_u64(P.tile_state + t, pack_state(P.epoch, kStAgg, total));
      __syncwarp();
      const uint64_t excl = lookback_exclusive(P.tile_state, t, P.epoch, total);   // (n < 2^32: the prefix fits the state word)
      if (lane == 0) {
        s_base_lo = uint32_t(excl);
        s_base_hi = uint32_t(excl >> 32);
        if (t == P.n_tiles - 1) *P.n_kept = excl + total;
      }
    }
    __syncthreads();
    const uint64_t base = uint64_t(s_base_lo) | (uint64_t(s_base_hi) << 32);
#pragma unroll
    for (int k = 0; k < kSelPer; ++k) {
      if (keepm & (1u << k)) {
        const uint64_t pos = base + s_off[k * kSelWarps + warp] + rank[k];
        if (pos < P.out_capacity) {
          if (P.wide) {
            st_rec(P.out + 2 * pos, lo[k], hi[k]);
          } else {
            P.out[2 * pos] = lo[k];
            P.out[2 * pos + 1] = hi[k];
          }
        }
      }
    }
    __syncthreads();                                         // s_tile, s_cnt, s_off, s_base are rewritten by the next tile
  }
}

}  // namespace tpcclus
