// tpcclus_kernels.cuh — sm_100a kernels of the TPC cluster finder (device side).
//
// Steps of SURVEY.md §8(a) and where they run:
//   S0  set-up               k_init   zero the per-bin entry counters and the run status
//   S1  charge-map fill      k_bin    TMA-staged digit chunks (16-byte pairs), D1 quantisation, digit ->
//                                     packed 4-byte entry in the list of every (sector,row,256-bin) digit
//                                     bin whose window holds it; write-combined: one 32-byte sector and
//                                     one global atomic per 8 entries
//                            k_tile   the bin's list is scattered into the (pad x time) charge map of the
//                                     tile, which lives in shared memory only                (tpcclus_tile.cuh)
//   S2  peak finding         k_tile   dense packed-u16x2 sweep of the map -> one flag byte per 8 cells
//   S3  peak count S(c)      k_tile   one thread per peak: other peaks of the 9x9 flag window, table-driven
//   S4  5x5 assembly         k_tile   one thread per peak, 25 charges straight from the map
//   S5  centroid / width     k_tile   exact integer moments from column / row weight sums; committer warp:
//                                     fp64 finish
//   S6  ordered compaction   k_tile   popc prefix inside the tile; committer warp: decoupled look-back across
//                                     tiles in (sector,row,time) ticket order, copy-out
//   S7  fragment ownership   k_tile   tiles cover exactly the core [b,e); halo rows never emit
//
// Definitions D1..D12 are those of SURVEY.md §8(c) (restated in DESIGN.md §2); the D-number
// is cited where each rule is implemented.  No code here is shared with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

// -DTPCCLUS_CHECKED (paper_2412_13755_b200/build.py: build(checked=True) -> libtpcclus_checked.so): every
// shared-memory and list index of the kernels is bounds-checked with a device assert.  This is the repo's own
// stand-in for compute-sanitizer memcheck, which is closed on this GPU pool (profiles/r2_sanitizer.md).
#ifdef TPCCLUS_CHECKED
#include <cassert>
#define TPC_ASSERT(x) assert(x)
#else
#define TPC_ASSERT(x) ((void)0)
#endif

namespace tpcclus {

#ifndef TPCCLUS_TILE_T
#define TPCCLUS_TILE_T 256
#endif
constexpr int      kTileT        = TPCCLUS_TILE_T;   // core time bins per tile (= one digit bin of k_bin)
constexpr int      kWorkThreads  = 2 * kTileT;       // worker warps of k_tile: one per 16 core rows
constexpr int      kThreads      = kWorkThreads + 32;   // + the committer warp
constexpr int      kTileCtasPerSm = kTileT == 256 ? 2 : 4;
constexpr int      kReach        = 5;     // D9: charges within Chebyshev distance 5 decide a cluster
constexpr int      kBoxH         = kTileT + 2 * kReach;   // map rows of a tile (266)
constexpr int      kBinT         = kTileT;   // core time bins per digit bin
constexpr int      kBinShift     = kTileT == 256 ? 8 : 7;
constexpr int      kBinBoxH      = kBinT + 2 * kReach;    // time rows a bin's window spans (266)
static_assert((1 << kBinShift) == kBinT && kBinT == kTileT, "a digit bin is one tile");
constexpr int      kColOff       = 2;     // map column of pad 0 (two zero columns each side: 5x5 window)
constexpr int      kListCap      = kWorkThreads < 256 ? kWorkThreads : 256;   // records per hand-over item (capacity of one staging buffer)
constexpr uint32_t kQClamp       = 16368; // D1
constexpr int      kMaxSectors   = 256;

struct RowInfo {              // one per pad row (device table), 32 bytes
  uint32_t list_off;          // element offset of this row's bins inside one sector's digit lists
  uint32_t cap;               // list capacity of one bin (multiple of 8): bin_occupancy_pct of the window's cells + padding margin
  uint16_t npads;
  uint16_t W;                 // smem map pitch in cells = roundup8(npads + 4)
  // k_tile's sweep over a tile of this row: strips of 8 cells x row segments
  uint16_t ns;                // strips per map row = W / 8
  uint16_t fpb;               // flag bytes per map row = flag_pitch_bytes(W)
  uint16_t segL;              // map rows flagged per segment
  uint16_t ntasks;            // ns * number of segments
  uint32_t rcp_ns;            // ceil(2^16 / ns): task / ns = (task * rcp_ns) >> 16 for task < 512 (ns <= 64)
  uint32_t sparse_max;        // k_tile: lists of up to this many entries take the digit-driven (sparse) path; <= 8 * kWorkThreads
  uint32_t pad_;
};
static_assert(sizeof(RowInfo) == 32, "RowInfo is 32 bytes");

struct DevStatus {            // device-side run status, copied to pinned host memory after the run
  unsigned long long n_dropped;
  unsigned long long n_clusters;
  unsigned int       ticket;  // tile ticket counter of k_tile
  unsigned int       n_overfull_bins;   // digit bins that received more entries than their capacity
};

struct BinParams {
  uint64_t n;                          // digits
  uint64_t sec_list_elems;             // list elements per sector
  int32_t  t_core_begin;               // b
  int32_t  t_lo, t_hi;                 // loaded range [lo,hi) in global time (D1)
  int32_t  t_base;                     // A19: global time = t_base + the digit's u16 time field
  uint32_t n_sectors, n_rows;
  uint32_t bins_per_row;               // bins per (sector,row) of this run = ceil((e-b)/kBinT)
  uint32_t bins_per_row_max;           // bins laid out per (sector,row)
  // k_bin (CTA-aggregated binning) only:
  const uint4* base16;                 // digit buffer aligned down to 16 bytes; digit i is 8-byte slot i + head
  uint32_t head;                       // 1 if the buffer starts in the upper half of a 16-byte pair
  uint32_t nb;                         // bins per sector of this run = n_rows * bins_per_row
  uint32_t total_chunks;               // cpref[n_sectors]
  uint32_t pad_;
  uint64_t pair_lo, pair_hi;           // pairs with both slots inside the buffer: [pair_lo, pair_hi)
  uint64_t off[kMaxSectors + 1];       // sector offsets (copied from the host array)
  uint32_t cpref[kMaxSectors + 1];     // k_bin: chunks of sectors < s (sector s has ceil(pairs / (kBinChunk/2)) chunks)
};

struct TileParams {
  const RowInfo*     rows;             // [n_rows]
  const uint32_t*    lists;            // packed digits, fixed-capacity bins
  const uint32_t*    counts;           // [n_tiles] digits appended per bin (may exceed cap: clamp)
  unsigned long long* tile_state;      // [n_tiles] decoupled look-back words
  DevStatus*         status;
  void*              out;              // tpcclus_cluster records
  uint64_t           out_capacity;
  uint64_t           sec_list_elems;
  uint32_t n_sectors, n_rows;
  uint32_t tiles_per_row;              // ceil((e-b)/kTileT)
  uint32_t n_tiles;
  int32_t  t_core_begin, t_core_end;   // [b,e)
  uint32_t tf_time_bins;
  uint32_t theta;                      // peak_min_q16
  uint32_t epoch;                      // run counter, tags tile_state words
  uint32_t map_bytes_max;              // smem bytes reserved for map + flag bytes
  uint32_t theta2;                     // theta | theta << 16
};

// ----------------------------------------------------------------------------------------
// small PTX wrappers (TMA bulk copy + mbarrier), sm_90+/sm_100a
// ----------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
  return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() {
  asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint64_t* bar, uint32_t bytes) {
  asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
               : "memory");
}
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
  asm volatile(
      "{\n"
      ".reg .pred p;\n"
      "WAIT_%=:\n"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n"
      "@p bra DONE_%=;\n"
      "bra WAIT_%=;\n"
      "DONE_%=:\n"
      "}\n" ::"r"(smem_u32(bar)),
      "r"(parity)
      : "memory");
}
// 1-D TMA bulk copy global -> shared (UBLKCP): 16-byte aligned addresses, size a multiple of 16.
__device__ __forceinline__ void tma_bulk_load(void* smem_dst, const void* gsrc, uint32_t bytes, uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::
          "r"(smem_u32(smem_dst)),
      "l"(reinterpret_cast<uint64_t>(gsrc)), "r"(bytes), "r"(smem_u32(bar))
      : "memory");
}
__device__ __forceinline__ void bar_sync_named(int id, int nthreads) {
  asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
  unsigned long long v;
  asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
  return v;
}
__device__ __forceinline__ void st_release_u64(unsigned long long* p, unsigned long long v) {
  asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ uint4 ld_stream_u4(const uint4* p) {   // streaming 16-byte load, no L1 allocation
  uint4 r;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(r.x), "=r"(r.y), "=r"(r.z), "=r"(r.w)
               : "l"(p));
  return r;
}

// ----------------------------------------------------------------------------------------
// S0: zero the per-tile digit counters of this run and the run status.
// ----------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_init(uint32_t* __restrict__ counts, uint32_t n_tiles,
                                              DevStatus* __restrict__ status) {
  const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
  if (i == 0) {
    status->n_dropped = 0ull;
    status->n_clusters = 0ull;
    status->ticket = 0u;
    status->n_overfull_bins = 0u;
  }
  const uint32_t n4 = (n_tiles + 3u) >> 2;                 // the array is padded to a multiple of 4
  for (uint32_t k = i; k < n4; k += gridDim.x * blockDim.x)
    reinterpret_cast<uint4*>(counts)[k] = make_uint4(0u, 0u, 0u, 0u);
}

// ----------------------------------------------------------------------------------------
// S1 (first half): digit binning.  One 16-byte load = two digits (BASELINE.json:north_star (2):
// "16-byte vectorised coalesced loads").  D1 quantisation; invalid digits dropped and counted.
// A valid digit at global time t is appended, as a packed entry with tl = its row inside the
// bin's 266-row window, to the list of every bin tb whose window [b + 256 tb - 5, b + 256 tb + 261)
// contains t (one bin, or two next to a bin seam).  Entries past a bin's capacity are discarded
// (memory-safe for duplicate cells) and the bin is reported (TPCCLUS_ERR_OCCUPANCY).
// ----------------------------------------------------------------------------------------
// packed list entry: pad (8 bits) | tl << 8 (row of the bin's window, 9 bits) | q16 << 17 (14 bits)
__device__ __forceinline__ uint32_t pack_digit(uint32_t pad, uint32_t tl, uint32_t q) { return pad | (tl << 8) | (q << 17); }
__device__ __forceinline__ uint32_t dig_pad(uint32_t d) { return d & 0xFFu; }
__device__ __forceinline__ uint32_t dig_tl(uint32_t d) { return (d >> 8) & 0x1FFu; }
__device__ __forceinline__ uint32_t dig_q(uint32_t d) { return d >> 17; }

__device__ __forceinline__ uint32_t quantise_q16(float charge) {
  // D1: q16 = clamp(rint(charge*16), 0, 16368).  cvt.rni.u32.f32 rounds half-even and saturates:
  // negative and NaN -> 0, huge -> 0xFFFFFFFF
  return min(__float2uint_rn(charge * 16.0f), kQClamp);
}

// append one packed digit to a bin, reserving R slots (R = 1 everywhere now; the other R-1 slots
// would be zero = "no digit")
template <int R>
__device__ __forceinline__ void bin_append(uint32_t* __restrict__ seclist, uint32_t* __restrict__ cnt, uint32_t dest0,
                                           uint32_t cap, uint32_t pk) {
  const uint32_t slot = atomicAdd(cnt, uint32_t(R));
  if (slot + uint32_t(R) <= cap) {
    TPC_ASSERT(pk != 0u);
    seclist[dest0 + slot] = pk;
#pragma unroll
    for (int x = 1; x < R; ++x) seclist[dest0 + slot + x] = 0u;
  }
}

template <int R>
__device__ __forceinline__ bool bin_one(uint32_t w0, uint32_t w1, uint64_t idx, uint32_t& sector,
                                        const BinParams& P, const RowInfo* srow, uint32_t* __restrict__ lists,
                                        uint32_t* __restrict__ counts) {
  while (idx >= P.off[sector + 1]) ++sector;     // digits are grouped per sector; rarely iterates
  const uint32_t row = w0 & 0xFFu, pad = (w0 >> 8) & 0xFFu;
  const int32_t time = int32_t(w0 >> 16) + P.t_base;              // A19
  const uint32_t q = quantise_q16(__uint_as_float(w1));
  if (q == 0u || row >= P.n_rows || time < P.t_lo || time >= P.t_hi) return false;
  const RowInfo ri = srow[row];
  if (pad >= ri.npads) return false;
  const int32_t u = time - P.t_core_begin;                       // >= -halo
  const int32_t tb_lo = max((u - kReach) >> kBinShift, 0);       // bins whose window [256 tb - 5, 256 tb + 261) holds u
  const int32_t tb_hi = min((u + kReach) >> kBinShift, int32_t(P.bins_per_row) - 1);
  uint32_t* seclist = lists + uint64_t(sector) * P.sec_list_elems;
  for (int32_t tb = tb_lo; tb <= tb_hi; ++tb) {
    const uint32_t tl = uint32_t(u - tb * kBinT + kReach);       // 0..265
    bin_append<R>(seclist, &counts[(sector * P.n_rows + row) * P.bins_per_row + uint32_t(tb)],
                  ri.list_off + uint32_t(tb) * ri.cap, ri.cap, pack_digit(pad, tl, q));
  }
  return true;
}

__global__ void __launch_bounds__(256) k_bin_direct(const uint2* __restrict__ digits, const __grid_constant__ BinParams P,
                                             const RowInfo* __restrict__ rows, uint32_t* __restrict__ lists,
                                             uint32_t* __restrict__ counts, DevStatus* __restrict__ status) {
  __shared__ RowInfo srow[256];
  for (uint32_t i = threadIdx.x; i < P.n_rows; i += blockDim.x) srow[i] = rows[i];
  __syncthreads();
  const uint64_t n = P.n;
  // the buffer is 8-byte aligned; peel one digit if it is not 16-byte aligned so that the
  // body can use 16-byte loads
  const uint64_t head = (reinterpret_cast<uintptr_t>(digits) & 8u) ? 1u : 0u;
  const uint64_t npairs = n > head ? (n - head) >> 1 : 0;
  const uint4* pairs = reinterpret_cast<const uint4*>(digits + head);
  uint32_t dropped = 0;
  const uint64_t tid = uint64_t(blockIdx.x) * blockDim.x + threadIdx.x;
  const uint64_t stride = uint64_t(gridDim.x) * blockDim.x;
  // sector of the first digit this thread touches (binary search), then monotone advance
  uint32_t sector = 0;
  {
    const uint64_t first = head + 2 * tid;
    uint32_t lo = 0, hi = P.n_sectors;           // invariant: off[lo] <= first (when first < n)
    while (hi - lo > 1) {
      const uint32_t mid = (lo + hi) >> 1;
      if (P.off[mid] <= first) lo = mid; else hi = mid;
    }
    sector = lo;
  }
  for (uint64_t i = tid; i < npairs; i += stride) {
    const uint4 v = ld_stream_u4(pairs + i);
    const uint64_t idx = head + 2 * i;
    dropped += bin_one<1>(v.x, v.y, idx, sector, P, srow, lists, counts) ? 0u : 1u;
    dropped += bin_one<1>(v.z, v.w, idx + 1, sector, P, srow, lists, counts) ? 0u : 1u;
  }
  if (tid == 0) {                                 // leftovers: the peeled head and an odd tail
    uint32_t s0 = 0;
    if (head && n > 0) dropped += bin_one<1>(digits[0].x, digits[0].y, 0, s0, P, srow, lists, counts) ? 0u : 1u;
    const uint64_t tail = head + 2 * npairs;
    if (tail < n) dropped += bin_one<1>(digits[tail].x, digits[tail].y, tail, s0, P, srow, lists, counts) ? 0u : 1u;
  }
  // warp-aggregated count of dropped digits
  dropped = __reduce_add_sync(0xffffffffu, dropped);
  if ((threadIdx.x & 31) == 0 && dropped) atomicAdd(&status->n_dropped, (unsigned long long)dropped);
}

// ----------------------------------------------------------------------------------------
// S1 (first half), write-combining: the production binning kernel.
//
// Why: appending digits one by one costs one scattered 4-byte store per list entry and, even
// when a CTA aggregates a chunk's reservations, about one global atomic per 2-4 entries; ncu
// shows both k_bin_direct and the chunk-aggregated variant pinned at ~45 % L1/L2 transaction
// throughput with every warp waiting (profiles/r1c_bin_ncu.md).  Here each CTA (one per SM) keeps an
// 8-entry (32-byte = one DRAM sector) buffer per bin of the sector it is reading in shared
// memory, and a bin costs ONE global atomic and ONE aligned 32-byte store per 8 entries:
//   A   every digit of the chunk (TMA-staged, double-buffered): quantise (D1), validate, rank
//       with a shared-memory atomic on the bin's fill count; ranks 0..7 go into the buffer, the
//       thread that takes rank 7 queues the bin for flushing; the digit's slot in the staging
//       area is overwritten by (entry, bin | rank << 12).  A digit within 5 bins of a bin seam
//       also enters the next bin (second-entry list; reserve-8 direct path when that is full).
//   B1  one thread per queued bin: reserve roundup8(count) slots with one global atomic, store
//       the 8 buffered entries as one sector, zero-fill the padding, reset the count
//   B2  entries that ranked >= 8 (more than a buffer's worth arrived within one chunk — rare
//       for shuffled input, the rule for sorted input) are stored at reservation + rank
// A CTA works through a contiguous range of chunks; buffers persist across the chunks of a
// sector and are flushed (padded to 8 with zero = "no digit" entries) when the sector changes.
// All reservations are multiples of 8, so every buffer flush is a 32-byte aligned store.
// ----------------------------------------------------------------------------------------
constexpr int      kBinThreads  = 1024;
constexpr int      kBinPer      = 6;                        // digits per thread per chunk
constexpr int      kBinChunk    = kBinThreads * kBinPer;    // 6144 digits = 48 KB of input
constexpr int      kBinSecCap   = 1024;                     // second (seam) entries kept per chunk
constexpr uint32_t kBinMaxNb    = 4096;                     // bins per sector (12-bit bin id)
constexpr uint32_t kBinFull     = 0xFFFFFFFFu;              // bin has no room (duplicates only)

__host__ __device__ inline uint32_t bin_smem_bytes(uint32_t nb) {
  const uint32_t nb4 = (nb + 3u) & ~3u;
  return 2u * uint32_t(kBinChunk) * 8u + nb4 * 32u + nb4 * 4u + nb4 * 4u + nb4 * 4u + nb4 * 2u + 2u * uint32_t(kBinSecCap) * 8u +
         3u * 256u * 4u + 96u + 128u;
}

// store a bin buffer (8 entries) at list position p: one aligned 32-byte sector on the production path; the
// reservations stop being multiples of 8 only after a single-entry append (second entries beyond kBinSecCap,
// i.e. time-sorted input), and then the entries go out one by one
__device__ __forceinline__ void store8(uint32_t* p, uint4 a, uint4 c) {
  if ((reinterpret_cast<uintptr_t>(p) & 31u) == 0u) {
    // ONE 256-bit store (sm_100): the sector goes through the LSU as one access instead of two
    asm volatile("st.global.v8.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8};" ::"l"(p), "r"(a.x), "r"(a.y), "r"(a.z), "r"(a.w),
                 "r"(c.x), "r"(c.y), "r"(c.z), "r"(c.w)
                 : "memory");
  } else {
    p[0] = a.x; p[1] = a.y; p[2] = a.z; p[3] = a.w;
    p[4] = c.x; p[5] = c.y; p[6] = c.z; p[7] = c.w;
  }
}

__global__ void __launch_bounds__(kBinThreads, 1) k_bin(const __grid_constant__ BinParams P,
                                                        const RowInfo* __restrict__ rows, uint32_t* __restrict__ lists,
                                                        uint32_t* __restrict__ counts, DevStatus* __restrict__ status) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  const uint32_t nb4 = (P.nb + 3u) & ~3u;
  uint8_t* sp = smem_raw;                                     // __align__(128); no static shared memory before it
  uint2* stage0 = reinterpret_cast<uint2*>(sp);               sp += 2u * uint32_t(kBinChunk) * 8u;   // two TMA destinations
  uint32_t* buf = reinterpret_cast<uint32_t*>(sp);            sp += nb4 * 32u;     // 8 entries per bin
  uint32_t* cnt = reinterpret_cast<uint32_t*>(sp);            sp += nb4 * 4u;      // fill count per bin
  uint2* sec = reinterpret_cast<uint2*>(sp);                  sp += 2u * uint32_t(kBinSecCap) * 8u;   // second entries, one list per staging buffer
  uint32_t* r_npads = reinterpret_cast<uint32_t*>(sp);        sp += 256 * 4;
  uint32_t* r_off = reinterpret_cast<uint32_t*>(sp);          sp += 256 * 4;
  uint32_t* r_cap = reinterpret_cast<uint32_t*>(sp);          sp += 256 * 4;
  uint64_t* mbar = reinterpret_cast<uint64_t*>(sp);           sp += 16;            // one per staging buffer
  uint32_t* s_ctl = reinterpret_cast<uint32_t*>(sp);          sp += 16;            // second entries of the chunk in staging buffer 0 / 1
  uint32_t* s_par = reinterpret_cast<uint32_t*>(sp);          sp += 32;            // per staging buffer: sector, slot_lo, slot_hi
  uint32_t* dst = reinterpret_cast<uint32_t*>(sp);            sp += nb4 * 4u;      // list offset of the bin's last reservation
  uint16_t* nfull = reinterpret_cast<uint16_t*>(sp);          sp += nb4 * 2u;      // whole sectors of that reservation
  uint32_t* nxt = reinterpret_cast<uint32_t*>(sp);            sp += nb4 * 4u;      // list offset of the sector reserved ahead for the bin

  const uint32_t tid = threadIdx.x;
  for (uint32_t i = tid; i < 256u; i += kBinThreads) {
    const bool in = i < P.n_rows;
    if (i < 64u) {                                            // npads - 1 as bytes, four rows per word
      uint32_t w = 0;
      for (uint32_t k = 0; k < 4u; ++k)
        if (4u * i + k < P.n_rows) w |= (uint32_t(rows[4u * i + k].npads) - 1u) << (8u * k);
      r_npads[i] = w;
    }
    r_off[i] = in ? rows[i].list_off : 0u;
    r_cap[i] = in ? rows[i].cap : 0u;
  }
  for (uint32_t i = tid; i < P.nb; i += kBinThreads) cnt[i] = 0u;
  if (tid == 0) {
    mbar_init(mbar, 1);
    mbar_init(mbar + 1, 1);
    fence_mbar_init();
    s_ctl[0] = 0u;
    s_ctl[1] = 0u;
  }
  uint32_t dropped = 0;
  // the (at most two) digits that do not sit in a full 16-byte pair: direct path, one thread
  if (blockIdx.x == 0 && tid == 32) {
    const uint2* dg = reinterpret_cast<const uint2*>(P.base16) + P.head;
    uint64_t edge[2];
    int ne = 0;
    if (P.head && P.n > 0) edge[ne++] = 0;
    if (((P.n + P.head) & 1ull) && P.n > 0 && !(P.head && P.n == 1)) edge[ne++] = P.n - 1;
    for (int k = 0; k < ne; ++k) {
      uint32_t s0 = 0;
      const uint2 v = dg[edge[k]];
      dropped += bin_one<1>(v.x, v.y, edge[k], s0, P, rows, lists, counts) ? 0u : 1u;
    }
  }

  constexpr uint32_t kPairs = kBinChunk / 2;
  // this CTA's contiguous range of chunks [k0, k1) of the sector-major chunk sequence
  const uint32_t k0 = uint32_t(uint64_t(blockIdx.x) * P.total_chunks / gridDim.x);
  const uint32_t k1 = uint32_t(uint64_t(blockIdx.x + 1) * P.total_chunks / gridDim.x);
  // pair range of chunk k of sector s (k is the global chunk index)
  auto chunk = [&](uint32_t k, uint32_t s, uint64_t& pa, uint32_t& np) {
    const uint64_t p0 = max((P.off[s] + P.head) >> 1, P.pair_lo);
    const uint64_t p1 = min((P.off[s + 1] + P.head + 1) >> 1, P.pair_hi);
    pa = p0 + uint64_t(k - P.cpref[s]) * kPairs;
    np = uint32_t(min(uint64_t(kPairs), p1 - pa));
  };
  auto sector_of = [&](uint32_t k, uint32_t s) -> uint32_t {
    while (k >= P.cpref[s + 1]) ++s;
    return s;
  };
  // one thread: start the TMA copies of chunk k (sector s) into staging buffer b and leave the
  // chunk's parameters for the CTA: slots [slot_lo, slot_hi) hold digits of sector s
  auto load = [&](uint32_t k, uint32_t s, uint32_t b) {
    uint64_t pa;
    uint32_t np;
    chunk(k, s, pa, np);
    // the buffer was last written through the generic proxy (phase A two chunks ago)
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    mbar_arrive_expect_tx(mbar + b, np * 16u);
    uint4* d = reinterpret_cast<uint4*>(stage0 + b * uint32_t(kBinChunk));
    for (uint32_t o = 0; o < np; o += 2048u)                 // <= 32 KB per bulk copy
      tma_bulk_load(d + o, P.base16 + pa + o, min(2048u, np - o) * 16u, mbar + b);
    const int64_t first = int64_t(2ull * pa) - int64_t(P.head);           // digit index of slot 0
    s_par[4u * b] = s;
    s_par[4u * b + 1u] = uint32_t(max(int64_t(P.off[s]) - first, int64_t(0)));
    s_par[4u * b + 2u] = uint32_t(min(int64_t(P.off[s + 1]) - first, int64_t(2u * np)));
  };
  const uint32_t bpr = P.bins_per_row;
  const uint32_t t_span = uint32_t(P.t_hi - P.t_lo);
  // phase B1 visits bins tid, tid + 1024, ... (P.nb <= 4 * kBinThreads): their list offsets and
  // capacities never change, and each keeps ONE SECTOR RESERVED AHEAD (nxt[bin]) so that a flush is
  // a plain store; the reservation that replaces it is an atomic whose result (res_g, valid in
  // res_m) is only looked at one chunk later — its latency is never waited for.
  uint32_t b_off[4], b_cap[4], res_g[4] = {0u, 0u, 0u, 0u}, res_m = 0u;
  auto apply_reservations = [&]() {
#pragma unroll
    for (int x = 0; x < 4; ++x)
      if (res_m & (1u << x))
        nxt[tid + uint32_t(x) * kBinThreads] = (res_g[x] + 8u <= b_cap[x]) ? b_off[x] + res_g[x] : kBinFull;
    res_m = 0u;
  };
  // entering sector s: one sector reserved for every bin
  auto reserve_all = [&](uint32_t s) {
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      const uint32_t bin = tid + uint32_t(x) * kBinThreads;
      if (bin < P.nb) {
        res_g[x] = atomicAdd(&counts[s * P.nb + bin], 8u);
        res_m |= 1u << x;
      }
    }
    apply_reservations();
  };
  // leaving sector s: every bin's partly filled buffer goes to its reserved sector, zero-padded
  // (an empty buffer too: the sector is part of the list now and must not keep stale entries)
  auto flush_all = [&](uint32_t s) {
    uint32_t* seclist = lists + uint64_t(s) * P.sec_list_elems;
    __syncthreads();                                          // phase B2 of the sector's last chunk (any thread) has filled the buffers
    apply_reservations();
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      const uint32_t bin = tid + uint32_t(x) * kBinThreads;
      if (bin < P.nb) {
        const uint32_t n = cnt[bin];                          // < 8: fuller bins were flushed in phase B1
        for (uint32_t y = n; y < 8u; ++y) buf[bin * 8u + y] = 0u;
        const uint4 a = *reinterpret_cast<const uint4*>(buf + bin * 8u);
        const uint4 c = *reinterpret_cast<const uint4*>(buf + bin * 8u + 4u);
        const uint32_t d = nxt[bin];
        if (d != kBinFull) {
          TPC_ASSERT(n < 8u && d >= b_off[x] && d + 8u <= b_off[x] + b_cap[x] && uint64_t(d) + 8u <= P.sec_list_elems);
          store8(seclist + d, a, c);
        }
        cnt[bin] = 0u;
      }
    }
    __syncthreads();
  };

  uint32_t s = 0, parbits = 0u;                            // bit b: wait parity of staging buffer b
  if (k0 < k1) {
    s = sector_of(k0, 0);
    if (tid == 0) load(k0, s, 0);
  }
  __syncthreads();
#pragma unroll
  for (int x = 0; x < 4; ++x) {
    const uint32_t bin = tid + uint32_t(x) * kBinThreads;
    const uint32_t row = min(bin / bpr, 255u), tb = bin - (bin / bpr) * bpr;
    b_cap[x] = r_cap[row];
    b_off[x] = r_off[row] + tb * b_cap[x];
  }
  if (k0 < k1) reserve_all(s);
  // ---- phase B2 of a chunk (entries ranked >= 8: into the reserved sectors, or back into the emptied buffer) is run
  //      at the START of the next iteration, in front of that chunk's phase A and without a barrier between them:
  //      B2 only writes buffer slots below the bin's fill count, phase A only takes ranks from the fill count up, and
  //      the two use different staging buffers and second-entry lists.  The slow, latency-bound B2 of some warps thus
  //      overlaps the issue-bound phase A of the others, and a chunk costs two barriers instead of three ----
  uint32_t pend = 0;                                         // this thread's entries of the previous chunk that wait for B2
  auto phase_b2 = [&](uint32_t bp, uint32_t* seclist) {      // bp: staging buffer of that chunk
    const uint2* stage2 = reinterpret_cast<const uint2*>(stage0 + bp * uint32_t(kBinChunk));
    auto place = [&](uint32_t pk, uint32_t y) {
      const uint32_t bin = y & 0xFFFu, r = y >> 12;
      const uint32_t nf8 = uint32_t(nfull[bin]) << 3;
      TPC_ASSERT(bin < P.nb && r >= 8u);
      if (r >= nf8) {
        TPC_ASSERT(r - nf8 < 8u);
        buf[bin * 8u + (r - nf8)] = pk;
      } else {
        const uint32_t d = dst[bin];
        TPC_ASSERT(d == kBinFull || uint64_t(d) + r < P.sec_list_elems);
        if (d != kBinFull) seclist[d + r] = pk;
      }
    };
    while (pend) {                    // most lanes have none: the loop runs as long as some lane has one
      const uint32_t e = __ffs(pend) - 1;
      pend &= pend - 1;
      const uint2 v = stage2[2u * ((e >> 1) * kBinThreads + tid) + (e & 1u)];
      place(v.x, v.y);
    }
    const uint2* secp = sec + bp * uint32_t(kBinSecCap);
    const uint32_t nsec = min(s_ctl[bp], uint32_t(kBinSecCap));
    for (uint32_t i = tid; i < nsec; i += kBinThreads) {
      const uint2 e = secp[i];
      if ((e.y >> 12) >= 8u) place(e.x, e.y);
    }
  };
  for (uint32_t k = k0; k < k1; ++k) {
    const uint32_t b = (k - k0) & 1u;
    if (k > k0) phase_b2(b ^ 1u, lists + uint64_t(s) * P.sec_list_elems);   // of chunk k - 1 (still sector s)
    {
      const uint32_t s_new = s_par[4u * b];
      if (s_new != s) {
        flush_all(s);
        s = s_new;
        reserve_all(s);
      }
    }
    const uint32_t slot_lo = s_par[4u * b + 1u], slot_hi = s_par[4u * b + 2u];
    const bool full_chunk = slot_lo == 0u && slot_hi == uint32_t(kBinChunk);   // no sector seam inside: no per-digit check
    const uint32_t cbase = s * P.nb;
    uint32_t* seclist = lists + uint64_t(s) * P.sec_list_elems;
    uint4* stage4 = reinterpret_cast<uint4*>(stage0 + b * uint32_t(kBinChunk));
    uint32_t* nsecp = s_ctl + b;                             // second entries of this chunk
    uint2* secb = sec + b * uint32_t(kBinSecCap);
    mbar_wait(mbar + b, (parbits >> b) & 1u);
    parbits ^= 1u << b;

    // rank an entry inside its bin; ranks 0..7 go to the bin's buffer
    auto insert = [&](uint32_t bin, uint32_t pk) -> uint32_t {
      TPC_ASSERT(bin < P.nb && pk != 0u);
      const uint32_t r = atomicAdd(&cnt[bin], 1u);
      if (r < 8u) buf[bin * 8u + r] = pk;
      return r;
    };
    // ---- phase A: quantise (D1), validate, rank.  An entry ranked >= 8 (its bin's buffer is full)
    //      overwrites its digit in the staging area and is remembered in `pend` for phase B2 ----
    uint2* stage2 = reinterpret_cast<uint2*>(stage4);
#pragma unroll
    for (int i = 0; i < kBinPer / 2; ++i) {
      const uint32_t pi = uint32_t(i) * kBinThreads + tid;
      const uint4 v = stage4[pi];
#pragma unroll
      for (int h = 0; h < 2; ++h) {
        const uint32_t w0 = h ? v.z : v.x, w1 = h ? v.w : v.y;
        const uint32_t j = 2u * pi + uint32_t(h);
        if (full_chunk || j - slot_lo < slot_hi - slot_lo) {
          const uint32_t row = w0 & 0xFFu, pad = (w0 >> 8) & 0xFFu;
          const int32_t time = int32_t(w0 >> 16) + P.t_base;        // A19
          const uint32_t q = quantise_q16(__uint_as_float(w1));
          const uint32_t last_pad = (r_npads[row >> 2] >> (8u * (row & 3u))) & 0xFFu;   // npads - 1
          if (q == 0u || uint32_t(time - P.t_lo) >= t_span || pad > last_pad || row >= P.n_rows) {
            ++dropped;
          } else {
            const int32_t u = time - P.t_core_begin;
            const int32_t tlo = max((u - kReach) >> kBinShift, 0);
            const int32_t thi = min((u + kReach) >> kBinShift, int32_t(bpr) - 1);
            if (tlo <= thi) {
              const uint32_t bin = row * bpr + uint32_t(tlo);
              const uint32_t pk = pack_digit(pad, uint32_t(u - (tlo << kBinShift) + kReach), q);
              const uint32_t r = insert(bin, pk);
              if (r >= 8u) {
                stage2[j] = make_uint2(pk, bin | (r << 12));
                pend |= 1u << (2 * i + h);
              }
              if (thi != tlo) {                               // also in the next bin's window
                const uint32_t pk2 = pk - (uint32_t(kBinT) << 8);
                const uint32_t k2 = atomicAdd(nsecp, 1u);
                TPC_ASSERT(bin + 1u < P.nb && uint32_t(thi) == uint32_t(tlo) + 1u);
                if (k2 < uint32_t(kBinSecCap)) {
                  secb[k2] = make_uint2(pk2, (bin + 1u) | (insert(bin + 1u, pk2) << 12));
                } else {                                      // second-entry list full: direct path
                  const uint32_t cap = r_cap[row];
                  bin_append<1>(seclist, &counts[cbase + bin + 1u], r_off[row] + uint32_t(tlo + 1) * cap, cap, pk2);
                }
              }
            }
          }
        }
      }
    }
    __syncthreads();                  // every entry is ranked (and phase B2 of the previous chunk is done): buffers and counts are complete
    if (tid == 0 && k + 1 < k1) load(k + 1, sector_of(k + 1, s), b ^ 1u);   // that buffer's last readers were the B2 above; lands during B1

    // ---- phase B1: bins holding a whole sector: store it into the sector reserved ahead, request the
    //      next reservation (one global atomic per flush, never waited for), keep the remainder ----
    if (tid == 0) s_ctl[b ^ 1u] = 0u; // the other buffer's counter is idle until the next chunk's phase A
    apply_reservations();             // (issued in the previous chunk's phase B1)
    uint32_t n4[4];                   // (the four fill counts are loaded before the first flush: independent round trips)
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      const uint32_t bin = tid + uint32_t(x) * kBinThreads;
      n4[x] = bin < P.nb ? cnt[bin] : 0u;
    }
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      const uint32_t bin = tid + uint32_t(x) * kBinThreads;
      const uint32_t n = n4[x];
      if (n >= 8u) {
        const uint4 a = *reinterpret_cast<const uint4*>(buf + bin * 8u);
        const uint4 c = *reinterpret_cast<const uint4*>(buf + bin * 8u + 4u);
        const uint32_t d = nxt[bin];
        if (d != kBinFull) {
          TPC_ASSERT(d >= b_off[x] && d + 8u <= b_off[x] + b_cap[x] && uint64_t(d) + 8u <= P.sec_list_elems);
          store8(seclist + d, a, c);
        }
        res_g[x] = atomicAdd(&counts[cbase + bin], 8u);       // the next sector, looked at one chunk later
        res_m |= 1u << x;
        const uint32_t nf = n >> 3;
        if (nf > 1u) {                                        // more than two sectors' worth arrived at once (sorted input)
          const uint32_t g2 = atomicAdd(&counts[cbase + bin], (nf - 1u) * 8u);
          dst[bin] = (g2 + (nf - 1u) * 8u <= b_cap[x]) ? b_off[x] + g2 - 8u : kBinFull;   // rank r >= 8 goes to dst + r
        }
        nfull[bin] = uint16_t(nf);
        cnt[bin] = n & 7u;            // entries ranked >= 8 * nfull move to the buffer's front in phase B2
      }
    }
    __syncthreads();                  // full buffers are out, nfull / dst are set for the chunk's phase B2 (run next iteration)
  }
  if (k0 < k1) {
    phase_b2((k1 - 1u - k0) & 1u, lists + uint64_t(s) * P.sec_list_elems);
    flush_all(s);
  }
  dropped = __reduce_add_sync(0xffffffffu, dropped);
  if ((tid & 31u) == 0u && dropped) atomicAdd(&status->n_dropped, (unsigned long long)dropped);
}

}  // namespace tpcclus

#include "tpcclus_tile.cuh"
#include "tpcclus_select.cuh"
