// tpcclus_kernels.cuh — sm_100a kernels of the TPC cluster finder (device side).
//
// Steps of SURVEY.md §8(a) and where they run:
//   S0  set-up               k_init   zero the per-bin entry counters and the run status
//   S1  charge-map fill      k_bin    TMA-staged digit chunks (16-byte pairs), D1 quantisation, digit ->
//                                     packed 4-byte entry in the list of every (sector,row,256-bin) digit
//                                     bin whose window holds it; write-combined: one 32-byte sector and
//                                     one global atomic per 8 entries
//                            k_tile   front warps: the bin's list is scattered into the (pad x time)
//                                     charge map of the tile, which lives in shared memory only
//   S2  peak finding         k_tile   front warps: digit-driven 3x3 ordered-maximum test on the smem map
//                                     -> flag bitmap; then each peak's 80-byte window is cut out
//   S3  peak count S(c)      k_tile   back warps: other peaks of the 9x9 flag window, table-driven
//   S4  5x5 assembly         k_tile   back warps: four lanes per peak (rotation classes)
//   S5  centroid / width     k_tile   back warps: exact integer moments; committer warp: fp64 finish
//   S6  ordered compaction   k_tile   front warps: popc prefix inside the tile; committer warp: decoupled
//                                     look-back across tiles in (sector,row,time) ticket order, copy-out
//   S7  fragment ownership   k_tile   tiles cover exactly the core [b,e); halo rows never emit
//
// Definitions D1..D12 are those of SURVEY.md §8(c) (restated in DESIGN.md §2); the D-number
// is cited where each rule is implemented.  No code here is shared with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <type_traits>

namespace tpcclus {

constexpr int      kThreads      = 640;   // CTA size of k_tile (two CTAs per SM)
constexpr int      kWorkThreads  = 608;   // warps 0..18: front (0..14) and back (15..18) warps; warp 19 commits
constexpr int      kTileT        = 256;   // core time bins per tile (= one digit bin of k_bin)
constexpr int      kReach        = 5;     // D9: charges within Chebyshev distance 5 decide a cluster
constexpr int      kBoxH         = kTileT + 2 * kReach;   // map rows of a tile (138)
constexpr int      kBinT         = 256;   // core time bins per digit bin (= two tiles: k_tile filters by half)
constexpr int      kBinShift     = 8;
constexpr int      kBinBoxH      = kBinT + 2 * kReach;    // time rows a bin's window spans (266)
static_assert((1 << kBinShift) == kBinT && kBinT == kTileT, "a digit bin is one tile");
constexpr int      kColOff       = 2;     // map column of pad 0 (two zero columns each side: 5x5 window)
constexpr int      kListCap      = 120;   // peaks per hand-over item (capacity of one window / staging buffer)
constexpr uint32_t kQClamp       = 16368; // D1
constexpr int      kMaxSectors   = 256;

struct RowInfo {              // one per pad row (device table)
  uint32_t list_off;          // element offset of this row's bins inside one sector's digit lists
  uint32_t cap;               // list capacity of one bin (multiple of 8): window cells * 5/4 + padding margin
  uint16_t npads;
  uint16_t W;                 // smem map pitch in cells = roundup8(npads + 4)
  uint32_t pad_;
};

struct DevStatus {            // device-side run status, copied to pinned host memory after the run
  unsigned long long n_dropped;
  unsigned long long n_clusters;
  unsigned int       ticket;  // tile ticket counter of k_tile
  unsigned int       pad_;
};

struct BinParams {
  uint64_t n;                          // digits
  uint64_t sec_list_elems;             // list elements per sector
  int32_t  t_core_begin;               // b
  int32_t  t_lo, t_hi;                 // loaded range [lo,hi) in global time (D1)
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
  uint32_t map_bytes_max;              // smem bytes reserved for map + flag bitmap
  uint32_t bm_words;                   // flag-bitmap words per tile row
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
  }
  const uint32_t n4 = (n_tiles + 3u) >> 2;                 // the array is padded to a multiple of 4
  for (uint32_t k = i; k < n4; k += gridDim.x * blockDim.x)
    reinterpret_cast<uint4*>(counts)[k] = make_uint4(0u, 0u, 0u, 0u);
}

// ----------------------------------------------------------------------------------------
// S1 (first half): digit binning.  One 16-byte load = two digits (BASELINE.json:north_star (2):
// "16-byte vectorised coalesced loads").  D1 quantisation; invalid digits dropped and counted.
// A valid digit at global time t is appended, as pad | tl<<8 | q16<<16 with tl its row inside
// the tile's 138-row window, to the list of every tile tt whose window
// [b + 128 tt - 5, b + 128 tt + 133) contains t (one tile, or two next to a tile seam).
// A bin has one slot per map cell, so it cannot overflow while D2's precondition (at most one
// digit per cell) holds; slots past the capacity are discarded (memory-safe for duplicates).
// ----------------------------------------------------------------------------------------
// packed list entry: pad (8 bits) | tl << 8 (row of the tile window, 9 bits) | q16 << 17 (14 bits)
__device__ __forceinline__ uint32_t pack_digit(uint32_t pad, uint32_t tl, uint32_t q) { return pad | (tl << 8) | (q << 17); }
__device__ __forceinline__ uint32_t dig_pad(uint32_t d) { return d & 0xFFu; }
__device__ __forceinline__ uint32_t dig_tl(uint32_t d) { return (d >> 8) & 0x1FFu; }
__device__ __forceinline__ uint32_t dig_q(uint32_t d) { return d >> 17; }

__device__ __forceinline__ uint32_t quantise_q16(float charge) {
  // D1: q16 = clamp(rint(charge*16), 0, 16368).  cvt.rni.u32.f32 rounds half-even and saturates:
  // negative and NaN -> 0, huge -> 0xFFFFFFFF
  return min(__float2uint_rn(charge * 16.0f), kQClamp);
}

// append one packed digit to a bin, reserving R slots (R = 1: k_bin_direct; R = 8: the odd
// entries of the write-combining kernel, whose reservations stay multiples of 8 — the other
// R-1 slots are zero = "no digit")
template <int R>
__device__ __forceinline__ void bin_append(uint32_t* __restrict__ seclist, uint32_t* __restrict__ cnt, uint32_t dest0,
                                           uint32_t cap, uint32_t pk) {
  const uint32_t slot = atomicAdd(cnt, uint32_t(R));
  if (slot + uint32_t(R) <= cap) {
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
  const int32_t time = int32_t(w0 >> 16);
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
constexpr uint32_t kBinNone     = 0xFFFFFFFFu;              // staging slot without a list entry

__host__ __device__ inline uint32_t bin_smem_bytes(uint32_t nb) {
  const uint32_t nb4 = (nb + 3u) & ~3u;
  return 2u * uint32_t(kBinChunk) * 8u + nb4 * 32u + nb4 * 4u + nb4 * 4u + nb4 * 4u + nb4 * 2u + uint32_t(kBinSecCap) * 8u +
         3u * 256u * 4u + 96u + 128u;
}

__device__ __forceinline__ void st_v4(uint32_t* p, uint4 v) { *reinterpret_cast<uint4*>(p) = v; }

__global__ void __launch_bounds__(kBinThreads, 1) k_bin(const __grid_constant__ BinParams P,
                                                        const RowInfo* __restrict__ rows, uint32_t* __restrict__ lists,
                                                        uint32_t* __restrict__ counts, DevStatus* __restrict__ status) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  const uint32_t nb4 = (P.nb + 3u) & ~3u;
  uint8_t* sp = smem_raw;                                     // __align__(128); no static shared memory before it
  uint2* stage0 = reinterpret_cast<uint2*>(sp);               sp += 2u * uint32_t(kBinChunk) * 8u;   // two TMA destinations
  uint32_t* buf = reinterpret_cast<uint32_t*>(sp);            sp += nb4 * 32u;     // 8 entries per bin
  uint32_t* cnt = reinterpret_cast<uint32_t*>(sp);            sp += nb4 * 4u;      // fill count per bin
  uint2* sec = reinterpret_cast<uint2*>(sp);                  sp += uint32_t(kBinSecCap) * 8u;
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
      dropped += bin_one<8>(v.x, v.y, edge[k], s0, P, rows, lists, counts) ? 0u : 1u;
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
          st_v4(seclist + d, a);
          st_v4(seclist + d + 4, c);
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
  for (uint32_t k = k0; k < k1; ++k) {
    const uint32_t b = (k - k0) & 1u;
    {
      const uint32_t s_new = s_par[4u * b];
      if (s_new != s) {
        flush_all(s);
        s = s_new;
        reserve_all(s);
      }
    }
    if (tid == 0 && k + 1 < k1) load(k + 1, sector_of(k + 1, s), b ^ 1u);   // lands while this chunk is processed
    const uint32_t slot_lo = s_par[4u * b + 1u], slot_hi = s_par[4u * b + 2u];
    const bool full_chunk = slot_lo == 0u && slot_hi == uint32_t(kBinChunk);   // no sector seam inside: no per-digit check
    const uint32_t cbase = s * P.nb;
    uint32_t* seclist = lists + uint64_t(s) * P.sec_list_elems;
    uint4* stage4 = reinterpret_cast<uint4*>(stage0 + b * uint32_t(kBinChunk));
    uint32_t* nsecp = s_ctl + b;                             // second entries of this chunk
    mbar_wait(mbar + b, (parbits >> b) & 1u);
    parbits ^= 1u << b;

    // rank an entry inside its bin; ranks 0..7 go to the bin's buffer
    auto insert = [&](uint32_t bin, uint32_t pk) -> uint32_t {
      const uint32_t r = atomicAdd(&cnt[bin], 1u);
      if (r < 8u) buf[bin * 8u + r] = pk;
      return r;
    };
    // ---- phase A: quantise (D1), validate, rank.  An entry ranked >= 8 (its bin's buffer is full)
    //      overwrites its digit in the staging area and is remembered in `pend` for phase B2 ----
    uint32_t pend = 0;
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
          const int32_t time = int32_t(w0 >> 16);
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
                if (k2 < uint32_t(kBinSecCap)) {
                  sec[k2] = make_uint2(pk2, (bin + 1u) | (insert(bin + 1u, pk2) << 12));
                } else {                                      // second-entry list full: reserve-8 direct path
                  const uint32_t cap = r_cap[row];
                  bin_append<8>(seclist, &counts[cbase + bin + 1u], r_off[row] + uint32_t(tlo + 1) * cap, cap, pk2);
                }
              }
            }
          }
        }
      }
    }
    __syncthreads();                  // every entry is ranked; buffers and counts are complete

    // ---- phase B1: bins holding a whole sector: store it into the sector reserved ahead, request the
    //      next reservation (one global atomic per flush, never waited for), keep the remainder ----
    if (tid == 0) s_ctl[b ^ 1u] = 0u; // the other buffer's counter is idle until the next chunk's phase A
    apply_reservations();             // (issued in the previous chunk's phase B1)
#pragma unroll
    for (int x = 0; x < 4; ++x) {
      const uint32_t bin = tid + uint32_t(x) * kBinThreads;
      const uint32_t n = bin < P.nb ? cnt[bin] : 0u;
      if (n >= 8u) {
        const uint4 a = *reinterpret_cast<const uint4*>(buf + bin * 8u);
        const uint4 c = *reinterpret_cast<const uint4*>(buf + bin * 8u + 4u);
        const uint32_t d = nxt[bin];
        if (d != kBinFull) {
          st_v4(seclist + d, a);
          st_v4(seclist + d + 4, c);
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
    __syncthreads();

    // ---- phase B2: entries ranked >= 8: into the reserved sectors, or back into the (now empty) buffer ----
    auto place = [&](uint32_t pk, uint32_t y) {
      const uint32_t bin = y & 0xFFFu, r = y >> 12;
      const uint32_t nf8 = uint32_t(nfull[bin]) << 3;
      if (r >= nf8) {
        buf[bin * 8u + (r - nf8)] = pk;
      } else {
        const uint32_t d = dst[bin];
        if (d != kBinFull) seclist[d + r] = pk;
      }
    };
    while (pend) {                    // most lanes have none: the loop runs as long as some lane has one
      const uint32_t e = __ffs(pend) - 1;
      pend &= pend - 1;
      const uint2 v = stage2[2u * ((e >> 1) * kBinThreads + tid) + (e & 1u)];
      place(v.x, v.y);
    }
    {
      const uint32_t nsec = min(*nsecp, uint32_t(kBinSecCap));
      for (uint32_t i = tid; i < nsec; i += kBinThreads) {
        const uint2 e = sec[i];
        if ((e.y >> 12) >= 8u) place(e.x, e.y);
      }
    }
    __syncthreads();                  // buffers, staging area and lists are reused by the next chunk
  }
  if (k0 < k1) flush_all(s);
  dropped = __reduce_add_sync(0xffffffffu, dropped);
  if ((tid & 31u) == 0u && dropped) atomicAdd(&status->n_dropped, (unsigned long long)dropped);
}

// ----------------------------------------------------------------------------------------
// S1 (second half) .. S7: fused tile kernel.
// ----------------------------------------------------------------------------------------
struct __align__(16) ClusterRec {   // byte-for-byte the tpcclus_cluster of include/tpcclus.h
  uint32_t w0;                      // sector | row<<8 | pad<<16 | flags<<24
  uint32_t time;
  uint32_t w2;                      // qmax_q16 | ncells<<16
  float qtot, dpad, dtime, sigma_pad, sigma_time;
};
static_assert(sizeof(ClusterRec) == 32, "cluster record is 32 bytes");

constexpr unsigned long long kStAgg = 1ull, kStPrefix = 2ull;
__device__ __forceinline__ unsigned long long pack_state(uint32_t epoch, unsigned long long st, uint32_t v) {
  return (uint64_t(epoch) << 34) | (st << 32) | uint64_t(v);
}

// Exclusive prefix of this tile's peak count over all earlier tiles (decoupled look-back;
// tiles are taken by ticket in (sector,row,time) order, so every earlier tile is owned by a
// CTA that is already running).  Called by one full warp.
__device__ __forceinline__ uint32_t lookback_exclusive(unsigned long long* state, uint32_t tile, uint32_t epoch,
                                                       uint32_t aggregate) {
  const uint32_t lane = threadIdx.x & 31;
  if (tile == 0) {
    if (lane == 0) st_release_u64(state, pack_state(epoch, kStPrefix, aggregate));
    return 0;
  }
  // the tile's own count (kStAgg) was published by its front warps right after the count phase
  uint32_t sum = 0;
  int64_t look = int64_t(tile) - 1;
  while (true) {
    const int64_t idx = look - lane;
    unsigned long long v;
    uint32_t okmask, pfxmask;
    do {   // wait until the 32 (or fewer) predecessors in the window have published something
      v = idx >= 0 ? ld_acquire_u64(state + idx) : pack_state(epoch, kStPrefix, 0);
      const bool valid = (uint32_t(v >> 34) == epoch) && (((v >> 32) & 3ull) != 0ull);
      okmask = __ballot_sync(0xffffffffu, valid);
      pfxmask = __ballot_sync(0xffffffffu, valid && (((v >> 32) & 3ull) == kStPrefix));
      // only lanes up to the nearest inclusive prefix have to be valid
      const uint32_t need = pfxmask ? ((2u << (__ffs(pfxmask) - 1)) - 1u) : 0xffffffffu;
      if ((okmask & need) == need) break;
    } while (true);
    const uint32_t upto = pfxmask ? uint32_t(__ffs(pfxmask) - 1) : 31u;
    const uint32_t contrib = lane <= upto ? uint32_t(v) : 0u;
    sum += __reduce_add_sync(0xffffffffu, contrib);
    if (pfxmask) break;
    look -= 32;
  }
  if (lane == 0) st_release_u64(state + tile, pack_state(epoch, kStPrefix, sum + aggregate));
  return sum;
}

// ----------------------------------------------------------------------------------------
// S3..S5, four lanes per peak.
//
// The 24 cells around a peak P split into four rotation classes of six: lane `sub` (0..3) owns
// the images under the quarter turn R_sub of the base cells
//     I0 = (1,0)  I1 = (1,1)                      inner ring (always members when charged, D5)
//     O0 = (2,-1) O1 = (2,0) O2 = (2,1) O3 = (2,2) outer ring (monotone descent, D5)
// written (a,b) = (pad, time) offsets in the lane's own frame; R_s(a,b) = (a cs - b sn, a sn + b cs)
// with (cs,sn) = (1,0),(0,1),(-1,0),(0,-1).  The inner cells 8-adjacent to O0..O3 are
// (1,-1),(1,0),(1,1) of the same frame, so a lane reads 7 charges.  Moments are summed in the
// lane frame with constant coefficients and rotated once.  D6's S(c) comes from the OTHER peaks
// of the 9x9 flag window: each one adds a table entry (one nibble per owned cell it is within
// distance 2 of, plus an "is this outer cell" bit).  The four partial sums are combined with two
// xor-shuffles; the record is staged as exact integers (RawRec) and finished by the committer warp.
// ----------------------------------------------------------------------------------------
constexpr int kNbrTabWords = 4 * 81;
constexpr uint32_t kShareL = 2520u;                      // D6: lcm(1..9)

// entry for lane frame s and another peak at window row k (time j-4+k), column i (pad p-4+i)
__device__ __forceinline__ uint32_t nbr_tab_entry(uint32_t idx) {
  const int s = int(idx / 81u), r = int(idx % 81u);
  const int u = r % 9 - 4, v = r / 9 - 4;               // (pad, time) offset of the other peak
  int up, vp;                                           // the same offset in the lane frame: R_s^-1 (u,v)
  if (s == 0)      { up = u;  vp = v; }
  else if (s == 1) { up = v;  vp = -u; }
  else if (s == 2) { up = -u; vp = -v; }
  else             { up = -v; vp = u; }
  const int ca[6] = {1, 1, 2, 2, 2, 2}, cb[6] = {0, 1, -1, 0, 1, 2};
  uint32_t e = 0;
  for (int c = 0; c < 6; ++c) {
    const int da = ca[c] - up, db = cb[c] - vp;
    if (da >= -2 && da <= 2 && db >= -2 && db <= 2) e += 1u << (4 * c);
    if (c >= 2 && da == 0 && db == 0) e |= 1u << (24 + c - 2);
  }
  return e;
}

struct __align__(16) RawRec {       // what the back warps stage: D7's exact integers; the committer turns it into ClusterRec
  uint32_t w0, time, w2;            // as in ClusterRec
  uint32_t W;                       // sum of weights, units of 1/(16*2520) ADC
  int32_t Mp, Mt;                   // sum w dp, sum w dt
  uint32_t Mpp, Mtt;                // sum w dp^2, sum w dt^2
};
static_assert(sizeof(RawRec) == 32, "raw record is 32 bytes");

// A peak's WINDOW: what S3..S5 need of the tile's map and flags, 80 bytes.  The front warps cut it
// out (four lanes per peak) so that the map can be reused for the next tile while the back warps
// still build this tile's clusters.  Layout (5 x uint4): [lane frame 0..3: the 8 charges
// qP|qIm, qI0|qI1, qO0|qO1, qO2|qO3 as u16 pairs] [G0, G1, G2, j<<16 | pad] with the 9x9 flag
// window packed three rows per word: bit 9*(k%3)+i of G[k/3] <-> row j-4+k, pad p-4+i, P cleared.
constexpr int kWinWords = 20;

// All 32 lanes call this; lanes 4g..4g+3 work on the same peak (j = map row, pad).
__device__ __forceinline__ void extract_window4(const uint16_t* __restrict__ map, const uint32_t* __restrict__ bm,
                                                uint32_t W, uint32_t bmw, uint32_t j, uint32_t pad, uint32_t sub,
                                                int32_t cs, int32_t sn, uint4* __restrict__ win) {
  const uint16_t* c = map + j * W + (pad + kColOff);
  const int32_t X = sn * int32_t(W) + cs, Y = cs * int32_t(W) - sn;     // steps of (a,b) in map cells
  const uint32_t qP = c[0];
  const uint32_t qIm = c[X - Y], qI0 = c[X], qI1 = c[X + Y];
  const uint32_t qO0 = c[2 * X - Y], qO1 = c[2 * X], qO2 = c[2 * X + Y], qO3 = c[2 * X + 2 * Y];
  win[sub] = make_uint4(qP | (qIm << 16), qI0 | (qI1 << 16), qO0 | (qO1 << 16), qO2 | (qO3 << 16));
  // flag rows: lane s reads rows s and s+4, lane 0 also row 8; OR-combined over the four lanes
  uint32_t G0 = 0, G1 = 0, G2 = 0;
  {
    const uint32_t sh = pad & 31u;
    const uint32_t* rowp = bm + (j - 4u) * bmw + (pad >> 5);
    auto row_bits = [&](uint32_t k) -> uint32_t {
      return __funnelshift_r(rowp[k * bmw], rowp[k * bmw + 1], sh) & 0x1FFu;
    };
    const uint32_t fa = row_bits(sub), fb = row_bits(sub + 4u), fc = sub == 0u ? row_bits(8u) : 0u;
    // row k -> word k/3, shift 9*(k%3)
    if (sub < 3u) G0 = fa << (9u * sub); else G1 = fa;                   // rows 0,1,2 | 3
    if (sub < 2u) G1 |= fb << (9u * (sub + 1u)); else G2 = fb << (9u * (sub - 2u));   // rows 4,5 | 6,7
    G2 |= fc << 18;                                                      // row 8
#pragma unroll
    for (int o = 1; o <= 2; o <<= 1) {
      G0 |= __shfl_xor_sync(0xffffffffu, G0, o);
      G1 |= __shfl_xor_sync(0xffffffffu, G1, o);
      G2 |= __shfl_xor_sync(0xffffffffu, G2, o);
    }
    G1 &= ~(1u << 13);                                                  // P itself (row 4, column 4)
  }
  if (sub == 3u) win[4] = make_uint4(G0, G1, G2, (j << 16) | pad);
}

// All 32 lanes call this; lanes 4g..4g+3 assemble the cluster of one window.  Returns the two
// 16-byte halves of the RawRec in every lane of the group.
__device__ __forceinline__ void assemble4(const uint4* __restrict__ win, const uint32_t* __restrict__ nbr_tab,
                                          const uint32_t* __restrict__ wtab, uint32_t sub, int32_t cs, int32_t sn,
                                          uint32_t sector_row /* sector | row << 8 */, uint32_t npads, int32_t t_row0,
                                          uint32_t tf_time_bins, uint4& lo, uint4& hi) {
  const uint4 ch = win[sub], fl = win[4];
  const uint32_t qP = ch.x & 0xFFFFu, qIm = ch.x >> 16, qI0 = ch.y & 0xFFFFu, qI1 = ch.y >> 16;
  const uint32_t qO0 = ch.z & 0xFFFFu, qO1 = ch.z >> 16, qO2 = ch.w & 0xFFFFu, qO3 = ch.w >> 16;
  uint32_t G0 = fl.x, G1 = fl.y, G2 = fl.z;
  const uint32_t pad = fl.w & 0xFFFFu;
  const int32_t tglob = t_row0 + int32_t(fl.w >> 16);                  // t_row0 = global time of map row 0
  uint32_t acc = 0;                                                     // nibble c: other peaks within distance 2 of cell c
  {
    const uint32_t* t = nbr_tab + sub * 81u;
    while (G0) { const uint32_t b = __ffs(G0) - 1; G0 &= G0 - 1; acc += t[b]; }
    while (G1) { const uint32_t b = __ffs(G1) - 1; G1 &= G1 - 1; acc += t[27 + b]; }
    while (G2) { const uint32_t b = __ffs(G2) - 1; G2 &= G2 - 1; acc += t[54 + b]; }
  }
  // D5 membership
  const bool mI0 = qI0 != 0u, mI1 = qI1 != 0u;
  const bool mO0 = qO0 != 0u && !((acc >> 24) & 1u) && (qIm >= qO0 || qI0 >= qO0);
  const bool mO1 = qO1 != 0u && !((acc >> 25) & 1u) && (qIm >= qO1 || qI0 >= qO1 || qI1 >= qO1);
  const bool mO2 = qO2 != 0u && !((acc >> 26) & 1u) && (qI0 >= qO2 || qI1 >= qO2);
  const bool mO3 = qO3 != 0u && !((acc >> 27) & 1u) && (qI1 >= qO3);
  // D6 weights w = Q * L / S, S = 1 + other peaks within distance 2
  uint32_t meta = 0;                                                    // ncells | n_saturated << 8 | n_split << 16
  auto weight = [&](bool m, uint32_t q, uint32_t nib) -> uint32_t {
    const uint32_t S = (acc >> (4 * nib)) & 15u;                        // S - 1
    if (m) meta += 1u + (q == kQClamp ? 0x100u : 0u) + (S ? 0x10000u : 0u);
    return m ? q * wtab[S] : 0u;
  };
  const uint32_t wI0 = weight(mI0, qI0, 0), wI1 = weight(mI1, qI1, 1);
  const uint32_t wO0 = weight(mO0, qO0, 2), wO1 = weight(mO1, qO1, 3);
  const uint32_t wO2 = weight(mO2, qO2, 4), wO3 = weight(mO3, qO3, 5);
  // D7 moments in the lane frame, then rotated (cs*sn = 0)
  const uint32_t wO = wO0 + wO1 + wO2 + wO3, wI = wI0 + wI1;
  uint32_t Wsum = wI + wO;
  const int32_t Ma = int32_t(wI + 2u * wO);
  const int32_t Mb = int32_t(wI1 + wO2 + 2u * wO3) - int32_t(wO0);
  const uint32_t Maa = wI + 4u * wO;
  const uint32_t Mbb = wI1 + wO0 + wO2 + 4u * wO3;
  int32_t Mp = cs * Ma - sn * Mb, Mt = sn * Ma + cs * Mb;
  uint32_t Mpp = cs ? Maa : Mbb, Mtt = cs ? Mbb : Maa;
#pragma unroll
  for (int o = 1; o <= 2; o <<= 1) {
    Wsum += __shfl_xor_sync(0xffffffffu, Wsum, o);
    Mp += __shfl_xor_sync(0xffffffffu, Mp, o);
    Mt += __shfl_xor_sync(0xffffffffu, Mt, o);
    Mpp += __shfl_xor_sync(0xffffffffu, Mpp, o);
    Mtt += __shfl_xor_sync(0xffffffffu, Mtt, o);
    meta += __shfl_xor_sync(0xffffffffu, meta, o);
  }
  Wsum += qP * kShareL;                                                 // D6: w(P) = L Q(P)
  uint32_t flags = 0;
  if (pad < 2u || pad + 2u >= npads) flags |= 1u;                       // D8 EDGE_PAD
  if (tglob < 2 || uint32_t(tglob) + 2u >= tf_time_bins) flags |= 2u;   // D8 EDGE_TIME
  if (qP == kQClamp || (meta & 0xFF00u)) flags |= 4u;                   // SATURATED
  if (meta >> 16) flags |= 8u;                                          // SPLIT
  lo = make_uint4(sector_row | (pad << 16) | (flags << 24), uint32_t(tglob),
                  qP | (((meta & 0xFFu) + 1u) << 16), Wsum);
  hi = make_uint4(uint32_t(Mp), uint32_t(Mt), Mpp, Mtt);
}

// ----------------------------------------------------------------------------------------
// S5 finish (D8): RawRec -> ClusterRec.  Evaluated in double from the exact integers and
// rounded once to float32.
// ----------------------------------------------------------------------------------------
// D8 on one record: RawRec halves -> ClusterRec halves
__device__ __forceinline__ void finish_rec(uint4& lo, uint4& hi) {
  const uint32_t W_ = lo.w;
  const int32_t Mp = int32_t(hi.x), Mt = int32_t(hi.y);
  const double Wd = double(W_);
  const long long Np = (long long)hi.z * (long long)W_ - (long long)Mp * (long long)Mp;
  const long long Nt = (long long)hi.w * (long long)W_ - (long long)Mt * (long long)Mt;
  lo.w = __float_as_uint(float(Wd / 40320.0));
  hi.x = __float_as_uint(float(double(Mp) / Wd));
  hi.y = __float_as_uint(float(double(Mt) / Wd));
  hi.z = __float_as_uint(float(sqrt(double(Np)) / Wd));
  hi.w = __float_as_uint(float(sqrt(double(Nt)) / Wd));
}

// D4 on the smem map for the digit (pad, tl, q): strictly greater than the 4 neighbours earlier
// in (time,pad) order, >= the 4 later ones.  map32: the map as 32-bit words (two cells).
__device__ __forceinline__ bool is_peak(const uint32_t* __restrict__ map32, uint32_t wpr, uint32_t pad, uint32_t tl,
                                        uint32_t q) {
  const uint32_t c = pad + kColOff;
  const uint32_t sh = (c & 1u) ? 0u : 16u;                      // cells c-1,c,c+1 start at bit sh of (w0,w1)
  const uint32_t* r = map32 + tl * wpr + ((c - 1u) >> 1);
  const uint32_t a0 = r[-int32_t(wpr)], a1 = r[1 - int32_t(wpr)];
  const uint32_t b0 = r[0], b1 = r[1];
  const uint32_t c0 = r[wpr], c1 = r[wpr + 1];
  const uint32_t A = __funnelshift_r(a0, a1, sh), Ar = (a1 >> sh) & 0xFFFFu;   // A = left | centre<<16
  const uint32_t B = __funnelshift_r(b0, b1, sh), Br = (b1 >> sh) & 0xFFFFu;
  const uint32_t C = __funnelshift_r(c0, c1, sh), Cr = (c1 >> sh) & 0xFFFFu;
  const uint32_t early = max(max(A & 0xFFFFu, A >> 16), max(Ar, B & 0xFFFFu));
  const uint32_t late = max(max(C & 0xFFFFu, C >> 16), max(Cr, Br));
  return q > early && q >= late;
}

// Front / back / committer pipeline inside one CTA of 20 warps:
//   front  (warps 0..14)  take tiles by ticket; zero the map, scatter the list (S1), D4 peak flags
//                         (S2), count + scan (S6 in-tile part), then cut each peak's WINDOW out of
//                         the map and flags into one of two window buffers — and go on to the next
//                         tile at once: nothing after this point needs the map
//   back   (warps 15..18) S3..S5 from the windows, four lanes per peak; RawRecs into one of two
//                         staging buffers
//   committer (warp 19)   decoupled look-back of the tile (S6), D8 finish, copy-out
// Hand-over is by named barriers (bar.arrive by the producers, bar.sync by the consumers):
//   kBarWinFull + b / kBarWinEmpty + b   front <-> back      (window buffer b and wmeta[b])
//   kBarFull + b    / kBarEmpty + b      back  <-> committer (staging buffer b and s_meta[b])
// A tile with more peaks than a buffer holds is handed over in several items; a tile without
// peaks still sends one empty item (its look-back has to publish a prefix).
constexpr int kFrontThreads = 480, kBackThreads = 128;
static_assert(kFrontThreads + kBackThreads == kWorkThreads && kFrontThreads >= kTileT + 1, "role split");
constexpr int kBarWork = 1, kBarFull = 2, kBarEmpty = 4, kBarWinFull = 6, kBarWinEmpty = 8;
constexpr uint32_t kStopTile = 0xFFFFFFFFu;
__device__ __forceinline__ void bar_arrive_named(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

__global__ void __launch_bounds__(kThreads, 2) k_tile(const __grid_constant__ TileParams P) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  // carve-up
  uint8_t* sp = smem_raw;                                     // __align__(128); no static shared memory before it
  uint8_t* mapraw = sp;                                     sp += P.map_bytes_max;   // map, then flag bitmap
  uint4* wins = reinterpret_cast<uint4*>(sp);               sp += 2 * kListCap * kWinWords * 4;   // two window buffers
  uint4* stage = reinterpret_cast<uint4*>(sp);              sp += 2 * kListCap * 32; // two RawRec staging buffers
  uint32_t* s_next = reinterpret_cast<uint32_t*>(sp);       sp += 16;            // next tile: index, sector, row, tile of the row
  uint32_t* s_misc = reinterpret_cast<uint32_t*>(sp);       sp += 32 * 4;        // [1..11] warp totals, [20] next peak group
  uint32_t* s_meta = reinterpret_cast<uint32_t*>(sp);       sp += 2 * 4 * 4;     // per staging buffer: tile, total, offset, count
  uint32_t* wmeta = reinterpret_cast<uint32_t*>(sp);        sp += 2 * 8 * 4;     // per window buffer: + sector|row<<8, npads, time of map row 0
  uint32_t* rowoff = reinterpret_cast<uint32_t*>(sp);       sp += (kTileT + 4) * 4;
  uint32_t* nbr_tab = reinterpret_cast<uint32_t*>(sp);      sp += kNbrTabWords * 4;
  uint32_t* wtab = reinterpret_cast<uint32_t*>(sp);         sp += 12 * 4;        // D6: L / S for S = 1..9

  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  const uint32_t bmw = P.bm_words;
  for (uint32_t i = tid; i < uint32_t(kNbrTabWords); i += kThreads) nbr_tab[i] = nbr_tab_entry(i);
  if (tid < 9u) wtab[tid] = kShareL / (tid + 1u);
  __syncthreads();
  const uint32_t sub = lane & 3u;                                      // four lanes per peak: lane frame R_sub
  const int32_t rot_cs = (sub == 0u) ? 1 : (sub == 2u) ? -1 : 0, rot_sn = (sub == 1u) ? 1 : (sub == 3u) ? -1 : 0;

  // s_misc[21 + 2b], [22 + 2b]: next group / groups done of the item in window buffer b; [25 + b]: the item
  // (sequence number) the back warps have opened in buffer b — front warps that find their next buffer
  // still busy help with that item instead of idling (dense tiles hand over many items per tile)
  if (tid < 2u) s_misc[25u + tid] = 0xFFFFFFFFu;
  // S3..S5 for the item in window buffer b: groups of 8 peaks, four lanes per peak, taken from a shared counter
  // (shared == false: only the back warps work on the item, groups dealt statically, no bookkeeping)
  auto assemble_item = [&](uint32_t b, auto shared_c, uint32_t bw) {
    constexpr bool shared = decltype(shared_c)::value;
    const uint32_t* m = wmeta + 8u * b;
    const uint32_t npass = m[3], sector_row = m[4], npads = m[5];
    const int32_t t_row0 = int32_t(m[6]);
    const uint4* wb = wins + b * uint32_t(kListCap * kWinWords / 4);
    uint4* stg = stage + b * (2u * kListCap);
    for (uint32_t g = bw;; g += uint32_t(kBackThreads / 32)) {
      if (shared) {
        if (lane == 0) g = atomicAdd(&s_misc[21u + 2u * b], 1u);
        g = __shfl_sync(0xffffffffu, g, 0);
      }
      if (g * 8u >= npass) break;
      const uint32_t i = g * 8u + (lane >> 2);
      uint4 lo4, hi4;
      assemble4(wb + min(i, npass - 1u) * uint32_t(kWinWords / 4), nbr_tab, wtab, sub, rot_cs, rot_sn, sector_row,
                npads, t_row0, P.tf_time_bins, lo4, hi4);
      if (i < npass && sub < 2u) stg[2u * i + sub] = sub ? hi4 : lo4;
      if (shared) {
        __threadfence_block();
        __syncwarp();
        if (lane == 0) atomicAdd(&s_misc[22u + 2u * b], 1u);
      }
    }
  };
  __syncthreads();

  if (warp == uint32_t(kWorkThreads / 32)) {
    // ================= committer warp: S6 look-back, S5 finish, copy-out =================
    uint32_t excl = 0;
    for (uint32_t q = 0;; ++q) {
      const uint32_t b = q & 1u;
      bar_sync_named(kBarFull + int(b), kBackThreads + 32);
      const uint32_t t = s_meta[4 * b];
      if (t == kStopTile) break;
      const uint32_t total = s_meta[4 * b + 1], off = s_meta[4 * b + 2], cnt = s_meta[4 * b + 3];
      if (off == 0u) {
        excl = lookback_exclusive(P.tile_state, t, P.epoch, total);
        if (lane == 0 && t == P.n_tiles - 1) P.status->n_clusters = (unsigned long long)excl + total;
      }
      const uint64_t g0 = uint64_t(excl) + off;                          // first record of this item
      const uint4* src = stage + b * (2u * kListCap);
      uint4* dst = reinterpret_cast<uint4*>(P.out) + 2 * g0;
      // S5 finish (D8), one record per lane: fp64 from the exact integers
      for (uint32_t r = lane; r < cnt; r += 32u) {
        if (g0 + r < P.out_capacity) {
          uint4 lo = src[2u * r], hi = src[2u * r + 1u];
          finish_rec(lo, hi);
          dst[2u * r] = lo;
          dst[2u * r + 1u] = hi;
        }
      }
      bar_arrive_named(kBarEmpty + int(b), kBackThreads + 32);
    }
    return;
  }

  if (warp >= uint32_t(kFrontThreads / 32)) {
    // ================= back warps: S3..S5 from the windows =================
    const uint32_t btid = tid - uint32_t(kFrontThreads);
    for (uint32_t q = 0;; ++q) {
      const uint32_t b = q & 1u;
      bar_sync_named(kBarWinFull + int(b), kWorkThreads);               // window buffer b and wmeta[b] are written
      if (q >= 2u) bar_sync_named(kBarEmpty + int(b), kBackThreads + 32);   // staging[b] has been copied out
      const uint32_t* m = wmeta + 8u * b;
      const uint32_t t = m[0];
      if (btid == 0) {
        s_meta[4 * b] = t;
        s_meta[4 * b + 1] = m[1];
        s_meta[4 * b + 2] = m[2];
        s_meta[4 * b + 3] = m[3];
      }
      if (t == kStopTile) {
        bar_arrive_named(kBarFull + int(b), kBackThreads + 32);
        break;
      }
      const bool shared = m[7] != 0u;                                   // a dense tile: front warps may help
      if (shared && btid == 0) *reinterpret_cast<volatile uint32_t*>(&s_misc[25u + b]) = q;   // open (staging[b] is ours)
      if (shared) assemble_item(b, std::true_type{}, 0u);
      else assemble_item(b, std::false_type{}, warp - uint32_t(kFrontThreads / 32));
      if (shared) {                                                     // groups taken by helpers may still be in flight
        const uint32_t ng = (m[3] + 7u) >> 3;
        while (*reinterpret_cast<volatile uint32_t*>(&s_misc[22u + 2u * b]) < ng) {}
      }
      bar_arrive_named(kBarWinEmpty + int(b), kWorkThreads);            // the windows are consumed
      bar_arrive_named(kBarFull + int(b), kBackThreads + 32);           // the records are staged
    }
    return;
  }

  // ================= front warps: S1, S2, in-tile S6, window cut-out =================
  // address and (clamped) length of a tile's digit list (tile = bin: kTileT == kBinT)
  auto tile_list = [&](uint32_t t, uint32_t sector, uint32_t row, uint32_t tt, const uint32_t*& src) -> uint32_t {
    const uint32_t cap = P.rows[row].cap;
    src = P.lists + uint64_t(sector) * P.sec_list_elems + P.rows[row].list_off + uint64_t(tt) * cap;
    return min(P.counts[t], cap);
  };
  // take the next tile in ticket order (one thread)
  auto fetch = [&]() {
    const uint32_t t = atomicAdd(&P.status->ticket, 1u);
    const uint32_t sr = t / P.tiles_per_row, sector = sr / P.n_rows;
    s_next[0] = t;
    s_next[1] = sector;
    s_next[2] = sr - sector * P.n_rows;         // row
    s_next[3] = t - sr * P.tiles_per_row;       // tile of the row
  };
  if (tid == 0) fetch();
  bar_sync_named(kBarWork, kFrontThreads);

  uint32_t q = 0;                                                      // hand-over items issued so far
  for (;;) {
    const uint32_t t = s_next[0];
    if (t >= P.n_tiles) break;
    const uint32_t sector = s_next[1], row = s_next[2], tt = s_next[3];
    const RowInfo ri = P.rows[row];
    const int32_t t0 = P.t_core_begin + int32_t(tt) * kTileT;           // global time of core row 0
    const uint32_t ncore = uint32_t(min(kTileT, P.t_core_end - t0));     // S7: only the core emits
    const uint32_t W = ri.W, wpr = W >> 1;
    uint16_t* map = reinterpret_cast<uint16_t*>(mapraw);
    uint32_t* bm = reinterpret_cast<uint32_t*>(mapraw + uint32_t(kBoxH) * W * 2u);   // W % 8 == 0: 16-byte aligned
    const uint32_t* src;
    const uint32_t n = tile_list(t, sector, row, tt, src);                                // k_bin: a multiple of 8; 0 entries are padding
    const uint4* src4 = reinterpret_cast<const uint4*>(src);
    const uint32_t n4 = n >> 2;

    // ---- D2: zero the tile's charge map and flag bitmap ----
    {
      const uint32_t nz = (uint32_t(kBoxH) * W * 2u + uint32_t(kBoxH) * bmw * 4u + 15u) >> 4;
      uint4* z = reinterpret_cast<uint4*>(mapraw);
      for (uint32_t i = tid; i < nz; i += kFrontThreads) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    bar_sync_named(kBarWork, kFrontThreads);
    if (tid == 0) fetch();                    // next tile's ticket (s_next is read again after later barriers)

    // ---- S1: scatter the list into the map (16-byte streaming loads, two in flight per thread) ----
    {
      auto put = [&](uint32_t d) {
        if (d) map[dig_tl(d) * W + dig_pad(d) + kColOff] = uint16_t(dig_q(d));   // 0 = padding
      };
      uint32_t i = tid;
      for (; i + kFrontThreads < n4; i += 2 * kFrontThreads) {
        const uint4 a = __ldg(src4 + i), c = __ldg(src4 + i + kFrontThreads);
        put(a.x); put(a.y); put(a.z); put(a.w);
        put(c.x); put(c.y); put(c.z); put(c.w);
      }
      if (i < n4) {
        const uint4 a = __ldg(src4 + i);
        put(a.x); put(a.y); put(a.z); put(a.w);
      }
      if (tid < (n & 3u)) put(__ldg(src + 4u * n4 + tid));               // k_bin_direct lists: any length
    }
    bar_sync_named(kBarWork, kFrontThreads);

    // ---- S2: D4 peak flags for map rows 1..kBoxH-2, digit-driven (the list is in L1/L2 now) ----
    {
      const uint32_t* map32 = reinterpret_cast<const uint32_t*>(map);
      // branch-free up to the flag store, so that the loads of several entries overlap: an entry that
      // cannot be a peak (below theta, halo row 0 / last, padding) is tested at a harmless cell instead
      auto test2 = [&](uint32_t d0, uint32_t d1) {
        uint32_t q0 = dig_q(d0), tl0 = dig_tl(d0), pad0 = dig_pad(d0);
        uint32_t q1 = dig_q(d1), tl1 = dig_tl(d1), pad1 = dig_pad(d1);
        const bool ok0 = q0 >= P.theta && tl0 - 1u < uint32_t(kBoxH - 2);
        const bool ok1 = q1 >= P.theta && tl1 - 1u < uint32_t(kBoxH - 2);
        if (!ok0) { tl0 = 1u; pad0 = 0u; }
        if (!ok1) { tl1 = 1u; pad1 = 0u; }
        const bool p0 = is_peak(map32, wpr, pad0, tl0, q0);
        const bool p1 = is_peak(map32, wpr, pad1, tl1, q1);
        if (ok0 && p0) atomicOr(&bm[tl0 * bmw + ((pad0 + 4u) >> 5)], 1u << ((pad0 + 4u) & 31u));
        if (ok1 && p1) atomicOr(&bm[tl1 * bmw + ((pad1 + 4u) >> 5)], 1u << ((pad1 + 4u) & 31u));
      };
      for (uint32_t i = tid; i < n4; i += kFrontThreads) {
        const uint4 a = __ldg(src4 + i);
        test2(a.x, a.y);
        test2(a.z, a.w);
      }
      if (tid < (n & 3u)) test2(__ldg(src + 4u * n4 + tid), 0u);
    }
    // pull the next tile's list towards L2 while this tile is counted and built
    {
      const uint32_t tn = s_next[0];
      if (tn < P.n_tiles) {
        const uint32_t* nsrc;
        const uint32_t nn = tile_list(tn, s_next[1], s_next[2], s_next[3], nsrc);
        for (uint32_t i = tid * 32u; i < nn; i += kFrontThreads * 32u)
          asm volatile("prefetch.global.L2 [%0];" ::"l"(nsrc + i));
      }
    }
    bar_sync_named(kBarWork, kFrontThreads);   // flags complete

    // ---- S6 (in-tile part): ordered count of the core rows, block scan ----
    uint32_t cnt = 0;
    if (tid < ncore) {
      const uint32_t* r = bm + (kReach + tid) * bmw;
      for (uint32_t w = 0; w < bmw; ++w) cnt += __popc(r[w]);
    }
    uint32_t incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= uint32_t(o)) incl += v;
    }
    if (lane == 31) s_misc[1 + warp] = incl;
    bar_sync_named(kBarWork, kFrontThreads);
    uint32_t wbase, total;
    {                                           // scan of the 15 warp totals, one per lane
      const uint32_t v = lane < uint32_t(kFrontThreads / 32) ? s_misc[1 + lane] : 0u;
      uint32_t ps = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, ps, o);
        if (lane >= uint32_t(o)) ps += u;
      }
      wbase = __shfl_sync(0xffffffffu, ps - v, warp);
      total = __shfl_sync(0xffffffffu, ps, kFrontThreads / 32 - 1);
    }
    if (tid <= kTileT) rowoff[tid] = (tid < kTileT) ? (wbase + incl - cnt) : total;
    // publish the tile's count early so that later tiles' look-backs never wait for this tile's build
    if (tid == 0 && t != 0u) st_release_u64(P.tile_state + t, pack_state(P.epoch, kStAgg, total));

    // ---- window cut-out, at most kListCap peaks per hand-over item ----
    uint32_t done = 0;
    do {
      const uint32_t b = q & 1u;
      if (q >= 2u) {
        // buffer b still holds item q-2: if it belongs to a dense tile, help the back warps once they have
        // opened it; then wait for its release
        if (wmeta[8u * b + 7u]) {
          while (*reinterpret_cast<volatile uint32_t*>(&s_misc[25u + b]) != q - 2u) __nanosleep(100);
          assemble_item(b, std::true_type{}, 0u);
        }
        bar_sync_named(kBarWinEmpty + int(b), kFrontThreads + kBackThreads);
      }
      const uint32_t npass = min(total - done, uint32_t(kListCap));
      if (tid == 0) {
        s_misc[20] = 0u;
        s_misc[21u + 2u * b] = 0u;
        s_misc[22u + 2u * b] = 0u;
        uint32_t* m = wmeta + 8u * b;
        m[0] = t;
        m[1] = total;
        m[2] = done;
        m[3] = npass;
        m[4] = sector | (row << 8);
        m[5] = ri.npads;
        m[6] = uint32_t(t0 - kReach);                                   // global time of map row 0
        m[7] = total > 3u * uint32_t(kListCap) ? 1u : 0u;               // dense tile: its items are shared with helpers
      }
      bar_sync_named(kBarWork, kFrontThreads);                          // rowoff and the group counter are ready
      // groups of 8 peaks, four lanes per peak, taken dynamically by the front warps
      uint4* wb = wins + b * uint32_t(kListCap * kWinWords / 4);
      for (;;) {
        uint32_t g = 0;
        if (lane == 0) g = atomicAdd(&s_misc[20], 1u);
        g = __shfl_sync(0xffffffffu, g, 0);
        if (g * 8u >= npass) break;
        const uint32_t i = min(g * 8u + (lane >> 2), npass - 1u);      // (a ragged group redoes the item's last peak)
        // locate peak number done + i of the tile (S6 order): its row by bisection of the row offsets
        // (the largest r with rowoff[r] <= k), then the (k - rowoff[r])-th set bit of the row's flags
        uint32_t k = done + i;
        uint32_t lo = 0, hi = uint32_t(kTileT);                         // rowoff[0] = 0 <= k < total = rowoff[kTileT]
#pragma unroll
        for (int it = 0; it < 8; ++it) {
          const uint32_t mid = (lo + hi) >> 1;
          if (rowoff[mid] <= k) lo = mid; else hi = mid;
        }
        static_assert(kTileT == 256, "eight bisection steps");
        k -= rowoff[lo];
        const uint32_t j = uint32_t(kReach) + lo;
        const uint32_t* fr = bm + j * bmw;
        uint32_t word = 0, wbit = 0;
        bool found = false;
        for (uint32_t w = 0; w < bmw; ++w) {
          const uint32_t x = fr[w], c = __popc(x);
          if (!found) {
            if (k < c) { word = x; wbit = w * 32u; found = true; } else k -= c;
          }
        }
        for (; k; --k) word &= word - 1u;                               // drop the k lowest flags
        const uint32_t pad = wbit + uint32_t(__ffs(word)) - 1u - 4u;
        extract_window4(map, bm, W, bmw, j, pad, sub, rot_cs, rot_sn, wb + i * uint32_t(kWinWords / 4));
      }
      bar_arrive_named(kBarWinFull + int(b), kFrontThreads + kBackThreads);
      ++q;
      done += npass;
      if (done < total) bar_sync_named(kBarWork, kFrontThreads);       // the group counter is reused
    } while (done < total);
    bar_sync_named(kBarWork, kFrontThreads);   // map, bitmap and s_next are stable until here
  }
  // stop item: the back warps pass it on to the committer
  {
    const uint32_t b = q & 1u;
    if (q >= 2u) bar_sync_named(kBarWinEmpty + int(b), kFrontThreads + kBackThreads);
    if (tid == 0) wmeta[8u * b] = kStopTile;
    bar_arrive_named(kBarWinFull + int(b), kFrontThreads + kBackThreads);
  }
}

}  // namespace tpcclus
