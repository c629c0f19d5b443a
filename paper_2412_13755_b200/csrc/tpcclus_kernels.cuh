// tpcclus_kernels.cuh — sm_100a kernels of the TPC cluster finder (device side).
//
// Steps of SURVEY.md §8(a) and where they run:
//   S0  map clear            k_clear      (HBM store-only)
//   S1  charge-map fill      k_scatter    (16-byte digit loads, 2-byte scattered stores)
//   S2  peak finding         k_cluster    phase A: TMA tile (+halo) -> smem, packed u16x2 3x3 ordered max
//   S3  peak count S(c)      k_cluster    phase C: 9x9 flag window from the smem flag bitmap
//   S4  5x5 assembly         k_cluster    phase C: one thread per peak, 25 charges from the smem tile
//   S5  centroid / width     k_cluster    phase C: exact integer moments, fp64 finish
//   S6  ordered compaction   k_cluster    phase B: popc prefix inside the tile + decoupled look-back
//                                         across tiles in (sector,row,time) ticket order
//   S7  fragment ownership   k_cluster    tiles cover exactly the core [b,e); halo rows are only read
//
// Definitions D1..D12 are those of SURVEY.md §8(c) (restated in DESIGN.md §2); the D-number
// is cited where each rule is implemented.  No code here is shared with oracle/.
#pragma once
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>

namespace tpcclus {

constexpr int      kThreads      = 256;   // CTA size of k_cluster
constexpr int      kTileT        = 128;   // core time bins per tile
constexpr int      kReach        = 5;     // D9: charges within Chebyshev distance 5 decide a cluster
constexpr int      kBoxH         = kTileT + 2 * kReach;   // tile rows staged in smem
constexpr int      kPadHalo      = 8;     // box starts at pad -8: the innermost TMA coordinate must be a multiple
                                          // of 16 bytes (measured: -2 raises 'illegal instruction'); 2 would do for 5x5
constexpr int      kPadTail      = 2;     // cells kept right of the last pad (5x5 window)
constexpr int      kStages       = 2;     // TMA double buffering
constexpr int      kListCap      = 1024;  // peaks processed per pass inside one tile
constexpr uint32_t kQClamp       = 16368; // D1
constexpr int      kMaxSectors   = 256;

struct RowInfo {              // one per pad row (device table)
  uint32_t map_off;           // element offset of this row's [H][pitch] block inside one sector's map
  uint16_t npads;
  uint16_t pitch;             // elements, multiple of 8 (TMA: global stride multiple of 16 bytes)
  uint16_t boxw;              // TMA box width in elements = roundup8(kPadHalo + npads + kPadTail)
  uint16_t nwords;            // active 2-cell word columns = ceil(npads/2)
};

struct DevStatus {            // device-side run status, copied to pinned host memory after the run
  unsigned long long n_dropped;
  unsigned long long n_clusters;
  unsigned int       ticket;  // tile ticket counter of k_cluster
  unsigned int       pad_;
};

struct ScatterParams {
  uint64_t n;                          // digits
  uint64_t sec_elems;                  // map elements per sector
  int32_t  t_origin;                   // global time of local map row 0 (= b - halo, may be negative)
  int32_t  t_lo, t_hi;                 // loaded range [lo,hi) in global time
  uint32_t n_sectors, n_rows;
  uint64_t off[kMaxSectors + 1];       // sector offsets (copied from the host array)
};

struct ClusterParams {
  const CUtensorMap* tmaps;            // [n_sectors*n_rows], global memory
  const RowInfo*     rows;             // [n_rows]
  unsigned long long* tile_state;      // [n_tiles] decoupled look-back words
  DevStatus*         status;
  void*              out;              // tpcclus_cluster records
  uint64_t           out_capacity;
  uint32_t n_sectors, n_rows;
  uint32_t tiles_per_row;              // ceil((e-b)/kTileT)
  uint32_t n_tiles;
  int32_t  t_core_begin, t_core_end;   // [b,e)
  int32_t  t_origin;                   // global time of local map row 0
  uint32_t tf_time_bins;
  uint32_t theta;                      // peak_min_q16
  uint32_t epoch;                      // run counter, tags tile_state words
  uint32_t tile_bytes_max;             // smem bytes reserved per stage
  uint32_t bm_words;                   // flag-bitmap words per tile row
};

// ----------------------------------------------------------------------------------------
// small PTX wrappers (TMA + mbarrier), sm_90+/sm_100a
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
// 2-D tiled TMA load global -> shared; out-of-range coordinates are zero-filled, which is
// exactly D2's "0 for every out-of-range pad or time".
__device__ __forceinline__ void tma_load_2d(void* smem_dst, const CUtensorMap* tmap, int x, int y,
                                            uint64_t* bar) {
  asm volatile(
      "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%3, %4}], [%2];" ::
          "r"(smem_u32(smem_dst)),
      "l"(reinterpret_cast<uint64_t>(tmap)), "r"(smem_u32(bar)), "r"(x), "r"(y)
      : "memory");
}
// The descriptors live in global memory (written once by the host in tpcclus_create); make them
// visible to the tensormap proxy of this SM before the first TMA that uses them.
__device__ __forceinline__ void tensormap_fence_acquire(const CUtensorMap* tmap) {
  asm volatile("fence.proxy.tensormap::generic.acquire.gpu [%0], 128;" ::"l"(reinterpret_cast<uint64_t>(tmap))
               : "memory");
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
// S0: clear the rows of the charge map that this run can read or write.
// grid = (n_sectors*n_rows, chunks); each (sector,row) block [rows_used][pitch] is contiguous.
// ----------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_clear(uint16_t* __restrict__ map, const RowInfo* __restrict__ rows,
                                               uint32_t n_rows, uint64_t sec_elems, uint32_t rows_used,
                                               DevStatus* __restrict__ status) {
  if (blockIdx.x == 0 && blockIdx.y == 0 && threadIdx.x == 0) {
    status->n_dropped = 0ull;
    status->n_clusters = 0ull;
    status->ticket = 0u;
  }
  const uint32_t sr = blockIdx.x;
  const uint32_t s = sr / n_rows, r = sr - s * n_rows;
  const RowInfo ri = rows[r];
  const uint64_t span16 = (uint64_t(rows_used) * ri.pitch) >> 3;       // 16-byte units (pitch % 8 == 0)
  uint4* base = reinterpret_cast<uint4*>(map + uint64_t(s) * sec_elems + ri.map_off);
  const uint4 z = make_uint4(0u, 0u, 0u, 0u);
  for (uint64_t i = uint64_t(blockIdx.y) * blockDim.x + threadIdx.x; i < span16;
       i += uint64_t(gridDim.y) * blockDim.x)
    base[i] = z;
}

// ----------------------------------------------------------------------------------------
// S1: digit scatter.  One 16-byte load = two digits (BASELINE.json:north_star (2): "16-byte
// vectorised coalesced loads").  D1 quantisation, D2 map fill, invalid digits dropped+counted.
// ----------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t quantise_q16(float charge) {
  // D1: q16 = clamp(rint(charge*16), 0, 16368); rint = round-half-even (cvt.rni); NaN -> 0
  const float x = rintf(charge * 16.0f);
  if (!(x > 0.0f)) return 0u;                    // also catches NaN
  return x >= float(kQClamp) ? kQClamp : uint32_t(x);
}

__device__ __forceinline__ bool scatter_one(uint32_t w0, uint32_t w1, uint64_t idx, uint32_t& sector,
                                            const ScatterParams& P, const RowInfo* srow,
                                            uint16_t* __restrict__ map) {
  while (idx >= P.off[sector + 1]) ++sector;     // digits are grouped per sector; rarely iterates
  const uint32_t row = w0 & 0xFFu, pad = (w0 >> 8) & 0xFFu;
  const int32_t time = int32_t(w0 >> 16);
  const uint32_t q = quantise_q16(__uint_as_float(w1));
  if (q == 0u || row >= P.n_rows || time < P.t_lo || time >= P.t_hi) return false;
  const RowInfo ri = srow[row];
  if (pad >= ri.npads) return false;
  const uint64_t e = uint64_t(sector) * P.sec_elems + ri.map_off + uint64_t(time - P.t_origin) * ri.pitch + pad;
  map[e] = uint16_t(q);
  return true;
}

__global__ void __launch_bounds__(256) k_scatter(const uint2* __restrict__ digits, const __grid_constant__ ScatterParams P,
                                                 const RowInfo* __restrict__ rows, uint16_t* __restrict__ map,
                                                 DevStatus* __restrict__ status) {
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
    dropped += scatter_one(v.x, v.y, idx, sector, P, srow, map) ? 0u : 1u;
    dropped += scatter_one(v.z, v.w, idx + 1, sector, P, srow, map) ? 0u : 1u;
  }
  if (tid == 0) {                                 // leftovers: the peeled head and an odd tail
    uint32_t s0 = 0;
    if (head && n > 0) dropped += scatter_one(digits[0].x, digits[0].y, 0, s0, P, srow, map) ? 0u : 1u;
    const uint64_t tail = head + 2 * npairs;
    if (tail < n) dropped += scatter_one(digits[tail].x, digits[tail].y, tail, s0, P, srow, map) ? 0u : 1u;
  }
  // warp-aggregated count of dropped digits
  dropped = __reduce_add_sync(0xffffffffu, dropped);
  if ((threadIdx.x & 31) == 0 && dropped) atomicAdd(&status->n_dropped, (unsigned long long)dropped);
}

// ----------------------------------------------------------------------------------------
// S2..S7: fused tile kernel.
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
  if (lane == 0) st_release_u64(state + tile, pack_state(epoch, kStAgg, aggregate));
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

__device__ __constant__ uint16_t kShareWeight[10] = {0, 2520, 1260, 840, 630, 504, 420, 360, 315, 280};  // D6: L/S

// One thread builds one cluster (S3..S5).  tile: smem charges [kBoxH][boxw]; bm: smem flag
// bitmap [kBoxH][bmw], bit (pad+4) of row j set iff the cell is a peak (D4).
__device__ __forceinline__ void build_cluster(const uint16_t* __restrict__ tile, const uint32_t* __restrict__ bm,
                                              uint32_t boxw, uint32_t bmw, uint32_t j, uint32_t pad,
                                              uint32_t sector, uint32_t row, uint32_t npads, int32_t tglob,
                                              uint32_t tf_time_bins, ClusterRec& rec) {
  // 5x5 charges around the peak: box column of pad p is p + kPadHalo
  uint32_t q[5][5];
  const uint16_t* c0 = tile + (j - 2) * boxw + (pad + kPadHalo - 2);
#pragma unroll
  for (int dt = 0; dt < 5; ++dt)
#pragma unroll
    for (int dp = 0; dp < 5; ++dp) q[dt][dp] = c0[dt * boxw + dp];

  // 9x9 peak-flag window: F[k] bit i  <->  row j-4+k, pad  p-4+i  (bitmap bit = pad + 4)
  uint32_t F[9];
  uint32_t others = 0;
  {
    const uint32_t sh = pad & 31u, wi = pad >> 5;
#pragma unroll
    for (int k = 0; k < 9; ++k) {
      const uint32_t* rowp = bm + (j - 4 + k) * bmw + wi;
      F[k] = __funnelshift_r(rowp[0], rowp[1], sh) & 0x1FFu;
      others |= (k == 4) ? (F[k] & ~0x10u) : F[k];
    }
  }

  const uint32_t qP = q[2][2];
  uint32_t W = qP * 2520u, Mpp = 0, Mtt = 0, ncells = 1, flags = 0;
  int32_t Mp = 0, Mt = 0;
  if (qP == kQClamp) flags |= 4u;
#pragma unroll
  for (int dt = -2; dt <= 2; ++dt)
#pragma unroll
    for (int dp = -2; dp <= 2; ++dp) {
      if (dp == 0 && dt == 0) continue;
      const uint32_t qc = q[dt + 2][dp + 2];
      bool member = qc != 0u;                                  // D5: a member has charge
      const bool outer = (dp == -2 || dp == 2 || dt == -2 || dt == 2);
      if (outer) {
        // D5: a peak is never a member; an inner-ring cell cannot be a peak (adjacent to P)
        member = member && !((F[dt + 4] >> (dp + 4)) & 1u);
        // D5 outer ring: some inner-ring cell 8-adjacent to c with Q(i) >= Q(c)
        bool desc = false;
#pragma unroll
        for (int it = -1; it <= 1; ++it)
#pragma unroll
          for (int ip = -1; ip <= 1; ++ip) {
            if (ip == 0 && it == 0) continue;
            if (ip - dp > 1 || dp - ip > 1 || it - dt > 1 || dt - it > 1) continue;
            desc = desc || (q[it + 2][ip + 2] >= qc);
          }
        member = member && desc;
      }
      if (member) {
        uint32_t S = 1;
        if (others) {                                          // D6: peaks within distance 2 of c
          S = 0;
#pragma unroll
          for (int jt = -2; jt <= 2; ++jt) S += __popc((F[dt + jt + 4] >> (dp + 2)) & 0x1Fu);
        }
        const uint32_t w = qc * uint32_t(kShareWeight[S]);     // D6 weight in 1/(16*2520) ADC
        W += w;                                                // D7 moments, exact integers
        Mp += int32_t(w) * dp;
        Mt += int32_t(w) * dt;
        Mpp += w * uint32_t(dp * dp);
        Mtt += w * uint32_t(dt * dt);
        ++ncells;
        if (S >= 2) flags |= 8u;
        if (qc == kQClamp) flags |= 4u;
      }
    }
  if (pad < 2u || pad + 2u >= npads) flags |= 1u;              // D8 EDGE_PAD
  if (tglob < 2 || uint32_t(tglob) + 2u >= tf_time_bins) flags |= 2u;   // D8 EDGE_TIME
  // D8: evaluated in double from the exact integers, rounded once to float32
  const double Wd = double(W);
  const long long Np = (long long)Mpp * (long long)W - (long long)Mp * (long long)Mp;
  const long long Nt = (long long)Mtt * (long long)W - (long long)Mt * (long long)Mt;
  rec.w0 = sector | (row << 8) | (pad << 16) | (flags << 24);
  rec.time = uint32_t(tglob);
  rec.w2 = qP | (ncells << 16);
  rec.qtot = float(Wd / 40320.0);
  rec.dpad = float(double(Mp) / Wd);
  rec.dtime = float(double(Mt) / Wd);
  rec.sigma_pad = float(sqrt(double(Np)) / Wd);
  rec.sigma_time = float(sqrt(double(Nt)) / Wd);
}

__global__ void __launch_bounds__(kThreads, 2) k_cluster(const __grid_constant__ ClusterParams P) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  // carve-up
  uint8_t* sp = smem_raw + ((128u - (smem_u32(smem_raw) & 127u)) & 127u);   // TMA destination: 128-byte aligned
  uint16_t* tile_buf[kStages];
#pragma unroll
  for (int s = 0; s < kStages; ++s) { tile_buf[s] = reinterpret_cast<uint16_t*>(sp); sp += P.tile_bytes_max; }
  uint64_t* mbar = reinterpret_cast<uint64_t*>(sp);         sp += 16 * 8;        // kStages used, keeps 128-byte alignment
  uint32_t* s_tile = reinterpret_cast<uint32_t*>(sp);       sp += 16 * 4;        // tile id per stage
  uint32_t* s_misc = reinterpret_cast<uint32_t*>(sp);       sp += 16 * 4;        // [0] exclusive prefix, [1..8] warp totals
  uint32_t* plist = reinterpret_cast<uint32_t*>(sp);        sp += kListCap * 4;
  RowInfo* srow = reinterpret_cast<RowInfo*>(sp);           sp += 256 * sizeof(RowInfo);
  uint32_t* rowoff = reinterpret_cast<uint32_t*>(sp);       sp += (kTileT + 4) * 4;
  uint32_t* bm = reinterpret_cast<uint32_t*>(sp);

  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  for (uint32_t i = tid; i < P.n_rows; i += kThreads) srow[i] = P.rows[i];
  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) mbar_init(&mbar[s], 1);
    fence_mbar_init();
  }
  __syncthreads();

  // issue the TMA load of the next ticketed tile into stage s (thread 0 only)
  auto fetch = [&](int s) {
    const uint32_t t = atomicAdd(&P.status->ticket, 1u);
    s_tile[s] = t;
    if (t < P.n_tiles) {
      const uint32_t sr = t / P.tiles_per_row, tt = t - sr * P.tiles_per_row;
      const uint32_t row = sr % P.n_rows;
      const RowInfo ri = srow[row];
      const int32_t t0 = P.t_core_begin + int32_t(tt) * kTileT;
      tensormap_fence_acquire(P.tmaps + sr);
      mbar_arrive_expect_tx(&mbar[s], uint32_t(kBoxH) * ri.boxw * 2u);
      tma_load_2d(tile_buf[s], P.tmaps + sr, -kPadHalo, (t0 - P.t_origin) - kReach, &mbar[s]);
    }
  };
  if (tid == 0) {
    for (int s = 0; s < kStages; ++s) fetch(s);
  }
  __syncthreads();

  uint32_t phase[kStages];
#pragma unroll
  for (int s = 0; s < kStages; ++s) phase[s] = 0;

  for (int stage = 0;; stage = (stage + 1) % kStages) {
    const uint32_t t = s_tile[stage];
    if (t >= P.n_tiles) break;
    const uint32_t sr = t / P.tiles_per_row, tt = t - sr * P.tiles_per_row;
    const uint32_t sector = sr / P.n_rows, row = sr - sector * P.n_rows;
    const RowInfo ri = srow[row];
    const int32_t t0 = P.t_core_begin + int32_t(tt) * kTileT;           // global time of core row 0
    const uint32_t ncore = uint32_t(min(kTileT, P.t_core_end - t0));     // S7: only the core emits
    const uint32_t bmw = P.bm_words;
    const uint16_t* tile = tile_buf[stage];

    // clear the flag bitmap while the TMA load is in flight
    for (uint32_t i = tid; i < kBoxH * bmw; i += kThreads) bm[i] = 0u;
    __syncthreads();
    mbar_wait(&mbar[stage], phase[stage]);
    phase[stage] ^= 1u;

    // ---------------- phase A (S2): D4 peak flags for tile rows 1 .. ncore+8 ----------------
    // Each thread owns one 2-cell word column and walks a strip of rows, keeping the 3-cell
    // horizontal maxima of the previous / current / next row in registers.
    {
      const uint32_t wpr = ri.boxw >> 1;                 // 32-bit words per tile row
      const uint32_t nw = ri.nwords;                     // active word columns (pads 0 .. npads-1)
      const uint32_t nstrips = kThreads / nw;
      const uint32_t strip = tid / nw, wc = tid - strip * nw;
      const uint32_t R = ncore + 2 * (kReach - 1);       // rows 1..R get flags
      const uint32_t rps = (R + nstrips - 1) / nstrips;
      const uint32_t jb = 1 + strip * rps, je = min(jb + rps, R + 1);
      if (strip < nstrips && jb < je) {
        const uint32_t* t32 = reinterpret_cast<const uint32_t*>(tile) + (wc + kPadHalo / 2);
        const uint32_t theta2 = P.theta | (P.theta << 16);
        auto load3 = [&](uint32_t j, uint32_t& X, uint32_t& L, uint32_t& Rr) {
          const uint32_t* p = t32 + j * wpr;
          const uint32_t xl = p[-1], xr = p[1];          // halo words left and right are zero
          X = p[0];
          L = __byte_perm(xl, X, 0x5432);                // (pad-1, pad) for the low half, ...
          Rr = __byte_perm(X, xr, 0x5432);               // (pad+1, pad+2)
        };
        uint32_t X, L, Rr, Xn, Ln, Rn;
        load3(jb - 1, X, L, Rr);
        uint32_t Hm = __vimax3_u16x2(L, X, Rr);          // 3-cell maxima of row j-1
        load3(jb, X, L, Rr);
        uint32_t H0 = __vimax3_u16x2(L, X, Rr);
        for (uint32_t j = jb; j < je; ++j) {
          load3(j + 1, Xn, Ln, Rn);
          const uint32_t Hp = __vimax3_u16x2(Ln, Xn, Rn);
          // D4: strictly greater than the 4 earlier neighbours (row j-1, and pad-1 in row j),
          // >= the 4 later ones (pad+1 in row j, row j+1), and >= theta.  With integers
          // Q > x  <=>  Q >= x+1.
          const uint32_t be = __vmaxu2(L, Hm) + 0x00010001u;
          const uint32_t bl = __vmaxu2(Rr, Hp);
          const uint32_t bound = __vimax3_u16x2(be, bl, theta2);
          const uint32_t pk = ((X | 0x80008000u) - bound) & 0x80008000u;   // bit15 of a half: Q >= bound
          if (pk) {
            const uint32_t bit0 = 2u * wc + 4u;                            // bitmap bit = pad + 4
            if (pk & 0x00008000u) atomicOr(&bm[j * bmw + (bit0 >> 5)], 1u << (bit0 & 31u));
            if (pk & 0x80000000u) atomicOr(&bm[j * bmw + ((bit0 + 1) >> 5)], 1u << ((bit0 + 1) & 31u));
          }
          Hm = H0; H0 = Hp; X = Xn; L = Ln; Rr = Rn;
        }
      }
    }
    __syncthreads();

    // ---------------- phase B (S6): ordered count, tile prefix, global prefix ----------------
    uint32_t cnt = 0;
    if (tid < ncore) {
      const uint32_t* r = bm + (kReach + tid) * bmw;
      for (uint32_t w = 0; w < bmw; ++w) cnt += __popc(r[w]);
    }
    // block exclusive scan over kTileT (<= kThreads) row counts
    uint32_t incl = cnt;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
      const uint32_t n = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= uint32_t(o)) incl += n;
    }
    if (lane == 31) s_misc[1 + warp] = incl;
    __syncthreads();
    uint32_t wbase = 0, total = 0;
#pragma unroll
    for (int w = 0; w < kThreads / 32; ++w) {
      const uint32_t v = s_misc[1 + w];
      if (uint32_t(w) < warp) wbase += v;
      total += v;
    }
    if (tid <= kTileT) rowoff[tid] = (tid < kTileT) ? (wbase + incl - cnt) : total;
    if (warp == 0) {
      const uint32_t excl = lookback_exclusive(P.tile_state, t, P.epoch, total);
      if (lane == 0) {
        s_misc[0] = excl;
        if (t == P.n_tiles - 1) P.status->n_clusters = (unsigned long long)excl + total;
      }
    }
    __syncthreads();
    const uint64_t gbase = s_misc[0];

    // ---------------- phase C (S3..S5): clusters, kListCap peaks per pass ----------------
    for (uint32_t done = 0; done < total;) {
      // rows [r0, r1) whose peaks fit in the list: rowoff[r1] - done <= kListCap
      // (a row holds at most 124 peaks, so every pass makes progress)
      if (tid < ncore) {
        const uint32_t ro = rowoff[tid], rn = ro + cnt;
        if (ro >= done && rn - done <= kListCap && cnt) {
          uint32_t k = ro - done;
          const uint32_t* r = bm + (kReach + tid) * bmw;
          for (uint32_t w = 0; w < bmw; ++w) {
            uint32_t bits = r[w];
            while (bits) {
              const uint32_t b = __ffs(bits) - 1;
              bits &= bits - 1;
              plist[k++] = ((kReach + tid) << 16) | (w * 32 + b - 4);    // (tile row, pad)
            }
          }
        }
      }
      __syncthreads();
      // number of peaks in this pass = largest rowoff[r] - done that is <= kListCap
      uint32_t npass = min(total - done, uint32_t(kListCap));
      if (total - done > kListCap) {
        // find the last row boundary within the cap (all threads compute the same value)
        uint32_t lo = 0, hi = ncore;               // rowoff is non-decreasing
        while (hi - lo > 1) {
          const uint32_t mid = (lo + hi) >> 1;
          if (rowoff[mid] - done <= kListCap && rowoff[mid] >= done) lo = mid; else hi = mid;
        }
        // rowoff[hi] may still fit
        npass = (rowoff[hi] >= done && rowoff[hi] - done <= kListCap) ? rowoff[hi] - done : rowoff[lo] - done;
      }
      for (uint32_t i = tid; i < npass; i += kThreads) {
        const uint32_t e = plist[i];
        const uint32_t j = e >> 16, pad = e & 0xFFFFu;
        const uint64_t g = gbase + done + i;
        if (g < P.out_capacity) {
          ClusterRec rec;
          build_cluster(tile, bm, ri.boxw, bmw, j, pad, sector, row, ri.npads, t0 + int32_t(j) - kReach,
                        P.tf_time_bins, rec);
          uint4* o = reinterpret_cast<uint4*>(reinterpret_cast<ClusterRec*>(P.out) + g);
          const uint4* s4 = reinterpret_cast<const uint4*>(&rec);
          o[0] = s4[0];
          o[1] = s4[1];
        }
      }
      done += npass;
      __syncthreads();
    }
    __syncthreads();
    // this stage's buffer is free: fetch the next tile into it
    if (tid == 0) fetch(stage);
    __syncthreads();
  }
}

}  // namespace tpcclus
