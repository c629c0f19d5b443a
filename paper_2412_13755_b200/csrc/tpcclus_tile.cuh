// tpcclus_tile.cuh — S1 (second half) .. S7: the fused tile kernel (device side).
//
// One tile = one digit bin of k_bin = one (sector, row, 256 core time bins) window of 266 map rows
// (the core plus the reach of 5 on each side, D9).  A CTA is 16 worker warps + 1 committer warp; two CTAs
// per SM; tiles are taken by an atomic ticket in (sector,row,time) order.  All worker warps go through
// the phases of a tile together (the second CTA of the SM fills the barrier gaps):
//
//   zero      the (pad x time) u16 charge map and the flag bytes, in shared memory            (D2)
//   scatter   the bin's list into the map, 16-byte loads from global memory                   (S1)
//   sweep     DENSE peak test (D3/D4): every lane owns a strip of 8 cells (one LDS.128) and walks down the
//             time rows; the 3x3 ordered maximum is separable — H3 = horizontal max of three per row, kept in
//             registers for three consecutive rows — and is evaluated on packed u16x2 words with the SIMD
//             min/max instructions (VIMNMX.U16x2, VIMNMX3.U16x2) and one half2 compare (HSET2: exact on these
//             bit patterns, every value is below 0x7C00); the eight flag bits of a strip go out as ONE
//             byte store, so the flag map needs neither atomics nor clearing                   (S2)
//   count     one thread per core row (the first eight warps): popc of its flag words, warp scan, and the row's
//             peaks written, in (time,pad) order, into the warp's segment of a peak list; the tile's count is
//             published for the look-back                                                      (S6, S7)
//   build     one thread per peak, dense over the tile's peaks in order: the 25 charges and the 9x9 flag window
//             straight from the map (S3..S5), exact integer moments, D8 finished in fp64 (Newton iterations from
//             fp32 seeds + an exact-residual correction instead of the library division / square root); the
//             finished 32-byte records go to a staging buffer
//   commit    the committer warp: decoupled look-back across tiles, ordered copy-out             (S6)
//
// Definitions D1..D12: SURVEY.md §8(c), restated in DESIGN.md §2.  No code here is shared with oracle/.
#pragma once
#include <cuda_fp16.h>
#ifdef TPCCLUS_PHASE_CLOCKS
#include <cstdio>
#endif

namespace tpcclus {

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
  // the tile's own count (kStAgg) was published by a worker right after the count phase
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
// shared-memory access by 32-bit shared-space address (no generic-address arithmetic in the hot loops)
// ----------------------------------------------------------------------------------------
__device__ __forceinline__ uint4 lds128(uint32_t a) {
  uint4 v;
  asm volatile("ld.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a));
  return v;
}
__device__ __forceinline__ uint32_t lds32(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ uint32_t lds16(uint32_t a) {
  uint32_t v;
  asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(a));
  return v;
}
__device__ __forceinline__ void sts8(uint32_t a, uint32_t v) { asm volatile("st.shared.u8 [%0], %1;" ::"r"(a), "r"(v)); }

// ----------------------------------------------------------------------------------------
// S5 finish (D8) in fp64 from D7's exact integers, rounded once to float32 — the same real-number definitions the
// oracle evaluates with the C library's double division and square root.  Here: a reciprocal of W and a square
// root by ONE Newton step from fp32 seeds (MUFU.RCP / MUFU.RSQ, 22 bits -> 44), each quotient and root closed
// with one exact-residual fma step (44 -> 88 bits before the rounding).  For these operand ranges (W < 2^31,
// |M| < 2^32, N < 2^63) the double results equal the correctly rounded ones (3e8 random cases on the host with
// seeds perturbed by up to 2^-21: 0 differences; every
// GPU parity test compares the records' bytes), at about a tenth of the instructions of the library routines
// with their special-case paths.  D12 itself only asks for 1e-6 relative / 1e-4 absolute.
// ----------------------------------------------------------------------------------------
__device__ __forceinline__ double recip_newton(double b) {               // 1 / b, b >= 1
  const double y = double(__fdividef(1.0f, float(b)));                   // 22 bits
  return fma(y, fma(-b, y, 1.0), y);                                     // 44 bits; div_corr's residual step does the rest
}
__device__ __forceinline__ double div_corr(double a, double b, double y) {   // a / b, y = 1 / b to 44 bits or better
  const double q = a * y;
  return fma(fma(-q, b, a), y, q);
}
__device__ __forceinline__ double sqrt_newton(double n) {                // sqrt(n), n >= 1
  const double y = double(rsqrtf(float(n)));
  double g = n * y, h = 0.5 * y;
  const double r = fma(-g, h, 0.5);                                      // one coupled step: 22 -> 44 bits
  g = fma(g, r, g);
  h = fma(h, r, h);
  return fma(fma(-g, g, n), h, g);                                       // exact residual: 44 -> 44 bits or better
}

// ----------------------------------------------------------------------------------------
// S3..S5, one thread per peak; returns the finished record (two 16-byte halves of a ClusterRec).
//
// The 25 cells of the 5x5 window are numbered k = 5 (dt+2) + (dp+2).  D6's S(c) comes from the OTHER peaks of
// the 9x9 flag window around P: each adds a table entry — one nibble per window cell it is within Chebyshev
// distance 2 of (25 nibbles = 4 words) — so S(c) - 1 is the cell's nibble of the sum.  Column and row sums of
// the weights give D7's moments with constant coefficients.
// ----------------------------------------------------------------------------------------
constexpr int kNbrTabWords = 81 * 4;
constexpr uint32_t kShareL = 2520u;                      // D6: lcm(1..9)

// word `idx & 3` of the entry for another peak at window row v+4 (time offset v), column u+4 (pad offset u)
__device__ __forceinline__ uint32_t nbr_tab_entry(uint32_t idx) {
  const int r = int(idx >> 2), word = int(idx & 3u);
  const int u = r % 9 - 4, v = r / 9 - 4;
  uint32_t e = 0;
  for (int n = 0; n < 8; ++n) {
    const int k = word * 8 + n;
    if (k >= 25) break;
    const int dt = k / 5 - 2, dp = k % 5 - 2;
    if (dp - u >= -2 && dp - u <= 2 && dt - v >= -2 && dt - v <= 2) e |= 1u << (4 * n);
  }
  return e;
}

// Flag bytes of a tile: row j of the map has a 4-byte zero prefix followed by one byte per strip of 8 map
// columns (bit b of byte s <-> column 8 s + b), padded with zero bytes to a multiple of 4.  Read as 32-bit
// words, the flag of pad p sits at bit index 32 + kColOff + p of the row; the zero prefix makes the 9-bit
// window that starts four pads to the left of a peak addressable without a branch for p < 4.
__host__ __device__ inline uint32_t flag_pitch_bytes(uint32_t W) { return 4u + (((W >> 3) + 3u) & ~3u); }

// Build the cluster of the peak at map row j, pad `pad` (one thread) from the tile's map (pitch W cells), its
// flag words (nfw per row), the neighbour table and the L/S table, all in shared memory.
__device__ __forceinline__ void build1(const uint16_t* __restrict__ map, const uint32_t* __restrict__ fw, uint32_t W, uint32_t nfw,
                                       uint32_t j, uint32_t pad, const uint4* __restrict__ tab, const uint32_t* __restrict__ wtab,
                                       uint32_t sector_row, uint32_t npads, int32_t t_row0, uint32_t tf_time_bins, uint4& lo,
                                       uint4& hi) {
  // ---- the 25 charges ----
  uint32_t q[25];
  {
    const uint16_t* c = map + j * W + (pad + uint32_t(kColOff));
#pragma unroll
    for (int dt = -2; dt <= 2; ++dt) {
      const uint16_t* rb = c + dt * int32_t(W);
#pragma unroll
      for (int dp = -2; dp <= 2; ++dp) q[(dt + 2) * 5 + dp + 2] = rb[dp];
    }
  }
  // ---- the 9x9 flag window: R[k] = flags of row j-4+k, bit i <-> pad p-4+i ----
  uint32_t R[9];
  {
    const uint32_t b0 = pad + (32u + uint32_t(kColOff) - 4u);           // bit index of pad p-4 inside a flag row
    const uint32_t sh = b0 & 31u;
    const uint32_t* a0 = fw + (j - 4u) * nfw + (b0 >> 5);
#pragma unroll
    for (int k = 0; k < 9; ++k) R[k] = __funnelshift_r(a0[uint32_t(k) * nfw], a0[uint32_t(k) * nfw + 1u], sh) & 0x1FFu;
    R[4] &= ~(1u << 4);                                                  // P itself
  }
  // ---- D6: other peaks of the window -> S(c) - 1 per cell (nibbles) ----
  uint32_t acc0 = 0, acc1 = 0, acc2 = 0, acc3 = 0;
  {
    uint32_t G0 = R[0] | (R[1] << 9) | (R[2] << 18), G1 = R[3] | (R[4] << 9) | (R[5] << 18), G2 = R[6] | (R[7] << 9) | (R[8] << 18);
    auto add = [&](uint32_t b) {
      const uint4 e = tab[b];
      acc0 += e.x; acc1 += e.y; acc2 += e.z; acc3 += e.w;
    };
    while (G0) { const uint32_t b = __ffs(G0) - 1; G0 &= G0 - 1; add(b); }
    while (G1) { const uint32_t b = __ffs(G1) - 1; G1 &= G1 - 1; add(27u + b); }
    while (G2) { const uint32_t b = __ffs(G2) - 1; G2 &= G2 - 1; add(54u + b); }
  }
  const uint32_t qP = q[12];
  uint32_t col[5] = {0u, 0u, 0u, 0u, 0u}, rowsum[5] = {0u, 0u, 0u, 0u, 0u};
  uint32_t ncells = 1u, nsplit = 0u;
#pragma unroll
  for (int k = 0; k < 25; ++k) {
    if (k == 12) continue;
    const int dt = k / 5 - 2, dp = k % 5 - 2;
    const uint32_t qc = q[k];
    // D5: has charge, is not a peak; outer ring: some 8-adjacent inner-ring cell has Q >= Q(c)
    bool m = qc != 0u && !((R[dt + 4] >> (dp + 4)) & 1u);
    if (dt == -2 || dt == 2 || dp == -2 || dp == 2) {
      uint32_t best = 0u;
#pragma unroll
      for (int it = -1; it <= 1; ++it)
#pragma unroll
        for (int ip = -1; ip <= 1; ++ip) {
          if (ip == 0 && it == 0) continue;
          if (ip - dp > 1 || dp - ip > 1 || it - dt > 1 || dt - it > 1) continue;
          best = max(best, q[(it + 2) * 5 + ip + 2]);
        }
      m = m && best >= qc;
    }
    // D6: w = Q * L / S
    const uint32_t accw = (k < 8) ? acc0 : (k < 16) ? acc1 : (k < 24) ? acc2 : acc3;
    const uint32_t nib = (accw >> (4 * (k & 7))) & 15u;                  // S - 1
    const uint32_t w = m ? qc * wtab[nib] : 0u;
    col[dp + 2] += w;
    rowsum[dt + 2] += w;
    if (m) {
      ncells += 1u;
      nsplit += nib;
    }
  }
  // D7 moments from the column / row sums
  const uint32_t Wsum = col[0] + col[1] + col[2] + col[3] + col[4] + qP * kShareL;   // D6: w(P) = L Q(P)
  const int32_t Mp = int32_t(2u * col[4] + col[3]) - int32_t(col[1] + 2u * col[0]);
  const int32_t Mt = int32_t(2u * rowsum[4] + rowsum[3]) - int32_t(rowsum[1] + 2u * rowsum[0]);
  const uint32_t Mpp = 4u * (col[0] + col[4]) + col[1] + col[3];
  const uint32_t Mtt = 4u * (rowsum[0] + rowsum[4]) + rowsum[1] + rowsum[3];
  const int32_t tglob = t_row0 + int32_t(j);                            // t_row0 = global time of map row 0
  uint32_t flags = 0;
  if (pad < 2u || pad + 2u >= npads) flags |= 1u;                       // D8 EDGE_PAD
  if (tglob < 2 || uint32_t(tglob) + 2u >= tf_time_bins) flags |= 2u;   // D8 EDGE_TIME
  if (qP == kQClamp) flags |= 4u;       // SATURATED: no member exceeds its peak (D4, D5), so a saturated member implies a saturated peak
  if (nsplit) flags |= 8u;                                              // SPLIT
  // D8
  const double Wd = double(Wsum);
  const double yW = recip_newton(Wd);
  const long long Np = (long long)Mpp * (long long)Wsum - (long long)Mp * (long long)Mp;
  const long long Nt = (long long)Mtt * (long long)Wsum - (long long)Mt * (long long)Mt;
  const float qtot = float(div_corr(Wd, 40320.0, 1.0 / 40320.0));
  const float dpad = float(div_corr(double(Mp), Wd, yW));
  const float dtime = float(div_corr(double(Mt), Wd, yW));
  const float spad = Np ? float(div_corr(sqrt_newton(double(Np)), Wd, yW)) : 0.0f;
  const float stime = Nt ? float(div_corr(sqrt_newton(double(Nt)), Wd, yW)) : 0.0f;
  lo = make_uint4(sector_row | (pad << 16) | (flags << 24), uint32_t(tglob), qP | (ncells << 16), __float_as_uint(qtot));
  hi = make_uint4(__float_as_uint(dpad), __float_as_uint(dtime), __float_as_uint(spad), __float_as_uint(stime));
}

// ----------------------------------------------------------------------------------------
// S2: the dense D4 sweep, packed u16x2.
//
// A word holds the cells (c, c+1) of one time row; "shifted" words S_i = (c-1, c) come from a byte
// permute of neighbouring words, so that for word i the left cells are S_i and the right cells S_{i+1}.
//   H3_i(j)  = max(S_i, w_i, S_{i+1})                       the three cells of row j around each cell
//   early    = max(H3_i(j-1), S_i(j))                       the 4 neighbours earlier in (time,pad) order
//   late     = max(H3_i(j+1), S_{i+1}(j))                   the 4 later ones
//   Peak     <=> Q >= theta and Q > early and Q >= late     (D4)
//            <=> Q >= max(early + 1, late, theta)
// The compare is a half2 compare on the raw bit patterns: all operands are <= 16369 < 0x7C00, i.e.
// non-negative finite fp16 values (denormals included) whose order is the integer order.
// The words left and right of a strip come from the neighbour lanes' registers: consecutive lanes hold
// consecutive strips (tasks), lanes 0 and 31 of a warp repeat the task before / after the warp's 30 and store
// nothing.  At a row's ends the neighbour word is zero by construction: the map's first two and last two
// columns are never written, and the neighbour lane holds the last (first) word of some row there.
// ----------------------------------------------------------------------------------------
__device__ __forceinline__ uint32_t shifted_pair(uint32_t w_left, uint32_t w) { return __byte_perm(w_left, w, 0x5432); }
__device__ __forceinline__ uint32_t ge_mask2(uint32_t a, uint32_t b) {   // 0xFFFF per half where a >= b
  return __hge2_mask(*reinterpret_cast<const __half2*>(&a), *reinterpret_cast<const __half2*>(&b));
}
__device__ __forceinline__ uint32_t bitsel(uint32_t k, uint32_t a, uint32_t b) { return (a & k) | (b & ~k); }

struct SweepRow {          // what the sweep keeps of one time row, per strip of 8 cells
  uint32_t C[4];           // the cells
  uint32_t Sr[4];          // S_{i+1}: the right neighbours
  uint32_t H3[4];          // horizontal max of three
  uint32_t E1[4];          // max(H3 of the row above, S_i) + 1: the early side, ready for the compare
};

// Load the strip at shared address a (row j), derive S / H3 (/ E1) into `cur`, and (kTest) return the flag byte
// of row j-1 (`prev`).
template <bool kE1, bool kTest>
__device__ __forceinline__ uint32_t sweep_step(uint32_t a, uint32_t theta2, const SweepRow& prev, SweepRow& cur) {
  const uint4 c = lds128(a);
  const uint32_t wl = __shfl_up_sync(0xffffffffu, c.w, 1), wr = __shfl_down_sync(0xffffffffu, c.x, 1);
  const uint32_t S0 = shifted_pair(wl, c.x), S1 = shifted_pair(c.x, c.y), S2 = shifted_pair(c.y, c.z),
                 S3 = shifted_pair(c.z, c.w), S4 = shifted_pair(c.w, wr);
  cur.C[0] = c.x; cur.C[1] = c.y; cur.C[2] = c.z; cur.C[3] = c.w;
  cur.Sr[0] = S1; cur.Sr[1] = S2; cur.Sr[2] = S3; cur.Sr[3] = S4;
  cur.H3[0] = __vimax3_u16x2(S0, c.x, S1);
  cur.H3[1] = __vimax3_u16x2(S1, c.y, S2);
  cur.H3[2] = __vimax3_u16x2(S2, c.z, S3);
  cur.H3[3] = __vimax3_u16x2(S3, c.w, S4);
  if (kE1) {
    cur.E1[0] = __vmaxu2(prev.H3[0], S0) + 0x00010001u;
    cur.E1[1] = __vmaxu2(prev.H3[1], S1) + 0x00010001u;
    cur.E1[2] = __vmaxu2(prev.H3[2], S2) + 0x00010001u;
    cur.E1[3] = __vmaxu2(prev.H3[3], S3) + 0x00010001u;
  }
  if constexpr (!kTest) {
    return 0u;
  } else {
  // row j-1: the late side needs H3 of this row
  uint32_t M[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const uint32_t X = __vimax3_u16x2(__vmaxu2(cur.H3[i], prev.Sr[i]), prev.E1[i], theta2);
    M[i] = ge_mask2(prev.C[i], X);
  }
  // gather the eight flags into one byte, bit b <-> column 8 s + b: word i's low half at bit 2i, high half at 2i+1
  const uint32_t x = bitsel(0x00020001u, M[0], M[1]);
  const uint32_t y = bitsel(0x00200010u, M[2], M[3]);
  const uint32_t sel = bitsel(0x000A0005u, x, y);
  return bitsel(0x55u, sel, sel >> 16);                                 // low byte is the flag byte
  }
}

// ----------------------------------------------------------------------------------------
// the kernel
// ----------------------------------------------------------------------------------------
constexpr int kBarWork = 1, kBarFull = 2, kBarEmpty = 4;
constexpr uint32_t kStopTile = 0xFFFFFFFFu;
constexpr int kWorkWarps = kWorkThreads / 32;
constexpr int kMapGuard = 16;                 // zero bytes in front of and behind the map (the sweep's edge loads)
static_assert(kWorkWarps * 16 == kTileT, "lanes 0..15 of every worker warp own one core row of a tile each");
static_assert(kListCap <= kWorkThreads, "one thread per peak of an item");
__device__ __forceinline__ void bar_arrive_named(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

#ifdef TPCCLUS_PHASE_CLOCKS   // debugging aid: per-phase cycle totals of a few CTAs (printf at kernel end)
#define PH_DECL long long ph_t = clock64(); long long ph_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
#define PH_MARK(i) { const long long ph_n = clock64(); ph_acc[i] += ph_n - ph_t; ph_t = ph_n; }
#define PH_DUMP(ntiles) if (threadIdx.x == 0 && (blockIdx.x % 97) == 0) printf("cta %d tiles %u cycles: zero %lld scatter %lld sweep %lld count %lld build %lld endbar %lld top %lld waitempty %lld\n", int(blockIdx.x), ntiles, ph_acc[0], ph_acc[1], ph_acc[2], ph_acc[3], ph_acc[7], ph_acc[5], ph_acc[6], ph_acc[4]);
#else
#define PH_DECL
#define PH_MARK(i)
#define PH_DUMP(n)
#endif

__global__ void __launch_bounds__(kThreads, kTileCtasPerSm) k_tile(const __grid_constant__ TileParams P) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  // carve-up
  uint8_t* sp = smem_raw;                                   // __align__(128); no static shared memory before it
  uint8_t* mapraw = sp;                                     sp += P.map_bytes_max;   // guard, map, guard, flag bytes
  uint4* stage = reinterpret_cast<uint4*>(sp);              sp += 2 * kListCap * 32; // two staging buffers of finished records
  uint32_t* nbr_tab = reinterpret_cast<uint32_t*>(sp);      sp += kNbrTabWords * 4;  // 16-byte aligned entries
  uint32_t* rowx = reinterpret_cast<uint32_t*>(sp);         sp += kTileT * 4;        // per core row: peaks of its warp's earlier rows
  uint32_t* wpre = reinterpret_cast<uint32_t*>(sp);         sp += kWorkWarps * kWorkWarps * 4;   // per warp: a copy of the warps' exclusive peak prefix
  uint32_t* s_next = reinterpret_cast<uint32_t*>(sp);       sp += 32;            // next tile: index, sector | row << 8, tile of the row, list length, list address
  uint32_t* wtot = reinterpret_cast<uint32_t*>(sp);         sp += 32 * 4;        // peaks per worker warp
  uint32_t* s_meta = reinterpret_cast<uint32_t*>(sp);       sp += 2 * 4 * 4;     // per staging buffer: tile, total, offset, count
  uint32_t* wtab = reinterpret_cast<uint32_t*>(sp);         sp += 16 * 4;        // D6: L / S for S = 1..9
  uint4* s_rows = reinterpret_cast<uint4*>(sp);                                  // the RowInfo table, 2 x 16 bytes per row

  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  for (uint32_t i = tid; i < uint32_t(kNbrTabWords); i += kThreads) nbr_tab[i] = nbr_tab_entry(i);
  if (tid < 16u) wtab[tid] = tid < 9u ? kShareL / (tid + 1u) : 0u;
  for (uint32_t i = tid; i < 2u * P.n_rows; i += kThreads) s_rows[i] = __ldg(reinterpret_cast<const uint4*>(P.rows) + i);
  for (uint32_t i = tid; i < uint32_t(kMapGuard) / 4u; i += kThreads) reinterpret_cast<uint32_t*>(mapraw)[i] = 0u;
  __syncthreads();

  if (warp == uint32_t(kWorkWarps)) {
    // ================= committer warp: S6 look-back and copy-out =================
    uint32_t excl = 0;
    for (uint32_t q = 0;; ++q) {
      const uint32_t b = q & 1u;
      bar_sync_named(kBarFull + int(b), kThreads);
      const uint32_t t = s_meta[4 * b];
      if (t == kStopTile) break;
      const uint32_t total = s_meta[4 * b + 1], off = s_meta[4 * b + 2], cnt = s_meta[4 * b + 3];
      if (off == 0u) {
        excl = lookback_exclusive(P.tile_state, t, P.epoch, total);
        if (lane == 0 && t == P.n_tiles - 1) P.status->n_clusters = (unsigned long long)excl + total;
      }
      TPC_ASSERT(cnt <= uint32_t(kListCap) && off + cnt <= total);
      const uint64_t g0 = uint64_t(excl) + off;                          // first record of this item
      const uint4* src = stage + b * (2u * kListCap);
      uint4* dst = reinterpret_cast<uint4*>(P.out) + 2 * g0;
      // ordered copy-out: consecutive lanes write consecutive 16-byte halves
      const uint64_t room = P.out_capacity > g0 ? P.out_capacity - g0 : 0ull;
      const uint32_t nh = 2u * uint32_t(min(uint64_t(cnt), room));
      for (uint32_t h = lane; h < nh; h += 32u) dst[h] = src[h];
      bar_arrive_named(kBarEmpty + int(b), kThreads);
    }
    return;
  }

  // ================= worker warps =================
  const uint32_t theta2 = P.theta2;
  const uint32_t map_s = smem_u32(mapraw) + uint32_t(kMapGuard);        // shared-space address of the map
  uint16_t* map = reinterpret_cast<uint16_t*>(mapraw + kMapGuard);
  // Tiles are taken by an atomic ticket in (sector,row,time) order, by thread 0, two tiles ahead: the ticket of
  // tile t+2 and the list length of tile t+1 are requested at the start of tile t and only looked at phases later,
  // so that neither round trip is ever waited for.  post() leaves what the CTA needs to start a tile in s_next.
  auto post = [&](uint32_t t, uint32_t count) {
    s_next[0] = t;
    if (t >= P.n_tiles) return;
    const uint32_t sr = t / P.tiles_per_row, sector = sr / P.n_rows, row = sr - sector * P.n_rows, tt = t - sr * P.tiles_per_row;
    const uint4 r0 = s_rows[2u * row];                                   // list_off, cap, ...
    const uint32_t cap = r0.y;
    const uint64_t src = reinterpret_cast<uint64_t>(P.lists + uint64_t(sector) * P.sec_list_elems + r0.x + uint64_t(tt) * cap);
    s_next[1] = sector | (row << 8);
    s_next[2] = tt;
    s_next[3] = min(count, cap);                                          // k_bin: a multiple of 8; 0 entries are padding
    if (count > cap) atomicAdd(&P.status->n_overfull_bins, 1u);           // -> TPCCLUS_ERR_OCCUPANCY
    s_next[4] = uint32_t(src);
    s_next[5] = uint32_t(src >> 32);
  };
  uint32_t tk1 = 0, tk2 = 0, cnt1 = 0;                                   // thread 0: tickets of the next two tiles, next list length
  if (tid == 0) {
    const uint32_t tk0 = atomicAdd(&P.status->ticket, 1u);
    tk1 = atomicAdd(&P.status->ticket, 1u);
    post(tk0, tk0 < P.n_tiles ? __ldg(P.counts + tk0) : 0u);
  }
  bar_sync_named(kBarWork, kWorkThreads);

  uint32_t q = 0;                                                      // hand-over items issued so far
  PH_DECL
  uint32_t ph_tiles = 0;
  for (;;) {
    const uint32_t t = s_next[0];
    if (t >= P.n_tiles) break;
    ++ph_tiles;
    const uint32_t sector_row = s_next[1], tt = s_next[2], n = s_next[3];
    const uint32_t* src = reinterpret_cast<const uint32_t*>(uint64_t(s_next[4]) | (uint64_t(s_next[5]) << 32));
    RowInfo ri;
    {
      static_assert(sizeof(RowInfo) == 32, "two 16-byte words");
      reinterpret_cast<uint4*>(&ri)[0] = s_rows[2u * (sector_row >> 8)];
      reinterpret_cast<uint4*>(&ri)[1] = s_rows[2u * (sector_row >> 8) + 1u];
    }
    const int32_t t0 = P.t_core_begin + int32_t(tt) * kTileT;           // global time of core row 0
    const uint32_t ncore = uint32_t(min(kTileT, P.t_core_end - t0));     // S7: only the core emits
    const uint32_t W = ri.W, pitch = 2u * W, fpb = ri.fpb, nfw = fpb >> 2;
    const uint32_t flag_off = uint32_t(kBoxH) * pitch + uint32_t(kMapGuard);   // flag bytes follow the map and its guard
    const uint32_t flag_s = map_s + flag_off;
    const uint32_t* fw = reinterpret_cast<const uint32_t*>(mapraw + kMapGuard + flag_off);
    const uint4* src4 = reinterpret_cast<const uint4*>(src);
    const uint32_t n4 = n >> 2;
    TPC_ASSERT(n <= ri.cap && (reinterpret_cast<uintptr_t>(src) & 15u) == 0u && tt < P.tiles_per_row &&
               flag_off + uint32_t(kBoxH) * fpb + uint32_t(kMapGuard) <= P.map_bytes_max);

    // the first two 16-byte loads of this thread's share of the list are issued before the map is zeroed, so that
    // their latency overlaps the zeroing and the barrier behind it
    uint4 pre_a = make_uint4(0u, 0u, 0u, 0u), pre_c = pre_a;
    uint32_t pre_tail = 0u;
    if (tid < n4) pre_a = __ldg(src4 + tid);
    if (tid + kWorkThreads < n4) pre_c = __ldg(src4 + tid + kWorkThreads);
    // A SPARSE tile (few enough entries that every thread holds its share of the list in registers: n <= 8 per
    // thread, and fewer than the row's sparse_max) is tested digit by digit instead of sweeping the map: the peak
    // test then costs per DIGIT, not per cell (the low-occupancy, pp-like path that skips the
    // dense scan; also the upper, emptier pad rows of the Pb-Pb configs).
    const bool sparse = n <= ri.sparse_max;
    // ---- D2: zero the tile's charge map, the guard behind it and the flag bytes ----
    {
      const uint32_t nz = (flag_off + uint32_t(kBoxH) * fpb + 15u) >> 4;
      uint4* z = reinterpret_cast<uint4*>(mapraw + kMapGuard);
      for (uint32_t i = tid; i < nz; i += kWorkThreads) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    PH_MARK(6)
    bar_sync_named(kBarWork, kWorkThreads);
    PH_MARK(0)
    if (tid == 0) {                           // requests for the tiles ahead (see above); nothing is waited for here
      cnt1 = tk1 < P.n_tiles ? __ldg(P.counts + tk1) : 0u;
      tk2 = atomicAdd(&P.status->ticket, 1u);
    }

    // ---- S1: scatter the list into the map (16-byte loads, two in flight per thread) ----
    {
      auto put = [&](uint32_t d) {
        const uint32_t tl = dig_tl(d);
        TPC_ASSERT(d == 0u || (tl < uint32_t(kBoxH) && dig_pad(d) < ri.npads && dig_q(d) >= 1u && dig_q(d) <= kQClamp));
        if (d && tl < uint32_t(kBoxH)) map[tl * W + dig_pad(d) + kColOff] = uint16_t(dig_q(d));   // 0 = padding
      };
      // (zero entries are skipped; short lists leave whole warps and every thread's second load empty)
      const bool has_a = (tid & ~31u) < n4, has_c = n4 > uint32_t(kWorkThreads) + (tid & ~31u);   // warp-uniform
      if (has_a) { put(pre_a.x); put(pre_a.y); put(pre_a.z); put(pre_a.w); }
      if (has_c) { put(pre_c.x); put(pre_c.y); put(pre_c.z); put(pre_c.w); }
      uint32_t i = tid + 2 * kWorkThreads;
      for (; i + kWorkThreads < n4; i += 2 * kWorkThreads) {
        const uint4 a = __ldg(src4 + i), c = __ldg(src4 + i + kWorkThreads);
        put(a.x); put(a.y); put(a.z); put(a.w);
        put(c.x); put(c.y); put(c.z); put(c.w);
      }
      if (i < n4) {
        const uint4 a = __ldg(src4 + i);
        put(a.x); put(a.y); put(a.z); put(a.w);
      }
      pre_tail = tid < (n & 3u) ? __ldg(src + 4u * n4 + tid) : 0u;       // k_bin_direct lists: any length
      if (n & 3u) put(pre_tail);
    }
    bar_sync_named(kBarWork, kWorkThreads);
    PH_MARK(1)
    if (tid == 0) {                           // (every thread has read this tile's s_next before the first barrier)
      post(tk1, cnt1);
      tk1 = tk2;
    }

    // ---- S2: dense D4 sweep -> flag bytes of map rows 1 .. kBoxH-2 ----
    // tasks = (strip s, row segment g): consecutive lanes take consecutive strips of one segment.  Segment g loads
    // rows jb .. jb + L + 1 and flags rows jb + 1 .. jb + L, jb = min(g L, kBoxH - 2 - L) (the last segment is moved
    // up so that nothing is read past the map; the rows it shares with its neighbour get the same bytes twice).
    if (!sparse) {
    for (uint32_t task0 = warp * 30u; task0 < ri.ntasks; task0 += uint32_t(kWorkWarps) * 30u) {   // (one pass for the usual rows)
      const uint32_t L = ri.segL, ns = ri.ns;
      const int32_t tsk = int32_t(task0 + lane) - 1;
      const bool owner = lane - 1u < 30u && uint32_t(tsk) < ri.ntasks;   // lanes 1..30 with a task of their own
      const uint32_t task = tsk < 0 ? ri.ntasks - 1u : (uint32_t(tsk) < ri.ntasks ? uint32_t(tsk) : 0u);
      const uint32_t g = (task * ri.rcp_ns) >> 16, s = task - g * ns;
      const uint32_t jb = min(g * L, uint32_t(kBoxH) - 2u - L);
      const uint32_t nout = owner ? L : 0u;
      uint32_t a = map_s + jb * pitch + 16u * s;
      uint32_t f = flag_s + (jb + 1u) * fpb + 4u + s;
      TPC_ASSERT(s < ns && 16u * s + 16u <= pitch && jb + L + 2u <= uint32_t(kBoxH) && 4u + s < fpb);
      SweepRow ra, rb;
      sweep_step<false, false>(a, theta2, ra, ra);
      a += pitch;
      sweep_step<true, false>(a, theta2, ra, rb);
      a += pitch;
      for (uint32_t m = 0; m < L; m += 2u) {
        const uint32_t b0 = sweep_step<true, true>(a, theta2, rb, ra);
        a += pitch;
        if (m < nout) sts8(f, b0);
        f += fpb;
        if (m + 1u >= L) break;
        const uint32_t b1 = sweep_step<true, true>(a, theta2, ra, rb);
        a += pitch;
        if (m + 1u < nout) sts8(f, b1);
        f += fpb;
      }
    }
    } else {
      // digit-driven D4: an entry is a peak iff Q >= theta, Q > the four neighbours earlier in (time,pad) order and
      // Q >= the four later ones (D3).  Rows 0 and kBoxH - 1 of the window never carry flags (as in the sweep).
      auto test = [&](uint32_t d) {
        const uint32_t tl = dig_tl(d), qv = dig_q(d);
        if (d == 0u || qv < P.theta || tl - 1u >= uint32_t(kBoxH) - 2u) return;
        const uint32_t col = dig_pad(d) + uint32_t(kColOff);
        const uint32_t a = map_s + 2u * (tl * W + col);
        const uint32_t up = a - pitch, dn = a + pitch;
        const uint32_t early = max(max(lds16(up - 2u), lds16(up)), max(lds16(up + 2u), lds16(a - 2u)));
        const uint32_t late = max(max(lds16(dn - 2u), lds16(dn)), max(lds16(dn + 2u), lds16(a + 2u)));
        if (qv > early && qv >= late)
          atomicOr(reinterpret_cast<uint32_t*>(mapraw + kMapGuard + flag_off) + tl * nfw + 1u + (col >> 5), 1u << (col & 31u));
      };
      if ((tid & ~31u) < n4) { test(pre_a.x); test(pre_a.y); test(pre_a.z); test(pre_a.w); }
      if (n4 > uint32_t(kWorkThreads) + (tid & ~31u)) { test(pre_c.x); test(pre_c.y); test(pre_c.z); test(pre_c.w); }
      if (n & 3u) test(pre_tail);
    }
    bar_sync_named(kBarWork, kWorkThreads);   // flags complete
    PH_MARK(2)
    // pull the next tile's list towards L2 while this tile is counted and built (thread 0 posted it after the
    // scatter barrier of this tile)
    if (s_next[0] < P.n_tiles) {
      const uint32_t nn = s_next[3];
      const uint32_t* nsrc = reinterpret_cast<const uint32_t*>(uint64_t(s_next[4]) | (uint64_t(s_next[5]) << 32));
      for (uint32_t i = tid * 32u; i < nn; i += kWorkThreads * 32u) asm volatile("prefetch.global.L2 [%0];" ::"l"(nsrc + i));
    }

    // ---- S6 (in-tile part): ordered count; lanes 0..15 of warp w own the core rows 16 w .. 16 w + 15 ----
    const uint32_t krow = warp * 16u + (lane & 15u);
    const uint32_t jrow = uint32_t(kReach) + krow;
    uint32_t cnt = 0;
    if (lane < 16u && krow < ncore) {
      const uint32_t* r = fw + jrow * nfw;
      for (uint32_t w = 1; w < nfw; ++w) cnt += __popc(r[w]);
    }
    uint32_t incl = cnt;
#pragma unroll
    for (int o = 1; o < 16; o <<= 1) {
      const uint32_t v = __shfl_up_sync(0xffffffffu, incl, o);
      if (lane >= uint32_t(o)) incl += v;
    }
    const uint32_t wcount = __shfl_sync(0xffffffffu, incl, 15);
    if (lane < 16u) rowx[krow] = incl - cnt;                             // peaks of this warp before this lane's row
    if (lane == 0) wtot[warp] = wcount;
    bar_sync_named(kBarWork, kWorkThreads);
    PH_MARK(3)
    uint32_t total;
    {
      const uint32_t v = lane < uint32_t(kWorkWarps) ? wtot[lane] : 0u;
      uint32_t ps = v;
#pragma unroll
      for (int o = 1; o < kWorkWarps; o <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, ps, o);
        if (lane >= uint32_t(o)) ps += u;
      }
      if (lane < uint32_t(kWorkWarps)) wpre[warp * uint32_t(kWorkWarps) + lane] = ps - v;   // this warp's own copy
      total = __shfl_sync(0xffffffffu, ps, kWorkWarps - 1);
      __syncwarp();
    }
    // publish the tile's count early so that later tiles' look-backs never wait for this tile's build
    if (tid == 0 && t != 0u) st_release_u64(P.tile_state + t, pack_state(P.epoch, kStAgg, total));

    // ---- S3..S5: one thread per peak, at most kListCap peaks per hand-over item ----
    const int32_t t_row0 = t0 - kReach;
    uint32_t done = 0;
    do {
      const uint32_t b = q & 1u;
      const uint32_t npass = min(total - done, uint32_t(kListCap));
      PH_MARK(4)
      if (q >= 2u) bar_sync_named(kBarEmpty + int(b), kThreads);        // staging[b] has been copied out
      PH_MARK(7)
      const uint32_t pk = tid;                                           // one thread per peak, dense
      if (pk < npass) {
        // locate peak number done + pk of the tile in (time,pad) order: its warp (largest w with wpre[w] <= x),
        // its row inside the warp's 16 (largest r with rowx[r] <= x'), then the x''-th set flag of that row
        uint32_t x = done + pk;
        const uint32_t* wp = wpre + warp * uint32_t(kWorkWarps);
        uint32_t wsel = 0;
#pragma unroll
        for (int st = kWorkWarps / 2; st >= 1; st >>= 1)
          if (wp[wsel + uint32_t(st)] <= x) wsel += uint32_t(st);
        x -= wp[wsel];
        const uint32_t* rx = rowx + wsel * 16u;
        uint32_t rsel = 0;
#pragma unroll
        for (int st = 8; st >= 1; st >>= 1)
          if (rx[rsel + uint32_t(st)] <= x) rsel += uint32_t(st);
        x -= rx[rsel];
        const uint32_t j = uint32_t(kReach) + wsel * 16u + rsel;
        TPC_ASSERT(wsel * 16u + rsel < ncore);
        const uint32_t* r = fw + j * nfw;
        uint32_t bits = 0, wbit = 0;
        bool found = false;
        for (uint32_t w = 1; w < nfw; ++w) {
          const uint32_t v = r[w], c = __popc(v);
          if (!found) {
            if (x < c) { bits = v; wbit = (w - 1u) * 32u; found = true; } else x -= c;
          }
        }
        for (; x; --x) bits &= bits - 1u;                               // drop the x lowest flags
        TPC_ASSERT(found && bits != 0u);
        const uint32_t pad = wbit + uint32_t(__ffs(bits)) - 1u - uint32_t(kColOff);
        TPC_ASSERT(pad < ri.npads && map[j * W + pad + kColOff] >= P.theta);
        uint4 lo4, hi4;
        build1(map, fw, W, nfw, j, pad, reinterpret_cast<const uint4*>(nbr_tab), wtab, sector_row, ri.npads, t_row0, P.tf_time_bins,
               lo4, hi4);
        uint4* stg = stage + b * (2u * kListCap) + 2u * pk;
        stg[0] = lo4;
        stg[1] = hi4;
      }
      if (tid == 0) {
        uint32_t* m = s_meta + 4u * b;
        m[0] = t;
        m[1] = total;
        m[2] = done;
        m[3] = npass;
      }
      bar_arrive_named(kBarFull + int(b), kThreads);                     // the records of this item are staged
      ++q;
      done += npass;
    } while (done < total);
    PH_MARK(4)
    bar_sync_named(kBarWork, kWorkThreads);   // map, flags and s_next are stable until here
    PH_MARK(5)
  }
  PH_DUMP(ph_tiles)
  (void)ph_tiles;
  // stop item
  {
    const uint32_t b = q & 1u;
    if (q >= 2u) bar_sync_named(kBarEmpty + int(b), kThreads);
    if (tid == 0) s_meta[4u * b] = kStopTile;
    bar_arrive_named(kBarFull + int(b), kThreads);
  }
}

}  // namespace tpcclus
