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
//   count     one lane per core row: popc of its flag words, warp scan, CTA scan -> the position of every
//             peak in (time,pad) order; the tile's count is published for the look-back       (S6, S7)
//   build     every warp builds the clusters of ITS 16 core rows, four lanes per peak, reading charges and
//             flags straight from the map (S3..S5); exact integer records (RawRec) go to a staging buffer
//   commit    the committer warp: decoupled look-back across tiles, D8 finish in fp64, ordered copy-out (S6)
//
// Definitions D1..D12: SURVEY.md §8(c), restated in DESIGN.md §2.  No code here is shared with oracle/.
#pragma once
#include <cuda_fp16.h>

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
// S3..S5, four lanes per peak.
//
// The 24 cells around a peak P split into four rotation classes of six: lane `sub` (0..3) owns
// the images under the quarter turn R_sub of the base cells
//     I0 = (1,0)  I1 = (1,1)                      inner ring (always members when charged, D5)
//     O0 = (2,-1) O1 = (2,0) O2 = (2,1) O3 = (2,2) outer ring (monotone descent, D5)
// written (a,b) = (pad, time) offsets in the lane's own frame; R_s(a,b) = (a cs - b sn, a sn + b cs)
// with (cs,sn) = (1,0),(0,1),(-1,0),(0,-1).  The inner cells 8-adjacent to O0..O3 are
// (1,-1),(1,0),(1,1) of the same frame, so a lane reads 7 charges besides P.  Moments are summed in
// the lane frame with constant coefficients and rotated once.  D6's S(c) comes from the OTHER peaks
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

struct __align__(16) RawRec {       // what the workers stage: D7's exact integers; the committer turns it into ClusterRec
  uint32_t w0, time, w2;            // as in ClusterRec
  uint32_t W;                       // sum of weights, units of 1/(16*2520) ADC
  int32_t Mp, Mt;                   // sum w dp, sum w dt
  uint32_t Mpp, Mtt;                // sum w dp^2, sum w dt^2
};
static_assert(sizeof(RawRec) == 32, "raw record is 32 bytes");

// Flag bytes of a tile: row j of the map has a 4-byte zero prefix followed by one byte per strip of 8 map
// columns (bit b of byte s <-> column 8 s + b), padded with zero bytes to a multiple of 4.  Read as 32-bit
// words, the flag of pad p sits at bit index 32 + kColOff + p of the row; the zero prefix makes the 9-bit
// window that starts four pads to the left of a peak addressable without a branch for p < 4.
__host__ __device__ inline uint32_t flag_pitch_bytes(uint32_t W) { return 4u + (((W >> 3) + 3u) & ~3u); }

// All 32 lanes call this; lanes 4g..4g+3 build the cluster of the peak at map row j, pad `pad`, from the
// tile's map and flag bytes.  Returns the two 16-byte halves of the RawRec in every lane of the group.
__device__ __forceinline__ void build4(const uint16_t* __restrict__ map, const uint32_t* __restrict__ fw, uint32_t W,
                                       uint32_t nfw, uint32_t j, uint32_t pad, const uint32_t* __restrict__ nbr_tab,
                                       const uint32_t* __restrict__ wtab, uint32_t sub, int32_t cs, int32_t sn,
                                       uint32_t sector_row /* sector | row << 8 */, uint32_t npads, int32_t t_row0,
                                       uint32_t tf_time_bins, uint4& lo, uint4& hi) {
  // ---- charges: P and the seven cells of this lane's rotation class ----
  const uint16_t* c = map + j * W + (pad + kColOff);
  const int32_t X = sn * int32_t(W) + cs, Y = cs * int32_t(W) - sn;     // steps of (a,b) in map cells
  const uint32_t qP = c[0];
  const uint32_t qIm = c[X - Y], qI0 = c[X], qI1 = c[X + Y];
  const uint32_t qO0 = c[2 * X - Y], qO1 = c[2 * X], qO2 = c[2 * X + Y], qO3 = c[2 * X + 2 * Y];
  // ---- the 9x9 flag window around P, three rows per word: bit 9*(k%3)+i of G[k/3] <-> row j-4+k, pad
  //      p-4+i.  Lane s reads rows s and s+4, lane 0 also row 8; OR-combined over the four lanes ----
  uint32_t G0 = 0, G1 = 0, G2 = 0;
  {
    const uint32_t b0 = pad + (32u + uint32_t(kColOff) - 4u);           // bit index of pad p-4
    const uint32_t sh = b0 & 31u;
    const uint32_t* rowp = fw + (j - 4u) * nfw + (b0 >> 5);
    auto row_bits = [&](uint32_t k) -> uint32_t {
      return __funnelshift_r(rowp[k * nfw], rowp[k * nfw + 1], sh) & 0x1FFu;
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
  const int32_t tglob = t_row0 + int32_t(j);                            // t_row0 = global time of map row 0
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

// Load row j of strip s, derive S / H3 / E1 (`cur`), and emit the flag byte of row j-1 (`prev`).
__device__ __forceinline__ uint32_t sweep_step(const uint16_t* __restrict__ map, uint32_t W, uint32_t j, uint32_t s,
                                               uint32_t ns, uint32_t lane, uint32_t theta2, const SweepRow& prev,
                                               SweepRow& cur) {
  const uint32_t cell0 = j * W + 8u * s;
  const uint4 c = *reinterpret_cast<const uint4*>(map + cell0);
  uint32_t wl = __shfl_up_sync(0xffffffffu, c.w, 1), wr = __shfl_down_sync(0xffffffffu, c.x, 1);
  const uint32_t* m32 = reinterpret_cast<const uint32_t*>(map) + (cell0 >> 1);
  if (s == 0u) wl = 0u; else if (lane == 0u) wl = m32[-1];              // (the map's columns 0,1 are zero anyway)
  if (s + 1u == ns) wr = 0u; else if (lane == 31u) wr = m32[4];
  const uint32_t S0 = shifted_pair(wl, c.x), S1 = shifted_pair(c.x, c.y), S2 = shifted_pair(c.y, c.z),
                 S3 = shifted_pair(c.z, c.w), S4 = shifted_pair(c.w, wr);
  cur.C[0] = c.x; cur.C[1] = c.y; cur.C[2] = c.z; cur.C[3] = c.w;
  cur.Sr[0] = S1; cur.Sr[1] = S2; cur.Sr[2] = S3; cur.Sr[3] = S4;
  cur.H3[0] = __vimax3_u16x2(S0, c.x, S1);
  cur.H3[1] = __vimax3_u16x2(S1, c.y, S2);
  cur.H3[2] = __vimax3_u16x2(S2, c.z, S3);
  cur.H3[3] = __vimax3_u16x2(S3, c.w, S4);
  cur.E1[0] = __vmaxu2(prev.H3[0], S0) + 0x00010001u;
  cur.E1[1] = __vmaxu2(prev.H3[1], S1) + 0x00010001u;
  cur.E1[2] = __vmaxu2(prev.H3[2], S2) + 0x00010001u;
  cur.E1[3] = __vmaxu2(prev.H3[3], S3) + 0x00010001u;
  // row j-1: late side needs H3 of this row
  uint32_t M[4];
#pragma unroll
  for (int i = 0; i < 4; ++i) {
    const uint32_t late = __vmaxu2(cur.H3[i], prev.Sr[i]);
    const uint32_t X = __vimax3_u16x2(prev.E1[i], late, theta2);
    M[i] = ge_mask2(prev.C[i], X);
  }
  // gather the eight flags into one byte, bit b <-> column 8 s + b: word i's low half at bit 2i, high half at 2i+1
  const uint32_t a = bitsel(0x00020001u, M[0], M[1]);
  const uint32_t b = bitsel(0x00200010u, M[2], M[3]);
  const uint32_t sel = bitsel(0x000A0005u, a, b);
  return bitsel(0x55u, sel, sel >> 16);                                 // low byte is the flag byte
}

// ----------------------------------------------------------------------------------------
// the kernel
// ----------------------------------------------------------------------------------------
constexpr int kBarWork = 1, kBarFull = 2, kBarEmpty = 4;
constexpr uint32_t kStopTile = 0xFFFFFFFFu;
constexpr int kWorkWarps = kWorkThreads / 32;
constexpr int kWarpList = 64;                 // peaks a warp lists per round (its 16 core rows)
static_assert(kWorkWarps * 16 == kTileT, "every worker warp owns 16 core rows of a tile");
__device__ __forceinline__ void bar_arrive_named(int id, int nthreads) {
  asm volatile("bar.arrive %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}

__global__ void __launch_bounds__(kThreads, 2) k_tile(const __grid_constant__ TileParams P) {
  extern __shared__ __align__(128) uint8_t smem_raw[];
  // carve-up
  uint8_t* sp = smem_raw;                                   // __align__(128); no static shared memory before it
  uint8_t* mapraw = sp;                                     sp += P.map_bytes_max;   // map, then flag bytes
  uint4* stage = reinterpret_cast<uint4*>(sp);              sp += 2 * kListCap * 32; // two RawRec staging buffers
  uint32_t* wlist = reinterpret_cast<uint32_t*>(sp);        sp += kWorkWarps * kWarpList * 4;
  uint32_t* s_next = reinterpret_cast<uint32_t*>(sp);       sp += 16;            // next tile: index, sector, row, tile of the row
  uint32_t* wtot = reinterpret_cast<uint32_t*>(sp);         sp += 32 * 4;        // peaks per worker warp
  uint32_t* s_meta = reinterpret_cast<uint32_t*>(sp);       sp += 2 * 4 * 4;     // per staging buffer: tile, total, offset, count
  uint32_t* nbr_tab = reinterpret_cast<uint32_t*>(sp);      sp += kNbrTabWords * 4;
  uint32_t* wtab = reinterpret_cast<uint32_t*>(sp);         sp += 12 * 4;        // D6: L / S for S = 1..9

  const uint32_t tid = threadIdx.x, lane = tid & 31u, warp = tid >> 5;
  for (uint32_t i = tid; i < uint32_t(kNbrTabWords); i += kThreads) nbr_tab[i] = nbr_tab_entry(i);
  if (tid < 9u) wtab[tid] = kShareL / (tid + 1u);
  __syncthreads();

  if (warp == uint32_t(kWorkWarps)) {
    // ================= committer warp: S6 look-back, S5 finish, copy-out =================
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
      bar_arrive_named(kBarEmpty + int(b), kThreads);
    }
    return;
  }

  // ================= worker warps =================
  const uint32_t sub = lane & 3u;                                      // four lanes per peak: lane frame R_sub
  const int32_t rot_cs = (sub == 0u) ? 1 : (sub == 2u) ? -1 : 0, rot_sn = (sub == 1u) ? 1 : (sub == 3u) ? -1 : 0;
  const uint32_t theta2 = P.theta | (P.theta << 16);
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
  bar_sync_named(kBarWork, kWorkThreads);

  uint32_t q = 0;                                                      // hand-over items issued so far
  for (;;) {
    const uint32_t t = s_next[0];
    if (t >= P.n_tiles) break;
    const uint32_t sector = s_next[1], row = s_next[2], tt = s_next[3];
    const RowInfo ri = P.rows[row];
    const int32_t t0 = P.t_core_begin + int32_t(tt) * kTileT;           // global time of core row 0
    const uint32_t ncore = uint32_t(min(kTileT, P.t_core_end - t0));     // S7: only the core emits
    const uint32_t W = ri.W, ns = W >> 3;
    const uint32_t fpb = flag_pitch_bytes(W), nfw = fpb >> 2;
    uint16_t* map = reinterpret_cast<uint16_t*>(mapraw);
    uint8_t* fl = mapraw + uint32_t(kBoxH) * W * 2u;                     // W % 8 == 0: 16-byte aligned
    const uint32_t* fw = reinterpret_cast<const uint32_t*>(fl);
    const uint32_t* src;
    const uint32_t n = tile_list(t, sector, row, tt, src);              // k_bin: a multiple of 8; 0 entries are padding
    const uint4* src4 = reinterpret_cast<const uint4*>(src);
    const uint32_t n4 = n >> 2;

    // ---- D2: zero the tile's charge map and flag bytes ----
    {
      const uint32_t nz = (uint32_t(kBoxH) * W * 2u + uint32_t(kBoxH) * fpb + 15u) >> 4;
      uint4* z = reinterpret_cast<uint4*>(mapraw);
      for (uint32_t i = tid; i < nz; i += kWorkThreads) z[i] = make_uint4(0u, 0u, 0u, 0u);
    }
    bar_sync_named(kBarWork, kWorkThreads);
    if (tid == 0) fetch();                    // next tile's ticket (s_next is read again after the tile's last barrier)

    // ---- S1: scatter the list into the map (16-byte loads, two in flight per thread) ----
    {
      auto put = [&](uint32_t d) {
        const uint32_t tl = dig_tl(d);
        if (d && tl < uint32_t(kBoxH)) map[tl * W + dig_pad(d) + kColOff] = uint16_t(dig_q(d));   // 0 = padding
      };
      uint32_t i = tid;
      for (; i + kWorkThreads < n4; i += 2 * kWorkThreads) {
        const uint4 a = __ldg(src4 + i), c = __ldg(src4 + i + kWorkThreads);
        put(a.x); put(a.y); put(a.z); put(a.w);
        put(c.x); put(c.y); put(c.z); put(c.w);
      }
      if (i < n4) {
        const uint4 a = __ldg(src4 + i);
        put(a.x); put(a.y); put(a.z); put(a.w);
      }
      if (tid < (n & 3u)) put(__ldg(src + 4u * n4 + tid));               // k_bin_direct lists: any length
    }
    bar_sync_named(kBarWork, kWorkThreads);

    // ---- S2: dense D4 sweep -> flag bytes of map rows 1 .. kBoxH-2 ----
    {
      // tasks = (strip s, row segment g): consecutive threads take consecutive strips of one segment, so that a
      // lane's horizontal neighbours are its neighbour lanes' registers
      constexpr uint32_t kRowsOut = uint32_t(kBoxH) - 2u;                // 264
      const uint32_t nseg_max = max(uint32_t(kWorkThreads) / ns, 1u);
      const uint32_t L = (kRowsOut + nseg_max - 1u) / nseg_max;          // rows per segment
      const uint32_t nseg = (kRowsOut + L - 1u) / L;
      const uint32_t ntasks = ns * nseg;
      for (uint32_t task0 = warp * 32u; task0 < ntasks; task0 += uint32_t(kWorkThreads)) {   // (one pass unless ns > kWorkThreads)
        const uint32_t task = task0 + lane;
        const bool active = task < ntasks;
        const uint32_t g = active ? task / ns : 0u, s = active ? task - g * ns : 0u;
        const uint32_t jbase = g * L;                                    // first row loaded; rows jbase+1 .. jbase+L are flagged
        const uint32_t jlast = min(jbase + L, kRowsOut);                 // last row flagged by this task
        SweepRow ra, rb;
#pragma unroll
        for (int i = 0; i < 4; ++i) { ra.C[i] = ra.Sr[i] = ra.H3[i] = ra.E1[i] = 0u; }
        rb = ra;
        // step k loads row jbase + k and flags row jbase + k - 1 (valid from k = 2 on)
        for (uint32_t k = 0; k < L + 2u; k += 2u) {
          {
            const uint32_t j = min(jbase + k, uint32_t(kBoxH) - 1u);
            const uint32_t byte = sweep_step(map, W, j, s, ns, lane, theta2, ra, rb);
            const uint32_t jo = jbase + k - 1u;
            if (active && k >= 2u && jo <= jlast) fl[jo * fpb + 4u + s] = uint8_t(byte);
          }
          {
            const uint32_t j = min(jbase + k + 1u, uint32_t(kBoxH) - 1u);
            const uint32_t byte = sweep_step(map, W, j, s, ns, lane, theta2, rb, ra);
            const uint32_t jo = jbase + k;
            if (active && k >= 1u && jo <= jlast) fl[jo * fpb + 4u + s] = uint8_t(byte);
          }
        }
      }
    }
    bar_sync_named(kBarWork, kWorkThreads);   // flags complete

    // ---- S6 (in-tile part): ordered count; lanes 0..15 of warp w own the core rows 16 w .. 16 w + 15 ----
    const uint32_t krow = warp * 16u + (lane & 15u);                     // core row of this lane (lanes 16..31 mirror 0..15)
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
    const uint32_t lexcl = incl - cnt;                                   // peaks of this warp before this lane's row
    const uint32_t wcount = __shfl_sync(0xffffffffu, incl, 15);
    if (lane == 0) wtot[warp] = wcount;
    bar_sync_named(kBarWork, kWorkThreads);
    uint32_t wbase, total;
    {
      const uint32_t v = lane < uint32_t(kWorkWarps) ? wtot[lane] : 0u;
      uint32_t ps = v;
#pragma unroll
      for (int o = 1; o < 32; o <<= 1) {
        const uint32_t u = __shfl_up_sync(0xffffffffu, ps, o);
        if (lane >= uint32_t(o)) ps += u;
      }
      wbase = __shfl_sync(0xffffffffu, ps - v, warp);
      total = __shfl_sync(0xffffffffu, ps, kWorkWarps - 1);
    }
    // publish the tile's count early so that later tiles' look-backs never wait for this tile's build
    if (tid == 0 && t != 0u) st_release_u64(P.tile_state + t, pack_state(P.epoch, kStAgg, total));

    // ---- S3..S5: every warp builds the clusters of its own rows; at most kListCap records per hand-over item ----
    const uint32_t sector_row = sector | (row << 8);
    const int32_t t_row0 = t0 - kReach;
    uint32_t done = 0;
    do {
      const uint32_t b = q & 1u;
      if (q >= 2u) bar_sync_named(kBarEmpty + int(b), kThreads);        // staging[b] has been copied out
      const uint32_t npass = min(total - done, uint32_t(kListCap));
      uint4* stg = stage + b * (2u * kListCap);
      // this warp's peaks are the tile's peaks wbase .. wbase + wcount - 1; those inside [done, done + npass) go now
      // (warp-local indices first .. last-1; empty when first >= last)
      const uint32_t first = done > wbase ? min(done - wbase, wcount) : 0u;
      const uint32_t last = done + npass > wbase ? min(done + npass - wbase, wcount) : 0u;
      for (uint32_t r0 = first; r0 < last; r0 += uint32_t(kWarpList)) {
        const uint32_t r1 = min(r0 + uint32_t(kWarpList), last);
        // list the warp's peaks r0 .. r1-1: the row owners walk their flag bits in ascending pad order
        uint32_t* wl = wlist + warp * uint32_t(kWarpList);
        __syncwarp();
        if (lane < 16u && cnt != 0u && lexcl < r1 && lexcl + cnt > r0) {
          const uint32_t* r = fw + jrow * nfw;
          uint32_t k = lexcl;
          for (uint32_t w = 1; w < nfw; ++w) {
            uint32_t bits = r[w];
            while (bits) {
              const uint32_t bpos = uint32_t(__ffs(bits)) - 1u;
              bits &= bits - 1u;
              if (k >= r0 && k < r1) wl[k - r0] = (jrow << 8) | ((w - 1u) * 32u + bpos - uint32_t(kColOff));
              ++k;
            }
          }
        }
        __syncwarp();
        for (uint32_t i0 = r0; i0 < r1; i0 += 8u) {
          const uint32_t i = min(i0 + (lane >> 2), r1 - 1u);             // (a ragged group redoes the last peak)
          const uint32_t e = wl[i - r0];
          uint4 lo4, hi4;
          build4(map, fw, W, nfw, e >> 8, e & 0xFFu, nbr_tab, wtab, sub, rot_cs, rot_sn, sector_row, ri.npads, t_row0,
                 P.tf_time_bins, lo4, hi4);
          if (i0 + (lane >> 2) < r1 && sub < 2u) stg[2u * (wbase + i - done) + sub] = sub ? hi4 : lo4;
        }
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
    bar_sync_named(kBarWork, kWorkThreads);   // map, flags and s_next are stable until here
  }
  // stop item
  {
    const uint32_t b = q & 1u;
    if (q >= 2u) bar_sync_named(kBarEmpty + int(b), kThreads);
    if (tid == 0) s_meta[4u * b] = kStopTile;
    bar_arrive_named(kBarFull + int(b), kThreads);
  }
}

}  // namespace tpcclus
