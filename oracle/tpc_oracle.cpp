// tpc_oracle.cpp — ORACLE: plain, slow, single-threaded CPU TPC cluster finder.
//
// THIS IS TEST INFRASTRUCTURE.  Only tests/, __graft_entry__.smoke() and bench.py's
// cpu_baseline / --impl reference leg may build, load or call it.  It shares no code,
// header, table or helper with the CUDA path under paper_2412_13755_b200/ and includes
// nothing from include/.  The record layouts below restate the 8-byte digit of
// BASELINE.json:configs[0] and the 32-byte cluster of SURVEY.md §8(b) independently.
//
// What it follows.  The paper (PAPER.md:110 §4, :142/:150 §4.2) only names TPC clustering;
// BASELINE.json:north_star names the five steps; SURVEY.md §8(c) D1..D12 fixes every
// detail and is the definition this file writes out step by step, in that order and
// notation (readings A1..A19 are listed in DESIGN.md §3).  Each block cites its D-number.
//
// Parity pins (tests/test_oracle_pins.py, tests/test_oracle_bruteforce.py,
// tests/test_oracle_invariants.py): hand-built maps P1..P9 with values worked out by hand
// in SURVEY.md §8(c), closed-form Gaussian widths (P8), exhaustive 3x3 / 4x4 and random
// 8x8 maps against an independently written set/path-form checker in Python with exact
// Fractions (B1, B2), and invariants I1..I9; the time base of long time frames (A19) by translation and
// fragment-seam invariance above bin 65536 (tests/test_oracle_timebase.py); the selection D13 by hand-worked
// records (tests/test_oracle_select.py).  No function here is "parity unpinned".
//
// Build: g++ -O2 -std=c++17 -shared -fPIC tpc_oracle.cpp -o libtpc_oracle.so
#include <cmath>
#include <cstdint>
#include <cstring>
#include <vector>

namespace {

struct Digit {            // BASELINE.json:configs[0] digit format, 8 bytes
  uint8_t  row;
  uint8_t  pad;
  uint16_t time;
  float    charge;
};
static_assert(sizeof(Digit) == 8, "digit is 8 bytes");

struct Cluster {          // SURVEY.md §8(b) cluster record, 32 bytes
  uint8_t  sector, row, pad, flags;
  uint32_t time;
  uint16_t qmax_q16;
  uint16_t ncells;
  float    qtot;
  float    dpad, dtime;
  float    sigma_pad, sigma_time;
};
static_assert(sizeof(Cluster) == 32, "cluster is 32 bytes");

constexpr int      kBorder = 5;        // D9: reach of a cluster is 5 cells
constexpr int64_t  kL      = 2520;     // D6: lcm(1..9)
constexpr uint16_t kQClamp = 16368;    // D1: 1023 ADC in 1/16 ADC

constexpr uint8_t FLAG_EDGE_PAD = 1, FLAG_EDGE_TIME = 2, FLAG_SATURATED = 4, FLAG_SPLIT = 8;

// One (pad x time) charge map of one row with a 5-cell zero border on every side (D2: zero
// for every out-of-range pad or time), so that no access below needs a bounds check.
struct RowMap {
  int npads = 0, ntime = 0;            // interior size
  int W = 0;                           // stride = npads + 2*kBorder
  std::vector<uint16_t> q;             // charges
  std::vector<uint8_t>  peak;          // D4 flags
  void init(int npads_, int ntime_) {
    npads = npads_; ntime = ntime_; W = npads + 2 * kBorder;
    q.assign(size_t(W) * size_t(ntime + 2 * kBorder), 0);
    peak.assign(q.size(), 0);
  }
  size_t idx(int p, int t) const { return size_t(t + kBorder) * size_t(W) + size_t(p + kBorder); }
  uint16_t Q(int p, int t) const { return q[idx(p, t)]; }
  bool     P(int p, int t) const { return peak[idx(p, t)] != 0; }
};

// D3: total order.  a > b  <=>  Q(a) > Q(b), or Q(a) == Q(b) and key(a) < key(b) with
// key = t*256 + p: among equal charges the cell earlier in (time, pad) order wins.
inline bool beats(uint16_t qa, int pa, int ta, uint16_t qb, int pb, int tb) {
  if (qa != qb) return qa > qb;
  const int64_t ka = int64_t(ta) * 256 + pa, kb = int64_t(tb) * 256 + pb;
  return ka < kb;
}

}  // namespace

extern "C" {

struct tpc_oracle_params {
  uint32_t n_sectors, n_rows;
  const uint16_t* npads;     // [n_rows]
  uint32_t tf_time_bins;
  uint32_t halo_bins;        // any value >= 0 here (the library rejects 1..4; invariant I7
                             // needs the oracle to be able to run with halo 4)
  uint16_t peak_min_q16;     // theta_peak (D11)
  uint16_t reserved;
  uint32_t t_time_base;      // A19: the digit's u16 time field counts from this global time bin,
                             // global time = t_time_base + digit.time; 0 for time frames of up to 65536 bins
};

struct tpc_oracle_stats {
  uint64_t n_digits_in;
  uint64_t n_digits_dropped;
  uint64_t n_duplicates;     // cells hit by more than one digit (D2 precondition violated)
  uint64_t n_clusters;       // clusters found (may exceed capacity)
  uint64_t sum_q16_loaded;   // sum of q16 over all loaded digits          } for invariant I1:
  uint64_t sum_W;            // sum of W over all emitted clusters         } sum_W <= 2520*sum_q16
};

// D1: q16 = clamp(rint(charge*16), 0, 16368); rint = round-half-to-even on the float32
// product (exact, x16 is a power of two).  NaN -> 0 (dropped).
uint16_t tpc_oracle_quantise(float charge) {
  if (std::isnan(charge)) return 0;
  const float x = std::nearbyintf(charge * 16.0f);   // default rounding mode: to nearest even
  if (!(x > 0.0f)) return 0;
  if (x >= float(kQClamp)) return kQClamp;
  return uint16_t(x);
}

// Run the cluster finder on one fragment.  Layout of the arguments as in the C-ABI of the
// product (digits grouped per sector by offsets[n_sectors+1], core [b,e) in global time
// bins); out may be null when cap == 0 (count only).  Returns 0, or -1 on bad arguments.
int tpc_oracle_run(const tpc_oracle_params* prm, const Digit* digits, uint64_t n,
                   const uint64_t* offsets, uint32_t b, uint32_t e,
                   Cluster* out, uint64_t cap, tpc_oracle_stats* st) {
  if (!prm || !prm->npads || !offsets || !st || (n && !digits)) return -1;
  if (!(b < e) || e > prm->tf_time_bins || prm->peak_min_q16 < 1) return -1;
  std::memset(st, 0, sizeof(*st));
  st->n_digits_in = n;

  // D9: loaded time range = [b-h, e+h) clipped to the TF.
  const int64_t lo = std::max<int64_t>(0, int64_t(b) - int64_t(prm->halo_bins));
  const int64_t hi = std::min<int64_t>(prm->tf_time_bins, int64_t(e) + int64_t(prm->halo_bins));
  const int ntime = int(hi - lo);
  const uint16_t theta = prm->peak_min_q16;

  uint64_t n_out = 0;
  for (uint32_t s = 0; s < prm->n_sectors; ++s) {
    if (offsets[s + 1] < offsets[s] || offsets[s + 1] > n) return -1;
    // Step 1 (D1, D2): validate, quantise, bucket by row, fill the dense maps.
    std::vector<RowMap> rows(prm->n_rows);
    for (uint32_t r = 0; r < prm->n_rows; ++r) rows[r].init(prm->npads[r], ntime);
    for (uint64_t i = offsets[s]; i < offsets[s + 1]; ++i) {
      const Digit& d = digits[i];
      const uint16_t q16 = tpc_oracle_quantise(d.charge);
      const int64_t tdig = int64_t(prm->t_time_base) + int64_t(d.time);   // A19: global time bin of the digit
      const bool ok = q16 != 0 && d.row < prm->n_rows && d.pad < prm->npads[d.row] &&
                      tdig >= lo && tdig < hi;
      if (!ok) { st->n_digits_dropped++; continue; }
      RowMap& m = rows[d.row];
      const size_t k = m.idx(d.pad, int(tdig - lo));
      if (m.q[k] != 0) st->n_duplicates++;
      m.q[k] = q16;
      st->sum_q16_loaded += q16;
    }

    for (uint32_t r = 0; r < prm->n_rows; ++r) {
      RowMap& m = rows[r];
      // Step 2 (D4): Peak(c) <=> Q(c) >= theta and c beats all 8 neighbours under D3.
      for (int t = 0; t < m.ntime; ++t)
        for (int p = 0; p < m.npads; ++p) {
          const uint16_t qc = m.Q(p, t);
          if (qc < theta) continue;
          bool is_peak = true;
          for (int dt = -1; dt <= 1 && is_peak; ++dt)
            for (int dp = -1; dp <= 1; ++dp) {
              if (dp == 0 && dt == 0) continue;
              if (!beats(qc, p, t, m.Q(p + dp, t + dt), p + dp, t + dt)) { is_peak = false; break; }
            }
          m.peak[m.idx(p, t)] = is_peak ? 1 : 0;
        }

      // Step 3: every peak whose time lies in the core, ascending (time, pad) (D9, D10).
      for (int t = 0; t < m.ntime; ++t) {
        const int64_t tg = lo + t;                  // global time bin
        if (tg < int64_t(b) || tg >= int64_t(e)) continue;
        for (int p = 0; p < m.npads; ++p) {
          if (!m.P(p, t)) continue;
          const uint16_t qP = m.Q(p, t);
          // D7 accumulators, exact integers.  The peak itself has weight Q(P)*L (D6).
          int64_t W = int64_t(qP) * kL, Mp = 0, Mt = 0, Mpp = 0, Mtt = 0;
          int ncells = 1;
          uint8_t flags = 0;
          if (qP == kQClamp) flags |= FLAG_SATURATED;
          for (int dt = -2; dt <= 2; ++dt)
            for (int dp = -2; dp <= 2; ++dp) {
              if (dp == 0 && dt == 0) continue;
              const uint16_t qc = m.Q(p + dp, t + dt);
              // D5: a member has charge, and a peak cell is never a member.
              if (qc == 0 || m.P(p + dp, t + dt)) continue;
              const int d = std::max(std::abs(dp), std::abs(dt));
              bool member;
              if (d == 1) {
                member = true;                      // inner ring: descent P->c is automatic
              } else {
                // outer ring: some inner-ring cell i 8-adjacent to c with Q(i) >= Q(c)
                member = false;
                for (int it = -1; it <= 1 && !member; ++it)
                  for (int ip = -1; ip <= 1; ++ip) {
                    if (ip == 0 && it == 0) continue;                       // i is in the inner ring
                    if (std::max(std::abs(ip - dp), std::abs(it - dt)) > 1) continue;  // adjacent to c
                    if (m.Q(p + ip, t + it) >= qc) { member = true; break; }
                  }
              }
              if (!member) continue;
              // D6: S(c) = number of peaks within Chebyshev distance 2 of c (counts P).
              int S = 0;
              for (int jt = -2; jt <= 2; ++jt)
                for (int jp = -2; jp <= 2; ++jp)
                  if (m.P(p + dp + jp, t + dt + jt)) ++S;
              const int64_t w = int64_t(qc) * (kL / S);     // S in 1..9 divides 2520
              W += w; Mp += w * dp; Mt += w * dt; Mpp += w * dp * dp; Mtt += w * dt * dt;
              ++ncells;
              if (S >= 2) flags |= FLAG_SPLIT;
              if (qc == kQClamp) flags |= FLAG_SATURATED;
            }
          // D8 flags.
          if (p < 2 || p >= m.npads - 2) flags |= FLAG_EDGE_PAD;
          if (tg < 2 || tg >= int64_t(prm->tf_time_bins) - 2) flags |= FLAG_EDGE_TIME;
          st->sum_W += uint64_t(W);
          if (n_out < cap && out) {
            // D8: evaluate in double from the exact integers, round once to float32.
            Cluster c;
            std::memset(&c, 0, sizeof(c));
            c.sector = uint8_t(s); c.row = uint8_t(r); c.pad = uint8_t(p); c.flags = flags;
            c.time = uint32_t(tg);
            c.qmax_q16 = qP;
            c.ncells = uint16_t(ncells);
            const double Wd = double(W);
            c.qtot = float(Wd / 40320.0);                           // 16 * 2520
            c.dpad = float(double(Mp) / Wd);
            c.dtime = float(double(Mt) / Wd);
            c.sigma_pad = float(std::sqrt(double(Mpp * W - Mp * Mp)) / Wd);
            c.sigma_time = float(std::sqrt(double(Mtt * W - Mt * Mt)) / Wd);
            out[n_out] = c;
          }
          ++n_out;
        }
      }
    }
  }
  st->n_clusters = n_out;
  return 0;
}

// Peak flags of ONE row of ONE sector over the loaded range of a fragment, for tests that
// compare peak flags cell by cell: flags_out[t_local*npads + pad] in {0,1}, t_local counted
// from max(0, b-halo).  Same steps 1 and 2 as above.  Returns the loaded length, or -1.
int64_t tpc_oracle_peak_flags(const tpc_oracle_params* prm, const Digit* digits, uint64_t n,
                              const uint64_t* offsets, uint32_t b, uint32_t e,
                              uint32_t sector, uint32_t row, uint8_t* flags_out, uint16_t* q_out) {
  if (!prm || !offsets || sector >= prm->n_sectors || row >= prm->n_rows) return -1;
  const int64_t lo = std::max<int64_t>(0, int64_t(b) - int64_t(prm->halo_bins));
  const int64_t hi = std::min<int64_t>(prm->tf_time_bins, int64_t(e) + int64_t(prm->halo_bins));
  RowMap m;
  m.init(prm->npads[row], int(hi - lo));
  for (uint64_t i = offsets[sector]; i < offsets[sector + 1] && i < n; ++i) {
    const Digit& d = digits[i];
    const uint16_t q16 = tpc_oracle_quantise(d.charge);
    const int64_t tdig = int64_t(prm->t_time_base) + int64_t(d.time);     // A19
    if (q16 == 0 || d.row != row || d.pad >= prm->npads[row] || tdig < lo || tdig >= hi) continue;
    m.q[m.idx(d.pad, int(tdig - lo))] = q16;
  }
  for (int t = 0; t < m.ntime; ++t)
    for (int p = 0; p < m.npads; ++p) {
      const uint16_t qc = m.Q(p, t);
      bool is_peak = qc >= prm->peak_min_q16;
      for (int dt = -1; dt <= 1 && is_peak; ++dt)
        for (int dp = -1; dp <= 1; ++dp) {
          if (dp == 0 && dt == 0) continue;
          if (!beats(qc, p, t, m.Q(p + dp, t + dt), p + dp, t + dt)) { is_peak = false; break; }
        }
      flags_out[size_t(t) * m.npads + p] = is_peak ? 1 : 0;
      if (q_out) q_out[size_t(t) * m.npads + p] = qc;
    }
  return hi - lo;
}

// D13 (reading A20; SURVEY.md §8(f) f-4 "cluster-quality cuts ... as parameters", "same
// code ... with appropriate selections and parameters"): an order-preserving selection over a finished cluster
// list.  A record is KEPT iff
//   qtot >= min_qtot  and  qmax_q16 >= min_qmax_q16  and  ncells >= min_ncells  and  (flags & reject_flags) == 0
//   and not (reject_single_pad  and sigma_pad  == 0)      -- all of the cluster's weight in one pad column
//   and not (reject_single_time and sigma_time == 0)      -- all of it in one time bin
// (sigma == 0 exactly iff the central second moment Mxx*W - Mx^2 is 0: D8 evaluates it from exact integers).
struct tpc_oracle_cuts {
  float    min_qtot;
  uint16_t min_qmax_q16;
  uint16_t min_ncells;
  uint8_t  reject_flags;
  uint8_t  reject_single_pad;
  uint8_t  reject_single_time;
  uint8_t  reserved;
};

// Returns the number of records kept; the first min(kept, cap) of them are written to out, in input order.
uint64_t tpc_oracle_select(const Cluster* in, uint64_t n, const tpc_oracle_cuts* cuts, Cluster* out, uint64_t cap) {
  uint64_t kept = 0;
  for (uint64_t i = 0; i < n; ++i) {
    const Cluster& c = in[i];
    bool keep = c.qtot >= cuts->min_qtot;
    keep = keep && c.qmax_q16 >= cuts->min_qmax_q16;
    keep = keep && c.ncells >= cuts->min_ncells;
    keep = keep && (c.flags & cuts->reject_flags) == 0;
    keep = keep && !(cuts->reject_single_pad && c.sigma_pad == 0.0f);
    keep = keep && !(cuts->reject_single_time && c.sigma_time == 0.0f);
    if (!keep) continue;
    if (kept < cap && out) out[kept] = c;
    ++kept;
  }
  return kept;
}

}  // extern "C"
