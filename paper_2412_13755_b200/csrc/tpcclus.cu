// tpcclus.cu — C-ABI of include/tpcclus.h on top of the sm_100a kernels in tpcclus_kernels.cuh.
//
// Host logic only: argument checks, geometry tables, launches, the host-staging pipeline.
// Every step of the path runs in the kernels.  The library links against the static CUDA
// runtime only and loads on a box without a GPU driver (where tpcclus_create then fails
// loudly with TPCCLUS_ERR_CUDA — there is no CPU fallback).
#include "../../include/tpcclus.h"
#include "tpcclus_kernels.cuh"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <new>
#include <vector>

using namespace tpcclus;

constexpr int kRing = TPCCLUS_MAX_PENDING;

// ---- tpcclus_select_static: k_select's scratch in a fixed device array instead of allocated memory ----
// Layout: word 0 (as u32) = the tile ticket; words 32.. = one decoupled look-back word per 1024-record tile.
// In host code this NAME is only a handle for cudaGetSymbolAddress (select_static_scratch below), never a device
// address.  Every device that loads the library holds its own copy (128.25 KB) until the process exits.
constexpr uint32_t kSelStaticHdr = 32;                                               // 256 bytes
constexpr uint32_t kSelStaticTiles = uint32_t(TPCCLUS_SELECT_STATIC_MAX_RECORDS / kSelTile);   // 16384
static_assert(TPCCLUS_SELECT_STATIC_MAX_RECORDS % kSelTile == 0, "whole tiles");
static __device__ __align__(256) unsigned long long g_sel_static[kSelStaticHdr + kSelStaticTiles];

static_assert(sizeof(tpcclus_digit) == 8, "digit is 8 bytes");
static_assert(sizeof(tpcclus_cluster) == 32 && sizeof(tpcclus_cluster) == sizeof(ClusterRec), "cluster is 32 bytes");

struct tpcclus_ctx {
  tpcclus_geometry g{};
  std::vector<uint16_t> npads;
  std::vector<RowInfo> rows;
  int device = 0;
  uint32_t tiles_per_row_max = 0; // ceil(max_core_bins / kTileT)
  uint32_t bins_per_row_max = 0;  // digit bins laid out per (sector,row): ceil(max_core_bins / kBinT)
  uint32_t max_bins = 0;
  uint64_t sec_list_elems = 0;    // digit-list elements per sector
  uint32_t max_tiles = 0;
  uint32_t map_bytes_max = 0, smem_bytes = 0;
  int tile_grid = 0;              // persistent grid of k_tile
  int bin_ctas_per_sm = 1;        // resident k_bin CTAs per SM (occupancy query)
  bool bin_aggregated = false;    // k_bin (CTA-aggregated) usable for this geometry, else k_bin_direct
  int n_sm = 0;
  uint32_t epoch = 0;
  uint64_t launches = 0;
  uint64_t dev_bytes = 0;
  // device
  uint32_t* d_lists = nullptr;    // fixed-capacity digit bins, one per (sector,row,time-tile)
  uint32_t* d_counts = nullptr;   // digits appended per bin in the current run
  RowInfo* d_rows = nullptr;
  unsigned long long* d_tile_state = nullptr;
  DevStatus* d_status = nullptr;
  // tpcclus_select (D13): scratch of its own
  unsigned long long* d_sel_state = nullptr;   // look-back words, one per 1024 records
  uint32_t sel_tiles_cap = 0, sel_epoch = 0;
  unsigned long long* d_sel_kept = nullptr;    // [0] records kept, [1] (as u32) the tile ticket
  unsigned long long* h_sel_kept = nullptr;    // pinned
  cudaEvent_t ev_sel = nullptr;
  bool sel_pending = false;
  uint64_t sel_cap = 0;
  // pinned host ring: one status slot per pending run (results are reported in FIFO order)
  DevStatus* h_status = nullptr;
  struct Pending { uint64_t n, cap; };
  Pending pending[kRing];
  cudaEvent_t ev_done[kRing] = {};
  cudaEvent_t ev_prof[kRing][TPCCLUS_N_KERNELS + 1] = {};   // around k_init / k_bin / k_tile when profiling
  bool slot_profiled[kRing] = {};
  uint64_t head = 0, tail = 0;          // runs reported / runs enqueued
  cudaStream_t last_stream = nullptr;
  bool profiling = false;
  double prof_ms[TPCCLUS_N_KERNELS] = {};
  uint64_t prof_runs = 0;
  // host staging (TPCCLUS_OPT_HOST_STAGING)
  tpcclus_digit* d_stage_digits[2] = {nullptr, nullptr};
  tpcclus_cluster* d_stage_out[2] = {nullptr, nullptr};
  cudaStream_t s_h2d = nullptr, s_run = nullptr, s_d2h = nullptr;
  cudaEvent_t ev_h2d[2] = {nullptr, nullptr}, ev_run[2] = {nullptr, nullptr}, ev_d2h[2] = {nullptr, nullptr};
};

namespace {

inline uint32_t roundup(uint32_t x, uint32_t m) { return (x + m - 1) / m * m; }

// Debugging aid, compiled in only with -DTPCCLUS_DEBUG_SYNC: synchronise after every launch and name the
// kernel that failed on stderr.  The library reads no environment variables.
#ifdef TPCCLUS_DEBUG_SYNC
void debug_check(cudaStream_t st, const char* what) {
  cudaError_t e = cudaStreamSynchronize(st);
  if (e == cudaSuccess) e = cudaGetLastError();
  std::fprintf(stderr, "[tpcclus] %s: %s\n", what, cudaGetErrorString(e));
}
#else
inline void debug_check(cudaStream_t, const char*) {}
#endif

#define CK(ctx, call)                                  \
  do {                                                 \
    cudaError_t e__ = (call);                          \
    if (e__ != cudaSuccess) return TPCCLUS_ERR_CUDA;    \
  } while (0)

// Device address of g_sel_static on the CURRENT device (and its SM count), looked up once per device with that
// device current.  Allocates nothing.
cudaError_t select_static_scratch(unsigned long long** ptr, int* n_sm) {
  constexpr int kMaxDev = 64;
  struct PerDevice { bool ready = false; unsigned long long* ptr = nullptr; int n_sm = 0; };
  static PerDevice table[kMaxDev];
  static std::mutex mu;
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess) return e;
  if (dev < 0 || dev >= kMaxDev) return cudaErrorInvalidDevice;
  std::lock_guard<std::mutex> lock(mu);
  PerDevice& d = table[dev];
  if (!d.ready) {
    unsigned long long* p = nullptr;
    int sms = 0;
    if ((e = cudaGetSymbolAddress(reinterpret_cast<void**>(&p), g_sel_static)) != cudaSuccess) return e;
    if ((e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return e;
    if (!p || sms < 1) return cudaErrorUnknown;
    d.ptr = p;
    d.n_sm = sms;
    d.ready = true;
  }
  *ptr = d.ptr;
  *n_sm = d.n_sm;
  return cudaSuccess;
}

template <typename T>
int dev_alloc(tpcclus_ctx* c, T** p, uint64_t bytes) {
  cudaError_t e = cudaMalloc(reinterpret_cast<void**>(p), bytes ? bytes : 16);
  if (e == cudaErrorMemoryAllocation) { cudaGetLastError(); return TPCCLUS_ERR_NOMEM; }
  if (e != cudaSuccess) return TPCCLUS_ERR_CUDA;
  c->dev_bytes += bytes;
  return TPCCLUS_OK;
}

}  // namespace

static int run_tf_host_enqueue(tpcclus_ctx* c, const tpcclus_fragment* fr, uint32_t nf, tpcclus_cluster* h_out,
                               uint64_t cap, tpcclus_run_stats* stats);

extern "C" {

const char* tpcclus_strerror(int code) {
  switch (code) {
    case TPCCLUS_OK: return "ok";
    case TPCCLUS_ERR_INVALID: return "invalid argument";
    case TPCCLUS_ERR_GEOMETRY: return "invalid geometry";
    case TPCCLUS_ERR_CAPACITY: return "cluster output capacity exceeded";
    case TPCCLUS_ERR_DIGIT: return "invalid digit in strict mode";
    case TPCCLUS_ERR_CUDA: return "CUDA error";
    case TPCCLUS_ERR_NOMEM: return "out of memory";
    case TPCCLUS_ERR_OCCUPANCY: return "digit bin overflow (bin_occupancy_pct too small for this input)";
    case TPCCLUS_ERR_TOO_LARGE: return "more records than tpcclus_select_static's fixed scratch holds (TPCCLUS_SELECT_STATIC_MAX_RECORDS)";
    default: return "unknown status";
  }
}

void tpcclus_destroy(tpcclus_ctx* c) {
  if (!c) return;
  cudaSetDevice(c->device);
  if (c->s_run) cudaStreamSynchronize(c->s_run);
  if (c->tail != c->head) cudaStreamSynchronize(c->last_stream);
  for (int i = 0; i < kRing; ++i) {
    if (c->ev_done[i]) cudaEventDestroy(c->ev_done[i]);
    for (int k = 0; k <= TPCCLUS_N_KERNELS; ++k) if (c->ev_prof[i][k]) cudaEventDestroy(c->ev_prof[i][k]);
  }
  if (c->sel_pending && c->ev_sel) cudaEventSynchronize(c->ev_sel);
  cudaFree(c->d_sel_state); cudaFree(c->d_sel_kept);
  if (c->h_sel_kept) cudaFreeHost(c->h_sel_kept);
  if (c->ev_sel) cudaEventDestroy(c->ev_sel);
  cudaFree(c->d_lists); cudaFree(c->d_counts); cudaFree(c->d_rows); cudaFree(c->d_tile_state); cudaFree(c->d_status);
  if (c->h_status) cudaFreeHost(c->h_status);
  for (int i = 0; i < 2; ++i) {
    cudaFree(c->d_stage_digits[i]); cudaFree(c->d_stage_out[i]);
    if (c->ev_h2d[i]) cudaEventDestroy(c->ev_h2d[i]);
    if (c->ev_run[i]) cudaEventDestroy(c->ev_run[i]);
    if (c->ev_d2h[i]) cudaEventDestroy(c->ev_d2h[i]);
  }
  if (c->s_h2d) cudaStreamDestroy(c->s_h2d);
  if (c->s_run) cudaStreamDestroy(c->s_run);
  if (c->s_d2h) cudaStreamDestroy(c->s_d2h);
  delete c;
}

int tpcclus_create(const tpcclus_geometry* g, int cuda_device, tpcclus_ctx** out) {
  if (!g || !out || !g->npads) return TPCCLUS_ERR_INVALID;
  *out = nullptr;
  if (g->n_sectors < 1 || g->n_sectors > (uint32_t)kMaxSectors || g->n_rows < 1 || g->n_rows > 256 ||
      g->tf_time_bins < 1 || g->tf_time_bins > TPCCLUS_MAX_TF_BINS || g->max_core_bins < 1 ||
      g->max_core_bins > g->tf_time_bins || (g->halo_bins >= 1 && g->halo_bins < TPCCLUS_MIN_HALO) ||
      g->halo_bins > 4096 || g->peak_min_q16 < 1 || g->peak_min_q16 > TPCCLUS_QMAX_Q16 ||
      g->bin_occupancy_pct > 100 || g->reserved_ != 0)
    return TPCCLUS_ERR_GEOMETRY;
  for (uint32_t r = 0; r < g->n_rows; ++r)
    if (g->npads[r] < 1 || g->npads[r] > TPCCLUS_MAX_NPADS) return TPCCLUS_ERR_GEOMETRY;

  tpcclus_ctx* c = new (std::nothrow) tpcclus_ctx();
  if (!c) return TPCCLUS_ERR_NOMEM;
  c->g = *g;
  c->npads.assign(g->npads, g->npads + g->n_rows);
  c->g.npads = c->npads.data();
  c->device = cuda_device;

  auto fail = [&](int rc) { tpcclus_destroy(c); return rc; };
  cudaError_t e = cudaSetDevice(cuda_device);
  if (e != cudaSuccess) return fail(TPCCLUS_ERR_CUDA);
  cudaDeviceProp prop;
  if (cudaGetDeviceProperties(&prop, cuda_device) != cudaSuccess) return fail(TPCCLUS_ERR_CUDA);
  if (prop.major < 10) return fail(TPCCLUS_ERR_CUDA);       // TMA + sm_100a code only; no fallback
  c->n_sm = prop.multiProcessorCount;

  // geometry tables: one digit bin per (sector, row, kBinT time bins).  Capacity: bin_occupancy_pct of the
  // cells of the bin's window (D2: at most one digit per cell, so 100 % cannot overflow) plus what k_bin's
  // whole-sector flushes pad with zero entries: at most 8 per bin for every CTA that works on the sector.
  // A bin that receives more than its capacity makes the run fail with TPCCLUS_ERR_OCCUPANCY.
  c->tiles_per_row_max = (g->max_core_bins + kTileT - 1) / kTileT;
  c->bins_per_row_max = (g->max_core_bins + kBinT - 1) / kBinT;
  const uint32_t bin_rows = std::min<uint32_t>(uint32_t(kBinBoxH), g->max_core_bins + 2 * g->halo_bins);
  const uint32_t occ_pct = g->bin_occupancy_pct ? g->bin_occupancy_pct : 50u;
  const uint32_t cap_margin = 8u * uint32_t(c->n_sm) + 64u;
  c->rows.resize(g->n_rows);
  uint64_t off = 0;
  uint32_t max_W = 0, max_npads = 0;
  for (uint32_t r = 0; r < g->n_rows; ++r) {
    RowInfo& ri = c->rows[r];
    ri.npads = c->npads[r];
    ri.W = uint16_t(roundup(ri.npads + 2 * kColOff, 8));
    ri.cap = roundup((bin_rows * ri.npads * occ_pct + 99u) / 100u + cap_margin, 8);
    ri.ns = uint16_t(ri.W / 8);
    ri.fpb = uint16_t(flag_pitch_bytes(ri.W));
    {
      // sweep tasks: as many row segments as the worker warps can take at once (30 tasks per warp: two lanes
      // repeat the neighbouring tasks), each flagging segL of the kBoxH - 2 rows that carry flags
      const uint32_t rows_out = uint32_t(kBoxH) - 2u;
      const uint32_t nseg_max = std::max<uint32_t>(uint32_t(kWorkWarps) * 30u / ri.ns, 1u);
      const uint32_t L = (rows_out + nseg_max - 1) / nseg_max;
      ri.segL = uint16_t(L);
      ri.ntasks = uint16_t(ri.ns * ((rows_out + L - 1) / L));
      ri.rcp_ns = (65536u + ri.ns - 1u) / ri.ns;
    }
    // the sparse path costs ~1.4 warp instructions per list entry, zeroing + sweeping the map ~85 per map column
    ri.sparse_max = std::min<uint32_t>(8u * uint32_t(kWorkThreads), 55u * ri.W);
    ri.pad_ = 0;
    ri.list_off = uint32_t(off);
    off += uint64_t(c->bins_per_row_max) * ri.cap;
    if (off > 0xFFFFFFFFull) return fail(TPCCLUS_ERR_GEOMETRY);   // list offsets inside a sector are 32-bit
    max_W = std::max<uint32_t>(max_W, ri.W);
    max_npads = std::max<uint32_t>(max_npads, ri.npads);
  }
  c->sec_list_elems = off;
  (void)max_npads;
  c->map_bytes_max = roundup(2u * uint32_t(kMapGuard) + uint32_t(kBoxH) * max_W * 2u + uint32_t(kBoxH) * flag_pitch_bytes(max_W), 16) + 16u;
  const uint64_t tiles = uint64_t(g->n_sectors) * g->n_rows * c->tiles_per_row_max;
  if (tiles > 0x7FFFFFF0ull) return fail(TPCCLUS_ERR_GEOMETRY);
  c->max_tiles = uint32_t(tiles);
  c->max_bins = g->n_sectors * g->n_rows * c->bins_per_row_max;
  c->smem_bytes = c->map_bytes_max + 2 * kListCap * 32 + kNbrTabWords * 4 + kTileT * 4 + kWorkWarps * kWorkWarps * 4 + 32 +
                  32 * 4 + 2 * 4 * 4 + 16 * 4 + g->n_rows * uint32_t(sizeof(RowInfo)) + 128;

  int rc;
  const uint64_t list_bytes = uint64_t(g->n_sectors) * c->sec_list_elems * 4;
  if ((rc = dev_alloc(c, &c->d_lists, list_bytes)) != TPCCLUS_OK) return fail(rc);
  if ((rc = dev_alloc(c, &c->d_counts, (uint64_t(c->max_bins) + 4) * 4)) != TPCCLUS_OK) return fail(rc);
  if ((rc = dev_alloc(c, &c->d_rows, g->n_rows * sizeof(RowInfo))) != TPCCLUS_OK) return fail(rc);
  if ((rc = dev_alloc(c, &c->d_tile_state, uint64_t(c->max_tiles) * 8)) != TPCCLUS_OK) return fail(rc);
  if ((rc = dev_alloc(c, &c->d_status, sizeof(DevStatus))) != TPCCLUS_OK) return fail(rc);
  if (cudaMallocHost(reinterpret_cast<void**>(&c->h_status), kRing * sizeof(DevStatus)) != cudaSuccess) return fail(TPCCLUS_ERR_NOMEM);
  for (int i = 0; i < kRing; ++i) {
    if (cudaEventCreateWithFlags(&c->ev_done[i], cudaEventDisableTiming) != cudaSuccess) return fail(TPCCLUS_ERR_CUDA);
    for (int k = 0; k <= TPCCLUS_N_KERNELS; ++k)
      if (cudaEventCreate(&c->ev_prof[i][k]) != cudaSuccess) return fail(TPCCLUS_ERR_CUDA);
  }
  // the bins start out as all "no digit" entries: whatever a later run leaves in slots it reserved but could
  // not fill is then either zero or a well-formed entry of this geometry (memory safety for duplicate cells)
  if (cudaMemset(c->d_lists, 0, list_bytes ? list_bytes : 16) != cudaSuccess) return fail(TPCCLUS_ERR_CUDA);
  if (cudaMemcpy(c->d_rows, c->rows.data(), g->n_rows * sizeof(RowInfo), cudaMemcpyHostToDevice) != cudaSuccess ||
      cudaMemset(c->d_tile_state, 0, uint64_t(c->max_tiles) * 8) != cudaSuccess ||
      cudaMemset(c->d_status, 0, sizeof(DevStatus)) != cudaSuccess)
    return fail(TPCCLUS_ERR_CUDA);

  // the attribute belongs to the function, not to this context: always allow the device maximum so that
  // contexts with different geometries can coexist
  if (c->smem_bytes > uint32_t(prop.sharedMemPerBlockOptin)) return fail(TPCCLUS_ERR_GEOMETRY);
  if (cudaFuncSetAttribute(k_tile, cudaFuncAttributeMaxDynamicSharedMemorySize, int(prop.sharedMemPerBlockOptin)) != cudaSuccess)
    return fail(TPCCLUS_ERR_CUDA);
  int occ = 0;
  if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_tile, kThreads, c->smem_bytes) != cudaSuccess || occ < 1)
    return fail(TPCCLUS_ERR_CUDA);
  c->tile_grid = occ * c->n_sm;
  {
    const uint32_t nb_max = g->n_rows * c->bins_per_row_max;
    c->bin_aggregated = nb_max <= kBinMaxNb && bin_smem_bytes(nb_max) <= uint32_t(prop.sharedMemPerBlockOptin) &&
                        !(g->options & TPCCLUS_OPT_BIN_DIRECT);
    if (c->bin_aggregated &&
        cudaFuncSetAttribute(k_bin, cudaFuncAttributeMaxDynamicSharedMemorySize, int(prop.sharedMemPerBlockOptin)) != cudaSuccess)
      return fail(TPCCLUS_ERR_CUDA);
    if (c->bin_aggregated) {
      int bocc = 0;
      if (cudaOccupancyMaxActiveBlocksPerMultiprocessor(&bocc, k_bin, kBinThreads, bin_smem_bytes(nb_max)) != cudaSuccess || bocc < 1)
        return fail(TPCCLUS_ERR_CUDA);
      c->bin_ctas_per_sm = 1;   // the bins' capacity margin (8 slots per CTA and bin) is sized for one CTA per SM
    }
  }

  if (g->options & TPCCLUS_OPT_HOST_STAGING) {
    for (int i = 0; i < 2; ++i) {
      if ((rc = dev_alloc(c, &c->d_stage_digits[i], g->max_digits * sizeof(tpcclus_digit))) != TPCCLUS_OK) return fail(rc);
      if ((rc = dev_alloc(c, &c->d_stage_out[i], g->max_clusters * sizeof(tpcclus_cluster))) != TPCCLUS_OK) return fail(rc);
      if (cudaEventCreateWithFlags(&c->ev_h2d[i], cudaEventDisableTiming) != cudaSuccess ||
          cudaEventCreateWithFlags(&c->ev_run[i], cudaEventDisableTiming) != cudaSuccess ||
          cudaEventCreateWithFlags(&c->ev_d2h[i], cudaEventDisableTiming) != cudaSuccess)
        return fail(TPCCLUS_ERR_CUDA);
    }
    if (cudaStreamCreateWithFlags(&c->s_h2d, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&c->s_run, cudaStreamNonBlocking) != cudaSuccess ||
        cudaStreamCreateWithFlags(&c->s_d2h, cudaStreamNonBlocking) != cudaSuccess)
      return fail(TPCCLUS_ERR_CUDA);
  }
  if (cudaDeviceSynchronize() != cudaSuccess) return fail(TPCCLUS_ERR_CUDA);
  *out = c;
  return TPCCLUS_OK;
}

int tpcclus_run(tpcclus_ctx* c, const tpcclus_digit* d_digits, uint64_t n, const uint64_t* h_off,
                uint32_t b, uint32_t e, tpcclus_cluster* d_out, uint64_t cap, void* cuda_stream) {
  return tpcclus_run_based(c, d_digits, n, h_off, 0u, b, e, d_out, cap, cuda_stream);
}

int tpcclus_run_based(tpcclus_ctx* c, const tpcclus_digit* d_digits, uint64_t n, const uint64_t* h_off, uint32_t t_base,
                      uint32_t b, uint32_t e, tpcclus_cluster* d_out, uint64_t cap, void* cuda_stream) {
  if (!c || !h_off || (n && !d_digits) || (cap && !d_out)) return TPCCLUS_ERR_INVALID;
  const tpcclus_geometry& g = c->g;
  if (!(b < e) || e > g.tf_time_bins || e - b > g.max_core_bins || n > g.max_digits || t_base > b) return TPCCLUS_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(d_digits) & 7u) || (reinterpret_cast<uintptr_t>(d_out) & 15u)) return TPCCLUS_ERR_INVALID;
  if (h_off[0] != 0 || h_off[g.n_sectors] != n) return TPCCLUS_ERR_INVALID;
  for (uint32_t s = 0; s < g.n_sectors; ++s)
    if (h_off[s + 1] < h_off[s]) return TPCCLUS_ERR_INVALID;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  if (c->tail - c->head >= uint64_t(kRing)) return TPCCLUS_ERR_INVALID;          // too many unreported runs
  if (c->tail != c->head && st != c->last_stream) return TPCCLUS_ERR_INVALID;    // pending runs share one stream
  CK(c, cudaSetDevice(c->device));
  const int slot = int(c->tail % kRing);
  const bool prof = c->profiling;
  c->slot_profiled[slot] = prof;
  if (prof) CK(c, cudaEventRecord(c->ev_prof[slot][0], st));

  const uint32_t tiles_per_row = (e - b + kTileT - 1) / kTileT;
  const uint32_t n_tiles = g.n_sectors * g.n_rows * tiles_per_row;
  const uint32_t bins_per_row = (e - b + kBinT - 1) / kBinT;
  const uint32_t n_bins = g.n_sectors * g.n_rows * bins_per_row;
  c->epoch = (c->epoch + 1) & 0x3FFFFFFFu;
  if (c->epoch == 0) {   // wrapped: stale words could alias, so wipe them once
    CK(c, cudaMemsetAsync(c->d_tile_state, 0, uint64_t(c->max_tiles) * 8, st));
    c->epoch = 1;
  }

  // S0: counters + status
  {
    const uint32_t blocks = std::min<uint32_t>((n_bins / 4 + 256) / 256, uint32_t(c->n_sm) * 8);
    k_init<<<std::max(blocks, 1u), 256, 0, st>>>(c->d_counts, n_bins, c->d_status);
    c->launches++;
    debug_check(st, "k_init");
    if (prof) CK(c, cudaEventRecord(c->ev_prof[slot][1], st));
  }
  // S1: binning
  if (n) {
    BinParams bp;
    bp.n = n;
    bp.sec_list_elems = c->sec_list_elems;
    bp.t_core_begin = int32_t(b);
    bp.t_base = int32_t(t_base);
    bp.t_lo = std::max<int32_t>(0, int32_t(b) - int32_t(g.halo_bins));
    bp.t_hi = int32_t(std::min<uint64_t>(g.tf_time_bins, uint64_t(e) + g.halo_bins));
    bp.n_sectors = g.n_sectors;
    bp.n_rows = g.n_rows;
    bp.bins_per_row = bins_per_row;
    bp.bins_per_row_max = c->bins_per_row_max;
    std::memcpy(bp.off, h_off, (g.n_sectors + 1) * sizeof(uint64_t));
    bp.nb = g.n_rows * bins_per_row;
    if (c->bin_aggregated && bp.nb <= kBinMaxNb) {
      // CTA-aggregated binning: chunks of kBinChunk digits, one sector per chunk
      bp.head = (reinterpret_cast<uintptr_t>(d_digits) & 8u) ? 1u : 0u;
      bp.base16 = reinterpret_cast<const uint4*>(reinterpret_cast<uintptr_t>(d_digits) - 8u * bp.head);
      bp.pair_lo = bp.head;
      bp.pair_hi = (n + bp.head) >> 1;
      uint32_t total = 0;
      for (uint32_t s = 0; s < g.n_sectors; ++s) {
        bp.cpref[s] = total;
        if (h_off[s + 1] <= h_off[s]) continue;
        const uint64_t p0 = std::max<uint64_t>((h_off[s] + bp.head) >> 1, bp.pair_lo);
        const uint64_t p1 = std::min<uint64_t>((h_off[s + 1] + bp.head + 1) >> 1, bp.pair_hi);
        if (p1 > p0) total += uint32_t((p1 - p0 + kBinChunk / 2 - 1) / (kBinChunk / 2));
      }
      bp.cpref[g.n_sectors] = total;
      bp.total_chunks = total;
      bp.pad_ = 0;
      const uint32_t blocks = uint32_t(std::min<uint64_t>(std::max<uint64_t>(total, 1), uint64_t(c->n_sm) * c->bin_ctas_per_sm));
      k_bin<<<blocks, kBinThreads, bin_smem_bytes(bp.nb), st>>>(bp, c->d_rows, c->d_lists, c->d_counts, c->d_status);
    } else {
      const uint64_t pairs = (n + 1) / 2;
      const uint32_t blocks = uint32_t(std::min<uint64_t>((pairs + 255) / 256, uint64_t(c->n_sm) * 16));
      k_bin_direct<<<std::max(blocks, 1u), 256, 0, st>>>(reinterpret_cast<const uint2*>(d_digits), bp, c->d_rows,
                                                         c->d_lists, c->d_counts, c->d_status);
    }
    c->launches++;
    debug_check(st, "k_bin");
  }
  if (prof) CK(c, cudaEventRecord(c->ev_prof[slot][2], st));
  // S1..S7: fused tile kernel
  {
    TileParams tp;
    tp.rows = c->d_rows;
    tp.lists = c->d_lists;
    tp.counts = c->d_counts;
    tp.tile_state = c->d_tile_state;
    tp.status = c->d_status;
    tp.out = d_out;
    tp.out_capacity = cap;
    tp.sec_list_elems = c->sec_list_elems;
    tp.n_sectors = g.n_sectors;
    tp.n_rows = g.n_rows;
    tp.tiles_per_row = tiles_per_row;
    tp.n_tiles = n_tiles;
    tp.t_core_begin = int32_t(b);
    tp.t_core_end = int32_t(e);
    tp.tf_time_bins = g.tf_time_bins;
    tp.theta = g.peak_min_q16;
    tp.epoch = c->epoch;
    tp.map_bytes_max = c->map_bytes_max;
    tp.theta2 = uint32_t(g.peak_min_q16) | (uint32_t(g.peak_min_q16) << 16);
    const int grid = int(std::min<uint32_t>(n_tiles, uint32_t(c->tile_grid)));
    k_tile<<<grid, kThreads, c->smem_bytes, st>>>(tp);
    c->launches++;
    debug_check(st, "k_tile");
  }
  if (prof) CK(c, cudaEventRecord(c->ev_prof[slot][3], st));
  CK(c, cudaGetLastError());
  CK(c, cudaMemcpyAsync(&c->h_status[slot], c->d_status, sizeof(DevStatus), cudaMemcpyDeviceToHost, st));
  CK(c, cudaEventRecord(c->ev_done[slot], st));
  c->last_stream = st;
  c->pending[slot].n = n;
  c->pending[slot].cap = cap;
  c->tail++;
  return TPCCLUS_OK;
}

int tpcclus_result(tpcclus_ctx* c, tpcclus_run_stats* stats) {
  if (!c || !stats) return TPCCLUS_ERR_INVALID;
  std::memset(stats, 0, sizeof(*stats));
  if (c->head == c->tail) { stats->status = TPCCLUS_ERR_INVALID; return TPCCLUS_ERR_INVALID; }
  cudaSetDevice(c->device);
  const int slot = int(c->head % kRing);
  cudaError_t e = cudaEventSynchronize(c->ev_done[slot]);
  c->head++;
  stats->n_digits_in = c->pending[slot].n;
  if (e != cudaSuccess) {
    stats->status = TPCCLUS_ERR_CUDA;
    stats->cuda_error = int(e);
    return TPCCLUS_ERR_CUDA;
  }
  if (c->slot_profiled[slot]) {
    for (int k = 0; k < TPCCLUS_N_KERNELS; ++k) {
      float ms = 0.f;
      if (cudaEventElapsedTime(&ms, c->ev_prof[slot][k], c->ev_prof[slot][k + 1]) == cudaSuccess) c->prof_ms[k] += ms;
    }
    c->prof_runs++;
  }
  stats->n_digits_dropped = c->h_status[slot].n_dropped;
  stats->n_clusters = c->h_status[slot].n_clusters;
  int rc = TPCCLUS_OK;
  if ((c->g.options & TPCCLUS_OPT_STRICT_DIGITS) && stats->n_digits_dropped) rc = TPCCLUS_ERR_DIGIT;
  else if (c->h_status[slot].n_overfull_bins) rc = TPCCLUS_ERR_OCCUPANCY;
  else if (stats->n_clusters > c->pending[slot].cap) rc = TPCCLUS_ERR_CAPACITY;
  stats->status = rc;
  return rc;
}

int tpcclus_set_profiling(tpcclus_ctx* c, int on) {
  if (!c) return TPCCLUS_ERR_INVALID;
  c->profiling = on != 0;
  if (on) { for (double& m : c->prof_ms) m = 0; c->prof_runs = 0; }
  return TPCCLUS_OK;
}

int tpcclus_get_profile(const tpcclus_ctx* c, double kernel_ms[TPCCLUS_N_KERNELS], uint64_t* n_runs) {
  if (!c || !kernel_ms || !n_runs) return TPCCLUS_ERR_INVALID;
  for (int k = 0; k < TPCCLUS_N_KERNELS; ++k) kernel_ms[k] = c->prof_ms[k];
  *n_runs = c->prof_runs;
  return TPCCLUS_OK;
}

int tpcclus_run_tf_host(tpcclus_ctx* c, const tpcclus_fragment* fr, uint32_t nf, tpcclus_cluster* h_out,
                        uint64_t cap, tpcclus_run_stats* stats) {
  if (!c || !fr || !stats || nf == 0 || (cap && !h_out) || c->head != c->tail) return TPCCLUS_ERR_INVALID;
  if (!(c->g.options & TPCCLUS_OPT_HOST_STAGING)) return TPCCLUS_ERR_INVALID;
  // every fragment is validated before anything is enqueued, so that no copy is in flight when an argument
  // error is reported
  for (uint32_t f = 0; f < nf; ++f) {
    const tpcclus_fragment& x = fr[f];
    if (x.n > c->g.max_digits || (x.n && !x.h_digits) || !x.h_sector_offsets) return TPCCLUS_ERR_INVALID;
    if (!(x.t_core_begin < x.t_core_end) || x.t_core_end > c->g.tf_time_bins ||
        x.t_core_end - x.t_core_begin > c->g.max_core_bins || x.t_time_base > x.t_core_begin || x.reserved_ != 0)
      return TPCCLUS_ERR_INVALID;
    if (x.h_sector_offsets[0] != 0 || x.h_sector_offsets[c->g.n_sectors] != x.n) return TPCCLUS_ERR_INVALID;
    for (uint32_t s2 = 0; s2 < c->g.n_sectors; ++s2)
      if (x.h_sector_offsets[s2 + 1] < x.h_sector_offsets[s2]) return TPCCLUS_ERR_INVALID;
  }
  CK(c, cudaSetDevice(c->device));
  for (uint32_t f = 0; f < nf; ++f) {
    std::memset(&stats[f], 0, sizeof(stats[f]));
    stats[f].status = TPCCLUS_ERR_INVALID;                  // "not run" until the fragment has been reported
  }
  const int rc_tf = run_tf_host_enqueue(c, fr, nf, h_out, cap, stats);
  // whatever happened, nothing of this call may still be reading the caller's buffers or writing h_out
  const cudaError_t e1 = cudaStreamSynchronize(c->s_h2d), e2 = cudaStreamSynchronize(c->s_run),
                    e3 = cudaStreamSynchronize(c->s_d2h);
  while (c->head != c->tail) { tpcclus_run_stats drop; tpcclus_result(c, &drop); }   // (only after an error)
  if (rc_tf == TPCCLUS_OK && (e1 != cudaSuccess || e2 != cudaSuccess || e3 != cudaSuccess)) return TPCCLUS_ERR_CUDA;
  return rc_tf;
}

}  // extern "C"

// The pipeline proper; the caller synchronises the three streams afterwards on every path.
static int run_tf_host_enqueue(tpcclus_ctx* c, const tpcclus_fragment* fr, uint32_t nf, tpcclus_cluster* h_out,
                               uint64_t cap, tpcclus_run_stats* stats) {
  int first_err = TPCCLUS_OK;
  uint64_t written = 0;
  // prologue: H2D of fragment 0
  CK(c, cudaMemcpyAsync(c->d_stage_digits[0], fr[0].h_digits, fr[0].n * sizeof(tpcclus_digit), cudaMemcpyHostToDevice, c->s_h2d));
  CK(c, cudaEventRecord(c->ev_h2d[0], c->s_h2d));
  for (uint32_t f = 0; f < nf; ++f) {
    const int slot = int(f & 1u);
    // kernels of fragment f: need its digits, and the slot's output buffer drained (D2H of f-2)
    CK(c, cudaStreamWaitEvent(c->s_run, c->ev_h2d[slot], 0));
    if (f >= 2) CK(c, cudaStreamWaitEvent(c->s_run, c->ev_d2h[slot], 0));
    int rc = tpcclus_run_based(c, c->d_stage_digits[slot], fr[f].n, fr[f].h_sector_offsets, fr[f].t_time_base,
                               fr[f].t_core_begin, fr[f].t_core_end, c->d_stage_out[slot], c->g.max_clusters, c->s_run);
    if (rc != TPCCLUS_OK) {
      stats[f].status = rc;
      return rc;
    }
    CK(c, cudaEventRecord(c->ev_run[slot], c->s_run));
    // overlap: H2D of fragment f+1 into the other slot (free once the kernels of f-1 are done)
    if (f + 1 < nf) {
      const int nslot = slot ^ 1;
      if (f >= 1) CK(c, cudaStreamWaitEvent(c->s_h2d, c->ev_run[nslot], 0));
      CK(c, cudaMemcpyAsync(c->d_stage_digits[nslot], fr[f + 1].h_digits, fr[f + 1].n * sizeof(tpcclus_digit),
                            cudaMemcpyHostToDevice, c->s_h2d));
      CK(c, cudaEventRecord(c->ev_h2d[nslot], c->s_h2d));
    }
    // the record count decides the D2H size and where the next fragment's list starts (D10)
    rc = tpcclus_result(c, &stats[f]);
    if (rc == TPCCLUS_ERR_CUDA) return rc;
    uint64_t ncopy = std::min<uint64_t>(stats[f].n_clusters, c->g.max_clusters);
    if (written + ncopy > cap) { ncopy = cap - written; rc = TPCCLUS_ERR_CAPACITY; stats[f].status = rc; }
    if (rc != TPCCLUS_OK && first_err == TPCCLUS_OK) first_err = rc;
    if (ncopy) {
      CK(c, cudaStreamWaitEvent(c->s_d2h, c->ev_run[slot], 0));
      CK(c, cudaMemcpyAsync(h_out + written, c->d_stage_out[slot], ncopy * sizeof(tpcclus_cluster), cudaMemcpyDeviceToHost, c->s_d2h));
    }
    CK(c, cudaEventRecord(c->ev_d2h[slot], c->s_d2h));
    written += ncopy;
  }
  return first_err;
}

extern "C" {

int tpcclus_run_host(tpcclus_ctx* c, const tpcclus_digit* h_digits, uint64_t n, const uint64_t* h_off, uint32_t b,
                     uint32_t e, tpcclus_cluster* h_out, uint64_t cap, tpcclus_run_stats* stats) {
  tpcclus_fragment f;
  f.h_digits = h_digits;
  f.n = n;
  f.h_sector_offsets = h_off;
  f.t_core_begin = b;
  f.t_core_end = e;
  f.t_time_base = 0;
  f.reserved_ = 0;
  return tpcclus_run_tf_host(c, &f, 1, h_out, cap, stats);
}

int tpcclus_select(tpcclus_ctx* c, const tpcclus_cluster* d_in, uint64_t n, const tpcclus_cuts* cuts,
                   tpcclus_cluster* d_out, uint64_t cap, void* cuda_stream) {
  if (!c || !cuts || (n && !d_in) || (cap && !d_out) || cuts->reserved_ != 0 || n > 0xFFFFFFFFull || c->sel_pending)
    return TPCCLUS_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(d_in) & 15u) || (reinterpret_cast<uintptr_t>(d_out) & 15u)) return TPCCLUS_ERR_INVALID;
  if (!(cuts->min_qtot == cuts->min_qtot)) return TPCCLUS_ERR_INVALID;          // NaN threshold
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  CK(c, cudaSetDevice(c->device));
  const uint32_t n_tiles = uint32_t((n + kSelTile - 1) / kSelTile);
  if (!c->d_sel_kept) {
    int rc;
    if ((rc = dev_alloc(c, &c->d_sel_kept, 16)) != TPCCLUS_OK) return rc;
    if (cudaMallocHost(reinterpret_cast<void**>(&c->h_sel_kept), 16) != cudaSuccess) return TPCCLUS_ERR_NOMEM;
    if (cudaEventCreateWithFlags(&c->ev_sel, cudaEventDisableTiming) != cudaSuccess) return TPCCLUS_ERR_CUDA;
  }
  if (n_tiles > c->sel_tiles_cap) {              // grow the look-back scratch (zeroed: epoch 0 is never used)
    CK(c, cudaStreamSynchronize(st));
    if (c->d_sel_state) { cudaFree(c->d_sel_state); c->dev_bytes -= uint64_t(c->sel_tiles_cap) * 8; c->d_sel_state = nullptr; }
    const uint32_t want = std::max<uint32_t>(n_tiles, 1024u);
    int rc;
    if ((rc = dev_alloc(c, &c->d_sel_state, uint64_t(want) * 8)) != TPCCLUS_OK) { c->sel_tiles_cap = 0; return rc; }
    CK(c, cudaMemset(c->d_sel_state, 0, uint64_t(want) * 8));
    c->sel_tiles_cap = want;
    c->sel_epoch = 0;
  }
  c->sel_epoch = (c->sel_epoch + 1) & 0x3FFFFFFFu;
  if (c->sel_epoch == 0) {
    CK(c, cudaMemsetAsync(c->d_sel_state, 0, uint64_t(c->sel_tiles_cap) * 8, st));
    c->sel_epoch = 1;
  }
  CK(c, cudaMemsetAsync(c->d_sel_kept, 0, 16, st));
  if (n_tiles) {
    SelectParams sp;
    sp.in = reinterpret_cast<const uint4*>(d_in);
    sp.out = reinterpret_cast<uint4*>(d_out);
    sp.tile_state = c->d_sel_state;
    sp.n_kept = c->d_sel_kept;
    sp.ticket = reinterpret_cast<unsigned int*>(c->d_sel_kept + 1);
    sp.n = n;
    sp.out_capacity = cap;
    sp.n_tiles = n_tiles;
    sp.epoch = c->sel_epoch;
    sp.min_qtot = cuts->min_qtot;
    sp.min_qmax_q16 = cuts->min_qmax_q16;
    sp.min_ncells = cuts->min_ncells;
    sp.reject_flags = cuts->reject_flags;
    sp.reject_single_pad = cuts->reject_single_pad ? 1u : 0u;
    sp.reject_single_time = cuts->reject_single_time ? 1u : 0u;
    sp.wide = ((reinterpret_cast<uintptr_t>(d_in) | reinterpret_cast<uintptr_t>(d_out)) & 31u) == 0u ? 1u : 0u;
    const uint32_t grid = std::min<uint32_t>(n_tiles, uint32_t(c->n_sm) * 8u);   // all resident: the look-back waits on earlier tiles
    k_select<<<grid, kSelThreads, 0, st>>>(sp);
    c->launches++;
    CK(c, cudaGetLastError());
  }
  CK(c, cudaMemcpyAsync(c->h_sel_kept, c->d_sel_kept, 8, cudaMemcpyDeviceToHost, st));
  CK(c, cudaEventRecord(c->ev_sel, st));
  c->sel_pending = true;
  c->sel_cap = cap;
  return TPCCLUS_OK;
}

int tpcclus_select_result(tpcclus_ctx* c, uint64_t* n_kept) {
  if (!c || !n_kept || !c->sel_pending) return TPCCLUS_ERR_INVALID;
  cudaSetDevice(c->device);
  c->sel_pending = false;
  if (cudaEventSynchronize(c->ev_sel) != cudaSuccess) return TPCCLUS_ERR_CUDA;
  *n_kept = *c->h_sel_kept;
  return *n_kept > c->sel_cap ? TPCCLUS_ERR_CAPACITY : TPCCLUS_OK;
}

int tpcclus_select_static(const tpcclus_cluster* d_in, uint64_t n, const tpcclus_cuts* cuts, tpcclus_cluster* d_out,
                          uint64_t cap, uint64_t* d_n_kept, void* cuda_stream) {
  if (!cuts || !d_n_kept || (n && !d_in) || (cap && !d_out) || cuts->reserved_ != 0) return TPCCLUS_ERR_INVALID;
  if ((reinterpret_cast<uintptr_t>(d_in) & 15u) || (reinterpret_cast<uintptr_t>(d_out) & 15u) ||
      (reinterpret_cast<uintptr_t>(d_n_kept) & 7u))
    return TPCCLUS_ERR_INVALID;
  if (!(cuts->min_qtot == cuts->min_qtot)) return TPCCLUS_ERR_INVALID;          // NaN threshold
  if (n > TPCCLUS_SELECT_STATIC_MAX_RECORDS) return TPCCLUS_ERR_TOO_LARGE;      // the array has no look-back word for more
  unsigned long long* scratch = nullptr;
  int n_sm = 0;
  if (select_static_scratch(&scratch, &n_sm) != cudaSuccess) return TPCCLUS_ERR_CUDA;
  cudaStream_t st = static_cast<cudaStream_t>(cuda_stream);
  const uint32_t n_tiles = uint32_t((n + kSelTile - 1) / kSelTile);
  // the array keeps the last call's contents: the ticket and the look-back words this call will use start at zero
  // (epoch 0 = "nothing published"; the call itself always runs as epoch 1)
  if (cudaMemsetAsync(scratch, 0, (uint64_t(kSelStaticHdr) + n_tiles) * 8, st) != cudaSuccess) return TPCCLUS_ERR_CUDA;
  if (cudaMemsetAsync(d_n_kept, 0, 8, st) != cudaSuccess) return TPCCLUS_ERR_CUDA;   // n = 0: no kernel writes it
  if (n_tiles) {
    SelectParams sp;
    sp.in = reinterpret_cast<const uint4*>(d_in);
    sp.out = reinterpret_cast<uint4*>(d_out);
    sp.tile_state = scratch + kSelStaticHdr;
    sp.n_kept = reinterpret_cast<unsigned long long*>(d_n_kept);
    sp.ticket = reinterpret_cast<unsigned int*>(scratch);
    sp.n = n;
    sp.out_capacity = cap;
    sp.n_tiles = n_tiles;
    sp.epoch = 1u;
    sp.min_qtot = cuts->min_qtot;
    sp.min_qmax_q16 = cuts->min_qmax_q16;
    sp.min_ncells = cuts->min_ncells;
    sp.reject_flags = cuts->reject_flags;
    sp.reject_single_pad = cuts->reject_single_pad ? 1u : 0u;
    sp.reject_single_time = cuts->reject_single_time ? 1u : 0u;
    sp.wide = ((reinterpret_cast<uintptr_t>(d_in) | reinterpret_cast<uintptr_t>(d_out)) & 31u) == 0u ? 1u : 0u;
    const uint32_t grid = std::min<uint32_t>(n_tiles, uint32_t(n_sm) * 8u);   // tiles are taken by ticket: any grid size is safe
    k_select<<<grid, kSelThreads, 0, st>>>(sp);
    if (cudaGetLastError() != cudaSuccess) return TPCCLUS_ERR_CUDA;
  }
  return TPCCLUS_OK;
}

uint64_t tpcclus_launch_count(const tpcclus_ctx* c) { return c ? c->launches : 0; }
uint64_t tpcclus_device_bytes(const tpcclus_ctx* c) { return c ? c->dev_bytes : 0; }

}  // extern "C"
