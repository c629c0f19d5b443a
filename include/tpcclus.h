/* tpcclus.h — C-ABI boundary of the B200-native TPC cluster finder.
 *
 * What the library computes
 * -------------------------
 * Cluster finding on zero-suppressed, continuous-readout TPC digits of one
 * time-frame fragment: charge-map fill, 3x3 local-maximum peak finding,
 * monotone-descent 5x5 cluster assembly, charge-weighted centroid and width,
 * ordered stream compaction.  The paper (PAPER.md:58 §3.1, :116 §4, :142 §4.2)
 * states the problem — ZS digits of a time frame in, reconstructed TPC clusters
 * out, the whole TF processed on one GPU with memory reused across steps — and
 * names no algorithm; the five steps come from BASELINE.json:north_star and the
 * exact definitions D1..D12 from SURVEY.md §8(c) (restated in DESIGN.md §2).
 *
 * Conventions
 * -----------
 *  - "host" / "device" is stated for every pointer.  No torch types, no C++
 *    types, no exceptions cross this boundary.
 *  - Every function returns an int status: 0 = TPCCLUS_OK, negative = error.
 *  - A context is not thread-safe; distinct contexts are independent.
 *  - Nothing is allocated inside tpcclus_run ("GPU memory reuse
 *    across processing steps became essential"); all scratch is sized in
 *    tpcclus_create from the geometry.
 *  - Determinism: the output bytes depend only on the SET of digits, the
 *    geometry and the core range — not on digit order inside a sector slice,
 *    launch configuration or run number.
 */
#ifndef TPCCLUS_H
#define TPCCLUS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes ------------------------------------------------------ */
#define TPCCLUS_OK             0
#define TPCCLUS_ERR_INVALID   -1  /* null / misaligned pointer, core range larger than max_core_bins,
                                     core outside the TF, offsets not monotone, n > max_digits       */
#define TPCCLUS_ERR_GEOMETRY  -2  /* n_sectors / n_rows out of 1..256, npads out of 1..256, zero sizes,
                                     halo_bins in 1..4 or > 4096, bin_occupancy_pct > 100,
                                     tf_time_bins > TPCCLUS_MAX_TF_BINS, digit bins beyond 2^32 entries
                                     per sector                                                       */
#define TPCCLUS_ERR_CAPACITY  -3  /* more clusters than out_capacity: the first out_capacity records
                                     are valid and ordered, stats.n_clusters is the number required
                                     (hit count fluctuates -> "safety margin")         */
#define TPCCLUS_ERR_DIGIT     -4  /* strict mode only: some digit was out of range / NaN / zero       */
#define TPCCLUS_ERR_CUDA      -5  /* stats.cuda_error holds the cudaError_t                           */
#define TPCCLUS_ERR_NOMEM     -6  /* device or pinned-host allocation failed in create                */
#define TPCCLUS_ERR_OCCUPANCY -7  /* some (sector,row,256-bin) digit bin received more digits than
                                     bin_occupancy_pct allows (scratch is sized ahead,
                                     with a margin): the run's records are incomplete; create the
                                     context with a larger bin_occupancy_pct                          */
#define TPCCLUS_ERR_TOO_LARGE -8  /* tpcclus_select_static only: n exceeds
                                     TPCCLUS_SELECT_STATIC_MAX_RECORDS, the size its fixed scratch
                                     array is built for; nothing was enqueued                         */

/* ---- cluster flag bits ---------------------------- */
#define TPCCLUS_FLAG_EDGE_PAD   0x01u /* peak pad < 2 or >= npads[row]-2                      */
#define TPCCLUS_FLAG_EDGE_TIME  0x02u /* peak time < 2 or >= tf_time_bins-2 (true TF ends)    */
#define TPCCLUS_FLAG_SATURATED  0x04u /* peak or a member has q16 == 16368 (1023 ADC)         */
#define TPCCLUS_FLAG_SPLIT      0x08u /* some member cell is shared with another peak (S>=2)  */

/* ---- geometry option bits ---------------------------------------------- */
#define TPCCLUS_OPT_STRICT_DIGITS 0x0001u /* an invalid digit makes the run fail with ERR_DIGIT
                                             instead of being dropped and counted             */
#define TPCCLUS_OPT_HOST_STAGING  0x0002u /* allocate the device staging buffers that
                                             tpcclus_run_host / tpcclus_run_tf_host need
                                             (2 x max_digits digits + 2 x max_clusters records) */
#define TPCCLUS_OPT_BIN_DIRECT    0x0004u /* route digits with the plain one-atomic-per-entry binning
                                             kernel (k_bin_direct) instead of the write-combining one;
                                             same output bytes, slower.  It is what geometries with
                                             more than 4096 digit bins per sector get anyway; the bit
                                             exists so that tests can cover that kernel             */

#define TPCCLUS_QMAX_Q16   16368u /* 1023 ADC in 1/16 ADC: the clamp of D1 */
#define TPCCLUS_MAX_NPADS  256u  /* the pad of a digit is a uint8 */
#define TPCCLUS_MAX_TF_BINS 16777216u /* 2^24 bins; a digit's uint16 time counts from the run's time base */
#define TPCCLUS_MAX_PENDING 64    /* runs that may be enqueued before their tpcclus_result */
#define TPCCLUS_MIN_HALO   5u     /* D9: a cluster depends on charges within Chebyshev distance 5 */

/* One zero-suppressed digit, 8 bytes (BASELINE.json:configs[0]: "uint8 row, uint8 pad,
 * uint16 time, float32 charge").  time counts from the run's time base: GLOBAL time bin inside
 * the TF = t_time_base + time (base 0 in tpcclus_run, so there it IS the global time bin; time
 * frames longer than 65536 bins — PAPER.md:118 §4 tested up to 256 orbits = 114048 bins — use
 * tpcclus_run_based with a base per fragment; DESIGN.md §3 A19).  The sector is not in the
 * record: digits arrive grouped per sector (see sector_offsets below). */
typedef struct {
  uint8_t  row;
  uint8_t  pad;
  uint16_t time;
  float    charge;   /* ADC counts; quantised by the library to q16 = clamp(rint(16*charge),0,16368) (D1) */
} tpcclus_digit;

/* One cluster, 32 bytes, one per peak (D8, D10).  Integer fields are bit-exact by contract;
 * the five floats are the real-number definitions of D8 evaluated from exact integer moments. */
typedef struct {
  uint8_t  sector, row, pad, flags; /* peak cell + TPCCLUS_FLAG_* bits                       */
  uint32_t time;                    /* peak cell, global TF time bin                          */
  uint16_t qmax_q16;                /* peak charge in 1/16 ADC                                */
  uint16_t ncells;                  /* 1..25 cells contributing (peak + members)              */
  float    qtot;                    /* ADC: sum of shared charge, W / (16*2520)               */
  float    dpad, dtime;             /* centroid minus peak cell, each in (-2, 2)              */
  float    sigma_pad, sigma_time;   /* sqrt of the charge-weighted central second moment      */
} tpcclus_cluster;

/* Detector shape and scratch sizing; read once by tpcclus_create (npads is copied). */
typedef struct {
  uint32_t n_sectors, n_rows;       /* 36, 152 in the configs; each 1..256                     */
  const uint16_t* npads;            /* HOST array [n_rows], each 1..TPCCLUS_MAX_NPADS          */
  uint32_t tf_time_bins;            /* whole-TF length, e.g. 57024; 1..TPCCLUS_MAX_TF_BINS    */
  uint32_t max_core_bins;           /* largest fragment core passed to run, e.g. 4096          */
  uint32_t halo_bins;               /* digits loaded each side of the core: 0 (single
                                       fragment) or >= TPCCLUS_MIN_HALO; 8 in configs[3]       */
  uint16_t peak_min_q16;            /* theta_peak >= 1 (D11); 64 = 4 ADC is the default used
                                       by the tests and the bench                              */
  uint16_t options;                 /* TPCCLUS_OPT_* bits                                      */
  uint64_t max_digits;              /* largest n passed to run                                 */
  uint64_t max_clusters;            /* sizing of the host-staging cluster buffers only         */
  uint32_t bin_occupancy_pct;       /* capacity of a digit bin in % of the cells of its window
                                       (266 time rows x npads): 0 = default 50, else 1..100.
                                       100 can never overflow (D2: one digit per cell); the
                                       densest config (C4) fills 35 %.  The digit bins are
                                       most of the context's memory: 4 bytes x pct/100 x
                                       1.04 x cells of the largest fragment    */
  uint32_t reserved_;               /* must be 0                                               */
} tpcclus_geometry;

typedef struct {
  uint64_t n_digits_in;             /* n of the run                                            */
  uint64_t n_digits_dropped;        /* invalid digits (row/pad/time out of range, NaN, q16==0) */
  uint64_t n_clusters;              /* clusters REQUIRED (may exceed out_capacity)             */
  int32_t  status;                  /* TPCCLUS_OK or the error of the run                      */
  int32_t  cuda_error;              /* cudaError_t when status == TPCCLUS_ERR_CUDA             */
} tpcclus_run_stats;

/* One fragment of a time frame held in HOST memory, for tpcclus_run_tf_host. */
typedef struct {
  const tpcclus_digit* h_digits;    /* HOST, n digits grouped per sector                       */
  uint64_t n;
  const uint64_t* h_sector_offsets; /* HOST [n_sectors+1]                                      */
  uint32_t t_core_begin, t_core_end;
  uint32_t t_time_base;             /* global time bin that digit.time counts from (0 for TFs
                                       of up to 65536 bins)                                    */
  uint32_t reserved_;               /* must be 0                                               */
} tpcclus_fragment;

typedef struct tpcclus_ctx tpcclus_ctx; /* opaque; owns all device scratch */

/* Create a context on CUDA device `cuda_device`.  Allocates, once, everything a run needs
 * (memory is reused across steps): the digit bins (one fixed-capacity list of
 * packed 4-byte entries per sector, row and 256 time bins of the largest fragment; ~5/4 slots
 * per cell of the bin's window), the bin counters, the tile look-back state and a pinned
 * status block.  The charge map itself only ever exists in shared memory.
 * Errors: ERR_INVALID (null), ERR_GEOMETRY, ERR_NOMEM, ERR_CUDA (no device / wrong arch). */
int tpcclus_create(const tpcclus_geometry* g, int cuda_device, tpcclus_ctx** out);

/* Enqueue one fragment on `cuda_stream` (a cudaStream_t passed as void*; NULL = default
 * stream).  Asynchronous: returns after the launches; call tpcclus_result for the outcome.
 *   d_digits          DEVICE, n records, 8-byte aligned, read-only, owned by the caller and
 *                     must stay valid until the run has finished.
 *   h_sector_offsets  HOST [n_sectors+1], monotone, off[0]==0, off[n_sectors]==n; digits of
 *                     sector s are d_digits[off[s] .. off[s+1]), in ANY order.  Read during
 *                     the call, not retained.
 *   t_core_begin/end  core [b,e) in global time bins, 0 <= b < e <= tf_time_bins,
 *                     e-b <= max_core_bins.  Digits with time in [b-halo, e+halo) (clipped to
 *                     the TF) are loaded, all others are dropped and counted; exactly the
 *                     clusters whose PEAK time lies in [b,e) are emitted (D9,
 *                     BASELINE.json:configs[3]).
 *   d_out             DEVICE, out_capacity records, 16-byte aligned, owned by the caller.
 *                     Record k is the k-th peak in ascending (sector,row,time,pad) (D10).
 * At most one digit per cell is a precondition (D2); the result for duplicate cells is
 * unspecified but memory-safe.  Up to TPCCLUS_MAX_PENDING runs may be enqueued before their
 * results are collected, all on the SAME stream (they share the digit bins and execute in
 * order; no host synchronisation is needed between the fragments of a time frame).
 * Errors (immediate): ERR_INVALID (also: too many pending runs, or a different stream while
 * runs are pending), ERR_CUDA.  Deferred to tpcclus_result: ERR_CAPACITY,
 * ERR_DIGIT, ERR_CUDA. */
int tpcclus_run(tpcclus_ctx* ctx, const tpcclus_digit* d_digits, uint64_t n,
                const uint64_t* h_sector_offsets,
                uint32_t t_core_begin, uint32_t t_core_end,
                tpcclus_cluster* d_out, uint64_t out_capacity, void* cuda_stream);

/* tpcclus_run for digits whose time field counts from t_time_base (DESIGN.md §3 A19): a digit's global
 * time bin is t_time_base + digit.time; t_core_begin / t_core_end and the records' time stay global.
 * Needed when tf_time_bins > 65536; a fragment's loaded range [b - halo, e + halo) must lie inside
 * [t_time_base, t_time_base + 65536) to be expressible.  tpcclus_run == tpcclus_run_based with base 0.
 * Errors as tpcclus_run; ERR_INVALID also when t_time_base > t_core_begin. */
int tpcclus_run_based(tpcclus_ctx* ctx, const tpcclus_digit* d_digits, uint64_t n,
                      const uint64_t* h_sector_offsets, uint32_t t_time_base,
                      uint32_t t_core_begin, uint32_t t_core_end,
                      tpcclus_cluster* d_out, uint64_t out_capacity, void* cuda_stream);

/* Wait for the OLDEST unreported run (FIFO) and report it.  Returns stats->status;
 * ERR_INVALID if no run is pending. */
int tpcclus_result(tpcclus_ctx* ctx, tpcclus_run_stats* stats);

/* Same operation with HOST buffers (pageable or pinned): copies the digits host->device,
 * runs, copies min(n_clusters, out_capacity) records device->host, synchronises.  Needs
 * TPCCLUS_OPT_HOST_STAGING; n <= max_digits; out_capacity is clipped to max_clusters. */
int tpcclus_run_host(tpcclus_ctx* ctx, const tpcclus_digit* h_digits, uint64_t n,
                     const uint64_t* h_sector_offsets,
                     uint32_t t_core_begin, uint32_t t_core_end,
                     tpcclus_cluster* h_out, uint64_t out_capacity, tpcclus_run_stats* stats);

/* A whole time frame from HOST memory, fragment by fragment ("streamed through device
 * memory", BASELINE.json:configs[3]): the host->device copy of fragment k+1
 * and the device->host copy of fragment k-1 overlap the kernels of fragment k (two staging
 * slots, three streams).  Fragment f writes its records to h_out + sum of the counts of the
 * fragments before it (D10: a TF's list is the concatenation of its fragments' lists);
 * stats[f] reports fragment f.  Returns the first non-OK fragment status, else OK.
 * h_out has out_capacity records in total. */
int tpcclus_run_tf_host(tpcclus_ctx* ctx, const tpcclus_fragment* frags, uint32_t n_frags,
                        tpcclus_cluster* h_out, uint64_t out_capacity,
                        tpcclus_run_stats* stats /* HOST [n_frags] */);

/* ---- quality selection (D13; "appropriate selections and parameters") --------
 * tpcclus_run rejects nothing: one record per peak (D10).  tpcclus_select is a separate, order-preserving pass over
 * a finished list.  A record is KEPT iff  qtot >= min_qtot  and  qmax_q16 >= min_qmax_q16  and
 * ncells >= min_ncells  and  (flags & reject_flags) == 0  and not (reject_single_pad and sigma_pad == 0: all of the
 * cluster's weight in one pad column)  and not (reject_single_time and sigma_time == 0). */
typedef struct {
  float    min_qtot;                /* ADC; 0 keeps all                                        */
  uint16_t min_qmax_q16;            /* 1/16 ADC                                                */
  uint16_t min_ncells;
  uint8_t  reject_flags;            /* TPCCLUS_FLAG_* bits that disqualify a cluster           */
  uint8_t  reject_single_pad;       /* 0 / 1                                                   */
  uint8_t  reject_single_time;      /* 0 / 1                                                   */
  uint8_t  reserved_;               /* must be 0                                               */
} tpcclus_cuts;

/* Enqueue the selection on `cuda_stream`: the kept records of d_in[0..n) go to d_out in the same order.
 *   d_in, d_out  DEVICE, 16-byte aligned, must not overlap; d_out holds out_capacity records.  When both are 32-byte
 *                aligned (any cudaMalloc'd buffer) a record moves as one 256-bit load and one 256-bit store, which is
 *                ~8 % faster than the two 16-byte halves used otherwise; the output is the same.
 *   n            < 2^32.
 * Asynchronous; tpcclus_select_result waits for it and returns the number of records kept (the number REQUIRED:
 * when it exceeds out_capacity the first out_capacity kept records are in d_out and the status is
 * TPCCLUS_ERR_CAPACITY).  One selection in flight per context; it uses scratch of its own (allocated on the first
 * call and whenever n grows — the only allocation outside tpcclus_create), so it may overlap the context's runs.
 * Errors: ERR_INVALID, ERR_NOMEM, ERR_CUDA. */
int tpcclus_select(tpcclus_ctx* ctx, const tpcclus_cluster* d_in, uint64_t n, const tpcclus_cuts* cuts,
                   tpcclus_cluster* d_out, uint64_t out_capacity, void* cuda_stream);
int tpcclus_select_result(tpcclus_ctx* ctx, uint64_t* n_kept /* HOST out */);

/* The same selection (D13) for callers that cannot allocate: code under CUDA graph capture, tight serving loops,
 * harnesses that forbid cudaMalloc.  It needs no context and calls no cudaMalloc / cudaFree / cudaMallocHost / event or
 * stream creation: the look-back words and the tile ticket that tpcclus_select keeps in allocated scratch live in ONE
 * fixed `static __device__` array inside the library (8 bytes per 1024 records + 256 bytes = 128.25 KB; every GPU that
 * loads the library holds it until the process exits).  Runs on the CURRENT device, on `cuda_stream`.
 *   d_in, d_out   DEVICE, 16-byte aligned, must not overlap; d_out holds out_capacity records.
 *   n             <= TPCCLUS_SELECT_STATIC_MAX_RECORDS, else TPCCLUS_ERR_TOO_LARGE (nothing enqueued).
 *   d_n_kept      DEVICE, 8-byte aligned, caller-owned: receives the number of records kept (the number REQUIRED: when it
 *                 exceeds out_capacity the first out_capacity kept records are in d_out); written in stream order,
 *                 also for n = 0.  The caller reads it back its own way (this call never synchronises).
 * Asynchronous: enqueues two memset nodes (the part of the array this call uses starts at zero; d_n_kept) and one
 * kernel, all capturable.  The first call on a device also looks the array's device address up
 * (cudaGetSymbolAddress, once per device): make one call — n = 0 will do — before starting a capture.
 * EVERY call on a device shares the array: two calls that overlap on the GPU (different streams without an
 * ordering between them, or concurrent branches of one graph) race on it and give undefined output; calls ordered
 * on one stream, or by events, are fine.  Output is byte-identical to tpcclus_select's.
 * Errors: ERR_INVALID (null / misaligned pointers, NaN threshold, reserved_ != 0), ERR_TOO_LARGE, ERR_CUDA. */
#define TPCCLUS_SELECT_STATIC_MAX_RECORDS 16777216ull   /* 2^24 records = 512 MB of cluster list */
int tpcclus_select_static(const tpcclus_cluster* d_in, uint64_t n, const tpcclus_cuts* cuts,
                          tpcclus_cluster* d_out, uint64_t out_capacity, uint64_t* d_n_kept /* DEVICE out */,
                          void* cuda_stream);

/* Per-kernel device timing (for the roofline figures of bench.py): while on, every run is
 * bracketed with CUDA events on ITS stream around k_init (S0), k_bin (S1 routing) and k_tile
 * (S1 fill .. S7); tpcclus_result adds the elapsed times up.  set_profiling(1) resets the sums. */
#define TPCCLUS_N_KERNELS 3
int tpcclus_set_profiling(tpcclus_ctx* ctx, int on);
int tpcclus_get_profile(const tpcclus_ctx* ctx, double kernel_ms[TPCCLUS_N_KERNELS] /* HOST out */, uint64_t* n_runs /* HOST out */);

/* Number of kernel launches this context has issued so far (for bench.py's gpu_launches). */
uint64_t tpcclus_launch_count(const tpcclus_ctx* ctx);

/* Bytes of device memory the context owns (digit bins + scratch + host-staging buffers). */
uint64_t tpcclus_device_bytes(const tpcclus_ctx* ctx);

/* Free everything.  NULL is allowed. */
void tpcclus_destroy(tpcclus_ctx* ctx);

/* Static string for a status code. */
const char* tpcclus_strerror(int code);

#ifdef __cplusplus
}
#endif
#endif /* TPCCLUS_H */
