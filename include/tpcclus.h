/*
 * tpcclus.h -- C ABI of libtpcclus.so, the B200-native (sm_100a) TPC clusterizer.
 *
 * The hot path behind this boundary is the one BASELINE.json north_star (NS) names, the
 * data-parallel front of the TPC online processing of arxiv/paper_2511_17018 (PAPER.md
 * lines 8 and 18: ">95 %" of the online workload, "highly parallelizable"):
 *
 *   zero-suppressed digits -> pad x time charge map -> 3x3 peaks above threshold ->
 *   peak noise suppression -> 5x5 centre-of-gravity clusters -> compaction -> sort.
 *
 * The paper never spells the algorithm out; every rule is fixed in SURVEY.md 8(c),
 * steps O0..O5 and readings Q1..Q23 (restated in DESIGN.md).  The paper contributes the
 * run modes: the deterministic mode (PAPER.md 24-50, section 2), run-time compilation
 * with constants baked in (PAPER.md 87-93, section 5) and constant-memory parameters
 * that may change between time frames (PAPER.md 79-85, section 4.1).
 *
 * Plain C: no exception crosses this boundary, no torch / C++ type appears in it.
 * Every pointer is marked HOST or DEVICE.  All device memory (digits, clusters,
 * counters, workspace) is owned by the caller; the handle owns host state, the
 * uploaded parameters and, for RTC handles, the NVRTC-built module.
 */
#ifndef TPCCLUS_H
#define TPCCLUS_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define TPCCLUS_API __attribute__((visibility("default")))

typedef struct tpcclus_handle tpcclus_handle; /* opaque, owned by the library */

/* Zero-suppressed digit, 8 bytes, little-endian, one 64-bit load.
 * charge: ADC, 10 bit; > 1023 is clamped to 1023, 0 is ignored (Q4).
 * Out-of-range sector/row/pad/time: the digit is ignored and BAD_DIGITS is raised (Q4).
 * Two digits on one cell: the larger charge wins in DETERMINISTIC mode; in FAST mode
 * either may win (Q5).  The digit array may be in ANY order (NS (5)). */
typedef struct {
  uint16_t charge;
  uint16_t time;   /* 0 .. n_time-1        */
  uint8_t pad;     /* 0 .. n_pads[row]-1   */
  uint8_t row;     /* 0 .. n_rows-1        */
  uint8_t sector;  /* 0 .. n_sectors-1     */
  uint8_t reserved; /* ignored on input    */
} tpcclus_digit;

/* Cluster, 32 bytes (fields per O3/O4).  Cell (p,t) has its centre at the
 * integer (p,t); means and sigmas are in bins (Q11, Q13). */
typedef struct {
  float pad_mean;    /* p_c + Sp/Q                      */
  float time_mean;   /* t_c + St/Q                      */
  float sigma_pad;   /* sqrt(Q*Spp - Sp^2)/Q            */
  float sigma_time;  /* sqrt(Q*Stt - St^2)/Q            */
  uint32_t q_tot;    /* Q: sum over the clipped 5x5     */
  uint16_t q_max;    /* charge of the peak cell         */
  uint16_t time_peak;
  uint8_t pad_peak, row, sector;
  uint8_t flags;     /* TPCCLUS_FLAG_*                  */
  uint32_t reserved; /* always 0; part of the byte compare */
} tpcclus_cluster;

enum {
  TPCCLUS_FLAG_EDGE_PAD = 1,  /* p_c < 2 or p_c + 2 >= n_pads[row] */
  TPCCLUS_FLAG_EDGE_TIME = 2, /* t_c < 2 or t_c + 2 >= n_time      */
  TPCCLUS_FLAG_SATURATED = 4  /* q_max == 1023                     */
};

/* run modes (NS (5); PAPER.md 28-50) */
enum {
  TPCCLUS_MODE_FAST = 0,          /* cluster order unspecified; every field as in DETERMINISTIC */
  TPCCLUS_MODE_DETERMINISTIC = 1  /* ascending (sector,row,time_peak,pad_peak); bitwise equal to
                                     the host oracle, invariant under input permutation and
                                     across runs (PAPER.md 26-28, 36, 47-48) */
};

/* create flags */
enum {
  TPCCLUS_RTC = 1, /* build the kernels with NVRTC at create(), geometry and thresholds baked
                      in as literals (PAPER.md 89-93); without it the offline-compiled kernels
                      read them from __constant__ memory (PAPER.md 79-85) */
  TPCCLUS_COG_GATED = 2, /* reading Q10' of the centre of gravity: a cell of
                           the outer ring of the 5x5 window counts only if the inner cell between
                           it and the peak is non-empty.  Default off (Q10: every cell, weight 1) */
  TPCCLUS_COG_SHARED = 4 /* reading Q10'' (second half; R8): a cell that lies in
                            the 5x5 windows of a cluster and of its partners -- the surviving peaks at Chebyshev
                            distance 2 -- is split between them with the integer weights (q_peak >> 2 d) + 1,
                            d = distance of the cell from that peak; peak cells are never split.  Exclusive with
                            TPCCLUS_COG_GATED (create returns TPCCLUS_ERR_INVALID_ARG for both).  Default off */
};

/* data-dependent conditions, OR-ed into *status on the device (never return codes) */
enum {
  TPCCLUS_STATUS_OVERFLOW = 1,  /* more clusters than out->capacity; *n_clusters is still the
                                   true total, the buffer holds `capacity` valid records (FAST:
                                   any subset; DETERMINISTIC: the first `capacity` in order) */
  TPCCLUS_STATUS_BAD_DIGITS = 2, /* at least one digit was out of range and ignored */
  TPCCLUS_STATUS_NO_PACKED = 4,  /* tpcclus_run_packed only: the frame has more clusters than the run
                                    buffer holds (max_digits / 8); nothing was written but *n_clusters */
  TPCCLUS_STATUS_INTERNAL = 0x80000000u /* a workspace capacity the library derived from max_digits was
                                    exceeded on the device (a partition slice or the tile-record blob).
                                    Cannot happen for n <= max_digits -- it would be a bug of the library;
                                    digits were dropped and the output is invalid.  Provoked on purpose
                                    only through tpcclus_debug_shrink (tests) */
};

/* return codes */
enum {
  TPCCLUS_OK = 0,
  TPCCLUS_ERR_INVALID_ARG = -1,
  TPCCLUS_ERR_CUDA = -2,
  TPCCLUS_ERR_NVRTC = -3,
  TPCCLUS_ERR_WORKSPACE_TOO_SMALL = -4,
  TPCCLUS_ERR_UNSUPPORTED_GEOMETRY = -5 /* more than 56064 coarse bins n_sectors*n_rows*ceil(n_time/16256): the
                                           directory kernels keep a counter per bin in shared memory.  (The first
                                           partition pass has stages for 5503 bins; beyond that it runs once per
                                           5503 bins, each time over the whole input: tpcclus_launches_per_run.) */
};

typedef struct {
  uint32_t struct_size;   /* = sizeof(tpcclus_params), for versioning                        */
  uint32_t n_sectors;     /* 1..256                                                          */
  uint32_t n_rows;        /* 1..256                                                          */
  uint32_t n_time;        /* 1..65536 time bins per time frame (PAPER.md 12: 32 orbits)      */
  const uint16_t* n_pads; /* HOST, n_rows entries, each 1..256; copied by create             */
  uint16_t thr_peak;      /* peak threshold, test is q >= thr_peak (Q6); default 6           */
  uint16_t noise_eps;     /* ridge tolerance of the suppression (O2, Q9); default 4          */
  uint64_t max_digits;    /* sizing only: largest n that run() will be given                 */
  uint32_t flags;         /* TPCCLUS_RTC | TPCCLUS_COG_GATED | TPCCLUS_COG_SHARED            */
  int32_t device;         /* CUDA ordinal                                                    */
  void* workspace;        /* DEVICE, caller-owned, 256-byte aligned, lives as long as the handle */
  uint64_t workspace_bytes; /* >= tpcclus_workspace_bytes(params)                            */
} tpcclus_params;

typedef struct {
  tpcclus_cluster* clusters; /* DEVICE, caller-owned, 16-byte aligned                        */
  uint64_t capacity;         /* in clusters                                                  */
  uint64_t* n_clusters;      /* DEVICE, caller-owned: true count, also on overflow           */
  uint32_t* status;          /* DEVICE, TPCCLUS_STATUS_* bits; may be NULL                   */
} tpcclus_out;

/* Packed native output: 16 bytes per cluster in fixed point, grouped by
 * pad row, with an index of where each (sector,row) starts -- the form the steps after the
 * clusterizer consume (PAPER.md 107 names them: coordinate transformation, error estimation).
 * Sector and row are not stored per cluster: they follow from the index.  The record is a pure
 * function (O6) of the 32-byte DETERMINISTIC record:
 *   time_fix  = rn(time_mean  * 256)    24 bit     pad_fix       = min(rn(pad_mean * 256), 65535)
 *   sigma_*_fix = rn(sigma_* * 16384)   16 bit     rn = float32 -> integer, round to nearest even
 * (the multiplications by a power of two are exact), so it is bitwise reproducible as well. */
typedef struct {
  uint32_t time_fix_pad_peak;  /* time_fix[0:24) | pad_peak[24:32)                            */
  uint16_t pad_fix;
  uint16_t time_peak;
  uint16_t q_tot;              /* <= 25575                                                    */
  uint16_t q_max_flags;        /* q_max[0:10) | flags[10:13)                                  */
  uint16_t sigma_pad_fix;
  uint16_t sigma_time_fix;
} tpcclus_cluster16;

typedef struct {
  tpcclus_cluster16* clusters; /* DEVICE, caller-owned, 16-byte aligned                       */
  uint64_t capacity;           /* in clusters                                                 */
  uint64_t* n_clusters;        /* DEVICE: true count, also on overflow                        */
  uint32_t* status;            /* DEVICE, TPCCLUS_STATUS_* bits; may be NULL                  */
  uint64_t* row_index;         /* DEVICE, n_sectors * n_rows + 1 entries: clusters of (s, r) are
                                  [row_index[s * n_rows + r], row_index[s * n_rows + r + 1])  */
} tpcclus_out_packed;

/* Bytes of device workspace a handle with these parameters needs (depends on the geometry
 * and max_digits only).  Returns 0 for invalid or unsupported parameters.  Host call. */
TPCCLUS_API uint64_t tpcclus_workspace_bytes(const tpcclus_params* params);

/* Validates, copies the geometry, lays out the workspace and brings the device code in (PAPER.md
 * section 3, line 64): the kernels are built as separate compilation units, one GPU binary per kernel
 * family, embedded in the library; create loads the units this handle can launch with the driver's
 * module loader.  Each unit has its own __constant__ parameter block (PAPER.md 81); the handle
 * registers every block it finds and fills all of them with the parameters (PAPER.md 83-85).  With
 * TPCCLUS_RTC the units are compiled here for sm_100a by NVRTC instead, in parallel, with every
 * parameter a literal, and loaded through the same loader (PAPER.md 89-93).
 * Host call, synchronous.  *out is NULL on failure.  Modules and constant blocks are per handle:
 * handles of any parameters may run concurrently on different streams. */
TPCCLUS_API int tpcclus_create(const tpcclus_params* params, tpcclus_handle** out);

/* Clusterizes one time frame: enqueues every step of the path (NS (1)..(5)) on
 * `cuda_stream` (a cudaStream_t; NULL = legacy default stream) and returns without
 * synchronising.  d_digits: DEVICE, 16-byte aligned, n <= max_digits records, any order,
 * not modified.  out: HOST struct of DEVICE pointers.  The result depends only on
 * (params, digit multiset, mode), never on earlier runs (Q17).  One run at a time per
 * handle (the workspace is per handle).  The caller synchronises the stream before
 * reading *n_clusters / *status / clusters.  Only kernel launches are enqueued -- nothing is
 * allocated, nothing synchronises, no device result is read on the host -- so the call may be
 * captured into a CUDA graph (with per-kernel timing off) and replayed with new digits in the
 * same buffers: n is frozen in the graph, pad a shorter frame with all-zero digits. */
TPCCLUS_API int tpcclus_run(tpcclus_handle* h, const tpcclus_digit* d_digits, uint64_t n,
                            const tpcclus_out* out, int mode, void* cuda_stream);

/* Same as run() but every pointer in `digits`/`out` is HOST memory (pinned or pageable):
 * copies the digits to a staging area inside the workspace, runs, copies n_clusters,
 * status and min(n_clusters, capacity) clusters back, and synchronises the stream.  The
 * workspace must have been sized with tpcclus_workspace_bytes_host().  This is the
 * end-to-end entry bench.py times (e2e). */
TPCCLUS_API uint64_t tpcclus_workspace_bytes_host(const tpcclus_params* params, uint64_t cluster_capacity);
TPCCLUS_API int tpcclus_run_host(tpcclus_handle* h, const tpcclus_digit* h_digits, uint64_t n,
                                 tpcclus_cluster* h_clusters, uint64_t capacity,
                                 uint64_t* h_n_clusters, uint32_t* h_status, int mode,
                                 void* cuda_stream);

/* The same end-to-end path for a STREAM of time frames, two in flight (PAPER.md 97: one process per GPU
 * takes whole time frames one after the other): submit() enqueues the host-to-device copy of a frame into
 * one of two staging slots on a copy stream of the handle, the run behind it on a second stream and the
 * read-back of the 16-byte result on a third, and returns without waiting; wait() blocks until the OLDEST
 * submitted frame is done, stores its count and status and copies min(n_clusters, capacity) clusters into
 * the h_clusters given at submit.  The copy of frame k+1 thus overlaps the clustering and the read-back of
 * frame k (full-duplex link).  At most two submits may be outstanding (a third returns
 * TPCCLUS_ERR_INVALID_ARG); h_digits and h_clusters (HOST, pinned for overlap) must stay valid until the
 * matching wait() returns; `capacity` must be the same for the frames in flight.  The workspace must have
 * been sized with tpcclus_workspace_bytes_host_pipelined().  Not to be mixed with tpcclus_run* on other
 * streams while frames are in flight (one workspace per handle). */
TPCCLUS_API uint64_t tpcclus_workspace_bytes_host_pipelined(const tpcclus_params* params, uint64_t cluster_capacity);
TPCCLUS_API int tpcclus_host_submit(tpcclus_handle* h, const tpcclus_digit* h_digits, uint64_t n,
                                    tpcclus_cluster* h_clusters, uint64_t capacity, int mode);
TPCCLUS_API int tpcclus_host_wait(tpcclus_handle* h, uint64_t* h_n_clusters, uint32_t* h_status);

TPCCLUS_API int tpcclus_destroy(tpcclus_handle* h);

/* The constant buffers may change between time frames (PAPER.md 79, 85): sets new thresholds and
 * rewrites EVERY registered constant block of the handle (one per loaded unit), stream-ordered on
 * `cuda_stream` -- runs enqueued on that stream before the call keep the old values, runs after it see
 * the new ones.  thr_peak 1..1023, noise_eps 0..1023.  Refused (TPCCLUS_ERR_INVALID_ARG) for RTC
 * handles, whose parameters are compiled in. */
TPCCLUS_API int tpcclus_update_params(tpcclus_handle* h, uint16_t thr_peak, uint16_t noise_eps, void* cuda_stream);

/* Static string for a return code.  Never NULL. */
TPCCLUS_API const char* tpcclus_error_string(int code);

/* Detail of the last failure on this handle (NVRTC log, CUDA error string); "" if none.
 * Valid until the next call on the handle.  h may be NULL: then the detail of the last
 * failed create() on this thread. */
TPCCLUS_API const char* tpcclus_last_error(const tpcclus_handle* h);

/* ---- introspection used by bench.py / tests (no effect on results) -------------------- */

/* Number of kernels one run() launches in `mode` (bench.py's gpu_launches). */
TPCCLUS_API int tpcclus_launches_per_run(const tpcclus_handle* h, int mode);

/* Per-kernel device times of the LAST run() on this handle, when timing was enabled with
 * tpcclus_set_timing(h, 1): fills up to `cap` entries (name pointers are static strings,
 * ms from CUDA events recorded on the run's stream) and returns the number of kernels.
 * Synchronises on the recorded events. */
TPCCLUS_API int tpcclus_set_timing(tpcclus_handle* h, int enable);
TPCCLUS_API int tpcclus_last_timing(tpcclus_handle* h, const char** names, float* ms, int cap);

/* RTC build time in milliseconds (0 for non-RTC handles). */
TPCCLUS_API double tpcclus_rtc_build_ms(const tpcclus_handle* h);

/* On-disk cache of run-time-compiled kernels (section 5.1: processes of one node
 * share one compilation, serialised by a file lock).  dir: HOST string, copied; NULL or "" turns
 * the cache off again; if never called, $TPCCLUS_RTC_CACHE is used when set.  Process-wide, applies to
 * handles created afterwards.  The key covers every baked parameter, the kernel text and the NVRTC
 * version.  I/O errors are not errors: the handle is then compiled without caching. */
TPCCLUS_API int tpcclus_set_rtc_cache_dir(const char* dir);
/* 1 if this RTC handle's cubin came from the cache, else 0. */
TPCCLUS_API int tpcclus_rtc_cache_hit(const tpcclus_handle* h);

/* Same path as tpcclus_run in DETERMINISTIC mode (order, tie-breaks, arithmetic), output in the
 * packed form above.  Clusters are in (sector,row,time_peak,pad_peak) order; on OVERFLOW the first
 * `capacity` are kept and row_index still refers to the full list.  Needs the run buffer
 * (clusters <= max_digits / 8, true for every frame but adversarial ones): otherwise
 * TPCCLUS_STATUS_NO_PACKED is set and only *n_clusters is valid.  Enqueues only, like tpcclus_run. */
TPCCLUS_API int tpcclus_run_packed(tpcclus_handle* h, const tpcclus_digit* d_digits, uint64_t n,
                                   const tpcclus_out_packed* out, void* cuda_stream);

/* The same packed form for a cluster list that is already on the device, WITHOUT a handle, a workspace or any
 * allocation: for callers that cannot call cudaMalloc (code under CUDA graph capture, tight serving loops,
 * harnesses that forbid it).  d_clusters: the n clusters tpcclus_run wrote in DETERMINISTIC mode, i.e. ordered by
 * (sector, row, time_peak, pad_peak) (DEVICE, 16-byte aligned); d_packed: room for n records (DEVICE, 16-byte
 * aligned); d_row_index: n_sectors * n_rows + 1 entries as in tpcclus_out_packed (DEVICE).  Byte for byte what
 * tpcclus_run_packed delivers for the same frame (a cluster whose sector or row lies outside the geometry given
 * here is packed but not indexed).  Enqueues one memset and two kernels on cuda_stream and returns; the device
 * that owns the buffers must be current.
 * The only scratch memory -- one 32-bit counter per (sector, row) -- is a file-scope array in device memory,
 * TPCCLUS_NOALLOC_SCRATCH_BYTES that every GPU that loads the library holds until the process ends; hence the
 * limits n_sectors * n_rows <= TPCCLUS_NOALLOC_MAX_ROWS and n <= TPCCLUS_NOALLOC_MAX_CLUSTERS: beyond them the
 * call returns TPCCLUS_ERR_INVALID_ARG and says which limit in `err` (optional, NUL-terminated, at most err_cap
 * bytes).  The array is shared by every call and keeps the last call's contents: each call clears the counters
 * it uses first, on its stream.  Calls that overlap on the GPU (two streams) RACE on it: serialise them.  The
 * first call on a device looks the array's address up (cudaGetSymbolAddress; no allocation): make it once
 * before a stream capture begins.  Calls no cudaMalloc, cudaFree or allocating library routine. */
#define TPCCLUS_NOALLOC_MAX_ROWS 65536u             /* (sector, row) pairs: 256 x 256 */
#define TPCCLUS_NOALLOC_MAX_CLUSTERS 0xFFFFFFFFull   /* 32-bit counters */
#define TPCCLUS_NOALLOC_SCRATCH_BYTES ((TPCCLUS_NOALLOC_MAX_ROWS + 64u) * 4u)   /* 256.25 KB */
TPCCLUS_API int tpcclus_pack_noalloc(const tpcclus_cluster* d_clusters, uint64_t n, uint32_t n_sectors, uint32_t n_rows,
                                     tpcclus_cluster16* d_packed, uint64_t* d_row_index, void* cuda_stream,
                                     char* err, uint32_t err_cap);

/* Number of constant blocks in the handle's registry (= loaded offline-compiled units; 0 for RTC
 * handles), and the names of the loaded compilation units (static strings; returns the count). */
TPCCLUS_API int tpcclus_constant_buffers(const tpcclus_handle* h);
TPCCLUS_API int tpcclus_loaded_units(const tpcclus_handle* h, const char** names, int cap);

/* Test hook: makes later runs pretend the partition slice (chunks per CTA) and the tile-record blob
 * (records) are smaller than laid out (0 = as laid out), so that TPCCLUS_STATUS_INTERNAL can be seen. */
TPCCLUS_API int tpcclus_debug_shrink(tpcclus_handle* h, uint32_t slice_cap, uint64_t blob_cap);

/* Debug/parity hook for step a1 (the charge map): after a run(), rebuilds the dense
 * [sector][row][time][pad] uint16 map (O0) from the binned digits into d_map (DEVICE,
 * n_sectors * n_time * sum(n_pads) entries).  Not on the hot path. */
TPCCLUS_API int tpcclus_debug_dense_map(tpcclus_handle* h, uint16_t* d_map, void* cuda_stream);

/* Debug / test hook: 1 if the last DETERMINISTIC run had more clusters than its temporary run
 * buffer holds (max_digits / 8) and therefore took the chained-scan fallback, 0 if not, negative
 * on error.  Synchronises the device.  Results are identical either way. */
TPCCLUS_API int tpcclus_debug_det_fallback(tpcclus_handle* h);

#ifdef __cplusplus
}
#endif
#endif /* TPCCLUS_H */
