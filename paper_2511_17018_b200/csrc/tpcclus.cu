// tpcclus.cu -- host side of libtpcclus.so: the C ABI of include/tpcclus.h.
//
// Orchestration only: parameter validation, workspace layout, the launch sequence of
// tpcclus_kernels.cuh, the module loader and the constant-buffer registry.  No step of the path
// runs on the host; without a CUDA device every entry point that would compute returns
// TPCCLUS_ERR_CUDA.
//
// How the device code gets here (section 3, lines 52-66, and section 5, lines 87-93):
//   * The kernel text is cut into COMPILATION UNITS, one per kernel family (TPC_U_* in the .cuh).
//     The build compiles each unit on its own, straight to a GPU binary (nvcc -cubin), and embeds
//     the binaries in this library; a handle loads them with cuModuleLoadData (PAPER.md 64).
//   * create(TPCCLUS_RTC) compiles the same units with NVRTC instead, every parameter a literal
//     (PAPER.md 89-93), and loads them through the very same loader (PAPER.md 91).
//   * Every offline-compiled unit carries its own copy of the __constant__ parameter block -- a
//     non-RDC unit cannot see another unit's symbol (PAPER.md 81).  The handle's registry looks the
//     symbol up in every module it loads, fills all copies at create and rewrites all of them when
//     the parameters change (tpcclus_update_params; PAPER.md 83-85).  Modules are per handle, so
//     handles with different parameters never share a constant block: any two handles may run
//     concurrently on different streams.
#include <cuda_runtime.h>
#include <dlfcn.h>
#include <fcntl.h>
#include <sys/file.h>
#include <unistd.h>

#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <mutex>
#include <string>
#include <thread>
#include <vector>

#include "../../include/tpcclus.h"
#define TPC_UNITS 0u   // declarations only: the kernels live in the embedded unit binaries
#include "tpcclus_kernels.cuh"

extern "C" const char tpcclus_kernel_source[];   // the kernel text, embedded at build time (PAPER.md 91)

// the unit binaries, embedded at build time (build/tpcclus_units.S: .incbin of build/unit_<name>.cubin)
// X(name, TPC_U_* bit, time halo the unit is compiled with): the units of reading Q10'' -- its tile kernels and
// the partition and debug units that feed them -- are built with TPC_HALO = 5 (paper_2511_17018_b200/build.py: UNITS)
#define TPC_UNIT_LIST(X)                                                                              \
  X(part_coarse, TPC_U_PART_COARSE, 3) X(dir, TPC_U_DIR, 3) X(part_fine, TPC_U_PART_FINE, 3)          \
  X(tiles_fast, TPC_U_TILES_FAST, 3) X(tiles_det, TPC_U_TILES_DET, 3) X(order, TPC_U_ORDER, 3)        \
  X(tiles_dump, TPC_U_TILES_DUMP, 3) X(tiles_fast_g, TPC_U_TILES_FAST_G, 3) X(tiles_det_g, TPC_U_TILES_DET_G, 3) \
  X(part_coarse_h5, TPC_U_PART_COARSE, 5) X(part_fine_h5, TPC_U_PART_FINE, 5) X(tiles_dump_h5, TPC_U_TILES_DUMP, 5) \
  X(tiles_fast_s, TPC_U_TILES_FAST_S, 5) X(tiles_det_s, TPC_U_TILES_DET_S, 5)
#define X(name, bit, halo) extern "C" const unsigned char tpcclus_cubin_##name[]; extern "C" const unsigned char tpcclus_cubin_##name##_end[];
TPC_UNIT_LIST(X)
#undef X

namespace {

constexpr uint32_t kMaxSmem = 232448;  // 227 KB: K1 needs 40 B per coarse bin + 12.8 KB (5472 bins at the full geometry)
constexpr int kMaxKernels = 12;

thread_local std::string g_create_error;

inline uint64_t align_up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

struct Layout {   // byte offsets into the workspace
  uint64_t counters, counters_bytes;   // zeroed at the head of every run
  uint64_t status, blob_cursor, slice_cnt;
  uint64_t used, bin_chunk_start, batch_start, batch_bin, dir, chunk_list, pool, blob, idx;
  uint64_t ticket, temp_cursor, det_flag, tile_state, tile_base, tile_cnt, tile_local, block_sum, block_prefix, row_off;
  uint64_t total;        // device-path workspace
  uint64_t host_digits;  // staging of run_host (beyond `total`)
  uint64_t host_out;     // n_clusters (8) + status (4)
  uint64_t host_clusters;
  uint64_t host_slot;    // bytes of one staging slot without its clusters (digits + result); the pipelined entry has two slots
};

struct Geometry {
  TpcParams prm;
  uint32_t g1;           // K1 grid = number of SMs
  uint32_t slice_cap;    // chunks per K1 CTA
  uint32_t k1_passes;    // K1 launches per run: ceil(n_bins / 5503)
  uint32_t n_tiles, n_scan_blocks;
  uint64_t n_chunks_max, n_batches_max, blob_cap, idx_cap;
  uint64_t max_digits;
  Layout lay;
};

int sm_count(int device) {
  int n = 0;
  if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || n <= 0) {
    cudaGetLastError();
    n = 148;   // B200; keeps workspace_bytes() usable on a box without a GPU
  }
  return n;
}

// Validates `p` and derives everything that depends on geometry and max_digits.
int make_geometry(const tpcclus_params* p, Geometry* g) {
  if (!p || p->struct_size != sizeof(tpcclus_params) || !p->n_pads) return TPCCLUS_ERR_INVALID_ARG;
  if (p->n_sectors < 1 || p->n_sectors > 256 || p->n_rows < 1 || p->n_rows > 256 || p->n_time < 1 ||
      p->n_time > 65536 || p->thr_peak < 1 || p->thr_peak > 1023 || p->noise_eps > 1023 || p->max_digits < 1 ||
      p->max_digits > (1ull << 31))
    return TPCCLUS_ERR_INVALID_ARG;
  memset(g, 0, sizeof *g);
  TpcParams& q = g->prm;
  q.n_sectors = p->n_sectors; q.n_rows = p->n_rows; q.n_time = p->n_time;
  uint32_t maxp = 0;
  for (uint32_t r = 0; r < p->n_rows; ++r) {
    if (p->n_pads[r] < 1 || p->n_pads[r] > 256) return TPCCLUS_ERR_INVALID_ARG;
    q.n_pads[r] = p->n_pads[r];
    if (p->n_pads[r] > maxp) maxp = p->n_pads[r];
  }
  q.n_tc = (p->n_time + TPC_TC - 1) / TPC_TC;
  uint64_t nb = (uint64_t)p->n_sectors * p->n_rows * q.n_tc;
  // K2..K4 keep one 4-byte counter per bin in shared memory (k_dir_scan: + 8 KB static): 56064 bins at most.
  if (nb > (kMaxSmem - 8192u) / 4u) return TPCCLUS_ERR_UNSUPPORTED_GEOMETRY;
  q.n_bins = (uint32_t)nb;
  // K1 has stages for 5503 bins; a larger geometry is binned in several passes over the input (R1)
  uint32_t k1_max = (uint32_t)nb;
  while (tpc_k1_smem_bytes(k1_max) > kMaxSmem) --k1_max;
  g->k1_passes = (uint32_t)((nb + k1_max - 1) / k1_max);
  q.k1_bins = (uint32_t)((nb + g->k1_passes - 1) / g->k1_passes);
  uint32_t tmin = p->n_time < TPC_TC ? p->n_time : TPC_TC;
  q.n_sl = (tmin + TPC_TS - 1) / TPC_TS;
  q.max_pads = maxp;
  q.pitch = (maxp + 2 * TPC_PG + 7) / 8 * 8;
  q.thr_peak = p->thr_peak; q.noise_eps = p->noise_eps;
  if ((p->flags & TPCCLUS_COG_GATED) && (p->flags & TPCCLUS_COG_SHARED)) return TPCCLUS_ERR_INVALID_ARG;   // one reading per handle
  q.cog_mode = (p->flags & TPCCLUS_COG_SHARED) ? 2u : (p->flags & TPCCLUS_COG_GATED) ? 1u : 0u;
  const uint32_t tt = TPC_TS + 2 * (q.cog_mode == 2u ? 5u : 3u);   // tile rows: the units of Q10'' carry a time halo of 5
  q.max_peaks = ((tt - 2 + 1) / 2) * ((maxp + 1) / 2);   // no two peaks are 8-neighbours; rows 1..TT-2 are scanned

  g->max_digits = p->max_digits;
  g->g1 = (uint32_t)sm_count(p->device);
  const uint64_t round = (uint64_t)TPC_K1_THREADS * TPC_K1_DPT;
  uint64_t per_cta = align_up((p->max_digits + g->g1 - 1) / g->g1, round);
  uint64_t dup = q.n_tc > 1 ? 2 : 1;   // K1 copies a digit into the next time-chunk at most once
  uint64_t cap = (per_cta * dup + TPC_CHUNK - 1) / TPC_CHUNK + nb;   // full chunks + one partial per bin
  if (cap > 0x0FFFFFFFull) return TPCCLUS_ERR_INVALID_ARG;
  g->slice_cap = (uint32_t)cap;
  g->n_chunks_max = (uint64_t)g->g1 * cap;
  if (g->n_chunks_max > (1ull << 26)) return TPCCLUS_ERR_INVALID_ARG;   // chunk ids are 26 bits in the chunk lists (4.3e9 records)
  g->n_batches_max = g->n_chunks_max / TPC_CPB + nb + 1;
  // K5 writes every record once; per batch at most 3 zero records in front of each of its n_sl + 1
  // A runs (16-byte alignment) and 7 at its end (32-byte alignment)
  g->blob_cap = p->max_digits * dup + g->n_batches_max * (3ull * (q.n_sl + 1) + 8ull) + 64;
  g->idx_cap = g->n_batches_max * q.n_sl;
  g->n_tiles = q.n_bins * q.n_sl;
  g->n_scan_blocks = (g->n_tiles + TPC_SCAN_PER_CTA - 1) / TPC_SCAN_PER_CTA;

  Layout& L = g->lay;
  uint64_t o = 0;
  auto take = [&](uint64_t bytes) { uint64_t r = o; o = align_up(o + bytes, 256); return r; };
  L.counters = o;
  L.status = take(4);
  L.blob_cursor = take(8);
  L.ticket = take(4);
  L.temp_cursor = take(8);
  L.det_flag = take(4);
  L.tile_state = take(8ull * g->n_tiles);   // DET chained scan: must start at 0 every run
  L.bin_chunk_start = take(4ull * (nb + 1));   // K2 accumulates the per-bin chunk totals here, K3 scans them in place
  L.counters_bytes = o - L.counters;
  L.slice_cnt = take(4ull * align_up(nb, 4) * g->g1);   // row pitch: a multiple of 4 entries
  L.used = take(4ull * g->g1);
  L.batch_start = take(4ull * (nb + 1));
  L.batch_bin = take(4ull * g->n_batches_max);
  L.dir = take(4ull * g->n_chunks_max);
  L.chunk_list = take(4ull * g->n_chunks_max);
  L.pool = take(256ull * g->n_chunks_max);
  L.blob = take(4ull * g->blob_cap);
  L.idx = take(8ull * g->idx_cap);
  L.tile_base = take(8ull * g->n_tiles);
  L.tile_cnt = take(4ull * g->n_tiles);
  L.tile_local = take(4ull * g->n_tiles);
  L.block_sum = take(4ull * g->n_scan_blocks);
  L.block_prefix = take(8ull * g->n_scan_blocks);
  L.row_off = take(8ull * (p->n_rows + 1));
  L.total = o;
  L.host_digits = take(8ull * p->max_digits);
  L.host_out = take(16);
  L.host_clusters = o;
  L.host_slot = L.host_clusters - L.host_digits;
  return TPCCLUS_OK;
}

// ---- driver API (module loader) and NVRTC entry points, resolved once per process ---------------
struct Drv {
  void* lib = nullptr;
  int (*cuModuleLoadData)(void**, const void*) = nullptr;
  int (*cuModuleUnload)(void*) = nullptr;
  int (*cuModuleGetFunction)(void**, void*, const char*) = nullptr;
  int (*cuModuleGetGlobal_v2)(unsigned long long*, size_t*, void*, const char*) = nullptr;
  int (*cuFuncSetAttribute)(void*, int, int) = nullptr;
  int (*cuLaunchKernel)(void*, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, void*, void**, void**) = nullptr;
  int (*cuGetErrorString)(int, const char**) = nullptr;
  bool ok = false;
  std::string why;
};
struct Nvrtc {
  void* lib = nullptr;
  int (*nvrtcCreateProgram)(void**, const char*, const char*, int, const char* const*, const char* const*) = nullptr;
  int (*nvrtcCompileProgram)(void*, int, const char* const*) = nullptr;
  int (*nvrtcGetCUBINSize)(void*, size_t*) = nullptr;
  int (*nvrtcGetCUBIN)(void*, char*) = nullptr;
  int (*nvrtcGetProgramLogSize)(void*, size_t*) = nullptr;
  int (*nvrtcGetProgramLog)(void*, char*) = nullptr;
  int (*nvrtcDestroyProgram)(void**) = nullptr;
  int (*nvrtcVersion)(int*, int*) = nullptr;
  bool ok = false;
  std::string why;
};

#define SYM(r, f) do { *(void**)(&(r).f) = dlsym((r).lib, #f); if (!(r).f) { all = false; (r).why = "missing symbol " #f; } } while (0)
Drv& drv() {
  static Drv r;
  static std::once_flag once;
  std::call_once(once, [] {
    r.lib = dlopen("libcuda.so.1", RTLD_NOW | RTLD_GLOBAL);
    if (!r.lib) { r.why = "dlopen(libcuda.so.1) failed"; return; }
    bool all = true;
    SYM(r, cuModuleLoadData); SYM(r, cuModuleUnload); SYM(r, cuModuleGetFunction); SYM(r, cuModuleGetGlobal_v2);
    SYM(r, cuFuncSetAttribute); SYM(r, cuLaunchKernel); SYM(r, cuGetErrorString);
    r.ok = all;
  });
  return r;
}
Nvrtc& nvrtc() {
  static Nvrtc r;
  static std::once_flag once;
  std::call_once(once, [] {
    // the toolkit's own NVRTC first (12.9: knows the 256-bit vector store), then whatever the process has
    for (const char* name : {"/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/targets/x86_64-linux/lib/libnvrtc.so.12",
                             "libnvrtc.so.12", "libnvrtc.so"}) {
      r.lib = dlopen(name, RTLD_NOW);
      if (r.lib) break;
    }
    if (!r.lib) { r.why = "dlopen(libnvrtc) failed"; return; }
    bool all = true;
    SYM(r, nvrtcCreateProgram); SYM(r, nvrtcCompileProgram); SYM(r, nvrtcGetCUBINSize); SYM(r, nvrtcGetCUBIN);
    SYM(r, nvrtcGetProgramLogSize); SYM(r, nvrtcGetProgramLog); SYM(r, nvrtcDestroyProgram); SYM(r, nvrtcVersion);
    r.ok = all;
  });
  return r;
}
#undef SYM
std::string drv_error(int rc) {
  const char* s = nullptr;
  drv().cuGetErrorString(rc, &s);
  return s ? s : "?";
}

// ---- compilation units and kernels -------------------------------------------------------------
enum UnitId { U_PART_COARSE, U_DIR, U_PART_FINE, U_TILES_FAST, U_TILES_DET, U_ORDER, U_TILES_DUMP, U_TILES_FAST_G, U_TILES_DET_G,
              U_PART_COARSE_H5, U_PART_FINE_H5, U_TILES_DUMP_H5, U_TILES_FAST_S, U_TILES_DET_S, U_COUNT_ };
struct UnitInfo { const char* name; uint32_t bit; uint32_t halo; const unsigned char* cubin; const unsigned char* cubin_end; };
#define X(name, bit, halo) {#name, bit, halo, tpcclus_cubin_##name, tpcclus_cubin_##name##_end},
const UnitInfo kUnits[U_COUNT_] = {TPC_UNIT_LIST(X)};
#undef X

// The kernels a handle launches (one slot each) and the unit that provides the slot's kernel for each
// reading of the centre of gravity: {Q10, Q10' gated, Q10'' shared}.
enum KernelId { K_RESET, K_PUBLISH, K_PART_COARSE, K_DIR_COUNT, K_DIR_SCAN, K_DIR_FILL, K_PART_FINE, K_TILES_FAST, K_TILES_FAST_E, K_TILES_DET,
                K_TILES_DET_TEMP, K_TILES_DET_TEMP_E, K_TILES_DUMP, K_SCAN_LOCAL, K_SCAN_SUMS, K_EMIT_ORDERED, K_EMIT_PACKED, K_COUNT_ };
struct KernelInfo { const char* name[3]; UnitId unit[3]; int smem; };   // smem: 0 none/static, 1 K1, 2 one word per bin, 5 K5, 6 K6
#define SAME3(x) {x, x, x}
const KernelInfo kKernels[K_COUNT_] = {
    {SAME3("k_reset"), SAME3(U_DIR), 0}, {SAME3("k_publish"), SAME3(U_DIR), 0},
    {SAME3("k_partition_coarse"), {U_PART_COARSE, U_PART_COARSE, U_PART_COARSE_H5}, 1},
    {SAME3("k_dir_count"), SAME3(U_DIR), 2}, {SAME3("k_dir_scan"), SAME3(U_DIR), 2}, {SAME3("k_dir_fill"), SAME3(U_DIR), 2},
    {SAME3("k_partition_fine"), {U_PART_FINE, U_PART_FINE, U_PART_FINE_H5}, 5},
    {{"k_cluster_tiles_fast", "k_cluster_tiles_fast_gated", "k_cluster_tiles_fast_shared"}, {U_TILES_FAST, U_TILES_FAST_G, U_TILES_FAST_S}, 6},
    // the same with the emitter warp, for sparse frames (reading Q10'' has none: the plain kernel)
    {{"k_cluster_tiles_fast_e", "k_cluster_tiles_fast_gated_e", "k_cluster_tiles_fast_shared"}, {U_TILES_FAST, U_TILES_FAST_G, U_TILES_FAST_S}, 6},
    {{"k_cluster_tiles_det", "k_cluster_tiles_det_gated", "k_cluster_tiles_det_shared"}, {U_TILES_DET, U_TILES_DET_G, U_TILES_DET_S}, 6},
    {{"k_cluster_tiles_det_temp", "k_cluster_tiles_det_temp_gated", "k_cluster_tiles_det_temp_shared"}, {U_TILES_DET, U_TILES_DET_G, U_TILES_DET_S}, 6},
    {{"k_cluster_tiles_det_temp_e", "k_cluster_tiles_det_temp_gated_e", "k_cluster_tiles_det_temp_shared"}, {U_TILES_DET, U_TILES_DET_G, U_TILES_DET_S}, 6},
    {SAME3("k_cluster_tiles_dump_map"), {U_TILES_DUMP, U_TILES_DUMP, U_TILES_DUMP_H5}, 6},
    {SAME3("k_scan_local"), SAME3(U_ORDER), 0}, {SAME3("k_scan_sums"), SAME3(U_ORDER), 0},
    {SAME3("k_emit_ordered"), SAME3(U_ORDER), 0}, {SAME3("k_emit_packed"), SAME3(U_ORDER), 0}};
#undef SAME3

}  // namespace

struct tpcclus_handle {
  Geometry g;
  tpcclus_params params;   // copy; n_pads points into g.prm
  char* ws = nullptr;
  bool is_rtc = false;
  int cog = 0;                     // reading of the centre of gravity: 0 Q10, 1 Q10' gated, 2 Q10'' shared
  uint32_t halo = 3;               // time halo of the handle's units (5 under Q10'')
  void* module[U_COUNT_] = {};     // one loaded GPU binary per compilation unit (PAPER.md 64)
  bool unit_cached[U_COUNT_] = {};
  void* fn[K_COUNT_] = {};
  // constant-buffer registry (PAPER.md 81-85): the device address of every module's parameter block
  struct ConstSym { UnitId unit; void* dptr; size_t bytes; };
  std::vector<ConstSym> consts;
  double rtc_ms = 0.0;
  bool rtc_cache_hit = false;
  uint32_t smem_k1 = 0, smem_k5 = 0, smem_k6 = 0;
  uint32_t grid_k5 = 0, grid_k6 = 0;
  uint32_t dbg_slice_cap = 0;      // test hook: a smaller K1 slice (tpcclus_debug_shrink)
  uint64_t dbg_blob_cap = 0;
  bool timing = false;
  int n_timed = 0;
  const char* timed_name[kMaxKernels] = {};
  cudaEvent_t ev[kMaxKernels + 1] = {};
  std::string err;
  bool ran = false;
  // two-deep host pipeline (tpcclus_host_submit / tpcclus_host_wait)
  struct Pipe {
    bool ready = false;
    cudaStream_t in = nullptr, comp = nullptr, out = nullptr;
    cudaEvent_t h2d[2] = {}, done[2] = {};
    uint64_t seq_submit = 0, seq_wait = 0;
    struct { tpcclus_cluster* h_clusters; uint64_t capacity; } job[2] = {};
    struct Res { uint64_t n; uint64_t s; }* res = nullptr;   // mapped pinned memory, one per slot: written by k_publish
    Res* res_dev = nullptr;
  } pipe;
};

namespace {

int fail(tpcclus_handle* h, int code, const std::string& detail) {
  if (h) h->err = detail; else g_create_error = detail;
  return code;
}
#define CUDA_TRY(h, expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { cudaGetLastError(); \
  return fail(h, TPCCLUS_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_)); } } while (0)

// The entry points select the handle's device and put the caller's back on every way out.
struct DeviceGuard {
  int prev = -1;
  bool switched = false;
  cudaError_t enter(int device) {
    if (cudaGetDevice(&prev) != cudaSuccess) { cudaGetLastError(); prev = -1; }
    if (prev == device) return cudaSuccess;
    cudaError_t e = cudaSetDevice(device);
    switched = e == cudaSuccess;
    return e;
  }
  ~DeviceGuard() { if (switched && prev >= 0) cudaSetDevice(prev); }
};

// One launch through the driver's module loader path: offline-compiled unit or NVRTC unit alike.
int launch(tpcclus_handle* h, KernelId k, dim3 grid, dim3 block, uint32_t smem, cudaStream_t st, void** args) {
  if (!h->fn[k]) return fail(h, TPCCLUS_ERR_CUDA, std::string("kernel not loaded: ") + kKernels[k].name[h->cog]);
  if (h->timing && h->n_timed < kMaxKernels) {
    if (h->n_timed == 0) cudaEventRecord(h->ev[0], st);
    h->timed_name[h->n_timed] = kKernels[k].name[h->cog];
  }
  int rc = drv().cuLaunchKernel(h->fn[k], grid.x, grid.y, grid.z, block.x, block.y, block.z, smem, st, args, nullptr);
  if (rc != 0) return fail(h, TPCCLUS_ERR_CUDA, std::string("cuLaunchKernel(") + kKernels[k].name[h->cog] + "): " + drv_error(rc));
  if (h->timing && h->n_timed < kMaxKernels) { ++h->n_timed; cudaEventRecord(h->ev[h->n_timed], st); }
  return TPCCLUS_OK;
}

// Text put in front of the kernel source for NVRTC: every parameter as a literal, and the unit.
std::string rtc_prologue(const TpcParams& q, uint32_t unit_bit, uint32_t halo) {
  char buf[256];
  std::string s = "#define TPC_RTC 1\n";
  snprintf(buf, sizeof buf, "#define TPC_UNITS %uu\n#define TPC_HALO %uu\n", unit_bit, halo); s += buf;
#define DEF(f) do { snprintf(buf, sizeof buf, "#define TPC_" #f " %uu\n", q.f); s += buf; } while (0)
  DEF(n_sectors); DEF(n_rows); DEF(n_time); DEF(n_tc); DEF(n_bins); DEF(n_sl); DEF(pitch); DEF(max_pads);
  DEF(thr_peak); DEF(noise_eps); DEF(max_peaks); DEF(cog_mode); DEF(k1_bins);
#undef DEF
  s += "__constant__ unsigned short TPC_NPADS_TABLE[256] = {";   // constant bank like the generic build's table: no 64-bit address registers
  for (int r = 0; r < 256; ++r) { snprintf(buf, sizeof buf, "%u,", (unsigned)q.n_pads[r]); s += buf; }
  s += "};\n";
  return s;
}

// NVRTC: kernel text -> cubin for sm_100a.  Thread-safe (one program per call); errors in *err.
int compile_cubin(const std::string& src, std::vector<char>* cubin, std::string* err) {
  Nvrtc& r = nvrtc();
  void* prog = nullptr;
  if (r.nvrtcCreateProgram(&prog, src.c_str(), "tpcclus_kernels.cu", 0, nullptr, nullptr) != 0) { *err = "nvrtcCreateProgram failed"; return TPCCLUS_ERR_NVRTC; }
  const char* opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", "-default-device", "-lineinfo", "--fmad=false", "--prec-div=true",
                        "--prec-sqrt=true", "--ftz=false", "-DTPC_NO_ST256=1"};
  int rc = r.nvrtcCompileProgram(prog, 8, opts);
  if (rc != 0) {   // older NVRTC: retry without the 256-bit store
    r.nvrtcDestroyProgram(&prog);
    prog = nullptr;
    if (r.nvrtcCreateProgram(&prog, src.c_str(), "tpcclus_kernels.cu", 0, nullptr, nullptr) != 0) { *err = "nvrtcCreateProgram failed"; return TPCCLUS_ERR_NVRTC; }
    rc = r.nvrtcCompileProgram(prog, 9, opts);
  }
  if (rc != 0) {
    size_t n = 0; r.nvrtcGetProgramLogSize(prog, &n);
    std::string log(n, '\0'); if (n) r.nvrtcGetProgramLog(prog, &log[0]);
    r.nvrtcDestroyProgram(&prog);
    *err = "nvrtcCompileProgram failed:\n" + log;
    return TPCCLUS_ERR_NVRTC;
  }
  size_t n = 0; r.nvrtcGetCUBINSize(prog, &n);
  cubin->resize(n);
  r.nvrtcGetCUBIN(prog, cubin->data());
  r.nvrtcDestroyProgram(&prog);
  return TPCCLUS_OK;
}

// On-disk cubin cache (PAPER.md 97: several processes per node share one run-time compilation,
// serialised by a file lock).  Key = hash of the exact text handed to NVRTC (prologue with every
// baked parameter and the unit + kernel source) and of the NVRTC version.  The compile happens under
// an exclusive flock on <key>.lock; the file is written under a temporary name and renamed, so a
// reader sees a whole file or none.  File = 24-byte header (magic, payload length, FNV-1a of the
// payload) + cubin: a truncated, corrupt or foreign file is deleted and compiled afresh.  Any I/O
// problem just means "compile, do not cache".
std::mutex g_cache_mutex;
std::string g_cache_dir;   // set by tpcclus_set_rtc_cache_dir or $TPCCLUS_RTC_CACHE

uint64_t fnv1a(const char* p, size_t n, uint64_t h = 1469598103934665603ull) {
  for (size_t i = 0; i < n; ++i) { h ^= (unsigned char)p[i]; h *= 1099511628211ull; }
  return h;
}
constexpr uint64_t kCacheMagic = 0x31434250434c4354ull;   // "TCLCPBC1"

bool read_cached(const std::string& path, std::vector<char>* out) {
  FILE* f = fopen(path.c_str(), "rb");
  if (!f) return false;
  uint64_t hdr[3] = {0, 0, 0};
  bool ok = fread(hdr, 1, sizeof hdr, f) == sizeof hdr && hdr[0] == kCacheMagic && hdr[1] > 0 && hdr[1] < (1ull << 30);
  if (ok) {
    out->resize((size_t)hdr[1]);
    ok = fread(out->data(), 1, out->size(), f) == out->size() && fgetc(f) == EOF && fnv1a(out->data(), out->size()) == hdr[2];
  }
  fclose(f);
  if (!ok) { out->clear(); remove(path.c_str()); }   // not ours, cut short or damaged: compile afresh
  return ok;
}

int cubin_for(const std::string& src, std::vector<char>* cubin, bool* hit, std::string* err) {
  *hit = false;
  std::string dir;
  { std::lock_guard<std::mutex> lk(g_cache_mutex); dir = g_cache_dir; }
  if (dir.empty()) { const char* e = getenv("TPCCLUS_RTC_CACHE"); if (e) dir = e; }
  if (dir.empty()) return compile_cubin(src, cubin, err);
  int vmaj = 0, vmin = 0;
  if (nvrtc().nvrtcVersion) nvrtc().nvrtcVersion(&vmaj, &vmin);
  uint64_t hsh = fnv1a(src.data(), src.size());
  char tag[64]; snprintf(tag, sizeof tag, "|nvrtc %d.%d|sm_100a", vmaj, vmin);
  hsh = fnv1a(tag, strlen(tag), hsh);
  char name[64]; snprintf(name, sizeof name, "/tpcclus_%016llx", (unsigned long long)hsh);
  const std::string base = dir + name, file = base + ".cubin", lock = base + ".lock";
  if (read_cached(file, cubin)) { *hit = true; return TPCCLUS_OK; }
  int fd = open(lock.c_str(), O_CREAT | O_RDWR, 0644);
  if (fd >= 0) flock(fd, LOCK_EX);   // whoever comes second waits here, then finds the file
  int rc = TPCCLUS_OK;
  if (fd >= 0 && read_cached(file, cubin)) {
    *hit = true;
  } else {
    rc = compile_cubin(src, cubin, err);
    if (rc == TPCCLUS_OK && fd >= 0) {
      char tmp[64]; snprintf(tmp, sizeof tmp, ".tmp%d_%llx", (int)getpid(), (unsigned long long)(uintptr_t)cubin);
      FILE* f = fopen((file + tmp).c_str(), "wb");
      if (f) {
        const uint64_t hdr[3] = {kCacheMagic, (uint64_t)cubin->size(), fnv1a(cubin->data(), cubin->size())};
        bool ok = fwrite(hdr, 1, sizeof hdr, f) == sizeof hdr && fwrite(cubin->data(), 1, cubin->size(), f) == cubin->size();
        ok = fclose(f) == 0 && ok;
        if (ok) rename((file + tmp).c_str(), file.c_str()); else remove((file + tmp).c_str());
      }
    }
  }
  if (fd >= 0) { flock(fd, LOCK_UN); close(fd); }
  return rc;
}

// Loads one unit's GPU binary into the handle, resolves its kernels, sizes their dynamic shared
// memory and REGISTERS its constant block (PAPER.md 83: "automatically register all constant memory
// symbols"), filling it with the handle's parameters.
int load_unit(tpcclus_handle* h, UnitId u, const void* image) {
  Drv& d = drv();
  int rc = d.cuModuleLoadData(&h->module[u], image);
  if (rc != 0) return fail(nullptr, TPCCLUS_ERR_CUDA, std::string("cuModuleLoadData(") + kUnits[u].name + "): " + drv_error(rc));
  for (int k = 0; k < K_COUNT_; ++k) {
    if (kKernels[k].unit[h->cog] != u) continue;
    if ((rc = d.cuModuleGetFunction(&h->fn[k], h->module[u], kKernels[k].name[h->cog])) != 0)
      return fail(nullptr, TPCCLUS_ERR_CUDA, std::string("cuModuleGetFunction(") + kKernels[k].name[h->cog] + "): " + drv_error(rc));
    const uint32_t smem = kKernels[k].smem == 1 ? h->smem_k1 : kKernels[k].smem == 5 ? h->smem_k5 : kKernels[k].smem == 6 ? h->smem_k6 : kKernels[k].smem == 2 ? 4u * h->g.prm.n_bins : 0u;
    const int CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES = 8;
    if (smem > 48u * 1024u && (rc = d.cuFuncSetAttribute(h->fn[k], CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)smem)) != 0)
      return fail(nullptr, TPCCLUS_ERR_CUDA, std::string("cuFuncSetAttribute(") + kKernels[k].name[h->cog] + "): " + drv_error(rc));
  }
  unsigned long long dptr = 0; size_t bytes = 0;
  if (d.cuModuleGetGlobal_v2(&dptr, &bytes, h->module[u], "c_prm") == 0) {   // RTC units have literals instead: nothing to register
    if (bytes != sizeof(TpcParams)) return fail(nullptr, TPCCLUS_ERR_CUDA, std::string("constant block of unit ") + kUnits[u].name + " has the wrong size");
    h->consts.push_back({u, (void*)(uintptr_t)dptr, bytes});
    cudaError_t e = cudaMemcpy((void*)(uintptr_t)dptr, &h->g.prm, sizeof(TpcParams), cudaMemcpyHostToDevice);
    if (e != cudaSuccess) { cudaGetLastError(); return fail(nullptr, TPCCLUS_ERR_CUDA, std::string("constant upload: ") + cudaGetErrorString(e)); }
  }
  return TPCCLUS_OK;
}

// Brings the listed units into the handle: embedded binaries (generic) or NVRTC builds (RTC; the
// units compile in parallel threads -- PAPER.md 64: "the compilation can be parallelized").
int load_units(tpcclus_handle* h, const std::vector<UnitId>& want) {
  if (!drv().ok) return fail(nullptr, TPCCLUS_ERR_CUDA, "driver API unavailable: " + drv().why);
  std::vector<UnitId> units;
  for (UnitId u : want) if (!h->module[u]) units.push_back(u);
  if (units.empty()) return TPCCLUS_OK;
  if (cudaFree(nullptr) != cudaSuccess) { cudaGetLastError(); return fail(nullptr, TPCCLUS_ERR_CUDA, "no CUDA context"); }
  if (!h->is_rtc) {
    for (UnitId u : units) { int rc = load_unit(h, u, kUnits[u].cubin); if (rc) return rc; }
    return TPCCLUS_OK;
  }
  if (!nvrtc().ok) return fail(nullptr, TPCCLUS_ERR_NVRTC, "RTC unavailable: " + nvrtc().why);
  auto t0 = std::chrono::steady_clock::now();
  // With the on-disk cache, processes that start together with the same parameters queue up here:
  // the first compiles all units, the others then find every unit in the cache (PAPER.md 97).
  int lock_fd = -1;
  {
    std::string dir;
    { std::lock_guard<std::mutex> lk(g_cache_mutex); dir = g_cache_dir; }
    if (dir.empty()) { const char* e = getenv("TPCCLUS_RTC_CACHE"); if (e) dir = e; }
    if (!dir.empty()) {
      const std::string pro = rtc_prologue(h->g.prm, 0u, h->halo);
      char name[64]; snprintf(name, sizeof name, "/tpcclus_handle_%016llx.lock", (unsigned long long)fnv1a(pro.data(), pro.size()));
      lock_fd = open((dir + name).c_str(), O_CREAT | O_RDWR, 0644);
      if (lock_fd >= 0) flock(lock_fd, LOCK_EX);
    }
  }
  struct Unlock { int fd; ~Unlock() { if (fd >= 0) { flock(fd, LOCK_UN); close(fd); } } } unlock{lock_fd};
  const size_t n = units.size();
  std::vector<std::vector<char>> cubins(n);
  std::vector<int> rcs(n, TPCCLUS_OK);
  std::vector<std::string> errs(n);
  std::vector<char> hits(n, 0);
  std::vector<std::thread> th;
  for (size_t i = 0; i < n; ++i)
    th.emplace_back([&, i] {
      bool hit = false;
      rcs[i] = cubin_for(rtc_prologue(h->g.prm, kUnits[units[i]].bit, kUnits[units[i]].halo) + tpcclus_kernel_source, &cubins[i], &hit, &errs[i]);
      hits[i] = hit;
    });
  for (auto& t : th) t.join();
  bool all_hit = true;
  for (size_t i = 0; i < n; ++i) {
    if (rcs[i]) return fail(nullptr, rcs[i], std::string("unit ") + kUnits[units[i]].name + ": " + errs[i]);
    all_hit = all_hit && hits[i];
  }
  for (size_t i = 0; i < n; ++i) {
    int rc = load_unit(h, units[i], cubins[i].data());
    if (rc) return rc;
    h->unit_cached[units[i]] = hits[i] != 0;
  }
  h->rtc_cache_hit = all_hit;
  h->rtc_ms += std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
  return TPCCLUS_OK;
}

}  // namespace

extern "C" {

uint64_t tpcclus_workspace_bytes(const tpcclus_params* p) {
  Geometry g;
  return make_geometry(p, &g) == TPCCLUS_OK ? g.lay.total : 0;
}

uint64_t tpcclus_workspace_bytes_host(const tpcclus_params* p, uint64_t cluster_capacity) {
  Geometry g;
  return make_geometry(p, &g) == TPCCLUS_OK ? g.lay.host_clusters + 32ull * cluster_capacity : 0;
}

int tpcclus_create(const tpcclus_params* p, tpcclus_handle** out) {
  if (!out) return TPCCLUS_ERR_INVALID_ARG;
  *out = nullptr;
  g_create_error.clear();
  Geometry g;
  int rc = make_geometry(p, &g);
  if (rc != TPCCLUS_OK) return fail(nullptr, rc, "invalid or unsupported parameters");
  if (!p->workspace || ((uintptr_t)p->workspace & 255u)) return fail(nullptr, TPCCLUS_ERR_INVALID_ARG, "workspace null or not 256-byte aligned");
  if (p->workspace_bytes < g.lay.total) return fail(nullptr, TPCCLUS_ERR_WORKSPACE_TOO_SMALL, "workspace too small");
  DeviceGuard dg;
  CUDA_TRY(nullptr, dg.enter(p->device));
  tpcclus_handle* h = new tpcclus_handle();
  h->g = g;
  h->params = *p;
  h->params.n_pads = h->g.prm.n_pads;
  h->ws = (char*)p->workspace;
  h->smem_k1 = tpc_k1_smem_bytes(g.prm.k1_bins);
  h->smem_k5 = tpc_k5_smem_bytes();
  h->cog = (int)g.prm.cog_mode;
  h->halo = h->cog == 2 ? 5u : 3u;
  h->smem_k6 = tpc_k6_smem_bytes(g.prm.pitch, g.prm.max_peaks, h->halo);
  h->grid_k5 = g.g1;
  h->grid_k6 = g.g1 * TPC_K6_CTAS < g.n_tiles ? g.g1 * TPC_K6_CTAS : g.n_tiles;
  h->is_rtc = (p->flags & TPCCLUS_RTC) != 0;
  auto bail = [&](int code) { std::string e = h->err.empty() ? g_create_error : h->err; tpcclus_destroy(h); g_create_error = e; return code; };
  // static table for the debug map hook
  std::vector<uint64_t> ro(p->n_rows + 1, 0);
  for (uint32_t r = 0; r < p->n_rows; ++r) ro[r + 1] = ro[r] + (uint64_t)p->n_time * p->n_pads[r];
  cudaError_t e = cudaMemcpy(h->ws + g.lay.row_off, ro.data(), 8ull * ro.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("cudaMemcpy(row_off): ") + cudaGetErrorString(e); return bail(TPCCLUS_ERR_CUDA); }
  // the units this handle can launch (the debug unit comes on demand); a handle of reading Q10' or Q10''
  // loads -- and, under RTC, compiles -- that reading's units instead of the plain ones
  rc = load_units(h, {kKernels[K_PART_COARSE].unit[h->cog], U_DIR, kKernels[K_PART_FINE].unit[h->cog],
                      kKernels[K_TILES_FAST].unit[h->cog], kKernels[K_TILES_DET].unit[h->cog], U_ORDER});
  if (rc != TPCCLUS_OK) return bail(rc);
  for (int i = 0; i <= kMaxKernels; ++i)
    if (cudaEventCreate(&h->ev[i]) != cudaSuccess) { cudaGetLastError(); g_create_error = "cudaEventCreate failed"; return bail(TPCCLUS_ERR_CUDA); }
  *out = h;
  return TPCCLUS_OK;
}

int tpcclus_destroy(tpcclus_handle* h) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  DeviceGuard dg;
  dg.enter(h->params.device);
  for (int i = 0; i <= kMaxKernels; ++i) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
  for (int u = 0; u < U_COUNT_; ++u) if (h->module[u]) drv().cuModuleUnload(h->module[u]);
  if (h->pipe.ready) {
    cudaStreamSynchronize(h->pipe.in); cudaStreamSynchronize(h->pipe.comp); cudaStreamSynchronize(h->pipe.out);
    for (int i = 0; i < 2; ++i) { cudaEventDestroy(h->pipe.h2d[i]); cudaEventDestroy(h->pipe.done[i]); }
    cudaStreamDestroy(h->pipe.in); cudaStreamDestroy(h->pipe.comp); cudaStreamDestroy(h->pipe.out);
    if (h->pipe.res) cudaFreeHost(h->pipe.res);
  }
  delete h;
  return TPCCLUS_OK;
}

// PAPER.md 79, 85: the constant buffers may change between time frames; the framework rewrites
// ALL registered copies, in stream order, so runs enqueued before keep the old values.
int tpcclus_update_params(tpcclus_handle* h, uint16_t thr_peak, uint16_t noise_eps, void* cuda_stream) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  h->err.clear();
  if (thr_peak < 1 || thr_peak > 1023 || noise_eps > 1023) return fail(h, TPCCLUS_ERR_INVALID_ARG, "tpcclus_update_params: threshold out of range");
  if (h->is_rtc) return fail(h, TPCCLUS_ERR_INVALID_ARG, "tpcclus_update_params: an RTC handle has its parameters compiled in (PAPER.md 89-91); create a new handle");
  DeviceGuard dg;
  CUDA_TRY(h, dg.enter(h->params.device));
  h->g.prm.thr_peak = thr_peak; h->g.prm.noise_eps = noise_eps;
  h->params.thr_peak = thr_peak; h->params.noise_eps = noise_eps;
  for (const auto& c : h->consts)   // pageable source: staged by the driver before the call returns
    CUDA_TRY(h, cudaMemcpyAsync(c.dptr, &h->g.prm, sizeof(TpcParams), cudaMemcpyHostToDevice, (cudaStream_t)cuda_stream));
  return TPCCLUS_OK;
}

int tpcclus_constant_buffers(const tpcclus_handle* h) { return h ? (int)h->consts.size() : TPCCLUS_ERR_INVALID_ARG; }

int tpcclus_loaded_units(const tpcclus_handle* h, const char** names, int cap) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  int n = 0;
  for (int u = 0; u < U_COUNT_; ++u)
    if (h->module[u]) { if (names && n < cap) names[n] = kUnits[u].name; ++n; }
  return n;
}

const char* tpcclus_error_string(int code) {
  switch (code) {
    case TPCCLUS_OK: return "ok";
    case TPCCLUS_ERR_INVALID_ARG: return "invalid argument";
    case TPCCLUS_ERR_CUDA: return "CUDA error";
    case TPCCLUS_ERR_NVRTC: return "NVRTC error";
    case TPCCLUS_ERR_WORKSPACE_TOO_SMALL: return "workspace too small";
    case TPCCLUS_ERR_UNSUPPORTED_GEOMETRY: return "unsupported geometry (too many coarse bins)";
    default: return "unknown error";
  }
}

const char* tpcclus_last_error(const tpcclus_handle* h) { return h ? h->err.c_str() : g_create_error.c_str(); }

int tpcclus_launches_per_run(const tpcclus_handle* h, int mode) {
  const int extra = h ? (int)h->g.k1_passes - 1 : 0;   // K1 once per pass (one, up to 5503 coarse bins)
  return (mode == TPCCLUS_MODE_DETERMINISTIC ? 11 : 7) + extra;   // K0..K6; DET: + K7, K8, K9 and the (normally idle) chained K6
}

int tpcclus_set_timing(tpcclus_handle* h, int enable) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  h->timing = enable != 0;
  h->n_timed = 0;
  return TPCCLUS_OK;
}

int tpcclus_last_timing(tpcclus_handle* h, const char** names, float* ms, int cap) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  int n = h->n_timed;
  if (n > 0 && cudaEventSynchronize(h->ev[n]) != cudaSuccess) { cudaGetLastError(); return TPCCLUS_ERR_CUDA; }
  for (int i = 0; i < n && i < cap; ++i) {
    if (names) names[i] = h->timed_name[i];
    if (ms) { ms[i] = 0.f; cudaEventElapsedTime(&ms[i], h->ev[i], h->ev[i + 1]); }
  }
  return n;
}

double tpcclus_rtc_build_ms(const tpcclus_handle* h) { return h ? h->rtc_ms : 0.0; }

int tpcclus_rtc_cache_hit(const tpcclus_handle* h) { return h && h->rtc_cache_hit ? 1 : 0; }

int tpcclus_set_rtc_cache_dir(const char* dir) {
  std::lock_guard<std::mutex> lk(g_cache_mutex);
  g_cache_dir = dir ? dir : "";
  return TPCCLUS_OK;
}

}  // extern "C"

// ---- the run ------------------------------------------------------------------------------
namespace {

struct RunPtrs {
  u32 *status, *slice_cnt, *used, *bin_chunk_start, *batch_start, *batch_bin, *dir, *chunk_list, *blob;
  u32 *ticket, *det_flag, *tile_cnt, *tile_local, *block_sum;
  u64 *blob_cursor, *idx, *tile_state, *temp_cursor, *tile_base, *block_prefix, *row_off;
  uint4* pool;
};
RunPtrs ptrs(tpcclus_handle* h) {
  const Layout& L = h->g.lay;
  char* w = h->ws;
  RunPtrs p;
  p.status = (u32*)(w + L.status); p.blob_cursor = (u64*)(w + L.blob_cursor);
  p.slice_cnt = (u32*)(w + L.slice_cnt); p.used = (u32*)(w + L.used);
  p.bin_chunk_start = (u32*)(w + L.bin_chunk_start); p.batch_start = (u32*)(w + L.batch_start); p.batch_bin = (u32*)(w + L.batch_bin);
  p.dir = (u32*)(w + L.dir); p.chunk_list = (u32*)(w + L.chunk_list); p.pool = (uint4*)(w + L.pool);
  p.blob = (u32*)(w + L.blob); p.idx = (u64*)(w + L.idx);
  p.ticket = (u32*)(w + L.ticket); p.tile_state = (u64*)(w + L.tile_state); p.row_off = (u64*)(w + L.row_off);
  p.temp_cursor = (u64*)(w + L.temp_cursor); p.det_flag = (u32*)(w + L.det_flag); p.tile_base = (u64*)(w + L.tile_base);
  p.tile_cnt = (u32*)(w + L.tile_cnt); p.tile_local = (u32*)(w + L.tile_local); p.block_sum = (u32*)(w + L.block_sum);
  p.block_prefix = (u64*)(w + L.block_prefix);
  return p;
}

// K1..K5: digits -> per-tile record runs.  Shared by run() and the debug map hook.
int enqueue_binning(tpcclus_handle* h, const tpcclus_digit* d_digits, uint64_t n, u32* status, u64* n_out_zero, cudaStream_t st) {
  const Geometry& g = h->g;
  RunPtrs p = ptrs(h);
  int rc;
  { uint4* cnt = (uint4*)(h->ws + g.lay.counters); u64 n16 = g.lay.counters_bytes / 16;   // (the layout is 256-byte granular)
    u32* st_ext = status != p.status ? status : nullptr;
    void* a[] = {&cnt, &n16, &st_ext, &n_out_zero};
    if ((rc = launch(h, K_RESET, dim3(g.g1), dim3(256), 0, st, a))) return rc; }
  const uint64_t round = (uint64_t)TPC_K1_THREADS * TPC_K1_DPT;
  u64 per_cta = align_up((n + g.g1 - 1) / g.g1, round);
  if (per_cta == 0) per_cta = round;
  const uint2* dig = (const uint2*)d_digits;
  u64 n64 = n;
  u32 slice_cap = h->dbg_slice_cap ? h->dbg_slice_cap : g.slice_cap;
  u64 blob_cap = h->dbg_blob_cap ? h->dbg_blob_cap : g.blob_cap;
  for (u32 pass = 0; pass < g.k1_passes; ++pass) {   // one pass, unless the geometry has more bins than K1 has stages for
    u32 bin_lo = pass * g.prm.k1_bins;
    void* a[] = {&dig, &n64, &per_cta, &p.pool, &p.dir, &p.used, &slice_cap, &status, &bin_lo};
    if ((rc = launch(h, K_PART_COARSE, dim3(g.g1), dim3(TPC_K1_THREADS), h->smem_k1, st, a))) return rc;
  }
  u32 smem_nb = 4u * g.prm.n_bins;
  { void* a[] = {&p.dir, &p.used, &slice_cap, &p.slice_cnt, &p.bin_chunk_start};
    if ((rc = launch(h, K_DIR_COUNT, dim3(g.g1), dim3(TPC_SCAN_THREADS), smem_nb, st, a))) return rc; }
  { void* a[] = {&p.bin_chunk_start, &p.batch_start, &p.batch_bin};
    if ((rc = launch(h, K_DIR_SCAN, dim3(1), dim3(TPC_SCAN_THREADS), smem_nb, st, a))) return rc; }
  // K4 fills the chunk lists range of bins by range of bins, one pass over the directory per 64 MB of lists (4 bytes per chunk)
  u32 k4_pass = (u32)((4ull * (n / TPC_CHUNK + (u64)g.prm.n_bins * g.g1) + (64ull << 20) - 1ull) / (64ull << 20));
  k4_pass = k4_pass < 1u ? 1u : k4_pass > 4u ? 4u : k4_pass;
  { void* a[] = {&p.dir, &p.used, &slice_cap, &p.slice_cnt, &p.bin_chunk_start, &p.chunk_list, &k4_pass};
    if ((rc = launch(h, K_DIR_FILL, dim3(g.g1), dim3(TPC_SCAN_THREADS), smem_nb, st, a))) return rc; }
  { void* a[] = {&p.pool, &p.dir, &p.chunk_list, &p.bin_chunk_start, &p.batch_start, &p.batch_bin, &p.blob, &p.blob_cursor, &blob_cap, &p.idx, &status};
    if ((rc = launch(h, K_PART_FINE, dim3(h->grid_k5), dim3(TPC_K5_THREADS), h->smem_k5, st, a))) return rc; }
  return TPCCLUS_OK;
}

}  // namespace

extern "C" {

// run() and run_packed(): `packed` != nullptr selects the packed output of the deterministic path.
static int run_impl(tpcclus_handle* h, const tpcclus_digit* d_digits, uint64_t n, const tpcclus_out* out,
                    const tpcclus_out_packed* packed, int mode, void* cuda_stream) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  h->err.clear();
  void* o_clusters = packed ? (void*)packed->clusters : out ? (void*)out->clusters : nullptr;
  const uint64_t o_capacity = packed ? packed->capacity : out ? out->capacity : 0;
  uint64_t* o_n = packed ? packed->n_clusters : out ? out->n_clusters : nullptr;
  uint32_t* o_status = packed ? packed->status : out ? out->status : nullptr;
  if ((!out && !packed) || !o_n || (!o_clusters && o_capacity) || (!d_digits && n) || n > h->g.max_digits ||
      (mode != TPCCLUS_MODE_FAST && mode != TPCCLUS_MODE_DETERMINISTIC) || ((uintptr_t)d_digits & 15u) ||
      ((uintptr_t)o_clusters & 15u) || ((uintptr_t)o_n & 7u) || (packed && (!packed->row_index || ((uintptr_t)packed->row_index & 7u))))
    return fail(h, TPCCLUS_ERR_INVALID_ARG, "tpcclus_run: bad argument");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard dg;
  CUDA_TRY(h, dg.enter(h->params.device));
  h->n_timed = 0;
  RunPtrs p = ptrs(h);
  u32* status = o_status ? o_status : p.status;
  int rc = enqueue_binning(h, d_digits, n, status, mode == TPCCLUS_MODE_FAST ? (u64*)o_n : nullptr, st);
  if (rc) return rc;

  K6Args a;
  a.blob = p.blob; a.idx = p.idx; a.batch_start = p.batch_start;
  a.out = (uint4*)o_clusters; a.capacity = o_capacity; a.n_clusters = (u64*)o_n; a.status = status;
  a.ticket = p.ticket; a.tile_state = p.tile_state;
  a.temp = p.pool; a.temp_cap = h->g.n_chunks_max * 8ull; a.temp_cursor = p.temp_cursor;   // the K1 pool is dead after K5
  a.tile_base = p.tile_base; a.tile_cnt = p.tile_cnt; a.det_flag = p.det_flag;
  a.dmap = nullptr; a.row_off = p.row_off;
  void* ka[] = {&a};
  // the readings Q10 and Q10' run with the emitter warp on sparse frames (K6): it only
  // serves tiles of at most 256 records, so a frame that averages 512 or more per tile starts without it
  const bool emitter = h->cog != 2 && n < 512ull * h->g.n_tiles;
  if (mode == TPCCLUS_MODE_FAST) {
    if ((rc = launch(h, emitter ? K_TILES_FAST_E : K_TILES_FAST, dim3(h->grid_k6), dim3(emitter ? TPC_K6_THREADS_E : TPC_K6_THREADS), h->smem_k6, st, ka))) return rc;
  } else {
    // ordered output (PAPER.md 47-50): runs into the temporary buffer, scan of the tile counts,
    // ordered copy.  Should the buffer be too small (more than max_digits/8 clusters) the flag is
    // set, K9 does nothing and the chained-scan K6 redoes the frame; otherwise that launch exits at once.
    const Geometry& g = h->g;
    if ((rc = launch(h, emitter ? K_TILES_DET_TEMP_E : K_TILES_DET_TEMP, dim3(h->grid_k6), dim3(emitter ? TPC_K6_THREADS_E : TPC_K6_THREADS), h->smem_k6, st, ka))) return rc;
    u32 nt = g.n_tiles, nblk = g.n_scan_blocks;
    { void* s[] = {&p.tile_cnt, &p.tile_local, &p.block_sum, &nt};
      if ((rc = launch(h, K_SCAN_LOCAL, dim3(nblk), dim3(TPC_SCAN_THREADS), 0, st, s))) return rc; }
    { u64* total = (u64*)o_n;
      void* s[] = {&p.block_sum, &p.block_prefix, &nblk, &total};
      if ((rc = launch(h, K_SCAN_SUMS, dim3(1), dim3(TPC_SCAN_THREADS), 0, st, s))) return rc; }
    uint4* o = (uint4*)o_clusters; u64 cap = o_capacity;
    if (packed) {
      u64* ri = (u64*)packed->row_index;
      void* s[] = {&a.temp, &p.tile_base, &p.tile_cnt, &p.tile_local, &p.block_prefix, &nt, &o, &cap, &ri, &p.det_flag, &status};
      if ((rc = launch(h, K_EMIT_PACKED, dim3(g.g1 * 8u), dim3(256), 0, st, s))) return rc;
    } else {
      void* s[] = {&a.temp, &p.tile_base, &p.tile_cnt, &p.tile_local, &p.block_prefix, &nt, &o, &cap, &p.det_flag, &status, &p.ticket};
      if ((rc = launch(h, K_EMIT_ORDERED, dim3(g.g1 * 8u), dim3(256), 0, st, s))) return rc;
      if ((rc = launch(h, K_TILES_DET, dim3(h->grid_k6), dim3(TPC_K6_THREADS), h->smem_k6, st, ka))) return rc;
    }
  }
  h->ran = true;
  return TPCCLUS_OK;
}

int tpcclus_run(tpcclus_handle* h, const tpcclus_digit* d_digits, uint64_t n, const tpcclus_out* out, int mode,
                void* cuda_stream) {
  return run_impl(h, d_digits, n, out, nullptr, mode, cuda_stream);
}

int tpcclus_run_packed(tpcclus_handle* h, const tpcclus_digit* d_digits, uint64_t n, const tpcclus_out_packed* out,
                       void* cuda_stream) {
  if (!out) return TPCCLUS_ERR_INVALID_ARG;
  return run_impl(h, d_digits, n, nullptr, out, TPCCLUS_MODE_DETERMINISTIC, cuda_stream);
}

int tpcclus_run_host(tpcclus_handle* h, const tpcclus_digit* h_digits, uint64_t n, tpcclus_cluster* h_clusters,
                     uint64_t capacity, uint64_t* h_n_clusters, uint32_t* h_status, int mode, void* cuda_stream) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  h->err.clear();
  const Layout& L = h->g.lay;
  if (!h_n_clusters || (!h_digits && n) || (!h_clusters && capacity) || n > h->g.max_digits ||
      h->params.workspace_bytes < L.host_clusters + 32ull * capacity)
    return fail(h, TPCCLUS_ERR_INVALID_ARG, "tpcclus_run_host: bad argument or workspace not sized with tpcclus_workspace_bytes_host");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard dg;
  CUDA_TRY(h, dg.enter(h->params.device));
  tpcclus_digit* d_dig = (tpcclus_digit*)(h->ws + L.host_digits);
  tpcclus_out o;
  o.clusters = (tpcclus_cluster*)(h->ws + L.host_clusters);
  o.capacity = capacity;
  o.n_clusters = (uint64_t*)(h->ws + L.host_out);
  o.status = (uint32_t*)(h->ws + L.host_out + 8);
  if (n) CUDA_TRY(h, cudaMemcpyAsync(d_dig, h_digits, 8ull * n, cudaMemcpyHostToDevice, st));
  int rc = tpcclus_run(h, d_dig, n, &o, mode, st);
  if (rc) return rc;
  struct { uint64_t n; uint32_t s; uint32_t pad; } res;
  CUDA_TRY(h, cudaMemcpyAsync(&res, o.n_clusters, 16, cudaMemcpyDeviceToHost, st));
  CUDA_TRY(h, cudaStreamSynchronize(st));
  *h_n_clusters = res.n;
  if (h_status) *h_status = res.s;
  uint64_t m = res.n < capacity ? res.n : capacity;
  if (m) {
    CUDA_TRY(h, cudaMemcpyAsync(h_clusters, o.clusters, 32ull * m, cudaMemcpyDeviceToHost, st));
    CUDA_TRY(h, cudaStreamSynchronize(st));
  }
  return TPCCLUS_OK;
}

uint64_t tpcclus_workspace_bytes_host_pipelined(const tpcclus_params* p, uint64_t cluster_capacity) {
  Geometry g;
  return make_geometry(p, &g) == TPCCLUS_OK ? g.lay.host_digits + 2ull * (g.lay.host_slot + align_up(32ull * cluster_capacity, 256)) : 0;
}

// Two frames in flight: the host-to-device copy of frame k+1 (its own stream, its own staging slot) runs
// while frame k is clusterized and its result travels back (PAPER.md 97: a process takes whole time frames
// one after the other; the link is the bottleneck of this entry, so keeping it busy is all that counts).
int tpcclus_host_submit(tpcclus_handle* h, const tpcclus_digit* h_digits, uint64_t n, tpcclus_cluster* h_clusters,
                        uint64_t capacity, int mode) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  h->err.clear();
  const Layout& L = h->g.lay;
  tpcclus_handle::Pipe& P = h->pipe;
  const uint64_t slot_bytes = L.host_slot + align_up(32ull * capacity, 256);
  if ((!h_digits && n) || (!h_clusters && capacity) || n > h->g.max_digits ||
      h->params.workspace_bytes < L.host_digits + 2ull * slot_bytes)
    return fail(h, TPCCLUS_ERR_INVALID_ARG, "tpcclus_host_submit: bad argument or workspace not sized with tpcclus_workspace_bytes_host_pipelined");
  if (P.seq_submit - P.seq_wait >= 2) return fail(h, TPCCLUS_ERR_INVALID_ARG, "tpcclus_host_submit: two frames are in flight, call tpcclus_host_wait first");
  DeviceGuard dg;
  CUDA_TRY(h, dg.enter(h->params.device));
  if (!P.ready) {
    CUDA_TRY(h, cudaStreamCreateWithFlags(&P.in, cudaStreamNonBlocking));
    CUDA_TRY(h, cudaStreamCreateWithFlags(&P.comp, cudaStreamNonBlocking));
    CUDA_TRY(h, cudaStreamCreateWithFlags(&P.out, cudaStreamNonBlocking));
    for (int i = 0; i < 2; ++i) {
      CUDA_TRY(h, cudaEventCreateWithFlags(&P.h2d[i], cudaEventDisableTiming));
      CUDA_TRY(h, cudaEventCreateWithFlags(&P.done[i], cudaEventDisableTiming));
    }
    CUDA_TRY(h, cudaHostAlloc((void**)&P.res, 2 * sizeof *P.res, cudaHostAllocMapped));
    CUDA_TRY(h, cudaHostGetDevicePointer((void**)&P.res_dev, P.res, 0));
    P.ready = true;
  }
  const int sl = (int)(P.seq_submit & 1);
  char* base = h->ws + L.host_digits + (uint64_t)sl * slot_bytes;
  tpcclus_digit* d_dig = (tpcclus_digit*)base;
  tpcclus_out o;
  o.n_clusters = (uint64_t*)(base + (L.host_out - L.host_digits));
  o.status = (uint32_t*)(base + (L.host_out - L.host_digits) + 8);
  o.clusters = (tpcclus_cluster*)(base + L.host_slot);
  o.capacity = capacity;
  // the slot's staging is free: wait() of the frame that used it two submits ago has returned
  if (n) CUDA_TRY(h, cudaMemcpyAsync(d_dig, h_digits, 8ull * n, cudaMemcpyHostToDevice, P.in));
  CUDA_TRY(h, cudaEventRecord(P.h2d[sl], P.in));
  CUDA_TRY(h, cudaStreamWaitEvent(P.comp, P.h2d[sl], 0));
  int rc = tpcclus_run(h, d_dig, n, &o, mode, P.comp);
  if (rc) return rc;
  { u64* hr = (u64*)&P.res_dev[sl]; const u64* nc = (const u64*)o.n_clusters; const u32* stp = o.status;
    void* a[] = {&hr, &nc, &stp};
    bool t = h->timing; h->timing = false;
    rc = launch(h, K_PUBLISH, dim3(1), dim3(32), 0, P.comp, a);
    h->timing = t;
    if (rc) return rc; }
  // wait() synchronises on this event before it reads anything back.  Nothing of frame k+1 may be queued on the
  // read-back stream ahead of frame k's clusters (a wait for frame k+1's run there cost the whole overlap).
  CUDA_TRY(h, cudaEventRecord(P.done[sl], P.comp));
  P.job[sl].h_clusters = h_clusters; P.job[sl].capacity = capacity;
  ++P.seq_submit;
  return TPCCLUS_OK;
}

int tpcclus_host_wait(tpcclus_handle* h, uint64_t* h_n_clusters, uint32_t* h_status) {
  if (!h || !h_n_clusters) return TPCCLUS_ERR_INVALID_ARG;
  h->err.clear();
  tpcclus_handle::Pipe& P = h->pipe;
  if (P.seq_wait == P.seq_submit) return fail(h, TPCCLUS_ERR_INVALID_ARG, "tpcclus_host_wait: nothing in flight");
  const Layout& L = h->g.lay;
  DeviceGuard dg;
  CUDA_TRY(h, dg.enter(h->params.device));
  const int sl = (int)(P.seq_wait & 1);
  CUDA_TRY(h, cudaEventSynchronize(P.done[sl]));   // the run is over; its 16-byte result is in the mapped host words
  *h_n_clusters = P.res[sl].n;
  if (h_status) *h_status = (uint32_t)P.res[sl].s;
  const uint64_t cap = P.job[sl].capacity, m = P.res[sl].n < cap ? P.res[sl].n : cap;
  if (m) {   // only the clusters that exist cross the link; meanwhile the next frame's digits are coming in
    const uint64_t slot_bytes = L.host_slot + align_up(32ull * cap, 256);
    const char* src = h->ws + L.host_digits + (uint64_t)sl * slot_bytes + L.host_slot;
    CUDA_TRY(h, cudaMemcpyAsync(P.job[sl].h_clusters, src, 32ull * m, cudaMemcpyDeviceToHost, P.out));
    CUDA_TRY(h, cudaStreamSynchronize(P.out));
  }
  ++P.seq_wait;
  return TPCCLUS_OK;
}

int tpcclus_debug_det_fallback(tpcclus_handle* h) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  uint32_t f = 0;
  DeviceGuard dg;
  CUDA_TRY(h, dg.enter(h->params.device));
  CUDA_TRY(h, cudaMemcpy(&f, h->ws + h->g.lay.det_flag, 4, cudaMemcpyDeviceToHost));   // synchronises
  return f != 0 ? 1 : 0;
}

int tpcclus_debug_shrink(tpcclus_handle* h, uint32_t slice_cap, uint64_t blob_cap) {
  if (!h || slice_cap > h->g.slice_cap || blob_cap > h->g.blob_cap) return TPCCLUS_ERR_INVALID_ARG;
  h->dbg_slice_cap = slice_cap;
  h->dbg_blob_cap = blob_cap;
  return TPCCLUS_OK;
}

int tpcclus_debug_dense_map(tpcclus_handle* h, uint16_t* d_map, void* cuda_stream) {
  if (!h || !d_map) return TPCCLUS_ERR_INVALID_ARG;
  if (!h->ran) return fail(h, TPCCLUS_ERR_INVALID_ARG, "tpcclus_debug_dense_map: no run() yet");
  cudaStream_t st = (cudaStream_t)cuda_stream;
  DeviceGuard dg;
  CUDA_TRY(h, dg.enter(h->params.device));
  int rc = load_units(h, {kKernels[K_TILES_DUMP].unit[h->cog]});   // the debug unit is loaded (RTC: compiled) on first use
  if (rc) { h->err = g_create_error; return rc; }
  const Geometry& g = h->g;
  RunPtrs p = ptrs(h);
  uint64_t cells = 0;
  for (uint32_t r = 0; r < g.prm.n_rows; ++r) cells += (uint64_t)g.prm.n_time * g.prm.n_pads[r];
  CUDA_TRY(h, cudaMemsetAsync(d_map, 0, 2ull * cells * g.prm.n_sectors, st));
  bool t = h->timing; h->timing = false;
  K6Args a;
  memset(&a, 0, sizeof a);
  a.blob = p.blob; a.idx = p.idx; a.batch_start = p.batch_start; a.status = p.status;
  a.dmap = d_map; a.row_off = p.row_off; a.ticket = p.ticket; a.tile_state = p.tile_state; a.det_flag = p.det_flag;
  CUDA_TRY(h, cudaMemsetAsync(p.ticket, 0, 4, st));   // the run before used the tickets up
  void* ka[] = {&a};
  rc = launch(h, K_TILES_DUMP, dim3(h->grid_k6), dim3(TPC_K6_THREADS), h->smem_k6, st, ka);
  h->timing = t;
  return rc;
}

}  // extern "C"
