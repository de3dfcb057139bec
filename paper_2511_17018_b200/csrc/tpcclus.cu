// tpcclus.cu -- host side of libtpcclus.so: the C ABI of include/tpcclus.h.
//
// Orchestration only: parameter validation, workspace layout, the launch sequence of
// tpcclus_kernels.cuh, the stream-ordered __constant__ upload (PAPER.md 85) and the NVRTC
// build of the same kernel text with constants baked in (PAPER.md 89-93; loaded through the
// driver's module loader like the paper's per-kernel binaries, PAPER.md 64, 91).
// No step of the path runs on the host; without a CUDA device every entry point that
// would compute returns TPCCLUS_ERR_CUDA.
#include <cuda_runtime.h>
#include <dlfcn.h>
#include <fcntl.h>
#include <sys/file.h>
#include <unistd.h>

#include <chrono>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <string>
#include <vector>

#include "../../include/tpcclus.h"
#include "tpcclus_kernels.cuh"

extern "C" const char tpcclus_kernel_source[];   // generated from tpcclus_kernels.cuh at build time

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
};

struct Geometry {
  TpcParams prm;
  uint32_t g1;           // K1 grid = number of SMs
  uint32_t slice_cap;    // chunks per K1 CTA
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
  if (nb > 65535 || tpc_k1_smem_bytes((uint32_t)nb) > kMaxSmem) return TPCCLUS_ERR_UNSUPPORTED_GEOMETRY;
  q.n_bins = (uint32_t)nb;
  uint32_t tmin = p->n_time < TPC_TC ? p->n_time : TPC_TC;
  q.n_sl = (tmin + TPC_TS - 1) / TPC_TS;
  q.max_pads = maxp;
  q.pitch = (maxp + 2 * TPC_HALO + 7) / 8 * 8;
  q.thr_peak = p->thr_peak; q.noise_eps = p->noise_eps;
  q.cog_gated = (p->flags & TPCCLUS_COG_GATED) ? 1u : 0u;
  q.max_peaks = ((TPC_TT - 2 + 1) / 2) * ((maxp + 1) / 2);   // no two peaks are 8-neighbours; rows 1..TT-2 are scanned

  g->max_digits = p->max_digits;
  g->g1 = (uint32_t)sm_count(p->device);
  const uint64_t round = (uint64_t)TPC_K1_THREADS * TPC_K1_DPT;
  uint64_t per_cta = align_up((p->max_digits + g->g1 - 1) / g->g1, round);
  uint64_t dup = q.n_tc > 1 ? 2 : 1;   // K1 copies a digit into the next time-chunk at most once
  uint64_t cap = (per_cta * dup + TPC_CHUNK - 1) / TPC_CHUNK + nb;   // full chunks + one partial per bin
  if (cap > 0x0FFFFFFFull) return TPCCLUS_ERR_INVALID_ARG;
  g->slice_cap = (uint32_t)cap;
  g->n_chunks_max = (uint64_t)g->g1 * cap;
  if (g->n_chunks_max > 0x00FFFFFFFFull) return TPCCLUS_ERR_INVALID_ARG;
  g->n_batches_max = g->n_chunks_max / TPC_CPB + nb + 1;
  g->blob_cap = p->max_digits * (dup + 2) + g->n_batches_max * 8ull * q.n_sl + 64;   // K5 halo copies + run padding
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
  return TPCCLUS_OK;
}

// ---- lazily loaded driver / NVRTC entry points (RTC handles only) ------------------------
struct Rtc {
  void* libcuda = nullptr; void* libnvrtc = nullptr;
  int (*cuModuleLoadData)(void**, const void*) = nullptr;
  int (*cuModuleUnload)(void*) = nullptr;
  int (*cuModuleGetFunction)(void**, void*, const char*) = nullptr;
  int (*cuFuncSetAttribute)(void*, int, int) = nullptr;
  int (*cuLaunchKernel)(void*, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, unsigned, void*, void**, void**) = nullptr;
  int (*cuGetErrorString)(int, const char**) = nullptr;
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

Rtc& rtc() {
  static Rtc r;
  static bool tried = false;
  if (tried) return r;
  tried = true;
  r.libcuda = dlopen("libcuda.so.1", RTLD_NOW | RTLD_GLOBAL);
  if (!r.libcuda) { r.why = "dlopen(libcuda.so.1) failed"; return r; }
  // the toolkit's own NVRTC first (12.9: knows the 256-bit vector store), then whatever the process has
  for (const char* name : {"/usr/local/cuda/lib64/libnvrtc.so.12", "/usr/local/cuda/targets/x86_64-linux/lib/libnvrtc.so.12",
                           "libnvrtc.so.12", "libnvrtc.so"}) {
    r.libnvrtc = dlopen(name, RTLD_NOW);
    if (r.libnvrtc) break;
  }
  if (!r.libnvrtc) { r.why = "dlopen(libnvrtc) failed"; return r; }
  bool all = true;
#define SYM(lib, f) do { *(void**)(&r.f) = dlsym(r.lib, #f); if (!r.f) { all = false; r.why = "missing symbol " #f; } } while (0)
  SYM(libcuda, cuModuleLoadData); SYM(libcuda, cuModuleUnload); SYM(libcuda, cuModuleGetFunction);
  SYM(libcuda, cuFuncSetAttribute); SYM(libcuda, cuLaunchKernel); SYM(libcuda, cuGetErrorString);
  SYM(libnvrtc, nvrtcCreateProgram); SYM(libnvrtc, nvrtcCompileProgram); SYM(libnvrtc, nvrtcGetCUBINSize);
  SYM(libnvrtc, nvrtcGetCUBIN); SYM(libnvrtc, nvrtcGetProgramLogSize); SYM(libnvrtc, nvrtcGetProgramLog);
  SYM(libnvrtc, nvrtcDestroyProgram); SYM(libnvrtc, nvrtcVersion);
#undef SYM
  r.ok = all;
  return r;
}

enum KernelId { K_PART_COARSE, K_DIR_COUNT, K_DIR_SCAN, K_DIR_FILL, K_PART_FINE, K_TILES_FAST, K_TILES_DET,
                K_TILES_DET_TEMP, K_TILES_DUMP, K_SCAN_LOCAL, K_SCAN_SUMS, K_EMIT_ORDERED, K_EMIT_PACKED,
                K_TILES_FAST_G, K_TILES_DET_G, K_TILES_DET_TEMP_G, K_COUNT_ };
const char* const kKernelNames[K_COUNT_] = {
    "k_partition_coarse", "k_dir_count", "k_dir_scan", "k_dir_fill", "k_partition_fine", "k_cluster_tiles_fast",
    "k_cluster_tiles_det", "k_cluster_tiles_det_temp", "k_cluster_tiles_dump_map", "k_scan_local", "k_scan_sums",
    "k_emit_ordered", "k_emit_packed", "k_cluster_tiles_fast_gated", "k_cluster_tiles_det_gated",
    "k_cluster_tiles_det_temp_gated"};
const void* const kKernelPtrs[K_COUNT_] = {
    (const void*)k_partition_coarse, (const void*)k_dir_count, (const void*)k_dir_scan, (const void*)k_dir_fill,
    (const void*)k_partition_fine, (const void*)k_cluster_tiles_fast, (const void*)k_cluster_tiles_det,
    (const void*)k_cluster_tiles_det_temp, (const void*)k_cluster_tiles_dump_map, (const void*)k_scan_local,
    (const void*)k_scan_sums, (const void*)k_emit_ordered, (const void*)k_emit_packed,
    (const void*)k_cluster_tiles_fast_gated, (const void*)k_cluster_tiles_det_gated,
    (const void*)k_cluster_tiles_det_temp_gated};

}  // namespace

struct tpcclus_handle {
  Geometry g;
  tpcclus_params params;   // copy; n_pads points into g.prm
  char* ws = nullptr;
  bool is_rtc = false;
  void* module = nullptr;
  void* fn[K_COUNT_] = {};
  double rtc_ms = 0.0;
  bool rtc_cache_hit = false;
  uint32_t smem_k1 = 0, smem_k5 = 0, smem_k6 = 0;
  uint32_t grid_k5 = 0, grid_k6 = 0;
  bool timing = false;
  int n_timed = 0;
  const char* timed_name[kMaxKernels] = {};
  cudaEvent_t ev[kMaxKernels + 1] = {};
  std::string err;
  bool ran = false;
};

namespace {

int fail(tpcclus_handle* h, int code, const std::string& detail) {
  if (h) h->err = detail; else g_create_error = detail;
  return code;
}
#define CUDA_TRY(h, expr) do { cudaError_t e_ = (expr); if (e_ != cudaSuccess) { cudaGetLastError(); \
  return fail(h, TPCCLUS_ERR_CUDA, std::string(#expr) + ": " + cudaGetErrorString(e_)); } } while (0)

// One launch, generic (runtime API, offline-compiled kernel) or RTC (driver API, NVRTC module).
int launch(tpcclus_handle* h, KernelId k, dim3 grid, dim3 block, uint32_t smem, cudaStream_t st, void** args) {
  if (h->timing && h->n_timed < kMaxKernels) {
    if (h->n_timed == 0) cudaEventRecord(h->ev[0], st);
    h->timed_name[h->n_timed] = kKernelNames[k];
  }
  if (h->is_rtc) {
    int rc = rtc().cuLaunchKernel(h->fn[k], grid.x, grid.y, grid.z, block.x, block.y, block.z, smem, st, args, nullptr);
    if (rc != 0) {
      const char* s = nullptr; rtc().cuGetErrorString(rc, &s);
      return fail(h, TPCCLUS_ERR_CUDA, std::string("cuLaunchKernel(") + kKernelNames[k] + "): " + (s ? s : "?"));
    }
  } else {
    cudaError_t e = cudaLaunchKernel(kKernelPtrs[k], grid, block, args, smem, st);
    if (e != cudaSuccess) {
      cudaGetLastError();
      return fail(h, TPCCLUS_ERR_CUDA, std::string("cudaLaunchKernel(") + kKernelNames[k] + "): " + cudaGetErrorString(e));
    }
  }
  if (h->timing && h->n_timed < kMaxKernels) { ++h->n_timed; cudaEventRecord(h->ev[h->n_timed], st); }
  return TPCCLUS_OK;
}

// Text put in front of the kernel source for NVRTC: every parameter as a literal.
std::string rtc_prologue(const TpcParams& q) {
  char buf[256];
  std::string s = "#define TPC_RTC 1\n";
#define DEF(f) do { snprintf(buf, sizeof buf, "#define TPC_" #f " %uu\n", q.f); s += buf; } while (0)
  DEF(n_sectors); DEF(n_rows); DEF(n_time); DEF(n_tc); DEF(n_bins); DEF(n_sl); DEF(pitch); DEF(max_pads);
  DEF(thr_peak); DEF(noise_eps); DEF(max_peaks); DEF(cog_gated);
#undef DEF
  s += "__device__ const unsigned short TPC_NPADS_TABLE[256] = {";
  for (int r = 0; r < 256; ++r) { snprintf(buf, sizeof buf, "%u,", (unsigned)q.n_pads[r]); s += buf; }
  s += "};\n";
  return s;
}

// NVRTC: kernel text -> cubin for sm_100a.
int compile_cubin(const std::string& src, std::vector<char>* cubin) {
  Rtc& r = rtc();
  void* prog = nullptr;
  if (r.nvrtcCreateProgram(&prog, src.c_str(), "tpcclus_kernels.cu", 0, nullptr, nullptr) != 0)
    return fail(nullptr, TPCCLUS_ERR_NVRTC, "nvrtcCreateProgram failed");
  const char* opts[] = {"--gpu-architecture=sm_100a", "-std=c++17", "-default-device", "-lineinfo", "--fmad=false", "--prec-div=true",
                        "--prec-sqrt=true", "--ftz=false", "-DTPC_NO_ST256=1"};
  int rc = r.nvrtcCompileProgram(prog, 8, opts);
  if (rc != 0) {   // older NVRTC: retry without the 256-bit store
    r.nvrtcDestroyProgram(&prog);
    prog = nullptr;
    if (r.nvrtcCreateProgram(&prog, src.c_str(), "tpcclus_kernels.cu", 0, nullptr, nullptr) != 0)
      return fail(nullptr, TPCCLUS_ERR_NVRTC, "nvrtcCreateProgram failed");
    rc = r.nvrtcCompileProgram(prog, 9, opts);
  }
  if (rc != 0) {
    size_t n = 0; r.nvrtcGetProgramLogSize(prog, &n);
    std::string log(n, '\0'); if (n) r.nvrtcGetProgramLog(prog, &log[0]);
    r.nvrtcDestroyProgram(&prog);
    return fail(nullptr, TPCCLUS_ERR_NVRTC, "nvrtcCompileProgram failed:\n" + log);
  }
  size_t n = 0; r.nvrtcGetCUBINSize(prog, &n);
  cubin->resize(n);
  r.nvrtcGetCUBIN(prog, cubin->data());
  r.nvrtcDestroyProgram(&prog);
  return TPCCLUS_OK;
}

// On-disk cubin cache (PAPER.md 97: several processes per node share one run-time compilation,
// serialised by a file lock).  Key = hash of the exact text handed to NVRTC (prologue with every
// baked parameter + kernel source) and of the NVRTC version.  The compile happens under an
// exclusive flock on <key>.lock; the cubin is written to a temporary name and renamed, so a
// reader sees a whole file or none.  Any I/O problem just means "compile, do not cache".
std::string g_cache_dir;   // set by tpcclus_set_rtc_cache_dir or $TPCCLUS_RTC_CACHE

bool read_file(const std::string& path, std::vector<char>* out) {
  FILE* f = fopen(path.c_str(), "rb");
  if (!f) return false;
  fseek(f, 0, SEEK_END);
  long n = ftell(f);
  fseek(f, 0, SEEK_SET);
  bool ok = n > 0;
  if (ok) { out->resize((size_t)n); ok = fread(out->data(), 1, (size_t)n, f) == (size_t)n; }
  fclose(f);
  return ok;
}

int cubin_for(const std::string& src, std::vector<char>* cubin, bool* hit) {
  *hit = false;
  std::string dir = g_cache_dir;
  if (dir.empty()) { const char* e = getenv("TPCCLUS_RTC_CACHE"); if (e) dir = e; }
  if (dir.empty()) return compile_cubin(src, cubin);
  int vmaj = 0, vmin = 0;
  if (rtc().nvrtcVersion) rtc().nvrtcVersion(&vmaj, &vmin);
  uint64_t hsh = 1469598103934665603ull;   // FNV-1a
  auto mix = [&](const char* p, size_t n) { for (size_t i = 0; i < n; ++i) { hsh ^= (unsigned char)p[i]; hsh *= 1099511628211ull; } };
  mix(src.data(), src.size());
  char tag[64]; snprintf(tag, sizeof tag, "|nvrtc %d.%d|sm_100a", vmaj, vmin); mix(tag, strlen(tag));
  char name[64]; snprintf(name, sizeof name, "/tpcclus_%016llx", (unsigned long long)hsh);
  const std::string base = dir + name, file = base + ".cubin", lock = base + ".lock";
  if (read_file(file, cubin)) { *hit = true; return TPCCLUS_OK; }
  int fd = open(lock.c_str(), O_CREAT | O_RDWR, 0644);
  if (fd >= 0) flock(fd, LOCK_EX);   // whoever comes second waits here, then finds the file
  int rc = TPCCLUS_OK;
  if (fd >= 0 && read_file(file, cubin)) {
    *hit = true;
  } else {
    rc = compile_cubin(src, cubin);
    if (rc == TPCCLUS_OK && fd >= 0) {
      char tmp[64]; snprintf(tmp, sizeof tmp, ".tmp%d", (int)getpid());
      FILE* f = fopen((file + tmp).c_str(), "wb");
      if (f) {
        bool ok = fwrite(cubin->data(), 1, cubin->size(), f) == cubin->size();
        ok = fclose(f) == 0 && ok;
        if (ok) rename((file + tmp).c_str(), file.c_str()); else remove((file + tmp).c_str());
      }
    }
  }
  if (fd >= 0) { flock(fd, LOCK_UN); close(fd); }
  return rc;
}

int build_rtc(tpcclus_handle* h) {
  Rtc& r = rtc();
  if (!r.ok) return fail(nullptr, TPCCLUS_ERR_NVRTC, "RTC unavailable: " + r.why);
  auto t0 = std::chrono::steady_clock::now();
  std::string src = rtc_prologue(h->g.prm) + tpcclus_kernel_source;
  std::vector<char> cubin;
  int rc = cubin_for(src, &cubin, &h->rtc_cache_hit);
  if (rc != TPCCLUS_OK) return rc;
  if (cudaFree(nullptr) != cudaSuccess) { cudaGetLastError(); return fail(nullptr, TPCCLUS_ERR_CUDA, "no CUDA context"); }
  if ((rc = r.cuModuleLoadData(&h->module, cubin.data())) != 0) {
    const char* s = nullptr; r.cuGetErrorString(rc, &s);
    return fail(nullptr, TPCCLUS_ERR_CUDA, std::string("cuModuleLoadData: ") + (s ? s : "?"));
  }
  for (int k = 0; k < K_COUNT_; ++k)
    if (r.cuModuleGetFunction(&h->fn[k], h->module, kKernelNames[k]) != 0)
      return fail(nullptr, TPCCLUS_ERR_NVRTC, std::string("cuModuleGetFunction: ") + kKernelNames[k]);
  const int CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES = 8;
  struct { int k; uint32_t b; } sm[] = {{K_PART_COARSE, h->smem_k1}, {K_PART_FINE, h->smem_k5}, {K_TILES_FAST, h->smem_k6},
                                        {K_TILES_DET, h->smem_k6}, {K_TILES_DET_TEMP, h->smem_k6}, {K_TILES_DUMP, h->smem_k6},
                                        {K_TILES_FAST_G, h->smem_k6}, {K_TILES_DET_G, h->smem_k6}, {K_TILES_DET_TEMP_G, h->smem_k6}};
  for (auto& e : sm)
    if (r.cuFuncSetAttribute(h->fn[e.k], CU_FUNC_ATTRIBUTE_MAX_DYNAMIC_SHARED_SIZE_BYTES, (int)e.b) != 0)
      return fail(nullptr, TPCCLUS_ERR_CUDA, std::string("cuFuncSetAttribute: ") + kKernelNames[e.k]);
  h->rtc_ms = std::chrono::duration<double, std::milli>(std::chrono::steady_clock::now() - t0).count();
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
  CUDA_TRY(nullptr, cudaSetDevice(p->device));
  tpcclus_handle* h = new tpcclus_handle();
  h->g = g;
  h->params = *p;
  h->params.n_pads = h->g.prm.n_pads;
  h->ws = (char*)p->workspace;
  h->smem_k1 = tpc_k1_smem_bytes(g.prm.n_bins);
  h->smem_k5 = tpc_k5_smem_bytes();
  h->smem_k6 = tpc_k6_smem_bytes(g.prm.pitch, g.prm.max_peaks);
  h->grid_k5 = g.g1;
  h->grid_k6 = g.g1 * TPC_K6_CTAS < g.n_tiles ? g.g1 * TPC_K6_CTAS : g.n_tiles;
  auto bail = [&](int code) { std::string e = h->err.empty() ? g_create_error : h->err; delete h; g_create_error = e; return code; };
  // static table for the debug map hook
  std::vector<uint64_t> ro(p->n_rows + 1, 0);
  for (uint32_t r = 0; r < p->n_rows; ++r) ro[r + 1] = ro[r] + (uint64_t)p->n_time * p->n_pads[r];
  cudaError_t e = cudaMemcpy(h->ws + g.lay.row_off, ro.data(), 8ull * ro.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("cudaMemcpy(row_off): ") + cudaGetErrorString(e); return bail(TPCCLUS_ERR_CUDA); }
  if (p->flags & TPCCLUS_RTC) {
    h->is_rtc = true;
    rc = build_rtc(h);
    if (rc != TPCCLUS_OK) return bail(rc);
  } else {
    struct { int k; uint32_t b; } sm[] = {{K_PART_COARSE, h->smem_k1}, {K_PART_FINE, h->smem_k5}, {K_TILES_FAST, h->smem_k6},
                                          {K_TILES_DET, h->smem_k6}, {K_TILES_DET_TEMP, h->smem_k6}, {K_TILES_DUMP, h->smem_k6},
                                        {K_TILES_FAST_G, h->smem_k6}, {K_TILES_DET_G, h->smem_k6}, {K_TILES_DET_TEMP_G, h->smem_k6}};
    for (auto& s : sm) {
      e = cudaFuncSetAttribute(kKernelPtrs[s.k], cudaFuncAttributeMaxDynamicSharedMemorySize, (int)s.b);
      if (e != cudaSuccess) { cudaGetLastError(); g_create_error = std::string("cudaFuncSetAttribute(") + kKernelNames[s.k] + "): " + cudaGetErrorString(e); return bail(TPCCLUS_ERR_CUDA); }
    }
  }
  for (int i = 0; i <= kMaxKernels; ++i)
    if (cudaEventCreate(&h->ev[i]) != cudaSuccess) { cudaGetLastError(); g_create_error = "cudaEventCreate failed"; return bail(TPCCLUS_ERR_CUDA); }
  *out = h;
  return TPCCLUS_OK;
}

int tpcclus_destroy(tpcclus_handle* h) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  for (int i = 0; i <= kMaxKernels; ++i) if (h->ev[i]) cudaEventDestroy(h->ev[i]);
  if (h->module) rtc().cuModuleUnload(h->module);
  delete h;
  return TPCCLUS_OK;
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
  (void)h;
  return mode == TPCCLUS_MODE_DETERMINISTIC ? 10 : 6;   // DET: + K7, K8, K9 and the (normally idle) chained K6
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
int enqueue_binning(tpcclus_handle* h, const tpcclus_digit* d_digits, uint64_t n, u32* status, cudaStream_t st) {
  const Geometry& g = h->g;
  RunPtrs p = ptrs(h);
  if (!h->is_rtc)   // PAPER.md 85: the constant buffer is rewritten for every time frame, in stream order
    CUDA_TRY(h, cudaMemcpyToSymbolAsync(c_prm, &g.prm, sizeof(TpcParams), 0, cudaMemcpyHostToDevice, st));
  CUDA_TRY(h, cudaMemsetAsync(h->ws + g.lay.counters, 0, g.lay.counters_bytes, st));
  if (status != p.status) CUDA_TRY(h, cudaMemsetAsync(status, 0, 4, st));
  const uint64_t round = (uint64_t)TPC_K1_THREADS * TPC_K1_DPT;
  u64 per_cta = align_up((n + g.g1 - 1) / g.g1, round);
  if (per_cta == 0) per_cta = round;
  const uint2* dig = (const uint2*)d_digits;
  u64 n64 = n;
  u32 slice_cap = g.slice_cap;
  int rc;
  { void* a[] = {&dig, &n64, &per_cta, &p.pool, &p.dir, &p.used, &slice_cap, &status};
    if ((rc = launch(h, K_PART_COARSE, dim3(g.g1), dim3(TPC_K1_THREADS), h->smem_k1, st, a))) return rc; }
  u32 smem_nb = 4u * g.prm.n_bins;
  { void* a[] = {&p.dir, &p.used, &slice_cap, &p.slice_cnt, &p.bin_chunk_start};
    if ((rc = launch(h, K_DIR_COUNT, dim3(g.g1), dim3(TPC_SCAN_THREADS), smem_nb, st, a))) return rc; }
  { void* a[] = {&p.bin_chunk_start, &p.batch_start, &p.batch_bin};
    if ((rc = launch(h, K_DIR_SCAN, dim3(1), dim3(TPC_SCAN_THREADS), smem_nb, st, a))) return rc; }
  { void* a[] = {&p.dir, &p.used, &slice_cap, &p.slice_cnt, &p.bin_chunk_start, &p.chunk_list};
    if ((rc = launch(h, K_DIR_FILL, dim3(g.g1), dim3(TPC_SCAN_THREADS), smem_nb, st, a))) return rc; }
  { void* a[] = {&p.pool, &p.dir, &p.chunk_list, &p.bin_chunk_start, &p.batch_start, &p.batch_bin, &p.blob, &p.blob_cursor, &p.idx, &status};
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
  CUDA_TRY(h, cudaSetDevice(h->params.device));
  h->n_timed = 0;
  RunPtrs p = ptrs(h);
  u32* status = o_status ? o_status : p.status;
  int rc = enqueue_binning(h, d_digits, n, status, st);
  if (rc) return rc;

  K6Args a;
  a.blob = p.blob; a.idx = p.idx; a.batch_start = p.batch_start;
  a.out = (uint4*)o_clusters; a.capacity = o_capacity; a.n_clusters = (u64*)o_n; a.status = status;
  a.ticket = p.ticket; a.tile_state = p.tile_state;
  a.temp = p.pool; a.temp_cap = h->g.n_chunks_max * 8ull; a.temp_cursor = p.temp_cursor;   // the K1 pool is dead after K5
  a.tile_base = p.tile_base; a.tile_cnt = p.tile_cnt; a.det_flag = p.det_flag;
  a.dmap = nullptr; a.row_off = p.row_off;
  void* ka[] = {&a};
  const bool gated = h->g.prm.cog_gated != 0u;   // reading Q10': its own kernel variants
  if (mode == TPCCLUS_MODE_FAST) {
    CUDA_TRY(h, cudaMemsetAsync(o_n, 0, 8, st));
    if ((rc = launch(h, gated ? K_TILES_FAST_G : K_TILES_FAST, dim3(h->grid_k6), dim3(TPC_K6_THREADS), h->smem_k6, st, ka))) return rc;
  } else {
    // ordered output (PAPER.md 47-50): runs into the temporary buffer, scan of the tile counts,
    // ordered copy.  Should the buffer be too small (more than max_digits/8 clusters) the flag is
    // set, K9 does nothing and the chained-scan K6 redoes the frame; otherwise that launch exits at once.
    const Geometry& g = h->g;
    if ((rc = launch(h, gated ? K_TILES_DET_TEMP_G : K_TILES_DET_TEMP, dim3(h->grid_k6), dim3(TPC_K6_THREADS), h->smem_k6, st, ka))) return rc;
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
      void* s[] = {&a.temp, &p.tile_base, &p.tile_cnt, &p.tile_local, &p.block_prefix, &nt, &o, &cap, &p.det_flag, &status};
      if ((rc = launch(h, K_EMIT_ORDERED, dim3(g.g1 * 8u), dim3(256), 0, st, s))) return rc;
      CUDA_TRY(h, cudaMemsetAsync(p.ticket, 0, 4, st));
      if ((rc = launch(h, gated ? K_TILES_DET_G : K_TILES_DET, dim3(h->grid_k6), dim3(TPC_K6_THREADS), h->smem_k6, st, ka))) return rc;
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
  CUDA_TRY(h, cudaSetDevice(h->params.device));
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

int tpcclus_debug_det_fallback(tpcclus_handle* h) {
  if (!h) return TPCCLUS_ERR_INVALID_ARG;
  uint32_t f = 0;
  CUDA_TRY(h, cudaMemcpy(&f, h->ws + h->g.lay.det_flag, 4, cudaMemcpyDeviceToHost));   // synchronises
  return f != 0 ? 1 : 0;
}

int tpcclus_debug_dense_map(tpcclus_handle* h, uint16_t* d_map, void* cuda_stream) {
  if (!h || !d_map) return TPCCLUS_ERR_INVALID_ARG;
  if (!h->ran) return fail(h, TPCCLUS_ERR_INVALID_ARG, "tpcclus_debug_dense_map: no run() yet");
  cudaStream_t st = (cudaStream_t)cuda_stream;
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
  int rc = launch(h, K_TILES_DUMP, dim3(h->grid_k6), dim3(TPC_K6_THREADS), h->smem_k6, st, ka);
  h->timing = t;
  return rc;
}

}  // extern "C"
