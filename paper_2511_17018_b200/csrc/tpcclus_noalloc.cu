// tpcclus_pack_noalloc: the packed 16-byte output of a cluster list that is
// already on the device, for callers that cannot allocate: code under CUDA graph capture, tight serving
// loops, harnesses that forbid cudaMalloc.  A variant of K9p (k_emit_packed): that kernel reads the per-tile
// run table and the tile-count scan out of the handle's workspace; this one takes the ordered list
// tpcclus_run(DETERMINISTIC) wrote, counts its clusters per (sector, row) and scans the counts -- and keeps
// those counts, its only scratch memory, in a file-scope array in device memory instead of a workspace:
// 256.25 KB that every GPU that loads the library holds until the process ends.  The entry point calls no
// cudaMalloc, no cudaFree and no allocating library routine: one cudaMemsetAsync and two kernel launches.
//
// The array is shared by all calls and keeps the last call's contents, so every call clears the counters it
// uses first, on the caller's stream.  Calls that overlap on the GPU (different streams, or threads on
// different streams) race on it: serialise them.
//
// Self-contained on purpose: shares no code with the handle-based path (tpcclus.cu, tpcclus_kernels.cuh),
// which this file does not change.
#include <cuda_runtime.h>

#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/tpcclus.h"

namespace {

typedef unsigned int u32;
typedef unsigned long long u64;

constexpr u32 kMaxRows = TPCCLUS_NOALLOC_MAX_ROWS;   // (sector, row) pairs: 256 x 256
constexpr u32 kScanThreads = 1024;
constexpr int kMaxDevices = 64;

// The scratch: one counter per (sector, row).  In host code this name is a host-side stand-in, not a device
// address: the address the kernels get comes from cudaGetSymbolAddress (scratch_of_current_device below).
static __device__ __align__(256) u32 g_noalloc_counts[kMaxRows + 64];

// ---- kernel 1: pack every cluster, count the clusters of every (sector, row) -------------------------------
// in: 32-byte clusters (include/tpcclus.h: tpcclus_cluster) = two 16-byte words
//   a = pad_mean, time_mean, sigma_pad, sigma_time (float32 bits)
//   b = q_tot, q_max | time_peak << 16, pad_peak | row << 8 | sector << 16 | flags << 24, 0
// out: the 16-byte record of tpcclus_cluster16 (same arithmetic as K9p: IEEE-RN multiply, round to nearest even)
__global__ void __launch_bounds__(256) k_pack_list(const uint4* __restrict__ in, u64 n, uint4* __restrict__ out,
                                                   u32* __restrict__ counts, u32 n_rows, u32 n_maps) {
  const u32 lane = threadIdx.x & 31u;
  const u64 stride = (u64)gridDim.x * blockDim.x;
  for (u64 i0 = (u64)blockIdx.x * blockDim.x + (threadIdx.x & ~31u); i0 < n; i0 += stride) {   // warp-uniform trip count
    const u64 i = i0 + lane;
    u32 key = 0xFFFFFFFFu;
    if (i < n) {
      const uint4 a = in[2ull * i], b = in[2ull * i + 1ull];
      const u32 time_fix = __float2uint_rn(__fmul_rn(__uint_as_float(a.y), 256.0f));
      u32 pad_fix = __float2uint_rn(__fmul_rn(__uint_as_float(a.x), 256.0f));
      if (pad_fix > 65535u) pad_fix = 65535u;
      const u32 sp = __float2uint_rn(__fmul_rn(__uint_as_float(a.z), 16384.0f));
      const u32 st = __float2uint_rn(__fmul_rn(__uint_as_float(a.w), 16384.0f));
      uint4 o;
      o.x = time_fix | ((b.z & 0xFFu) << 24);
      o.y = pad_fix | (b.y & 0xFFFF0000u);
      o.z = (b.x & 0xFFFFu) | (((b.y & 0x3FFu) | ((b.z >> 24) << 10)) << 16);
      o.w = sp | (st << 16);
      out[i] = o;
      const u32 k = ((b.z >> 16) & 0xFFu) * n_rows + ((b.z >> 8) & 0xFFu);
      if (((b.z >> 8) & 0xFFu) < n_rows && k < n_maps) key = k;   // (a cluster of another geometry is packed, not indexed)
    }
    // The list is ordered by (sector, row): the lanes of a warp hold a few runs of equal keys.  One atomic per run.
    const u32 prev = __shfl_up_sync(0xFFFFFFFFu, key, 1);
    const u32 heads = __ballot_sync(0xFFFFFFFFu, lane == 0u || key != prev);
    if ((heads >> lane) & 1u) {
      const u32 after = heads & ~((2u << lane) - 1u);                 // heads behind this lane
      const u32 len = (after ? (u32)__ffs((int)after) - 1u : 32u) - lane;
      if (key != 0xFFFFFFFFu) atomicAdd(&counts[key], len);
    }
  }
}

// ---- kernel 2 (one CTA): row_index[m] = clusters of the maps before m, [n_maps] = all of them --------------
__global__ void __launch_bounds__(kScanThreads) k_row_index(const u32* __restrict__ counts, u32 n_maps, u64* __restrict__ row_index) {
  __shared__ u64 s_sum[kScanThreads];
  const u32 per = (n_maps + kScanThreads - 1u) / kScanThreads;
  const u32 lo = threadIdx.x * per;
  u32 hi = lo + per;
  if (hi > n_maps) hi = n_maps;
  u64 mine = 0ull;
  for (u32 m = lo; m < hi; ++m) mine += counts[m];
  s_sum[threadIdx.x] = mine;
  __syncthreads();
  for (u32 d = 1u; d < kScanThreads; d <<= 1) {   // inclusive scan of the per-thread sums
    const u64 v = threadIdx.x >= d ? s_sum[threadIdx.x - d] : 0ull;
    __syncthreads();
    s_sum[threadIdx.x] += v;
    __syncthreads();
  }
  u64 at = s_sum[threadIdx.x] - mine;
  for (u32 m = lo; m < hi; ++m) { row_index[m] = at; at += counts[m]; }
  if (threadIdx.x == kScanThreads - 1u) row_index[n_maps] = s_sum[threadIdx.x];
}

void say(char* err, uint32_t cap, const char* msg) {
  if (err && cap) snprintf(err, cap, "%s", msg);
}

// Set-up, once per device, with that device current: the device address of the scratch array.
u32* scratch_of_current_device(int* rc_cuda) {
  static std::mutex mu;
  static u32* ptr[kMaxDevices] = {};
  int dev = -1;
  cudaError_t e = cudaGetDevice(&dev);
  if (e != cudaSuccess || dev < 0 || dev >= kMaxDevices) { *rc_cuda = e != cudaSuccess ? (int)e : (int)cudaErrorInvalidDevice; return nullptr; }
  std::lock_guard<std::mutex> g(mu);
  if (!ptr[dev]) {
    void* p = nullptr;
    e = cudaGetSymbolAddress(&p, g_noalloc_counts);
    if (e != cudaSuccess || !p) { *rc_cuda = e != cudaSuccess ? (int)e : (int)cudaErrorInvalidSymbol; return nullptr; }
    ptr[dev] = (u32*)p;
  }
  return ptr[dev];
}

}  // namespace

extern "C" TPCCLUS_API int tpcclus_pack_noalloc(const tpcclus_cluster* d_clusters, uint64_t n, uint32_t n_sectors, uint32_t n_rows,
                                                tpcclus_cluster16* d_packed, uint64_t* d_row_index, void* cuda_stream,
                                                char* err, uint32_t err_cap) {
  char buf[200];
  if (err && err_cap) err[0] = 0;
  if (n_sectors < 1 || n_sectors > 256 || n_rows < 1 || n_rows > 256 || (uint64_t)n_sectors * n_rows > kMaxRows) {
    snprintf(buf, sizeof buf, "tpcclus_pack_noalloc: %u sectors x %u rows is beyond the %u (sector,row) pairs (256 x 256) the static scratch array holds",
             n_sectors, n_rows, kMaxRows);
    say(err, err_cap, buf);
    return TPCCLUS_ERR_INVALID_ARG;
  }
  if (n > TPCCLUS_NOALLOC_MAX_CLUSTERS) {
    snprintf(buf, sizeof buf, "tpcclus_pack_noalloc: %llu clusters is beyond the maximum of %llu (32-bit counters in the static scratch array)",
             (unsigned long long)n, (unsigned long long)TPCCLUS_NOALLOC_MAX_CLUSTERS);
    say(err, err_cap, buf);
    return TPCCLUS_ERR_INVALID_ARG;
  }
  if (!d_row_index || ((uintptr_t)d_row_index & 7u) || (n && (!d_clusters || !d_packed)) || ((uintptr_t)d_clusters & 15u) || ((uintptr_t)d_packed & 15u)) {
    say(err, err_cap, "tpcclus_pack_noalloc: null or misaligned buffer (clusters and packed records 16 bytes, row index 8 bytes)");
    return TPCCLUS_ERR_INVALID_ARG;
  }
  int rc_cuda = 0;
  u32* counts = scratch_of_current_device(&rc_cuda);
  if (!counts) {
    snprintf(buf, sizeof buf, "tpcclus_pack_noalloc: cudaGetSymbolAddress of the scratch array failed: %s", cudaGetErrorString((cudaError_t)rc_cuda));
    say(err, err_cap, buf);
    cudaGetLastError();
    return TPCCLUS_ERR_CUDA;
  }
  cudaStream_t st = (cudaStream_t)cuda_stream;
  const u32 n_maps = n_sectors * n_rows;
  cudaError_t e = cudaMemsetAsync(counts, 0, 4ull * n_maps, st);   // the array keeps the last call's counts
  if (e == cudaSuccess && n) {
    u64 blocks = (n + 255ull) / 256ull;
    if (blocks > 148ull * 8ull) blocks = 148ull * 8ull;
    k_pack_list<<<(unsigned)blocks, 256, 0, st>>>((const uint4*)d_clusters, n, (uint4*)d_packed, counts, n_rows, n_maps);
    e = cudaGetLastError();
  }
  if (e == cudaSuccess) {
    k_row_index<<<1, kScanThreads, 0, st>>>(counts, n_maps, (u64*)d_row_index);
    e = cudaGetLastError();
  }
  if (e != cudaSuccess) {
    snprintf(buf, sizeof buf, "tpcclus_pack_noalloc: %s", cudaGetErrorString(e));
    say(err, err_cap, buf);
    return TPCCLUS_ERR_CUDA;
  }
  return TPCCLUS_OK;
}
