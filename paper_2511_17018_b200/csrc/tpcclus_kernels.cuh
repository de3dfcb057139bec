// tpcclus_kernels.cuh -- device code of the B200-native TPC clusterizer (sm_100a).
//
// ONE source for both builds (PAPER.md 89-93, section 5): nvcc compiles it offline with
// the geometry/thresholds read from a __constant__ parameter block (PAPER.md 79-85), and
// create(TPCCLUS_RTC) hands the very same text to NVRTC with `#define TPC_RTC 1` and one
// `#define TPC_<field> <literal>` per parameter in front, so every PRM(x) below becomes a
// literal and the dead branches (e.g. the time-chunk duplication) fold away.
// Self-contained on purpose: no #include, so NVRTC needs no header search path.
//
// The path (rules: SURVEY.md 8(c) O0..O5):
//   K1 partition_coarse  digits(8 B) -> 4-byte records binned by (sector,row,time-chunk)
//   K2 dir_count / K3 dir_scan / K4 dir_fill   chunk directory -> per-bin chunk lists
//   K5 partition_fine    per bin: batch-local counting sort by time slab (+3-bin halo copy)
//   K6 cluster_tiles     per (sector,row,slab) tile: charge map in shared memory (O0),
//                        3x3 peaks (O1), suppression (O2), 5x5 CoG (O3,O4), compaction,
//                        ordered emission (O5)
#pragma once

// ---- compilation units (PAPER.md 64, section 3: "one source file per kernel", compiled straight to a
// GPU binary and loaded with cuModuleLoad).  TPC_UNITS is a bit mask of the kernel families this
// translation unit emits; the build compiles the text once per unit (csrc/tpcclus_unit.cu), every
// unit gets the register allocation that suits it and its own copy of the constant block, which
// the host's registry finds and fills (PAPER.md 81-85).  0 = declarations only (the host side).
#define TPC_U_PART_COARSE 0x001u   // k_partition_coarse
#define TPC_U_DIR 0x002u           // k_dir_count, k_dir_scan, k_dir_fill
#define TPC_U_PART_FINE 0x004u     // k_partition_fine
#define TPC_U_TILES_FAST 0x008u    // k_cluster_tiles_fast
#define TPC_U_TILES_DET 0x010u     // k_cluster_tiles_det_temp, k_cluster_tiles_det
#define TPC_U_ORDER 0x020u         // k_scan_local, k_scan_sums, k_emit_ordered, k_emit_packed
#define TPC_U_TILES_DUMP 0x040u    // k_cluster_tiles_dump_map (debug hook of step a1)
#define TPC_U_TILES_FAST_G 0x080u  // reading Q10' variants
#define TPC_U_TILES_DET_G 0x100u
#define TPC_U_TILES_FAST_S 0x200u  // reading Q10'' variants (compiled with TPC_HALO = 5, like the partition units they run behind)
#define TPC_U_TILES_DET_S 0x400u
#ifndef TPC_UNITS
#define TPC_UNITS 0xFFFFFFFFu
#endif

typedef unsigned int u32;
typedef unsigned long long u64;
typedef unsigned short u16;
typedef unsigned char u8;

// ---- fixed design constants ------------------------------------
#ifndef TPC_TS
#define TPC_TS 128u            // time bins a tile owns
#endif
#ifndef TPC_HALO
#define TPC_HALO 3u            // time halo: peaks at distance 2 need charges at distance 3 (O2); the units of reading
#endif                         // Q10'' are compiled with 5 (survivors at distance 2 need peaks at 4, charges at 5)
#define TPC_PG 3u              // zero guard pads on each side of a map row (no pad-edge branches)
#define TPC_TT (TPC_TS + 2u * TPC_HALO)   // rows of a tile in shared memory
#ifndef TPC_TC
#define TPC_TC 16256u          // time bins per coarse time-chunk: 127*128, +6 halo < 2^14
#endif
#define TPC_STAGE 8u           // records (32 B) staged per coarse bin in K1
#define TPC_CHUNK 64u          // records per pool chunk (256 B)
#define TPC_CPB 256u           // chunks per K5 batch (<= 16384 records)
#define TPC_K1_THREADS 1024
#define TPC_K1_DPT 4           // digits per thread per round
#define TPC_K5_THREADS 1024
#define TPC_SCAN_THREADS 1024
#define TPC_SCAN_PER_CTA 4096u

#define TPC_STATUS_OVERFLOW 1u
#define TPC_STATUS_BAD_DIGITS 2u
#define TPC_STATUS_INTERNAL 0x80000000u   // a capacity the host derived from max_digits was exceeded: a bug, results invalid

struct TpcParams {
  u32 n_sectors, n_rows, n_time;
  u32 n_tc;        // coarse time-chunks = ceil(n_time / TPC_TC)
  u32 n_bins;      // NB = n_sectors * n_rows * n_tc
  u32 n_sl;        // tiles (slabs) per bin = ceil(min(n_time, TPC_TC) / TPC_TS)
  u32 pitch;       // u16 cells per tile row = roundup8(max_pads + 6)
  u32 max_pads;
  u32 thr_peak, noise_eps;
  u32 max_peaks;   // capacity of the per-tile peak list
  u32 cog_mode;    // 0 = Q10, 1 = Q10' gated, 2 = Q10'' shared (host side only: selects the kernel variants)
  u32 k1_bins;     // coarse bins one K1 launch holds stages for: n_bins, or n_bins / passes (rounded up) beyond the shared-memory budget
  u16 n_pads[256];
};

// ---- declarations the host side shares (sizes of the dynamic shared memory, kernel arguments) ----
#define TPC_STATUS_NO_PACKED 4u
#define TPC_K1_FQ 2048u      // flush-queue entries (u16 bin ids)
#define TPC_K1_SPILL 512u    // spill entries per buffer (2 x u32)
__host__ __device__ inline u32 tpc_k1_smem_bytes(u32 nb) {
  return (nb * (TPC_STAGE + 2u) + 4u * TPC_K1_SPILL + 8u) * 4u + TPC_K1_FQ * 2u;
}
#ifndef TPC_NSLMAX
#define TPC_NSLMAX 128u   // >= slabs per bin: TPC_TC / TPC_TS = 127
#endif
#define TPC_NKEY (2u * TPC_NSLMAX + 32u)   // sort keys: 2 per slab + A of the slab after the last; multiple of 32
#define TPC_K5_BUF (TPC_CPB * TPC_CHUNK + 4u * TPC_NSLMAX + 8u)   // u32 words: the records of a batch + alignment gaps + end padding
__host__ __device__ inline u32 tpc_k5_smem_bytes() { return (TPC_K5_BUF + 2u * TPC_NKEY + 8u) * 4u; }
#define TPC_MODE_FAST 0
#define TPC_MODE_DET 1        // chained scan inside K6 (fallback: any number of clusters)
#define TPC_MODE_DET_TEMP 2   // runs into the temporary buffer, K7-K9 order them (the usual path)
#define TPC_MODE_DUMP_MAP 3
#ifndef TPC_K6_CONSUMERS
#define TPC_K6_CONSUMERS 256u                   // threads that compute
#endif
#define TPC_K6_THREADS (TPC_K6_CONSUMERS + 32u)  // + the producer warp
#define TPC_K6_THREADS_E (TPC_K6_THREADS + 32u)   // FAST kernels of the readings Q10 and Q10': + the emitter warp (K6, sparse tiles)
#define TPC_K6_BLK 256u                          // clusters of the temporary buffer a CTA reserves at a time (DET, sparse tiles)
#define TPC_K6_RING 64u                          // clusters in flight between the consumers and the emitter warp
#ifndef TPC_K6_CAP
#define TPC_K6_CAP 4096u                         // records staged per round (16 KB)
#endif
#define TPC_K6_CAPU (TPC_K6_CAP / 4u)            // ... in 16-byte units
#ifndef TPC_K6_CTAS
#define TPC_K6_CTAS 3                            // resident CTAs per SM (shared memory and registers)
#endif

struct K6Args {
  const u32* blob; const u64* idx; const u32* batch_start;
  uint4* out; u64 capacity; u64* n_clusters; u32* status;
  u32* ticket;        // next tile to hand out (zeroed per run)
  u64* tile_state;    // DET: chained scan of the tile counts, [n_tiles], zeroed per run
  uint4* temp; u64 temp_cap; u64* temp_cursor;   // DET_TEMP: run buffer (the dead K1 pool), in clusters
  u64* tile_base; u32* tile_cnt; u32* det_flag;  // DET_TEMP: per-tile (place, count); flag = buffer too small
  u16* dmap; const u64* row_off;   // DUMP_MAP only: row_off[r] = cells of rows < r in one sector; [n_rows] = per sector
};

#define TPC_K6_GROUP 4u   // tiles (consecutive slabs of one bin) a ticket covers
#define TPC_K6_PMW 9u
__host__ __device__ inline u32 tpc_k6_smem_bytes(u32 pitch, u32 max_peaks, u32 halo) {   // halo: the TPC_HALO of the handle's units
  const u32 tt = TPC_TS + 2u * halo;
  return (TPC_K6_CAP + tt * pitch / 2u + TPC_K6_RING * 8u + 4u + 4u + 2u + tt * (8u + TPC_K6_PMW) + tt + 2u + 16u + (max_peaks + 1u) / 2u) * 4u + 128u;
}

#ifdef TPC_RTC
#define PRM(x) (TPC_##x)
#define PRM_NPADS(r) (TPC_NPADS_TABLE[r])   // emitted by the host in front of this text
#else
#if TPC_UNITS != 0u
// One constant block per compilation unit (a non-RDC unit cannot see another unit's symbol:
// PAPER.md 81).  extern "C": the host's registry looks the symbol up by this name in every module
// it loads and keeps all copies up to date (PAPER.md 83-85).
extern "C" { __constant__ TpcParams c_prm; }
#endif
#define PRM(x) (c_prm.x)
#define PRM_NPADS(r) (c_prm.n_pads[r])
#endif
#if TPC_UNITS != 0u   // ---- device code ------------------------------------------------------------

// ---- shared-memory sizes (bytes); the host launches with exactly these --------------------

// ---- small PTX helpers -------------------------------------------------------------------
__device__ __forceinline__ uint2 ld_stream_u2(const uint2* p) {   // read-once input: keep out of L1
  uint2 v;
  asm volatile("ld.global.nc.L1::no_allocate.v2.u32 {%0,%1}, [%2];" : "=r"(v.x), "=r"(v.y) : "l"(p));
  return v;
}
__device__ __forceinline__ uint4 ld_stream_u4(const uint4* p) {
  uint4 v;
  asm volatile("ld.global.nc.L1::no_allocate.v4.u32 {%0,%1,%2,%3}, [%4];"
               : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "l"(p));
  return v;
}
__device__ __forceinline__ void st_256(void* p, uint4 a, uint4 b) {   // one 32-byte sector, one request
#ifdef TPC_NO_ST256   // an NVRTC older than 12.9 has no 256-bit vector store
  ((uint4*)p)[0] = a; ((uint4*)p)[1] = b;
  return;
#endif
  asm volatile("st.global.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(a.x), "r"(a.y), "r"(a.z),
               "r"(a.w), "r"(b.x), "r"(b.y), "r"(b.z), "r"(b.w) : "memory");
}
__device__ __forceinline__ u32 lane_id() { return threadIdx.x & 31u; }

// ==========================================================================================
// K1  partition_coarse  (NS (1) "digit -> charge-map scatter", first half: O0's validity,
//     clamp and zero rules, and the routing of each digit to its (sector,row) map)
//
// One persistent CTA per SM.  Shared memory holds a 32-byte write-combining stage per
// coarse bin; a full stage leaves as ONE 32-byte sector store into a 256-byte chunk that
// is private to (CTA, bin), so there is no global atomic and no histogram pre-pass.
// The chunk directory dir[] (bin<<8 | records) is turned into per-bin lists by K2..K4.
//
// A round = 4096 digits, two block barriers:
//   insert : slot = atomicAdd(cnt[bin]); slot < 8 -> the record goes into the stage; the
//            writer of slot 7 queues the bin for flushing; slot >= 8 (the stage is full until
//            the flush) -> the record is parked in a small spill list, its slot stays reserved
//            and it is written at the head of the next round (slot - 8).
//   flush  : the queue is worked off densely, two lanes per 32-byte stage, cnt[bin] -= 8.
// Any skew is legal: when the spill list or the flush queue is full a thread keeps its
// record in registers and the round repeats (flush, slot -= 8) until everything is placed.
//
// record (4 B):  pad[0:8) | u[8:22) | q[22:32)   with u = time - tc*TPC_TC + 3  (14 bit)
// ==========================================================================================

struct K1Smem {   // layout computed identically on the host (tpc_k1_smem_bytes)
  u32* stage;     // [NB][8]
  u32* cnt;       // [NB]  records reserved in the stage (may exceed 8 until the flush)
  u32* pos;       // [NB]  (chunk_local << 4) | sectors_filled(0..8)
  u32* spill;     // [2][warps][TPC_K1_WSP][2]  {rec, bin | slot << 16}
  u32* misc;      // [0] next chunk
  u16* fq;        // [warps][TPC_K1_WFQ]
  u32 bin_lo;     // first bin of this pass (bins are local to the pass in shared memory, global in dir[])
};
__device__ __forceinline__ K1Smem k1_smem(u32* base, u32 nb, u32 bin_lo) {   // fixed-size arrays first: constant offsets
  K1Smem s;
  s.bin_lo = bin_lo;
  s.misc = base;
  s.spill = s.misc + 8;
  s.fq = (u16*)(s.spill + 4u * TPC_K1_SPILL);
  s.stage = (u32*)(s.fq + TPC_K1_FQ);
  s.cnt = s.stage + nb * TPC_STAGE;
  s.pos = s.cnt + nb;
  return s;
}

// Moves the full stage of `bin` into the pool: lane pair (even, odd) = the two 16-byte halves.
// Called with all 32 lanes; `act` marks the pairs that carry a bin.
__device__ __forceinline__ void k1_flush_pair(const K1Smem& s, bool act, u32 bin, u32 slice_base, u32 slice_cap,
                                              uint4* pool, u32* dir) {
  const u32 half = threadIdx.x & 1u;
  u32 sector = 0xFFFFFFFFu;   // index of the 32-byte sector inside this CTA's slice
  if (act && half == 0u) {
    const u32 p = s.pos[bin];
    u32 fill = p & 15u, c = p >> 4;
    if (fill == 8u) {
      c = atomicAdd(&s.misc[0], 1u);
      fill = 0u;
      if (c < slice_cap) dir[slice_base + c] = ((bin + s.bin_lo) << 8) | TPC_CHUNK;
    }
    s.pos[bin] = (c << 4) | (fill + 1u);
    s.cnt[bin] -= 8u;   // one flush per bin and phase: no other thread touches cnt[bin] here
    if (c < slice_cap) sector = c * 8u + fill;
  }
  sector = __shfl_sync(0xFFFFFFFFu, sector, (int)(lane_id() & ~1u));
  if (act && sector != 0xFFFFFFFFu) {
    const uint4 v = ((const uint4*)s.stage)[bin * 2u + half];
    pool[((u64)slice_base * 8u + sector) * 2u + half] = v;
  }
}
__device__ __forceinline__ void k1_flush_single(const K1Smem& s, u32 bin, u32 slice_base, u32 slice_cap, uint4* pool, u32* dir) {
  const u32 p = s.pos[bin];
  u32 fill = p & 15u, c = p >> 4;
  if (fill == 8u) {
    c = atomicAdd(&s.misc[0], 1u);
    fill = 0u;
    if (c < slice_cap) dir[slice_base + c] = ((bin + s.bin_lo) << 8) | TPC_CHUNK;
  }
  s.pos[bin] = (c << 4) | (fill + 1u);
  s.cnt[bin] -= 8u;
  const uint4* st = (const uint4*)(s.stage + bin * TPC_STAGE);
  if (c < slice_cap) st_256(pool + ((u64)(slice_base + c) * 16u + fill * 2u), st[0], st[1]);
}

#define TPC_K1_WFQ (TPC_K1_FQ / (TPC_K1_THREADS / 32))        // flush-queue entries per warp (64)
#define TPC_K1_WSP (TPC_K1_SPILL / (TPC_K1_THREADS / 32))     // spill entries per warp and buffer (16)

// One pass = insert phase + flush phase (two block barriers).  Entries k with bit k of `pend`
// set are still to be placed; FIRST = they have no reserved slot yet.  The flush queue and
// the spill list are private to the warp and filled with ballots, so the only shared-memory
// atomics are the slot reservations.  `nsp` = entries this warp parked in the previous pass.
// Returns (block-uniform) whether any thread still has a pending entry.  `between` runs after
// this warp's share of the flush and before the closing barrier: register-only work of the
// next round (its decode) goes there, where it fills the issue slots the flush -- a few warps
// on dependent shared-memory chains -- leaves idle.
struct K1Nothing { __device__ __forceinline__ void operator()() const {} };
template <int K, bool FIRST, class F = K1Nothing>
__device__ __forceinline__ bool k1_pass(const K1Smem& s, u32& cur, u32& nsp, const u32 (&bin)[K], const u32 (&rec)[K],
                                        u32 (&slot)[K], u32& pend, u32 slice_base, u32 slice_cap,
                                        uint4* pool, u32* dir, F between = F()) {
  u32 tid_ = threadIdx.x;
  asm volatile("" : "+r"(tid_));   // opaque: read the thread id once instead of re-deriving everything from S2R under register pressure
  const u32 lane = tid_ & 31u, warp = tid_ >> 5, lt = (1u << lane) - 1u;
  u16* fq = s.fq + warp * TPC_K1_WFQ;
  u32* sp_in = s.spill + ((cur * (TPC_K1_THREADS / 32) + warp) * TPC_K1_WSP) * 2u;
  u32* sp_out = s.spill + (((cur ^ 1u) * (TPC_K1_THREADS / 32) + warp) * TPC_K1_WSP) * 2u;
  u32 lf = 0u, drain_bin = 0u, nfq = 0u, nout = 0u;
  auto queue = [&](bool fl, u32 b, int bit) {   // warp-wide: every lane calls it
    const u32 m = __ballot_sync(0xFFFFFFFFu, fl);
    if (fl) {
      const u32 i = nfq + __popc(m & lt);
      if (i < TPC_K1_WFQ) fq[i] = (u16)b;
      else { lf |= 1u << bit; if (bit == K) drain_bin = b; }   // queue full: flush it myself
    }
    nfq += __popc(m);
  };
  {   // records parked in the previous pass: their bin was flushed since, slot - 8 < 8
    bool fl = false;
    u32 b = 0u;
    if (lane < nsp) {
      const u32 r = sp_in[2u * lane], w = sp_in[2u * lane + 1u];
      b = w & 0xFFFFu;
      const u32 sl = (w >> 16) - 8u;
      s.stage[b * TPC_STAGE + sl] = r;
      fl = sl == TPC_STAGE - 1u;
    }
    queue(fl, b, K);
  }
#pragma unroll
  for (int k = 0; k < K; ++k) {   // reserve: independent atomics first
    if (FIRST) slot[k] = (pend & (1u << k)) ? atomicAdd(&s.cnt[bin[k]], 1u) : 0xFFFFFFFFu;
    else slot[k] = (pend & (1u << k)) ? slot[k] - 8u : 0xFFFFFFFFu;
  }
#pragma unroll
  for (int k = 0; k < K; ++k) {
    const u32 sl = slot[k];
    if (sl < TPC_STAGE) { s.stage[bin[k] * TPC_STAGE + sl] = rec[k]; pend &= ~(1u << k); }
    queue(sl == TPC_STAGE - 1u, bin[k], k);
    const bool sp = sl >= TPC_STAGE && sl < 2u * TPC_STAGE;   // the stage is full until the flush: park it
    const u32 m = __ballot_sync(0xFFFFFFFFu, sp);
    if (sp) {
      const u32 i = nout + __popc(m & lt);
      if (i < TPC_K1_WSP) { sp_out[2u * i] = rec[k]; sp_out[2u * i + 1u] = bin[k] | (sl << 16); pend &= ~(1u << k); }
    }
    nout += __popc(m);
  }
  nsp = nout < TPC_K1_WSP ? nout : TPC_K1_WSP;
  __syncthreads();
  // ---- flush phase: every warp works off its own queue, one lane pair per 32-byte stage ----
  if (nfq > TPC_K1_WFQ) nfq = TPC_K1_WFQ;
  for (u32 j0 = 0u; j0 < nfq; j0 += 16u) {
    const u32 j = j0 + (lane >> 1);
    const bool act = j < nfq;
    k1_flush_pair(s, act, act ? (u32)fq[j] : 0u, slice_base, slice_cap, pool, dir);
  }
  if (lf) {   // the queue was full
#pragma unroll
    for (int k = 0; k < K; ++k)
      if (lf & (1u << k)) k1_flush_single(s, bin[k], slice_base, slice_cap, pool, dir);
    if (lf & (1u << K)) k1_flush_single(s, drain_bin, slice_base, slice_cap, pool, dir);
  }
  cur ^= 1u;
  between();
  return __syncthreads_or((int)pend) != 0;
}

// GENERAL: several coarse time-chunks (halo copies into the neighbouring chunk's bin) and / or several passes over
// the input (only the bins [bin_lo, bin_lo + k1_bins) of this pass are staged); false: one chunk, one pass
template <bool MULTI_TC>
__device__ __forceinline__ void k1_rounds(const K1Smem& s, const uint2* __restrict__ digits, u64 n, u32 n_rounds, u32 slice_base,
                                          u32 slice_cap, uint4* pool, u32* dir, u32& cur, u32& nsp, bool& bad) {
  const u32 S = PRM(n_sectors), R = PRM(n_rows), T = PRM(n_time), NTC = PRM(n_tc), KB = PRM(k1_bins);
  // The input is cut into (2 x warps x CTAs) regions of n_rounds x 64 digits; load h of warp w
  // walks region (2w + h) * CTAs + cta, 512 contiguous bytes per round (lane l: digits 2l, 2l+1).
  // A round of this CTA therefore draws from 64 places spread over the whole frame, so that
  // time- or sector-ordered input (readout order) fills the stages as evenly as shuffled
  // input does (measured: readout-ordered CFG[4] 26.3 -> 8.8 ms; shuffled 8.6 -> 9.0 ms).
  // Digits past the end read as 0 = "charge 0, ignored": no bounds checks in the decode.
  u64 off[TPC_K1_DPT / 2];
#pragma unroll
  for (int h = 0; h < TPC_K1_DPT / 2; ++h)
    off[h] = ((u64)((TPC_K1_DPT / 2) * (threadIdx.x >> 5) + h) * gridDim.x + blockIdx.x) * n_rounds * 64u + 2u * lane_id();
  // block-uniform: every region of this CTA lies inside the input (all CTAs but the last few)
  const bool inside = ((u64)((TPC_K1_DPT / 2) * (TPC_K1_THREADS / 32) - 1) * gridDim.x + blockIdx.x + 1u) * n_rounds * 64u <= n;
  auto fetch = [&](u32 j, uint4 (&d)[TPC_K1_DPT / 2]) {
    if (inside && j < n_rounds) {
#pragma unroll
      for (int h = 0; h < TPC_K1_DPT / 2; ++h) d[h] = ld_stream_u4((const uint4*)(digits + off[h] + (u64)j * 64u));
      return;
    }
#pragma unroll
    for (int h = 0; h < TPC_K1_DPT / 2; ++h) {
      const u64 i = off[h] + (u64)j * 64u;
      if (j < n_rounds && i + 1u < n) d[h] = ld_stream_u4((const uint4*)(digits + i));
      else if (j < n_rounds && i < n) { const uint2 v = ld_stream_u2(digits + i); d[h] = make_uint4(v.x, v.y, 0u, 0u); }
      else d[h] = make_uint4(0u, 0u, 0u, 0u);
    }
  };
  // O0's validity / clamp / zero rules and the routing of one round's digits
  auto decode = [&](const uint4 (&curd)[TPC_K1_DPT / 2], u32 (&bin)[TPC_K1_DPT], u32 (&rec)[TPC_K1_DPT], u32& pend,
                    u32 (&dbin)[TPC_K1_DPT], u32 (&drec)[TPC_K1_DPT], u32& dpend) {
    pend = 0u; dpend = 0u;
#pragma unroll
    for (int k = 0; k < TPC_K1_DPT; ++k) {
      const u32 w0 = (k & 1) ? curd[k >> 1].z : curd[k >> 1].x, w1 = (k & 1) ? curd[k >> 1].w : curd[k >> 1].y;
      u32 q = w0 & 0xFFFFu;
      const u32 t = w0 >> 16, pad = w1 & 0xFFu, row = (w1 >> 8) & 0xFFu, sec = (w1 >> 16) & 0xFFu;
      // O0 / Q4: out of range -> ignored + flagged (pad >= n_pads[row] is caught by K5, where the row is uniform)
      const bool valid = sec < S && row < R && t < T;
      bad |= !valid;
      q = q > 1023u ? 1023u : q;                                  // Q4: clamp
      // Q4: a digit with charge 0 is ignored -- but O0 tests its range first, and the pad is only known to be
      // in range in K5: such a digit travels there as a record with q = 0, is checked and dropped.  Only the
      // all-zero word (charge 0 at sector 0, row 0, pad 0, time 0: in range, nothing to flag; also what the
      // padding behind the input's end reads as) ends here.  Zero suppression makes both cases rare upstream.
      const bool ok = valid && (w0 | w1) != 0u;
      u32 tc = 0u, v = t;
      if (MULTI_TC) { tc = t / TPC_TC; v = t - tc * TPC_TC; }
      const u32 b0 = MULTI_TC ? (sec * R + row) * NTC + tc : sec * R + row;
      const bool mine = ok && (!MULTI_TC || b0 - s.bin_lo < KB);   // (unsigned: also false below bin_lo)
      bin[k] = mine ? b0 - (MULTI_TC ? s.bin_lo : 0u) : 0u;
      rec[k] = pad | ((v + TPC_HALO) << 8) | (q << 22);
      pend |= mine ? (1u << k) : 0u;
      if (MULTI_TC) {   // halo copy into the neighbouring time-chunk's bin
        dbin[k] = 0u; drec[k] = 0u;
        if (ok && v < TPC_HALO && tc > 0u && b0 - 1u - s.bin_lo < KB) {
          dbin[k] = b0 - 1u - s.bin_lo; drec[k] = pad | ((v + TPC_TC + TPC_HALO) << 8) | (q << 22); dpend |= 1u << k;
        } else if (ok && v + TPC_HALO >= TPC_TC && tc + 1u < NTC && b0 + 1u - s.bin_lo < KB) {
          dbin[k] = b0 + 1u - s.bin_lo; drec[k] = pad | ((v + TPC_HALO - TPC_TC) << 8) | (q << 22); dpend |= 1u << k;
        }
      }
    }
  };
  uint4 nxt[TPC_K1_DPT / 2];
  fetch(0u, nxt);
  if (!MULTI_TC) {
    // Software pipeline: the digits of round j+1 are decoded inside round j's flush phase and the
    // loads of round j+2 issued behind them, so a round is insert | barrier | flush + decode | barrier.
    u32 bin[TPC_K1_DPT], rec[TPC_K1_DPT], slot[TPC_K1_DPT], nbin[TPC_K1_DPT], nrec[TPC_K1_DPT], unused[TPC_K1_DPT];
    u32 pend, npend = 0u, dp;
    decode(nxt, bin, rec, pend, unused, unused, dp);
    fetch(1u, nxt);
    for (u32 j = 0u; j < n_rounds; ++j) {
      auto next_round = [&]() {
        decode(nxt, nbin, nrec, npend, unused, unused, dp);   // past the end: all zero, nothing pending
        fetch(j + 2u, nxt);
      };
      if (k1_pass<TPC_K1_DPT, true>(s, cur, nsp, bin, rec, slot, pend, slice_base, slice_cap, pool, dir, next_round))
        while (k1_pass<TPC_K1_DPT, false>(s, cur, nsp, bin, rec, slot, pend, slice_base, slice_cap, pool, dir)) {}
#pragma unroll
      for (int k = 0; k < TPC_K1_DPT; ++k) { bin[k] = nbin[k]; rec[k] = nrec[k]; }
      pend = npend;
    }
  } else
  for (u32 j = 0u; j < n_rounds; ++j) {
    uint4 curd[TPC_K1_DPT / 2];
#pragma unroll
    for (int h = 0; h < TPC_K1_DPT / 2; ++h) curd[h] = nxt[h];
    fetch(j + 1u, nxt);   // prefetch the next round while this one is binned
    u32 bin[TPC_K1_DPT], rec[TPC_K1_DPT], slot[TPC_K1_DPT], dbin[TPC_K1_DPT], drec[TPC_K1_DPT];
    u32 pend = 0u, dpend = 0u;
    decode(curd, bin, rec, pend, dbin, drec, dpend);
    if (k1_pass<TPC_K1_DPT, true>(s, cur, nsp, bin, rec, slot, pend, slice_base, slice_cap, pool, dir))
      while (k1_pass<TPC_K1_DPT, false>(s, cur, nsp, bin, rec, slot, pend, slice_base, slice_cap, pool, dir)) {}
    if (__syncthreads_or((int)dpend)) {
      if (k1_pass<TPC_K1_DPT, true>(s, cur, nsp, dbin, drec, slot, dpend, slice_base, slice_cap, pool, dir))
        while (k1_pass<TPC_K1_DPT, false>(s, cur, nsp, dbin, drec, slot, dpend, slice_base, slice_cap, pool, dir)) {}
    }
  }
}

#if TPC_UNITS & TPC_U_PART_COARSE
extern "C" __global__ void __launch_bounds__(TPC_K1_THREADS, 1)
k_partition_coarse(const uint2* __restrict__ digits, u64 n, u64 per_cta, uint4* __restrict__ pool,
                   u32* __restrict__ dir, u32* __restrict__ used, u32 slice_cap, u32* __restrict__ status, u32 bin_lo) {
  // A geometry with more coarse bins than shared memory has stages for (5503) is binned in several passes over the
  // input, pass p staging the bins [p * k1_bins, (p + 1) * k1_bins): `bin_lo` = the first of them.  A pass
  // continues this CTA's slice of the pool where the pass before stopped (used[]).
  extern __shared__ __align__(128) u32 smem_u32[];
  const u32 nb = PRM(k1_bins);
  const K1Smem s = k1_smem(smem_u32, nb, bin_lo);
  for (u32 i = threadIdx.x; i < nb; i += TPC_K1_THREADS) { s.pos[i] = 8u; s.cnt[i] = 0u; }
  if (threadIdx.x < 8) s.misc[threadIdx.x] = (threadIdx.x == 0 && bin_lo != 0u) ? used[blockIdx.x] : 0u;
  __syncthreads();

  const u32 slice_base = blockIdx.x * slice_cap;
  const u32 n_rounds = (u32)(per_cta / (TPC_K1_THREADS * TPC_K1_DPT));   // per_cta is a multiple of the round
  u32 cur = 0u, nsp = 0u;
  bool bad = false;
  if (PRM(n_tc) > 1u || PRM(k1_bins) < PRM(n_bins)) k1_rounds<true>(s, digits, n, n_rounds, slice_base, slice_cap, pool, dir, cur, nsp, bad);
  else { K1Smem s0 = s; s0.bin_lo = 0u;   // (known to be 0 here: keeps the add out of the flush of the common instance)
         k1_rounds<false>(s0, digits, n, n_rounds, slice_base, slice_cap, pool, dir, cur, nsp, bad); }
  if (bad) atomicOr(status, TPC_STATUS_BAD_DIGITS);
  {   // records still parked in the spill lists
    u32 bin[1] = {0u}, rec[1] = {0u}, slot[1] = {0u}, pend = 0u;
    while (__syncthreads_or((int)nsp)) k1_pass<1, false>(s, cur, nsp, bin, rec, slot, pend, slice_base, slice_cap, pool, dir);
  }
  __syncthreads();
  // drain: every bin's partial stage goes to its current (or a fresh) chunk, unused slots zeroed;
  // fix the record count of that last chunk in the directory.
  for (u32 b = threadIdx.x; b < nb; b += TPC_K1_THREADS) {
    const u32 m = s.cnt[b];   // 0..7 staged
    const u32 p = s.pos[b];
    u32 fill = p & 15u, c = p >> 4;
    if (m != 0u) {
      if (fill == 8u) { c = atomicAdd(&s.misc[0], 1u); fill = 0u; }
      u32* stw = s.stage + b * TPC_STAGE;
      for (u32 k = m; k < TPC_STAGE; ++k) stw[k] = 0u;
      const uint4* st = (const uint4*)stw;
      if (c < slice_cap) {
        st_256(pool + ((u64)(slice_base + c) * 16u + fill * 2u), st[0], st[1]);
        dir[slice_base + c] = ((b + bin_lo) << 8) | (fill * 8u + m);
      }
    } else if (fill != 8u && fill != 0u) {
      if (c < slice_cap) dir[slice_base + c] = ((b + bin_lo) << 8) | (fill * 8u);
    }
  }
  __syncthreads();
  if (threadIdx.x == 0) {
    u32 u = s.misc[0];
    if (u > slice_cap) { u = slice_cap; atomicOr(status, TPC_STATUS_INTERNAL); }   // cannot happen (bound in DESIGN.md; provoked by tpcclus_debug_shrink)
    used[blockIdx.x] = u;
  }
}
#endif

// ==========================================================================================
// K2..K4  chunk directory -> per-bin chunk lists (bookkeeping of the scatter; ~2.6e7 chunks
// at CFG[4], 4 bytes each).  One CTA per K1 slice with a shared-memory histogram, so there
// are no global atomics on hot addresses: K2 counts chunks per (slice, bin) and adds its row
// to the per-bin totals (one spread reduction per non-empty entry), K3 -- a single CTA -- scans
// the NB totals into bin and batch offsets, K4 derives its slice's cursors from the count
// matrix (slices of one bin follow each other) and places the chunk ids.  The order of chunks inside
// a (slice, bin) group is whatever the shared atomics give: nothing downstream depends on
// it (the map build is a max, O0/Q5).
// ==========================================================================================
// K0: the per-run counters (status, cursors, ticket, chained-scan states, per-bin totals) start at zero, and so
// do the caller's status word and -- in FAST mode -- its cluster count.  A kernel, not cudaMemsetAsync: a memset
// of this size goes to a copy engine, where it would queue behind the 13 GB host-to-device copy of the NEXT
// frame of the host pipeline (tpcclus_host_submit) and hold up this frame's run for 230 ms.
#if TPC_UNITS & TPC_U_DIR
extern "C" __global__ void __launch_bounds__(256)
k_reset(uint4* __restrict__ counters, u64 n16, u32* __restrict__ status, u64* __restrict__ n_out) {
  for (u64 i = (u64)blockIdx.x * 256u + threadIdx.x; i < n16; i += (u64)gridDim.x * 256u) counters[i] = make_uint4(0u, 0u, 0u, 0u);
  if (blockIdx.x == 0 && threadIdx.x == 0) {
    if (status) *status = 0u;
    if (n_out) *n_out = 0ull;
  }
}
#endif
// The result of a frame of the host pipeline (count, status) goes to the host through a store into mapped pinned
// memory: a 16-byte device-to-host cudaMemcpyAsync can land on the copy engine that is busy with the next
// frame's 13 GB host-to-device copy and would then wait for all of it.
#if TPC_UNITS & TPC_U_DIR
extern "C" __global__ void k_publish(u64* __restrict__ host_res, const u64* __restrict__ n_clusters, const u32* __restrict__ status) {
  if (threadIdx.x == 0 && blockIdx.x == 0) {
    host_res[1] = (u64)*status;
    __threadfence_system();
    host_res[0] = *n_clusters;
    __threadfence_system();
  }
}
#endif
#if TPC_UNITS & TPC_U_DIR
extern "C" __global__ void __launch_bounds__(TPC_SCAN_THREADS)
k_dir_count(const u32* __restrict__ dir, const u32* __restrict__ used, u32 slice_cap, u32* __restrict__ slice_cnt,
            u32* __restrict__ bin_total) {   // bin_total = bin_chunk_start, zeroed at the head of the run
  extern __shared__ __align__(128) u32 smem_u32[];
  const u32 nb = PRM(n_bins);
  for (u32 i = threadIdx.x; i < nb; i += TPC_SCAN_THREADS) smem_u32[i] = 0u;
  __syncthreads();
  const u32 n = used[blockIdx.x];
  const u32* d = dir + (u64)blockIdx.x * slice_cap;
  for (u32 c = threadIdx.x; c < n; c += TPC_SCAN_THREADS) atomicAdd(&smem_u32[d[c] >> 8], 1u);
  __syncthreads();
  for (u32 i = threadIdx.x; i < nb; i += TPC_SCAN_THREADS) {
    const u32 c = smem_u32[i];
    slice_cnt[(u64)blockIdx.x * ((nb + 3u) & ~3u) + i] = c;   // row pitch: a multiple of 4 entries (K4 reads 16 bytes)
    if (c != 0u) atomicAdd(&bin_total[i], c);   // integer sum: the order does not matter
  }
}
#endif

// single CTA: exclusive scans over the bins.
//   bin_chunk_start[b] = sum_{b'<b} nchunks[b']          (NB+1 entries)
//   batch_start[b]     = sum_{b'<b} ceil(nchunks[b']/CPB) (NB+1 entries; [NB] = total batches)
//   batch_bin[k]       = the bin batch k belongs to
// On entry bin_chunk_start[b] holds nchunks[b] (summed over the slices by K2).
#if TPC_UNITS & TPC_U_DIR
extern "C" __global__ void __launch_bounds__(TPC_SCAN_THREADS)
k_dir_scan(u32* __restrict__ bin_chunk_start, u32* __restrict__ batch_start, u32* __restrict__ batch_bin) {
  extern __shared__ __align__(128) u32 smem_u32[];   // [nb] chunks per bin
  __shared__ u32 s_a[TPC_SCAN_THREADS], s_b[TPC_SCAN_THREADS];
  const u32 nb = PRM(n_bins);
  for (u32 b = threadIdx.x; b < nb; b += TPC_SCAN_THREADS) smem_u32[b] = bin_chunk_start[b];
  __syncthreads();
  const u32 per = (nb + TPC_SCAN_THREADS - 1u) / TPC_SCAN_THREADS;
  const u32 lo = threadIdx.x * per;
  u32 hi = lo + per;
  if (hi > nb) hi = nb;
  u32 sa = 0u, sb = 0u;
  for (u32 b = lo; b < hi; ++b) { u32 c = smem_u32[b]; sa += c; sb += (c + TPC_CPB - 1u) / TPC_CPB; }
  s_a[threadIdx.x] = sa; s_b[threadIdx.x] = sb;
  __syncthreads();
  for (u32 d = 1u; d < TPC_SCAN_THREADS; d <<= 1) {   // Hillis-Steele inclusive scan
    u32 va = 0u, vb = 0u;
    if (threadIdx.x >= d) { va = s_a[threadIdx.x - d]; vb = s_b[threadIdx.x - d]; }
    __syncthreads();
    s_a[threadIdx.x] += va; s_b[threadIdx.x] += vb;
    __syncthreads();
  }
  u32 ea = s_a[threadIdx.x] - sa, eb = s_b[threadIdx.x] - sb;   // exclusive prefix of this thread's range
  for (u32 b = lo; b < hi; ++b) {
    u32 c = smem_u32[b];
    bin_chunk_start[b] = ea; batch_start[b] = eb;
    const u32 nbt = (c + TPC_CPB - 1u) / TPC_CPB;
    for (u32 k = 0u; k < nbt; ++k) batch_bin[eb + k] = b;   // batch -> its bin, for K5
    ea += c; eb += nbt;
  }
  if (threadIdx.x == TPC_SCAN_THREADS - 1u) { bin_chunk_start[nb] = s_a[threadIdx.x]; batch_start[nb] = s_b[threadIdx.x]; }
}
#endif

#if TPC_UNITS & TPC_U_DIR
extern "C" __global__ void __launch_bounds__(TPC_SCAN_THREADS)
k_dir_fill(const u32* __restrict__ dir, const u32* __restrict__ used, u32 slice_cap,
           const u32* __restrict__ slice_cnt, const u32* __restrict__ bin_chunk_start, u32* __restrict__ chunk_list, u32 n_pass) {
  extern __shared__ __align__(128) u32 smem_u32[];   // [nb] cursors of this slice
  const u32 nb = PRM(n_bins);
  // cursor of slice s in bin i = bin start + the counts of the slices before it = bin end - the
  // counts of the slices from s on: whichever is the shorter column walk (the matrix sits in L2)
  const u32 s = blockIdx.x, ns = gridDim.x, nq = (nb + 3u) >> 2;   // 16-byte words per matrix row
  const bool fwd = 2u * s <= ns;
  const u32 k0 = fwd ? 0u : s, k1 = fwd ? s : ns;
  const uint4* m4 = (const uint4*)slice_cnt;
  for (u32 j = threadIdx.x; j < nq; j += TPC_SCAN_THREADS) {   // four bins per thread and load
    uint4 acc = make_uint4(0u, 0u, 0u, 0u);
#pragma unroll 8
    for (u32 k = k0; k < k1; ++k) {
      const uint4 v = m4[(u64)k * nq + j];
      acc.x += v.x; acc.y += v.y; acc.z += v.z; acc.w += v.w;
    }
    const u32 a[4] = {acc.x, acc.y, acc.z, acc.w};
#pragma unroll
    for (u32 e = 0u; e < 4u; ++e) {
      const u32 i = 4u * j + e;   // entries past nb are row padding
      if (i < nb) smem_u32[i] = fwd ? bin_chunk_start[i] + a[e] : bin_chunk_start[i + 1u] - a[e];
    }
  }
  __syncthreads();
  const u32 n = used[blockIdx.x];
  const u32 id0 = blockIdx.x * slice_cap;
  // (bound by the scattered 4-byte stores: eight directory loads in flight per thread changed nothing)
  // In n_pass passes over the slice's directory (the host picks one pass per 64 MB of lists: 2 at CFG[4]), each
  // placing the chunks of one range of bins: all CTAs together then write into 1/n_pass of the lists at a time, so
  // that the eight 4-byte stores into one 32-byte sector meet in L2 instead of going to DRAM one by one (the 104 MB
  // of lists of CFG[4], written in one pass, do not: 0.36 ms; in two passes 0.26 ms, a pass costing 0.09 ms).
  const u32 per_pass = (nb + n_pass - 1u) / n_pass;
  for (u32 pass = 0u; pass < n_pass; ++pass) {
    const u32 lo = pass * per_pass;
    for (u32 c0 = threadIdx.x; c0 < n; c0 += 4u * TPC_SCAN_THREADS) {   // four directory entries in flight per thread
      u32 d[4];
#pragma unroll
      for (int k = 0; k < 4; ++k) { const u32 c = c0 + (u32)k * TPC_SCAN_THREADS; d[k] = c < n ? dir[id0 + c] : 0xFFFFFFFFu; }
#pragma unroll
      for (int k = 0; k < 4; ++k) {
        // entry = chunk id [0:26) | (records - 1) [26:32): K5 gets the count with the id instead of from a scattered 4-byte read of dir[]
        const u32 c = c0 + (u32)k * TPC_SCAN_THREADS;
        if ((d[k] >> 8) - lo < per_pass) chunk_list[atomicAdd(&smem_u32[d[k] >> 8], 1u)] = (id0 + c) | (((d[k] & 0xFFu) - 1u) << 26);
      }
    }
  }
}
#endif

// ==========================================================================================
// K7/K8/K9  deterministic mode, ordered output (O5 / PAPER.md 47-50: an ordered scan and an
// ordered copy after the kernel whose output order depends on the concurrency).  K6 emits each
// tile's clusters, already in (time,pad) order, as one run at an atomically allocated place of
// a temporary buffer and records (place, count) per tile; K7/K8 scan the counts; K9 copies the
// runs to their final places in tile order.
// ==========================================================================================
#if TPC_UNITS & TPC_U_ORDER
extern "C" __global__ void __launch_bounds__(TPC_SCAN_THREADS)
k_scan_local(const u32* __restrict__ in, u32* __restrict__ out_local, u32* __restrict__ block_sum, u32 n) {
  __shared__ u32 s[TPC_SCAN_THREADS];
  const u32 base = blockIdx.x * TPC_SCAN_PER_CTA + threadIdx.x * 4u;
  u32 v[4], t = 0u;
#pragma unroll
  for (int k = 0; k < 4; ++k) { v[k] = (base + k < n) ? in[base + k] : 0u; t += v[k]; }
  s[threadIdx.x] = t;
  __syncthreads();
  for (u32 d = 1u; d < TPC_SCAN_THREADS; d <<= 1) {
    u32 a = threadIdx.x >= d ? s[threadIdx.x - d] : 0u;
    __syncthreads();
    s[threadIdx.x] += a;
    __syncthreads();
  }
  u32 e = s[threadIdx.x] - t;
#pragma unroll
  for (int k = 0; k < 4; ++k) { if (base + k < n) out_local[base + k] = e; e += v[k]; }
  if (threadIdx.x == TPC_SCAN_THREADS - 1u) block_sum[blockIdx.x] = s[threadIdx.x];
}
#endif

// single CTA: block_prefix[i] = sum_{j<i} block_sum[j] (64 bit); *total = grand total.
#if TPC_UNITS & TPC_U_ORDER
extern "C" __global__ void __launch_bounds__(TPC_SCAN_THREADS)
k_scan_sums(const u32* __restrict__ block_sum, u64* __restrict__ block_prefix, u32 nblocks, u64* __restrict__ total) {
  __shared__ u64 s[TPC_SCAN_THREADS];
  __shared__ u64 carry;
  if (threadIdx.x == 0) carry = 0ull;
  __syncthreads();
  for (u32 base = 0u; base < nblocks; base += TPC_SCAN_THREADS) {
    u32 i = base + threadIdx.x;
    u64 v = i < nblocks ? (u64)block_sum[i] : 0ull;
    s[threadIdx.x] = v;
    __syncthreads();
    for (u32 d = 1u; d < TPC_SCAN_THREADS; d <<= 1) {
      u64 a = threadIdx.x >= d ? s[threadIdx.x - d] : 0ull;
      __syncthreads();
      s[threadIdx.x] += a;
      __syncthreads();
    }
    if (i < nblocks) block_prefix[i] = carry + s[threadIdx.x] - v;
    __syncthreads();
    if (threadIdx.x == TPC_SCAN_THREADS - 1u) carry += s[threadIdx.x];
    __syncthreads();
  }
  if (threadIdx.x == 0) *total = carry;
}
#endif


// K9: one warp per tile, 16 bytes per lane.  Skipped as a whole (flag set) when the temporary
// buffer was too small: the chained-scan variant of K6 then redoes the frame (k6_chain).
#if TPC_UNITS & TPC_U_ORDER
extern "C" __global__ void __launch_bounds__(256)
k_emit_ordered(const uint4* __restrict__ temp, const u64* __restrict__ tile_base, const u32* __restrict__ tile_cnt,
               const u32* __restrict__ tile_local, const u64* __restrict__ block_prefix, u32 n_tiles,
               uint4* __restrict__ out, u64 capacity, const u32* __restrict__ flag, u32* __restrict__ status, u32* __restrict__ ticket) {
  if (blockIdx.x == 0 && threadIdx.x == 0) *ticket = 0u;   // fresh tickets for the chained-scan K6 that follows (normally idle)
  if (*flag != 0u) return;
  const u32 lane = threadIdx.x & 31u;
  bool over = false;
  for (u32 tile = blockIdx.x * 8u + (threadIdx.x >> 5); tile < n_tiles; tile += gridDim.x * 8u) {
    const u32 cnt = tile_cnt[tile];
    if (cnt == 0u) continue;
    const u64 src = tile_base[tile] * 2ull;
    const u64 dst0 = block_prefix[tile / TPC_SCAN_PER_CTA] + tile_local[tile];
    u64 keep = capacity > dst0 ? capacity - dst0 : 0ull;   // Q22: the first `capacity` clusters stay, in order
    if (keep < cnt) over = true; else keep = cnt;
    for (u32 i = lane; i < (u32)keep * 2u; i += 32u) out[dst0 * 2ull + i] = temp[src + i];
  }
  if (over) atomicOr(status, TPC_STATUS_OVERFLOW);
}
#endif

// K9p: the packed variant of K9 (O6: 16-byte fixed-point record) plus
// the per-row index.  One warp per tile, one cluster per lane; the first tile of every pad row
// also writes where that row starts.  When the run buffer was too small (flag) nothing is
// written but the NO_PACKED status bit.
#if TPC_UNITS & TPC_U_ORDER
extern "C" __global__ void __launch_bounds__(256)
k_emit_packed(const uint4* __restrict__ temp, const u64* __restrict__ tile_base, const u32* __restrict__ tile_cnt,
              const u32* __restrict__ tile_local, const u64* __restrict__ block_prefix, u32 n_tiles,
              uint4* __restrict__ out, u64 capacity, u64* __restrict__ row_index, const u32* __restrict__ flag,
              u32* __restrict__ status) {
  if (*flag != 0u) {
    if (blockIdx.x == 0 && threadIdx.x == 0) atomicOr(status, TPC_STATUS_NO_PACKED);
    return;
  }
  const u32 lane = threadIdx.x & 31u;
  const u32 tiles_per_row = PRM(n_tc) * PRM(n_sl);   // bins of one (sector,row) are consecutive
  bool over = false;
  for (u32 tile = blockIdx.x * 8u + (threadIdx.x >> 5); tile <= n_tiles; tile += gridDim.x * 8u) {
    const u64 dst0 = tile < n_tiles ? block_prefix[tile / TPC_SCAN_PER_CTA] + tile_local[tile]
                                    : block_prefix[(n_tiles - 1u) / TPC_SCAN_PER_CTA] + tile_local[n_tiles - 1u] + tile_cnt[n_tiles - 1u];
    if (lane == 0u && tile % tiles_per_row == 0u) row_index[tile / tiles_per_row] = dst0;   // incl. the end sentinel
    if (tile == n_tiles) break;
    const u32 cnt = tile_cnt[tile];
    if (cnt == 0u) continue;
    const u64 src = tile_base[tile] * 2ull;
    u64 keep = capacity > dst0 ? capacity - dst0 : 0ull;   // Q22: the first `capacity` clusters stay, in order
    if (keep < cnt) over = true; else keep = cnt;
    for (u32 i = lane; i < (u32)keep; i += 32u) {
      const uint4 a = temp[src + 2ull * i], b = temp[src + 2ull * i + 1ull];
      // a = pad_mean, time_mean, sigma_pad, sigma_time (float32 bits); b = q_tot, q_max | time_peak << 16,
      // pad_peak | row << 8 | sector << 16 | flags << 24, 0
      const u32 time_fix = __float2uint_rn(__fmul_rn(__uint_as_float(a.y), 256.0f));
      u32 pad_fix = __float2uint_rn(__fmul_rn(__uint_as_float(a.x), 256.0f));
      if (pad_fix > 65535u) pad_fix = 65535u;
      const u32 sp = __float2uint_rn(__fmul_rn(__uint_as_float(a.z), 16384.0f));
      const u32 st = __float2uint_rn(__fmul_rn(__uint_as_float(a.w), 16384.0f));
      uint4 o;
      o.x = time_fix | ((b.z & 0xFFu) << 24);
      o.y = pad_fix | (b.y & 0xFFFF0000u);                                  // pad_fix | time_peak << 16
      o.z = (b.x & 0xFFFFu) | (((b.y & 0x3FFu) | ((b.z >> 24) << 10)) << 16);   // q_tot | (q_max | flags << 10) << 16
      o.w = sp | (st << 16);
      out[dst0 + i] = o;
    }
  }
  if (over) atomicOr(status, TPC_STATUS_OVERFLOW);
}
#endif

// ==========================================================================================
// K5  partition_fine  (NS (1), second half: group every record with the tile(s) whose shared-
//     memory charge map needs it)
//
// A batch = up to TPC_CPB chunks (<= 16384 records) of ONE coarse bin.  The CTA counting-sorts
// the batch in shared memory and writes it as one contiguous blob.  Sort key = 2 * slab + (m >= 6)
// with u = slab * TS + m: each slab is split into its first 6 rows (A) and the rest (B), so the
// layout is  A0 B0 A1 B1 A2 ...  and tile `sl`, which needs u in [sl*TS, sl*TS + TS + 6), reads
// the CONTIGUOUS range A_sl B_sl A_sl+1.  The border rows A are shared by two tiles instead of
// being copied: no halo duplicates, one shared atomic per record.  Every A starts on a 4-record
// (16-byte, the bulk-copy alignment) boundary, zero records filling the gap after the B before,
// so a tile's range starts aligned; rounding its end up to 16 bytes can only reach into B_sl+1,
// whose records (other slab parity, m >= 6) K6 recognises as foreign.  One index entry per
// (tile, batch): pos[0:40) | count[40:64).  The batch end is padded with zero records to 32 B.
// index layout: idx[n_sl * batch_start[b] + sl * nbatch_b + kb], so a tile finds the runs
// of all batches of its bin in one contiguous read.
//
// tile record (4 B):  pad[0:8) | f[8:16) | q[16:26)   f = m | (slab & 1) << 7      (0 = padding)
// For tile sl, tl = f ^ ((sl & 1) << 7) is the row in its map: own slab -> m, next slab -> TS + m;
// tl >= TPC_TT means "not mine".  Tile sl OWNS rows tl in [3, TS+3).
// ==========================================================================================

// sort key of a record with u = slab * TS + m: 2 * slab + (m >= 2 HALO).  For 128-bin slabs without a compare:
// (u >> 7) + ((u + 128 - 2 HALO) >> 7), the second term being slab + (m >= 2 HALO).
__device__ __forceinline__ u32 k5_key(u32 u) {
  return TPC_TS == 128u ? (u >> 7) + ((u + 128u - 2u * TPC_HALO) >> 7) : 2u * (u / TPC_TS) + ((u % TPC_TS) >= 2u * TPC_HALO ? 1u : 0u);
}
#if TPC_UNITS & TPC_U_PART_FINE
extern "C" __global__ void __launch_bounds__(TPC_K5_THREADS, 1)
k_partition_fine(const uint4* __restrict__ pool, const u32* __restrict__ dir, const u32* __restrict__ chunk_list,
                 const u32* __restrict__ bin_chunk_start, const u32* __restrict__ batch_start,
                 const u32* __restrict__ batch_bin, u32* __restrict__ blob, u64* __restrict__ blob_cursor, u64 blob_cap,
                 u64* __restrict__ idx, u32* __restrict__ status) {
  extern __shared__ __align__(128) u32 smem_u32[];
  u32* buf = smem_u32;                       // [TPC_K5_BUF]
  u32* s_cnt = buf + TPC_K5_BUF;             // [NKEY] records per key
  u32* s_off = s_cnt + TPC_NKEY;             // [NKEY + 1] start of every key's run
  __shared__ u64 s_gbase;
  const u32 nb = PRM(n_bins), nsl = PRM(n_sl);
  const u32 n_batches = batch_start[nb];
  bool bad = false;

  // The loads of a batch are issued one batch ahead, so that their latency (batch -> bin ->
  // chunk list -> chunk: four dependent levels) hides behind the placing and dumping of the
  // batch before: `look` fetches the scalars, `ids` the chunk ids, `pieces` the records.
  struct Batch { u32 b, kb, nbatch_b, c0, nch; };
  auto look = [&](u32 batch, Batch& t) {
    t.nch = 0u;
    if (batch >= n_batches) return;
    t.b = batch_bin[batch];
    const u32 bs = batch_start[t.b];
    t.kb = batch - bs;
    t.nbatch_b = batch_start[t.b + 1] - bs;
    t.c0 = bin_chunk_start[t.b] + t.kb * TPC_CPB;
    u32 c1 = t.c0 + TPC_CPB;
    const u32 ce = bin_chunk_start[t.b + 1];
    if (c1 > ce) c1 = ce;
    t.nch = c1 - t.c0;
  };
  auto ids = [&](const Batch& t, u32 (&cid)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const u32 ch = (threadIdx.x + (u32)i * TPC_K5_THREADS) >> 4;
      cid[i] = ch < t.nch ? chunk_list[t.c0 + ch] : 0xFFFFFFFFu;
    }
  };
  auto pieces = [&](const u32 (&cid)[4], uint4 (&v)[4], u32 (&nrec)[4]) {
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const u32 sub = (threadIdx.x + (u32)i * TPC_K5_THREADS) & 15u;
      v[i] = make_uint4(0u, 0u, 0u, 0u);
      nrec[i] = cid[i];   // the count sits in the entry's top bits; decoded where it is used (measured: 4.93 -> 4.66 ms against decoding it here)
      if (cid[i] != 0xFFFFFFFFu) v[i] = ld_stream_u4(pool + (u64)(cid[i] & 0x03FFFFFFu) * 16u + sub);
    }
  };
  Batch cur_b, nxt_b;
  u32 cidn[4], nrecn[4];
  uint4 vn[4];
  look(blockIdx.x, cur_b);
  ids(cur_b, cidn);
  pieces(cidn, vn, nrecn);
  look(blockIdx.x + gridDim.x, nxt_b);
  if (threadIdx.x < TPC_NKEY) s_cnt[threadIdx.x] = 0u;
  __syncthreads();

  // Three block barriers per batch: count | scan | place | dump.  The counters are cleared in the
  // place phase (the scan was their last reader) and the dump of a batch needs no barrier after
  // it: the next writers of buf / s_off / s_gbase (the scan warp) sit behind the barrier that
  // follows the next count, which every thread reaches only after its dump.
  for (u32 batch = blockIdx.x; batch < n_batches; batch += gridDim.x) {
    const u32 b = cur_b.b, kb = cur_b.kb, nbatch_b = cur_b.nbatch_b;
    const u32 npads = PRM_NPADS((b / PRM(n_tc)) % PRM(n_rows));   // one bin = one pad row

    // ---- <= 16 records per thread: count per key, remember the rank -------------------------
    u32 rec[16];
    u32 rank[8];
    // Does this warp's share of the batch look time-ordered (its first 32 records in one slab)?
    // Only then is it worth testing every warp step for a common key (see below).
    int agg;
    __match_all_sync(0xFFFFFFFFu, ((vn[0].x >> 8) & 0x3FFFu) / TPC_TS, &agg);
#pragma unroll
    for (int i = 0; i < 4; ++i) {
      const u32 sub = (threadIdx.x + (u32)i * TPC_K5_THREADS) & 15u;
      // K1 writes whole 32-byte sectors and zero-fills the last one: a piece is valid or not as a whole
      uint4 v = vn[i];
      if (nrecn[i] == 0xFFFFFFFFu || sub * 4u >= (nrecn[i] >> 26) + 1u) v = make_uint4(0u, 0u, 0u, 0u);
      u32 r4[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
      for (int j = 0; j < 4; ++j) {
        u32 r = r4[j];   // q >= 1 in every valid record, so 0 = none
        if ((r & 0xFFu) >= npads && r != 0u) { r = 0u; bad = true; }   // O0 / Q4: pad out of range -> ignored + flagged
        u32 rk = 0u;
        {
          const u32 u = (r >> 8) & 0x3FFFu;
          const u32 key = r != 0u ? k5_key(u) : 0xFFFFFFFFu;   // <= 2 * nsl (u < TC + 2 HALO)
          // time-ordered input (readout order) puts the 32 records of a warp step into ONE run: then a
          // single atomic serves the warp; otherwise (shuffled input: ~28 different keys) one per record
          int same = 0;
          if (agg) __match_all_sync(0xFFFFFFFFu, key, &same);
          if (same) {
            if (key != 0xFFFFFFFFu) {
              u32 base = 0u;
              if (lane_id() == 0u) base = atomicAdd(&s_cnt[key], 32u);
              rk = __shfl_sync(0xFFFFFFFFu, base, 0) + lane_id();
            }
          } else if (r != 0u) {
            rk = atomicAdd(&s_cnt[key], 1u);
          }
        }
        rec[i * 4 + j] = r;
        if (j & 1) rank[i * 2 + (j >> 1)] |= rk << 16; else rank[i * 2 + (j >> 1)] = rk;
      }
    }
    ids(nxt_b, cidn);   // chunk ids of the next batch: in flight during the scan and the placing
    // the bulk stores of the batch before must have read buf before the scan warp writes it again
    if (threadIdx.x >= TPC_K5_THREADS - 32u) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncthreads();
    // ---- exclusive scan of the run lengths (one warp, NKEY/32 keys = NKEY/64 slabs per lane);
    //      every slab's A run starts on a multiple of 4 records ----------------------------------
    u64 gb = 0ull;   // lane 31: the batch's place in the blob; stored after the place phase, so that
                     // the round trip of the atomic hides behind it instead of holding up the barrier
    if (threadIdx.x < 32) {
      u32 la[TPC_NKEY / 64u], lb[TPC_NKEY / 64u], t = 0u;
#pragma unroll
      for (int k = 0; k < (int)(TPC_NKEY / 64u); ++k) {
        const u32 key = 2u * (threadIdx.x * (TPC_NKEY / 64u) + (u32)k);
        la[k] = s_cnt[key]; lb[k] = s_cnt[key + 1u];
        t += (la[k] + lb[k] + 3u) & ~3u;
      }
      u32 inc = t;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) { u32 o = __shfl_up_sync(0xFFFFFFFFu, inc, d); if ((int)threadIdx.x >= d) inc += o; }
      u32 e = inc - t;
#pragma unroll
      for (int k = 0; k < (int)(TPC_NKEY / 64u); ++k) {
        const u32 key = 2u * (threadIdx.x * (TPC_NKEY / 64u) + (u32)k);
        s_off[key] = e; s_off[key + 1u] = e + la[k];
        const u32 end = e + la[k] + lb[k];
        e += (la[k] + lb[k] + 3u) & ~3u;
        for (u32 g = end; g < e; ++g) buf[g] = 0u;   // the gap before the next A (nobody else writes there)
      }
      if (threadIdx.x == 31) {
        s_off[TPC_NKEY] = inc;
        gb = atomicAdd(blob_cursor, (u64)((inc + 7u) & ~7u));   // batches start 32-byte aligned
      }
    }
    __syncthreads();
    // ---- place ------------------------------------------------------------------------------
#pragma unroll
    for (int k = 0; k < 16; ++k) {
      const u32 r = rec[k];
      if (r != 0u) {
        const u32 u = (r >> 8) & 0x3FFFu;
        const u32 key = k5_key(u);
        const u32 rk = (rank[k >> 1] >> ((k & 1) * 16)) & 0xFFFFu;
        // tile record: pad | (m | parity << 7) << 8 | q << 16.  With 128-bin slabs m | parity << 7 is simply the low byte of u,
        // which already sits in bits [8:16) of the coarse record
        const u32 f = TPC_TS == 128u ? (r & 0xFFFFu) : ((r & 0xFFu) | (((u % TPC_TS) | (((u / TPC_TS) & 1u) << 7)) << 8));
        buf[s_off[key] + rk] = f | ((r >> 22) << 16);
      }
    }
    if (threadIdx.x >= TPC_K5_THREADS - TPC_NKEY) s_cnt[threadIdx.x - (TPC_K5_THREADS - TPC_NKEY)] = 0u;   // for the next batch
    pieces(cidn, vn, nrecn);   // records of the next batch: in flight during the dump
    cur_b = nxt_b;
    look(batch + 2u * gridDim.x, nxt_b);
    const u32 total = s_off[TPC_NKEY];
    if (threadIdx.x < 8u && total + threadIdx.x < ((total + 7u) & ~7u)) buf[total + threadIdx.x] = 0u;   // end padding
    if (threadIdx.x == 31u) s_gbase = gb;
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");   // this thread's writes to buf -> visible to the bulk copy
    __syncthreads();
    // ---- dump the sorted batch + its index entries -----------------------------------------
    // The copy shared -> global is handed to the bulk-copy engine (the last warp issues it, 4 KB per
    // lane): it costs no LSU wavefronts -- the resource the count and place phases are bound by --
    // and runs while the CTA already counts the next batch.
    const u64 gbase = s_gbase;                 // a multiple of 8 records (32 B)
    // the blob is sized for every record once plus the alignment gaps (host: blob_cap); should a batch
    // not fit -- it cannot -- nothing is written, its tiles get empty runs and the status says so
    const bool fits = gbase + (u64)((total + 7u) & ~7u) <= blob_cap;
    if (!fits && threadIdx.x == 0) atomicOr(status, TPC_STATUS_INTERNAL);
    if (fits && threadIdx.x >= TPC_K5_THREADS - 32u) {
      const u32 bytes = ((total + 7u) >> 3) * 32u, off = (threadIdx.x & 31u) * 4096u;
      if (off < bytes) {
        const u32 nby = bytes - off < 4096u ? bytes - off : 4096u;
        asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"((const char*)(blob + gbase) + off),
                     "r"((u32)__cvta_generic_to_shared(buf) + off), "r"(nby) : "memory");
      }
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    if (threadIdx.x < nsl) {   // tile sl reads A_sl B_sl A_sl+1
      const u32 sl = threadIdx.x;
      const u32 beg = s_off[2u * sl], end = s_off[2u * sl + 3u];   // beg is a multiple of 4
      idx[(u64)nsl * batch_start[b] + (u64)sl * nbatch_b + kb] = fits ? (gbase + beg) | ((u64)(end - beg) << 40) : 0ull;
    }
  }
  if (threadIdx.x >= TPC_K5_THREADS - 32u) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  if (bad) atomicOr(status, TPC_STATUS_BAD_DIGITS);
}
#endif

// ==========================================================================================
// K6  cluster_tiles  (NS (1) last step + (2) + (3) + (4); rules O0..O5 of SURVEY.md 8(c))
//
// Persistent CTAs of 8 consumer warps + 1 producer warp; one tile = (bin, slab) at a time.
// The producer warp stages the tile's record runs into shared memory with 1-D bulk copies
// (cp.async.bulk -> mbarrier complete_tx) one tile ahead of the consumers, so no consumer
// ever waits on a global load.  The consumers build the tile's charge map in shared memory
// as u16 [TPC_TT][pitch] with 3 zero guard pads on each side (O0), find the 3x3 peaks with a
// dense scan on packed u16x2 words (O1: a rolling 3-row window per word column, 2 cells per
// max.u16x2), mark peaks with bit 15, run the suppression per listed peak (O2), mark the
// survivors in a per-row pad bitmask -- which ranks every cluster in (time, pad) order inside
// the tile without a sort -- and finalise the 5x5 sums (O3/O4).  The base of the tile comes
// from one atomic (FAST) or from a single-pass chained scan of the tile counts (DETERMINISTIC,
// k6_chain below).  Tiles are handed out by ticket, in increasing order.
// ==========================================================================================
// ---- mbarrier / bulk-copy / packed-max helpers (PTX; SASS: SYNCS.*, UBLKCP, VIMNMX3.U16x2) --
__device__ __forceinline__ u32 smem_addr(const void* p) { u64 a; asm("cvta.to.shared.u64 %0, %1;" : "=l"(a) : "l"(p)); return (u32)a; }
__device__ __forceinline__ void mbar_init(u64* bar, u32 count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(u64* bar, u32 bytes) {
  asm volatile("mbarrier.expect_tx.relaxed.cta.shared::cta.b64 [%0], %1;" ::"r"(smem_addr(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(u64* bar) {
  asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ void mbar_wait(u64* bar, u32 parity) {
  u32 ok;
  do {
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_addr(bar)), "r"(parity) : "memory");
  } while (!ok);
}
__device__ __forceinline__ void mbar_wait_backoff(u64* bar, u32 parity) {   // the producer's wait: do not steal issue slots
  u32 ok;
  for (;;) {
    asm volatile("{\n.reg .pred p;\nmbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\nselp.u32 %0, 1, 0, p;\n}"
                 : "=r"(ok) : "r"(smem_addr(bar)), "r"(parity) : "memory");
    if (ok) break;
    asm volatile("nanosleep.u32 200;" ::: "memory");
  }
}
__device__ __forceinline__ void bulk_g2s(void* dst, const void* src, u32 bytes, u64* bar) {
  asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];"
               ::"r"(smem_addr(dst)), "l"(src), "r"(bytes), "r"(smem_addr(bar)) : "memory");
}
__device__ __forceinline__ u32 vmax2(u32 a, u32 b) { u32 d; asm("max.u16x2 %0, %1, %2;" : "=r"(d) : "r"(a), "r"(b)); return d; }
// barrier 1 = the consumer threads only (the producer warp never joins it)
__device__ __forceinline__ void csync() { asm volatile("bar.sync 1, %0;" ::"n"(TPC_K6_CONSUMERS) : "memory"); }
__device__ __forceinline__ u32 csync_popc(bool v) {   // barrier + number of threads with v set
  u32 r;
  asm volatile("{\n.reg .pred p;\nsetp.ne.u32 p, %1, 0;\nbar.red.popc.u32 %0, 1, %2, p;\n}"
               : "=r"(r) : "r"((u32)v), "n"(TPC_K6_CONSUMERS) : "memory");
  return r;
}
__device__ __forceinline__ u32 csync_or(u32 v) {
  u32 r;
  asm volatile("{\n.reg .pred p, q;\nsetp.ne.u32 p, %1, 0;\nbar.red.or.pred q, 1, %2, p;\nselp.u32 %0, 1, 0, q;\n}"
               : "=r"(r) : "r"(v), "n"(TPC_K6_CONSUMERS) : "memory");
  return r;
}

struct K6Smem {
  u32* rec;        // [TPC_K6_CAP] staged records of one round
  u16* tile; u32* tile32;
  u64* bar;        // [0] full (producer -> consumers), [1] empty (consumers -> producer)
  u64* base;
  u32* pmask;      // [TT][9]  O1 peaks, bit = pad + HALO = the cell's index in its map row
  u32* rowmask;    // [TT][8]  O2 survivors, bit = pad
  u32* rowpre; u32* misc; u16* peaks;
  uint4* ring;     // [TPC_K6_RING][2] integer sums of a sparse tile's clusters on their way to the emitter warp (FAST)
  u32* rctl;       // [0] entries reserved  [1] entries consumed  [2] the consumers are done
};
// misc: [0] n_peaks  [1],[2] DET: next and end of the CTA's block of the temporary buffer  [3] first tile of the stage  [4] tiles in the stage  [5] row | sector << 8 |
//       n_pads << 16  [6] time of row 0 of the first tile  [7] its slab  [8+2m],[9+2m] offset and
//       size (16-byte units) of tile m's records in `rec`
__device__ __forceinline__ K6Smem k6_smem(u32* p) {
  K6Smem s;
  s.rec = p; p += TPC_K6_CAP;
  s.tile32 = p; s.tile = (u16*)p; p += TPC_TT * PRM(pitch) / 2u;
  s.ring = (uint4*)p; p += TPC_K6_RING * 8u;   // (16-byte aligned: the two areas before it are multiples of 16 bytes)
  s.rctl = p; p += 4;
  s.bar = (u64*)p; p += 4;
  s.base = (u64*)p; p += 2;
  s.pmask = p; p += TPC_TT * TPC_K6_PMW;   // pmask and rowmask are contiguous: zeroed together
  s.rowmask = p; p += TPC_TT * 8u;
  s.rowpre = p; p += TPC_TT + 2u;
  s.misc = p; p += 16;
  s.peaks = (u16*)p;
  return s;
}

// ---- DET: single-pass chained scan of the tile counts (decoupled look-back) ---------------
// tile_state[t] = flag[62:64) | value[0:62): flag 1 = the tile's own count, flag 2 = the inclusive
// prefix up to and including t.  Tiles are handed out by ticket in increasing order, so every
// tile a CTA waits for was started by a CTA that is running: no co-residency assumption.
// The result is a pure function of the counts, i.e. of the input set (an ordered scan
// in place of atomics).  Called by one full warp; returns the exclusive prefix of `tile`.
// relaxed is enough: the 64-bit word carries everything (flag and value), nothing else is published with it
__device__ __forceinline__ u64 ld_state_u64(const u64* p) { u64 v; asm volatile("ld.relaxed.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory"); return v; }
__device__ __forceinline__ void st_state_u64(u64* p, u64 v) { asm volatile("st.relaxed.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory"); }
__device__ __forceinline__ u64 k6_chain(u64* state, u32 tile, u32 count) {
  const u32 lane = lane_id();
  if (lane == 0u) st_state_u64(state + tile, (1ull << 62) | (u64)count);
  u64 excl = 0ull;
  for (long long j = (long long)tile - 1; j >= 0; j -= 32) {
    const long long i = j - (long long)lane;
    u64 v = i >= 0 ? ld_state_u64(state + i) : (2ull << 62);   // before tile 0: prefix 0
    while (__any_sync(0xFFFFFFFFu, (v >> 62) == 0ull)) { if ((v >> 62) == 0ull) v = ld_state_u64(state + i); }
    const u32 pm = __ballot_sync(0xFFFFFFFFu, (v >> 62) == 2ull);
    const u32 first = pm ? (u32)__ffs((int)pm) - 1u : 31u;   // nearest tile that already has its prefix
    u64 c = lane <= first ? (v & ((1ull << 62) - 1ull)) : 0ull;
#pragma unroll
    for (int d = 16; d >= 1; d >>= 1) c += __shfl_xor_sync(0xFFFFFFFFu, c, d);
    excl += c;
    if (pm) break;
  }
  if (lane == 0u) st_state_u64(state + tile, (2ull << 62) | (excl + (u64)count));
  return excl;
}

// Tile row of a K5 record for the tile of slab `sl`: own slab -> m, next slab -> TS + m (its first
// 6 rows close this tile); anything >= TPC_TT is a foreign record (up to 3 of them follow a run).
__device__ __forceinline__ u32 k6_row(u32 r, u32 sl) {
  const u32 x = ((r >> 8) & 0xFFu) ^ ((sl & 1u) << 7);   // bit 7: the record belongs to the next slab
  return TPC_TS == 128u ? x : (x & 127u) + (x >> 7) * TPC_TS;
}

// Producer warp: stages round `round` of a tile -- the 16-byte units [round*CAPU, (round+1)*CAPU)
// of the concatenation of the tile's runs (one run per K5 batch of the bin, 16-byte aligned,
// possibly followed by up to 3 foreign records: k6_row) -- and arrives on the full barrier.  Returns the tile's total units.
__device__ __forceinline__ u32 k6_stage(const K6Smem& s, const K6Args& a, u64 ib, u32 nbatch, u32 round, u64 e0) {
  const u32 lane = lane_id();
  const u32 lo = round * TPC_K6_CAPU, hi = lo + TPC_K6_CAPU;
  u32 pos = 0u;
  for (u32 g0 = 0u; g0 < nbatch; g0 += 32u) {
    const u32 g = g0 + lane;
    u64 e = g0 == 0u ? e0 : (g < nbatch ? a.idx[ib + g] : 0ull);   // e0: the first 32 entries, loaded ahead
    const u32 units = ((u32)(e >> 40) + 3u) >> 2;
    const u64 src = e & ((1ull << 40) - 1ull);
    u32 inc = units;
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) { u32 o = __shfl_up_sync(0xFFFFFFFFu, inc, d); if ((int)lane >= d) inc += o; }
    const u32 b = pos + inc - units, en = pos + inc;      // stream range of this run
    const u32 c0 = b > lo ? b : lo, c1 = en < hi ? en : hi;
    const u32 n = c1 > c0 ? c1 - c0 : 0u;
    const u32 tot = __reduce_add_sync(0xFFFFFFFFu, n);
    if (tot != 0u) {
      if (lane == 0u) mbar_expect_tx(&s.bar[0], tot * 16u);
      __syncwarp();
      if (n != 0u) bulk_g2s(s.rec + (c0 - lo) * 4u, a.blob + src + (u64)(c0 - b) * 4u, n * 16u, &s.bar[0]);
    }
    pos += __shfl_sync(0xFFFFFFFFu, inc, 31);
  }
  if (lane == 0u) { s.misc[8] = 0u; s.misc[9] = pos; mbar_arrive(&s.bar[0]); }
  return pos;
}

__device__ __forceinline__ uint4 lds_volatile_u4(const uint4* p) {
  uint4 v;
  asm volatile("ld.volatile.shared.v4.u32 {%0,%1,%2,%3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"((u32)__cvta_generic_to_shared(p)) : "memory");
  return v;
}
template <int V> struct TpcInt { static constexpr int v = V; };

// O4: the five exact integer sums of a cluster -> its 32 bytes (IEEE-RN float32 operations only, Q12/Q13).  In:
// c0 = (Q, Sp, St, Spp), c1 = (Stt, qmax | time << 16, pad | row << 8 | sector << 16 | flags << 24, any).
__device__ __forceinline__ void k6_finalise(uint4& c0, uint4& c1) {
  const u32 Q = c0.x, Spp = c0.w, Stt = c1.x;
  const int Sp = (int)c0.y, St = (int)c0.z;
  const int Vp = (int)(Q * Spp) - Sp * Sp, Vt = (int)(Q * Stt) - St * St;
  const float fQ = __uint2float_rn(Q);
  const float pm = __fadd_rn(__uint2float_rn(c1.z & 0xFFu), __fdiv_rn(__int2float_rn(Sp), fQ));
  const float tm = __fadd_rn(__uint2float_rn(c1.y >> 16), __fdiv_rn(__int2float_rn(St), fQ));
  const float sp = __fdiv_rn(__fsqrt_rn(__int2float_rn(Vp)), fQ);
  const float st = __fdiv_rn(__fsqrt_rn(__int2float_rn(Vt)), fQ);
  c0 = make_uint4(__float_as_uint(pm), __float_as_uint(tm), __float_as_uint(sp), __float_as_uint(st));
  c1 = make_uint4(Q, c1.y, c1.z, 0u);
}
// COG: the reading of the centre of gravity -- 0 = Q10 (every cell, weight 1), 1 = Q10' (outer ring gated),
// 2 = Q10'' (charge shared with the surviving peaks on the outer ring; needs TPC_HALO >= 5)
template <int MODE, int COG, bool EMIT>
__device__ __forceinline__ void k6_body(const K6Args& a, u32* smem) {
  const K6Smem s = k6_smem(smem);
  const u32 nb = PRM(n_bins), nsl = PRM(n_sl), pitch = PRM(pitch);
  const u32 n_tiles = nb * nsl;
  const u32 thr = PRM(thr_peak), eps = PRM(noise_eps);
  const u32 tile_words = TPC_TT * pitch / 2u;
  const u32 tid = threadIdx.x;
  // rows whose peaks are listed and tested for survival: the owned rows; under Q10'' two more on each
  // side, whose survivors the owned clusters share charge with (they are emitted by their own tiles)
  static_assert(COG != 2 || TPC_HALO >= 5u, "reading Q10'' needs a time halo of 5");
  constexpr u32 LIST_LO = COG == 2 ? TPC_HALO - 2u : TPC_HALO, LIST_HI = COG == 2 ? TPC_TS + TPC_HALO + 2u : TPC_TS + TPC_HALO;

  if (tid == 0) {
    mbar_init(&s.bar[0], 1u);                       // full: the producer's arrive (+ tx bytes)
    mbar_init(&s.bar[1], TPC_K6_CONSUMERS / 32u);   // empty: one arrive per consumer warp
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
  }
  for (u32 i = tid; i < TPC_K6_RING * 2u; i += TPC_K6_CONSUMERS) s.ring[i] = make_uint4(0u, 0u, 0u, 0u);
  if (tid < 4u) s.rctl[tid] = 0u;
  if (tid == 0) { s.misc[1] = 0u; s.misc[2] = 0u; }   // DET: the CTA's block of the temporary buffer [next, end)
  __syncthreads();

  // The emitter warp (FAST, readings Q10 and Q10'): a sparse tile has its ~4 peaks in ONE warp, and the other
  // seven waited at barrier E while that warp walked global atomic -> division -> square root -> store (41 % of
  // the samples of the pp-like frame).  The consumers now leave the integer sums of such a cluster in a ring in
  // shared memory -- entry i: slot i % RING, valid once word 7 holds its tag i / RING + 1 -- and this warp, which
  // is outside their barriers, finalises, reserves and writes.  No consumer ever waits for it: a warp that finds
  // the ring full emits its clusters itself, as the tiles with more than one record per thread always do.
  // The kernels *_e have the warp; the host launches them when the frame averages less than 512 records per tile.
  // DET_TEMP has it as well: there the consumers know every cluster's place (the tile's run is cut from a block of
  // the temporary buffer that the CTA holds, its rank comes from the warp that holds the tile's peaks), so the entry
  // carries the place -- c0 = (Q | Spp << 15, Sp, St, place) -- and the emitter only finalises and stores.
  static_assert(!EMIT || ((MODE == TPC_MODE_FAST || MODE == TPC_MODE_DET_TEMP) && COG != 2), "the emitter warp serves FAST and DET_TEMP of the readings Q10, Q10'");
  if (EMIT && tid >= TPC_K6_CONSUMERS + 32u) {
    const u32 lane = lane_id();
    u32 t = 0u;   // entries consumed
    u32 nap = 100u;
    for (;;) {
      const u32 i = t + lane, slot = i % TPC_K6_RING;
      uint4 c1 = lds_volatile_u4(&s.ring[2u * slot + 1u]);
      const u32 vm = __ballot_sync(0xFFFFFFFFu, c1.w == i / TPC_K6_RING + 1u);
      const u32 nv = vm == 0xFFFFFFFFu ? 32u : (u32)__ffs((int)~vm) - 1u;   // the valid entries at the head
      if (nv == 0u) {
        if (*(volatile u32*)&s.rctl[2] != 0u && t == *(volatile u32*)&s.rctl[0]) break;   // the consumers are done and nothing is left
        __nanosleep(nap);
        if (nap < 1600u) nap *= 2u;
        continue;
      }
      nap = 100u;
      uint4 c0 = make_uint4(1u, 0u, 0u, 0u);
      if (lane < nv) c0 = lds_volatile_u4(&s.ring[2u * slot]);
      __syncwarp();
      t += nv;
      u64 base = 0ull;
      if (MODE == TPC_MODE_DET_TEMP) {
        if (lane == 0u) *(volatile u32*)&s.rctl[1] = t;   // the slots are free again
        if (lane < nv) {
          const u64 o = c0.w;
          c0 = make_uint4(c0.x & 0x7FFFu, c0.y, c0.z, c0.x >> 15);
          k6_finalise(c0, c1);
          if (o < a.temp_cap) { a.temp[o * 2u] = c0; a.temp[o * 2u + 1u] = c1; }
        }
        continue;
      }
      if (lane == 0u) { *(volatile u32*)&s.rctl[1] = t; base = atomicAdd(a.n_clusters, (u64)nv); }   // the slots are free again
      if (lane < nv) k6_finalise(c0, c1);
      base = __shfl_sync(0xFFFFFFFFu, base, 0);
      if (lane < nv) {
        const u64 o = base + lane;
        if (o < a.capacity) { a.out[o * 2u] = c0; a.out[o * 2u + 1u] = c1; }
        else atomicOr(a.status, TPC_STATUS_OVERFLOW);
      }
    }
    return;
  }
  if (tid >= TPC_K6_CONSUMERS) {
    // ---- producer warp -----------------------------------------------------------------------
    // A ticket = up to TPC_K6_GROUP consecutive slabs of one bin, handed out in increasing order.
    // Small tiles (sparse frames) are staged together, one bulk copy per run and one barrier
    // phase for the whole group, so that the staging latency is paid once per group; a tile
    // that does not fit is staged alone, in as many rounds as it needs.  The loads for a stage
    // (ticket, batch table, index entries, L2 prefetch of the runs) are issued before the wait
    // for the buffer, i.e. while the consumers still work on the stage before.
    u32 ph = 1u;   // a fresh barrier passes a wait on parity 1: the buffer starts out free
    const u32 lane = lane_id();
    const u32 gpb = (nsl + TPC_K6_GROUP - 1u) / TPC_K6_GROUP, n_tickets = nb * gpb;
    for (;;) {
      u32 t = 0u;
      if (lane == 0u) t = atomicAdd(a.ticket, 1u);
      t = __shfl_sync(0xFFFFFFFFu, t, 0);
      if (t >= n_tickets) break;
      const u32 b = t / gpb, sl0 = (t - b * gpb) * TPC_K6_GROUP;
      const u32 cnt = nsl - sl0 < TPC_K6_GROUP ? nsl - sl0 : TPC_K6_GROUP;
      const u32 bs0 = a.batch_start[b];
      const u32 nbatch = a.batch_start[b + 1] - bs0;
      const u64 ib0 = (u64)nsl * bs0 + (u64)sl0 * nbatch;
      const u32 tile0 = b * nsl + sl0;
      const u32 tc = b % PRM(n_tc), sr = b / PRM(n_tc);
      const u32 row = sr % PRM(n_rows), sector = sr / PRM(n_rows);
      const u32 geo = row | (sector << 8) | ((u32)PRM_NPADS(row) << 16);
      const int t0 = (int)(tc * TPC_TC + sl0 * TPC_TS) - (int)TPC_HALO;   // time of row 0 of the first tile
      bool grouped = false;
      u64 e = 0ull;
      u32 units = 0u, inc = 0u;
      const u32 m = lane >> 3, kb = lane & 7u;   // grouped: lane = (tile m of the group, batch kb)
      if (nbatch <= 8u && cnt > 1u) {
        if (m < cnt && kb < nbatch) e = a.idx[ib0 + (u64)m * nbatch + kb];
        units = ((u32)(e >> 40) + 3u) >> 2;
        inc = units;
#pragma unroll
        for (int d = 1; d < 32; d <<= 1) { u32 o = __shfl_up_sync(0xFFFFFFFFu, inc, d); if ((int)lane >= d) inc += o; }
        grouped = __shfl_sync(0xFFFFFFFFu, inc, 31) <= TPC_K6_CAPU;
      }
      if (grouped) {
        const u32 tot = __shfl_sync(0xFFFFFFFFu, inc, 31);
        const void* src = a.blob + (e & ((1ull << 40) - 1ull));
        if (units != 0u) asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src), "r"(units * 16u) : "memory");
        const u32 off = inc - units;                                     // this run's place in rec
        const u32 t_end = __shfl_sync(0xFFFFFFFFu, inc, (int)(lane | 7u));   // end of this tile's runs
        const u32 t_beg = __shfl_sync(0xFFFFFFFFu, off, (int)(lane & ~7u));
        mbar_wait_backoff(&s.bar[1], ph); ph ^= 1u;
        if (kb == 0u && m < TPC_K6_GROUP) { s.misc[8u + 2u * m] = t_beg; s.misc[9u + 2u * m] = m < cnt ? t_end - t_beg : 0u; }
        if (lane == 0u) { s.misc[3] = tile0; s.misc[4] = cnt; s.misc[5] = geo; s.misc[6] = (u32)t0; s.misc[7] = sl0; if (tot != 0u) mbar_expect_tx(&s.bar[0], tot * 16u); }
        __syncwarp();
        if (units != 0u) bulk_g2s(s.rec + off * 4u, src, units * 16u, &s.bar[0]);
        __syncwarp();
        if (lane == 0u) mbar_arrive(&s.bar[0]);
      } else {
        for (u32 k = 0u; k < cnt; ++k) {
          const u64 ib = ib0 + (u64)k * nbatch;
          const u64 e0 = lane < nbatch ? a.idx[ib + lane] : 0ull;
          const u32 bytes = (((u32)(e0 >> 40) + 3u) >> 2) * 16u;
          if (bytes != 0u)
            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(a.blob + (e0 & ((1ull << 40) - 1ull))), "r"(bytes) : "memory");
          mbar_wait_backoff(&s.bar[1], ph); ph ^= 1u;
          if (lane == 0u) { s.misc[3] = tile0 + k; s.misc[4] = 1u; s.misc[5] = geo; s.misc[6] = (u32)(t0 + (int)(k * TPC_TS)); s.misc[7] = sl0 + k; }   // published by the arrive in k6_stage
          const u32 total = k6_stage(s, a, ib, nbatch, 0u, e0);
          for (u32 round = 1u; round * TPC_K6_CAPU < total; ++round) {
            mbar_wait_backoff(&s.bar[1], ph); ph ^= 1u;
            k6_stage(s, a, ib, nbatch, round, e0);
          }
        }
      }
    }
    mbar_wait_backoff(&s.bar[1], ph);   // tell the consumers there is nothing left
    if (lane == 0u) { s.misc[3] = 0xFFFFFFFFu; s.misc[4] = 0u; mbar_arrive(&s.bar[0]); }
    return;
  }

  // ---- consumers -------------------------------------------------------------------------------
  // Per tile, five block barriers (A..G below).  The map, pmask and rowmask are zeroed at the
  // tail of the previous tile, so barrier A doubles as "zeroing done".
  u32 ph = 0u;
  const u32 zero_words = tile_words / 4u;
  auto zero_tile = [&]() {
    uint4* z = (uint4*)s.tile32;
    for (u32 i = tid; i < zero_words; i += TPC_K6_CONSUMERS) z[i] = make_uint4(0u, 0u, 0u, 0u);
    for (u32 i = tid; i < TPC_TT * (8u + TPC_K6_PMW); i += TPC_K6_CONSUMERS) s.pmask[i] = 0u;
    if (tid == 0) s.misc[0] = 0u;
  };
  zero_tile();
  for (;;) {
    mbar_wait(&s.bar[0], ph); ph ^= 1u;
    const u32 tile0 = s.misc[3], ntl = s.misc[4];
    if (tile0 == 0xFFFFFFFFu) break;   // block-uniform
   for (u32 mt = 0u; mt < ntl; ++mt) {   // the tiles of this stage
    const u32 tile = tile0 + mt, total = s.misc[9u + 2u * mt];
    const u32* const rec = s.rec + s.misc[8u + 2u * mt] * 4u;
    u32* const s_rec_w = s.rec + s.misc[8u + 2u * mt] * 4u;   // (the peak test keeps its candidate list in the consumed records)
    const bool last = mt + 1u == ntl;   // the staged records are released after the last tile's use of them
    if (total == 0u) {   // block-uniform: nothing in this tile; the map stays zero
      __syncwarp();
      if (last && lane_id() == 0u) mbar_arrive(&s.bar[1]);
      if (MODE == TPC_MODE_DET_TEMP && tid == 0) a.tile_cnt[tile] = 0u;
      if (MODE == TPC_MODE_DET && tid >= TPC_K6_CONSUMERS - 32u) {   // an empty tile is still a link of the chain
        const u64 ex = k6_chain(a.tile_state, tile, 0u);
        if (tile == n_tiles - 1u && lane_id() == 0u) *a.n_clusters = ex;
      }
      continue;
    }
    // the producer (which has the time for the divisions) decoded the tile: all tiles of a stage share the bin
    const u32 geo = s.misc[5];
    const u32 row = geo & 0xFFu, sector = (geo >> 8) & 0xFFu, npads = geo >> 16;
    const int t_base = (int)s.misc[6] + (int)(mt * TPC_TS);   // time of tile row 0
    const u32 sl = s.misc[7] + mt;                            // slab of this tile inside its bin
    csync();   // A: the previous tile is done with the map, and the map is zero
    u32 my_r = 0u;   // sparse tile: this thread's record, if it lies in the tile
    // ---- O0: scatter the tile's records ------------------------------------------------------
    for (u32 round = 0u;;) {
      u32 nu = total - round * TPC_K6_CAPU;
      if (nu > TPC_K6_CAPU) nu = TPC_K6_CAPU;
      const uint4* r4 = (const uint4*)rec;
      if (MODE == TPC_MODE_FAST || round == 0u) {   // plain stores: FAST may keep either of two digits on one
                                                    // cell (Q5); DET: the map is still empty in round 0, the loop below settles it
        if (nu * 4u <= TPC_K6_CONSUMERS) {   // a sparse tile: one record per thread, spread over all warps
          const u32 r = tid < nu * 4u ? rec[tid] : 0u;
          const u32 tl = k6_row(r, sl);
          if (r >= (1u << 16) && tl < TPC_TT) { s.tile[tl * pitch + (r & 0xFFu) + TPC_PG] = (u16)((r >> 16) & 0x3FFu); my_r = r; }   // (q = 0: Q4, ignored)
        } else
        for (u32 u = tid; u < nu; u += TPC_K6_CONSUMERS) {
          const uint4 v = r4[u];
          const u32 rr[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
          for (int k = 0; k < 4; ++k)
            if (rr[k] >= (1u << 16)) {   // q >= 1; not batch padding (0) nor a zero-charge digit (Q4: ignored; K5 has checked its range)
              const u32 tl = k6_row(rr[k], sl);
              if (tl < TPC_TT) s.tile[tl * pitch + (rr[k] & 0xFFu) + TPC_PG] = (u16)((rr[k] >> 16) & 0x3FFu);
            }
        }
      }
      if (MODE != TPC_MODE_FAST && total > TPC_K6_CAPU) {   // (a single-round tile checks in its peak pass instead)
        // Q5, deterministic: two digits on one cell -> the maximum, whatever the order and however
        // many staging rounds the tile takes: from here on a cell is only ever raised, and the pass
        // repeats until no record is larger than its cell.  Duplicate-free input: one confirming pass.
        if (round == 0u) csync();
        for (;;) {   // passes are separated by the barrier inside csync_or
          u32 any = 0u;
          for (u32 u = tid; u < nu; u += TPC_K6_CONSUMERS) {
            const uint4 v = r4[u];
            const u32 rr[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const u32 tl = k6_row(rr[k], sl);
              if (rr[k] != 0u && tl < TPC_TT) {
                const u32 cell = tl * pitch + (rr[k] & 0xFFu) + TPC_PG;
                const u16 q = (u16)((rr[k] >> 16) & 0x3FFu);
                if (s.tile[cell] < q) { s.tile[cell] = q; any = 1u; }
              }
            }
          }
          if (!csync_or(any)) break;
        }
      }
      ++round;
      if (round * TPC_K6_CAPU >= total) break;
      __syncwarp();
      if (lane_id() == 0u) mbar_arrive(&s.bar[1]);   // this warp is done with the staged records
      mbar_wait(&s.bar[0], ph); ph ^= 1u;
    }
    // a tile staged in one round (the usual case) keeps its records for the peak test below
#ifdef TPC_X_DENSE
    const bool sparse = total * 4u <= TPC_K6_CONSUMERS && MODE != TPC_MODE_DUMP_MAP;
#else
    const bool sparse = total <= TPC_K6_CAPU && MODE != TPC_MODE_DUMP_MAP;
#endif
    if (!sparse) { __syncwarp(); if (last && lane_id() == 0u) mbar_arrive(&s.bar[1]); }
    csync();   // C: the map is complete

    if (MODE == TPC_MODE_DUMP_MAP) {
      const u64 sector_cells = a.row_off[PRM(n_rows)];
      for (u32 i = tid; i < TPC_TS * npads; i += TPC_K6_CONSUMERS) {
        u32 tl = i / npads + TPC_HALO, p = i % npads;
        int t = t_base + (int)tl;
        if (t < (int)PRM(n_time))
          a.dmap[(u64)sector * sector_cells + a.row_off[row] + (u64)t * npads + p] = s.tile[tl * pitch + p + TPC_PG];
      }
      csync();
      zero_tile();
      continue;
    }

    // ---- O1: 3x3 peaks, record-driven (the tile's records are still staged) -----------------
    // Every record with q >= thr_peak in rows 1..TT-2 tests its own cell: the two words holding
    // (x-1, x, x+1) of the rows above, at and below are loaded and aligned with a funnel shift;
    // q > the 4 neighbours earlier in (t,p) order and q >= the 4 later ones (O1).  Cost follows
    // the occupancy, not the tile area; a tile that needed several staging rounds takes the
    // dense scan below instead.  A peak sets its bit in pmask (which also removes duplicates of
    // one cell); the peaks of owned rows go into the list the later phases walk.
    bool d_done = false;   // block-uniform: barrier D already passed
    if (sparse) {
      const u32 nW = pitch >> 1;
      const uint4* r4 = (const uint4*)rec;
      // `check` (DET): also verify that no cell holds less than one of its records -- the plain
      // stores of the scatter may have left a smaller duplicate on top (Q5)
      const u32 nrec = total * 4u;
      // K records of one thread: K = 4 (a 16-byte piece, the loads of the four in flight together)
      // or K = 1 (a sparse tile: one record per thread, spread over all warps)
      auto peak_recs = [&](auto kt, const u32* rr, const bool check) -> u32 {
        constexpr int K = decltype(kt)::v;
        u32 viol = 0u;
        {
          // the four records of a piece are independent: their loads are issued together, in two
          // stages -- the own row first (two thirds of the candidates already lose against a pad
          // neighbour there), then the rows above and below for those still in the race; the others
          // read word 0, a broadcast that costs no bank conflict
          u32 pu[K], nu[K], pm[K], nm[K], pd[K], nd[K];
          bool cand[K];
#pragma unroll
          for (int k = 0; k < K; ++k) {
            const u32 q = (rr[k] >> 16) & 0x3FFu, tl = k6_row(rr[k], sl), pad = rr[k] & 0xFFu;
            cand[k] = q >= thr && tl - 1u < TPC_TT - 2u;   // (q = 0 for run padding)
            if (check && !cand[k] && rr[k] != 0u && tl < TPC_TT && s.tile[tl * pitch + pad + TPC_PG] < q) viol = 1u;
            const u32 x = pad + TPC_PG, h = x & 1u, sh = 16u - 16u * h;
            const u32* w = s.tile32 + (cand[k] ? tl * nW + (x >> 1) - 1u + h : 0u);
            pm[k] = __funnelshift_r(w[0], w[1], sh); nm[k] = (w[1] >> sh) & 0xFFFFu;
          }
#pragma unroll
          for (int k = 0; k < K; ++k) {
            const u32 q = (rr[k] >> 16) & 0x3FFu, tl = k6_row(rr[k], sl), pad = rr[k] & 0xFFu;
            if (check && cand[k] && (pm[k] >> 16) < q) viol = 1u;   // the cell holds a smaller duplicate of this record (Q5)
            cand[k] = cand[k] && (pm[k] >> 16) == q && q > (pm[k] & 0xFFFFu) && q >= nm[k];   // (!= q: a smaller duplicate of this cell)
            const u32 x = pad + TPC_PG, h = x & 1u, sh = 16u - 16u * h;
            const u32* w = s.tile32 + (cand[k] ? (tl - 1u) * nW + (x >> 1) - 1u + h : 0u);
            pu[k] = __funnelshift_r(w[0], w[1], sh); nu[k] = (w[1] >> sh) & 0xFFFFu;
            w += 2u * nW;
            pd[k] = __funnelshift_r(w[0], w[1], sh); nd[k] = (w[1] >> sh) & 0xFFFFu;
          }
#pragma unroll
          for (int k = 0; k < K; ++k) {
            const u32 q = (rr[k] >> 16) & 0x3FFu, tl = k6_row(rr[k], sl), pad = rr[k] & 0xFFu;
            const u32 e = max(max(pu[k] & 0xFFFFu, pu[k] >> 16), nu[k]);
            const u32 l = max(max(pd[k] & 0xFFFFu, pd[k] >> 16), nd[k]);
            if (cand[k] && q > e && q >= l) {
              const u32 bit = 1u << ((pad + TPC_PG) & 31u);
              const u32 old = atomicOr(&s.pmask[tl * TPC_K6_PMW + ((pad + TPC_PG) >> 5)], bit);
              if (!(old & bit) && tl >= LIST_LO && tl < LIST_HI) {   // a halo-row peak is emitted by its own tile
                const u32 i = atomicAdd(&s.misc[0], 1u);
                s.peaks[i] = (u16)((tl << 8) | pad);
              }
            }
          }
        }
        return viol;
      };
      // Tiles with more than one record per thread: two stages with a compaction in between, so that
      // the rows above and below are only fetched -- by full warps -- for the records that won their own
      // row.  Stage 1 (all records, 16-byte pieces): q >= thr, q > left, q >= right, and the cell holds
      // this very charge (a smaller duplicate of the cell is out).  Its survivors, one record in five, are
      // written back IN PLACE: warp w reads records [1024 k + 128 w, + 128) in its k-th step and keeps its
      // list in those same regions, in order -- it never holds more survivors than it has read, so the
      // list only ever covers records the warp has consumed itself: no other buffer, no block barrier.
      // Stage 2 walks the list, 64 entries per warp step; a peak sets its bit in pmask and the peaks of
      // owned rows join the tile's list with one shared atomic per warp step.
      auto peak_big = [&]() {
        const u32 lane = lane_id(), lt = (1u << lane) - 1u, wbase = (tid >> 5) * 128u;
        u32 nlist = 0u;   // warp-uniform
        for (u32 u0 = (tid >> 5) * 32u; u0 < total; u0 += TPC_K6_CONSUMERS) {
          const u32 u = u0 + lane;
          uint4 v = make_uint4(0u, 0u, 0u, 0u);
          if (u < total) v = r4[u];
          const u32 rr[4] = {v.x, v.y, v.z, v.w};
          u32 pm[4], nm[4];
          bool cand[4];
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const u32 q = (rr[k] >> 16) & 0x3FFu, tl = k6_row(rr[k], sl), pad = rr[k] & 0xFFu;
            cand[k] = q >= thr && tl - 1u < TPC_TT - 2u;   // (q = 0 for run padding)
            const u32 x = pad + TPC_PG, h = x & 1u, sh = 16u - 16u * h;
            const u32* w = s.tile32 + (cand[k] ? tl * nW + (x >> 1) - 1u + h : 0u);   // the others: word 0, a broadcast
            pm[k] = __funnelshift_r(w[0], w[1], sh); nm[k] = (w[1] >> sh) & 0xFFFFu;
          }
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const u32 q = (rr[k] >> 16) & 0x3FFu;
            const bool win = cand[k] && (pm[k] >> 16) == q && q > (pm[k] & 0xFFFFu) && q >= nm[k];
            const u32 m = __ballot_sync(0xFFFFFFFFu, win);   // (the ballot needs every lane's piece: all loads of this step are done)
            if (win) {
              const u32 p = nlist + __popc(m & lt);
              s_rec_w[(p >> 7) * (TPC_K6_CONSUMERS * 4u) + wbase + (p & 127u)] = rr[k];
            }
            nlist += __popc(m);
          }
        }
        __syncwarp();
        for (u32 p0 = 0u; p0 < nlist; p0 += 64u) {
          u32 r2[2], pu[2], nu[2], pd[2], nd[2];
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            const u32 p = p0 + 32u * (u32)k + lane;
            r2[k] = p < nlist ? s_rec_w[(p >> 7) * (TPC_K6_CONSUMERS * 4u) + wbase + (p & 127u)] : 0u;
          }
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            const u32 tl = k6_row(r2[k], sl), pad = r2[k] & 0xFFu;
            const u32 x = pad + TPC_PG, h = x & 1u, sh = 16u - 16u * h;
            const u32* w = s.tile32 + (r2[k] != 0u ? (tl - 1u) * nW + (x >> 1) - 1u + h : 0u);
            pu[k] = __funnelshift_r(w[0], w[1], sh); nu[k] = (w[1] >> sh) & 0xFFFFu;
            w += 2u * nW;
            pd[k] = __funnelshift_r(w[0], w[1], sh); nd[k] = (w[1] >> sh) & 0xFFFFu;
          }
#pragma unroll
          for (int k = 0; k < 2; ++k) {
            const u32 q = (r2[k] >> 16) & 0x3FFu, tl = k6_row(r2[k], sl), pad = r2[k] & 0xFFu;
            const u32 e = max(max(pu[k] & 0xFFFFu, pu[k] >> 16), nu[k]);
            const u32 l = max(max(pd[k] & 0xFFFFu, pd[k] >> 16), nd[k]);
            bool own = false;
            if (r2[k] != 0u && q > e && q >= l) {
              const u32 bit = 1u << ((pad + TPC_PG) & 31u);
              const u32 old = atomicOr(&s.pmask[tl * TPC_K6_PMW + ((pad + TPC_PG) >> 5)], bit);
              own = !(old & bit) && tl >= LIST_LO && tl < LIST_HI;   // a halo-row peak is emitted by its own tile
            }
            const u32 m = __ballot_sync(0xFFFFFFFFu, own);
            if (m) {
              u32 base = 0u;
              if (lane == 0u) base = atomicAdd(&s.misc[0], (u32)__popc(m));
              base = __shfl_sync(0xFFFFFFFFu, base, 0);
              if (own) s.peaks[base + __popc(m & lt)] = (u16)((tl << 8) | pad);
            }
          }
        }
      };
      // DET: have the plain stores of the scatter left a smaller duplicate on top of a cell (Q5)?
      auto settle = [&]() {   // raise every cell to the maximum of its records; ends behind a barrier
        for (;;) {
          u32 any = 0u;
          for (u32 u = tid; u < total; u += TPC_K6_CONSUMERS) {
            const uint4 v = r4[u];
            const u32 rr[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const u32 tl = k6_row(rr[k], sl);
              if (rr[k] != 0u && tl < TPC_TT) {
                const u32 cell = tl * pitch + (rr[k] & 0xFFu) + TPC_PG;
                const u16 q = (u16)((rr[k] >> 16) & 0x3FFu);
                if (s.tile[cell] < q) { s.tile[cell] = q; any = 1u; }
              }
            }
          }
          if (!csync_or(any)) break;
        }
      };
      if (nrec > TPC_K6_CONSUMERS) {
        if (MODE != TPC_MODE_FAST) {
          // the in-place list would destroy the records the settling needs: verify first (one more pass
          // over the records and one more barrier per tile than FAST -- the price of Q5 in this mode)
          u32 viol = 0u;
          for (u32 u = tid; u < total; u += TPC_K6_CONSUMERS) {
            const uint4 v = r4[u];
            const u32 rr[4] = {v.x, v.y, v.z, v.w};
            u32 c4[4];
#pragma unroll
            for (int k = 0; k < 4; ++k) {
              const u32 tl = k6_row(rr[k], sl);
              c4[k] = s.tile[(tl < TPC_TT ? tl * pitch : 0u) + (rr[k] & 0xFFu) + TPC_PG];
            }
#pragma unroll
            for (int k = 0; k < 4; ++k)
              if (rr[k] != 0u && k6_row(rr[k], sl) < TPC_TT && c4[k] < ((rr[k] >> 16) & 0x3FFu)) viol = 1u;
          }
          if (csync_or(viol)) settle();   // rare: duplicates in this tile
        }
        peak_big();
      } else if (MODE == TPC_MODE_FAST) {
        const u32 r1[1] = {tid < nrec ? rec[tid] : 0u};
        peak_recs(TpcInt<1>(), r1, false);
      } else {
        d_done = true;
        const u32 r1[1] = {tid < nrec ? rec[tid] : 0u};
        if (csync_or(peak_recs(TpcInt<1>(), r1, true))) {   // rare: duplicates in this tile.  Settle the maxima, forget the peaks, test again.
          settle();
          for (u32 i = tid; i < TPC_TT * TPC_K6_PMW; i += TPC_K6_CONSUMERS) s.pmask[i] = 0u;
          if (tid == 0) s.misc[0] = 0u;
          csync();
          peak_recs(TpcInt<1>(), r1, false);
          csync();
        }
      }
      __syncwarp();
      if (last && lane_id() == 0u) mbar_arrive(&s.bar[1]);   // this warp is done with the staged records
    } else
    // ---- O1: 3x3 peaks, dense scan on packed u16x2 words ----------------------------------
    // A thread owns a group of 4 word columns (8 cells, one 128-bit load per row) of a strip of
    // rows and walks down the time axis with a rolling 3-row window.  For the word C of row r:
    // L / R = the same two cells shifted one pad left / right, H(r) = max(L, C, R).  A cell is a
    // peak iff q > the 4 neighbours earlier in (t,p) order and q >= the 4 later ones (O1), i.e.
    // q > M1 = max(H(r-1), L(r)) and q >= M2 = max(H(r+1), R(r), thr_peak); an empty cell never
    // passes (M2 >= 1).  Charges have 10 bits, so each 16-bit half carries a guard bit: with
    // G = 0x80008000, (C | G) - M1 - 0x00010001 and (C | G) - M2 keep their guard bits exactly where
    // the comparison holds, with plain 32-bit adds and no borrow between the halves.  The 8 result
    // bits of a row are one byte of pmask (bit = cell index): a byte store, no atomics.  Rows
    // 1..TT-2 are tested: the owned rows plus the halo rows whose peaks O2 needs.  Guard cells are 0
    // and can never be flagged.  The peaks of owned rows are listed afterwards, from pmask.
    {
      const u32 nW = pitch >> 1;
      const u32 ng = ((npads + TPC_PG - 1u) >> 3) + 1u;   // 8-cell groups up to the last real pad's cell (npads + 2)
      const u32 strips = TPC_K6_CONSUMERS / ng;          // >= 1: npads <= 256 -> ng <= 33
      const u32 rp = (TPC_TT - 2u + strips - 1u) / strips;
      const u32 si = tid / ng, g = tid - si * ng;
      const u32 thr2 = thr | (thr << 16);
      const u32 r0 = 1u + si * rp;
      u32 r1 = r0 + rp;
      if (r1 > TPC_TT - 1u) r1 = TPC_TT - 1u;
      if (si < strips && r0 < r1) {
        const bool hasl = g != 0u, hasr = 4u * g + 4u < nW;
        struct Row { u32 C[4], S[5], H[4]; };
        auto load = [&](const u32* q, Row& w) {
          const uint4 v = *(const uint4*)q;
          const u32 a = hasl ? q[-1] : 0u, b = hasr ? q[4] : 0u;
          w.C[0] = v.x; w.C[1] = v.y; w.C[2] = v.z; w.C[3] = v.w;
          w.S[0] = __funnelshift_l(a, v.x, 16); w.S[1] = __funnelshift_l(v.x, v.y, 16);
          w.S[2] = __funnelshift_l(v.y, v.z, 16); w.S[3] = __funnelshift_l(v.z, v.w, 16);
          w.S[4] = __funnelshift_l(v.w, b, 16);
#pragma unroll
          for (int k = 0; k < 4; ++k) w.H[k] = vmax2(vmax2(w.S[k], w.C[k]), w.S[k + 1]);
        };
        u8* const pmb = (u8*)s.pmask + g;
        auto test = [&](const Row& up, const Row& mid, const Row& dn, u32 r) {
          u32 byte = 0u;
#pragma unroll
          for (int k = 0; k < 4; ++k) {
            const u32 M1 = vmax2(up.H[k], mid.S[k]);
            const u32 M2 = vmax2(vmax2(dn.H[k], mid.S[k + 1]), thr2);
            const u32 cg = mid.C[k] | 0x80008000u;
            const u32 x = ((cg - M1 - 0x00010001u) & (cg - M2) & 0x80008000u) >> 15;   // bit 0: the low cell is a peak, bit 16: the high cell
            byte |= ((x | (x >> 15)) & 3u) << (2 * k);
          }
          pmb[r * (TPC_K6_PMW * 4u)] = (u8)byte;
        };
        const u32* q = s.tile32 + (r0 - 1u) * nW + 4u * g;
        Row ra, rb, rc;
        load(q, ra); q += nW;
        load(q, rb); q += nW;
        for (u32 r = r0;;) {   // unrolled by 3 so the window rotates by renaming, not by moves
          load(q, rc); test(ra, rb, rc, r); if (++r >= r1) break; q += nW;
          load(q, ra); test(rb, rc, ra, r); if (++r >= r1) break; q += nW;
          load(q, rb); test(rc, ra, rb, r); if (++r >= r1) break; q += nW;
        }
      }
      csync();   // D': pmask complete
      // the peaks of the owned rows, listed from pmask: a warp per 32 mask words, one shared atomic per warp step
      const u32 nwp = ((npads + TPC_PG - 1u) >> 5) + 1u;   // mask words that can hold a peak
      const u32 inv = 65536u / nwp + 1u;                      // i / nwp for i < 2^11 (exact: nwp <= 9)
      const u32 lane = lane_id(), lt = (1u << lane) - 1u;
      for (u32 i0 = (tid >> 5) * 32u; i0 < (LIST_HI - LIST_LO) * nwp; i0 += TPC_K6_CONSUMERS) {
        const u32 i = i0 + lane;
        const u32 rw = (i * inv) >> 16, wd = i - rw * nwp;
        u32 w = i < (LIST_HI - LIST_LO) * nwp ? s.pmask[(rw + LIST_LO) * TPC_K6_PMW + wd] : 0u;
        for (;;) {
          const u32 m = __ballot_sync(0xFFFFFFFFu, w != 0u);
          if (!m) break;
          u32 base = 0u;
          if (lane == 0u) base = atomicAdd(&s.misc[0], (u32)__popc(m));
          base = __shfl_sync(0xFFFFFFFFu, base, 0);
          if (w != 0u) {
            const u32 bpos = (u32)__ffs((int)w) - 1u;
            w &= w - 1u;
            s.peaks[base + __popc(m & lt)] = (u16)(((rw + LIST_LO) << 8) | (wd * 32u + bpos - TPC_PG));
          }
        }
      }
    }
    if (!d_done) csync();   // D: peak set complete
    const u32 npk = s.misc[0];

    // ---- O2: suppression of the owned peaks against the un-updated peak set -----------------
    auto suppressed = [&](const u32 e) -> bool {
      const u32 tl = e >> 8, pad = e & 0xFFu;
      // the 5x5 ring of peak bits around (tl, pad): 5 bits per row, bit k <-> dp = k - 2
      const u32 w0 = (pad + TPC_PG - 2u) >> 5, sh = (pad + TPC_PG - 2u) & 31u;   // bit of (pad - 2) = cell index pad + HALO - 2
      u32 ring = 0u;
#pragma unroll
      for (int dt = -2; dt <= 2; ++dt) {
        const u32* pm = s.pmask + (tl + dt) * TPC_K6_PMW + w0;
        const u32 win = __funnelshift_r(pm[0], pm[1], sh) & ((dt == -2 || dt == 2) ? 0x1Fu : 0x11u);
        ring |= win << (5 * (dt + 2));
      }
      bool dead = false;
      if (ring) {   // some peak at Chebyshev distance exactly 2
        const u16* c = s.tile + tl * pitch + pad + TPC_PG;
        const u32 qc = c[0];
        u32 nq[3][3];
#pragma unroll
        for (int dt = -1; dt <= 1; ++dt)
#pragma unroll
          for (int dp = -1; dp <= 1; ++dp) nq[dt + 1][dp + 1] = c[dt * (int)pitch + dp];
#pragma unroll
        for (int dt = -2; dt <= 2; ++dt)
#pragma unroll
          for (int dp = -2; dp <= 2; ++dp) {
            if (dt != -2 && dt != 2 && dp != -2 && dp != 2) continue;
            if (!((ring >> (5 * (dt + 2) + dp + 2)) & 1u)) continue;
            const u32 q2 = c[dt * (int)pitch + dp];
            const bool beats = q2 > qc || (q2 == qc && (dt < 0 || (dt == 0 && dp < 0)));   // P:36 total order
            if (!beats) continue;
#pragma unroll
            for (int mt = -1; mt <= 1; ++mt)
#pragma unroll
              for (int mp = -1; mp <= 1; ++mp) {
                if (mt == 0 && mp == 0) continue;
                if (mt - dt > 1 || dt - mt > 1 || mp - dp > 1 || dp - mp > 1) continue;
                if (nq[mt + 1][mp + 1] + eps >= qc) dead = true;
              }
          }
      }
      return dead;
    };
    uint4 o0 = make_uint4(0u, 0u, 0u, 0u), o1 = make_uint4(0u, 0u, 0u, 0u);
    const auto owned = [&](u32 e) -> bool { return COG != 2 || ((e >> 8) >= TPC_HALO && (e >> 8) < TPC_TS + TPC_HALO); };
    const auto survivor = [&](u32 e) -> bool { return (s.rowmask[(e >> 8) * 8u + ((e & 0xFFu) >> 5)] >> (e & 31u)) & 1u; };
    // Q10'' (R8): the sums O3 with the charge of every cell that a partner's window also holds
    // split by the integer weights w_p(x) = (q_p >> 2 cheb(p, x)) + 1.  Partners = the survivors on the
    // outer ring of the window, read from rowmask (complete: barrier F).  Peak cells are never split.
    auto shared_sums = [&](u32 tl, u32 pad, const u16* c, u32& Q, int& Sp, int& St, u32& Spp, u32& Stt) -> bool {
      const u32 st0 = (pad > 2u ? pad : 2u) - 2u, w0 = st0 >> 5, sh = st0 & 31u;   // window bits pad-2 .. pad+2 of the survivor rows
      u32 ring = 0u;
#pragma unroll
      for (int dt = -2; dt <= 2; ++dt) {
        const u32* rm = s.rowmask + (tl + dt) * 8u + w0;
        u32 win = __funnelshift_r(rm[0], w0 < 7u ? rm[1] : 0u, sh);
        if (pad < 2u) win <<= 2u - pad;   // pads -2, -1 do not exist
        ring |= (win & ((dt == -2 || dt == 2) ? 0x1Fu : 0x11u)) << (5 * (dt + 2));
      }
      if (ring == 0u) return false;
      const u32 qc = c[0];
      u32 q5[25], den[25], kill = 0u;
#pragma unroll
      for (int k = 0; k < 25; ++k) {
        const int dt = k / 5 - 2, dp = k % 5 - 2, d = max(abs(dt), abs(dp));
        q5[k] = c[dt * (int)pitch + dp];
        den[k] = (qc >> (2 * d)) + 1u;
      }
      while (ring) {
        const int b = __ffs((int)ring) - 1;
        ring &= ring - 1u;
        const int et = b / 5 - 2, ep = b - (b / 5) * 5 - 2;
        const u32 qp = c[et * (int)pitch + ep];
#pragma unroll
        for (int k = 0; k < 25; ++k) {
          const int dt = k / 5 - 2, dp = k % 5 - 2;
          const int d2 = max(abs(et - dt), abs(ep - dp));
          if (d2 <= 2) den[k] += (qp >> (2 * d2)) + 1u;
          if (d2 == 0) kill |= 1u << k;
        }
      }
#pragma unroll
      for (int k = 0; k < 25; ++k) {
        const int dt = k / 5 - 2, dp = k % 5 - 2, d = max(abs(dt), abs(dp));
        const u32 wc = (qc >> (2 * d)) + 1u;
        u32 sh_q = q5[k];
        if (k != 12 && den[k] != wc) sh_q = q5[k] * wc / den[k];
        if ((kill >> k) & 1u) sh_q = 0u;
        Q += sh_q; Sp += (int)sh_q * dp; St += (int)sh_q * dt;
        Spp += sh_q * (u32)(dp * dp); Stt += sh_q * (u32)(dt * dt);
      }
      return true;
    };
    // O3 for one surviving peak: the integer sums, (c0, c1) = (Q, Sp, St, Spp), (Stt, words 1 and 2 of the cluster's
    // second half, 0); O4 = k6_finalise
    auto cog_int = [&](u32 e, uint4& c0, uint4& c1) {
      const u32 tl = e >> 8, pad = e & 0xFFu;
      const u16* c = s.tile + tl * pitch + pad + TPC_PG;
      // exact integer sums (Q12): per-row partial sums first, so the 25 loads and the adds of
      // different rows are independent (short dependency chains; any order gives the same bits)
      u32 Q = 0u, Spp = 0u, Stt = 0u;
      int Sp = 0, St = 0;
      bool done = false;
      if (COG == 2) done = shared_sums(tl, pad, c, Q, Sp, St, Spp, Stt);   // Q10'': false when the peak has no partner
      if (done) {
      } else if (COG != 1) {   // Q10: every in-range cell, weight 1 (the reading is a kernel variant: no run-time test)
#pragma unroll
        for (int dt = -2; dt <= 2; ++dt) {
          const u16* cr = c + dt * (int)pitch;
          const u32 a = cr[-2], b = cr[-1], m = cr[0], d = cr[1], e2 = cr[2];
          const u32 rq = (a + b) + (m + d) + e2;
          const int rsp = (int)(2u * e2 + d) - (int)(2u * a + b);
          const u32 rspp = 4u * (a + e2) + (b + d);
          Q += rq; Sp += rsp; Spp += rspp;
          St += (int)rq * dt; Stt += rq * (u32)(dt * dt);
        }
      } else {                 // Q10': an outer-ring cell counts only if the inner cell towards the peak holds charge
        u32 w5[5][5];
#pragma unroll
        for (int dt = -2; dt <= 2; ++dt)
#pragma unroll
          for (int dp = -2; dp <= 2; ++dp) w5[dt + 2][dp + 2] = c[dt * (int)pitch + dp];
#pragma unroll
        for (int dt = -2; dt <= 2; ++dt)
#pragma unroll
          for (int dp = -2; dp <= 2; ++dp)
            if (dt == -2 || dt == 2 || dp == -2 || dp == 2) {
              const int it = dt < -1 ? -1 : (dt > 1 ? 1 : dt), ip = dp < -1 ? -1 : (dp > 1 ? 1 : dp);
              if (w5[it + 2][ip + 2] == 0u) w5[dt + 2][dp + 2] = 0u;
            }
#pragma unroll
        for (int dt = -2; dt <= 2; ++dt) {
          const u32 a = w5[dt + 2][0], b = w5[dt + 2][1], m = w5[dt + 2][2], d = w5[dt + 2][3], e2 = w5[dt + 2][4];
          const u32 rq = (a + b) + (m + d) + e2;
          const int rsp = (int)(2u * e2 + d) - (int)(2u * a + b);
          const u32 rspp = 4u * (a + e2) + (b + d);
          Q += rq; Sp += rsp; Spp += rspp;
          St += (int)rq * dt; Stt += rq * (u32)(dt * dt);
        }
      }
      const u32 qc = c[0];
      const int t = t_base + (int)tl;
      u32 fl = 0u;
      if (pad < 2u || pad + 2u >= npads) fl |= 1u;
      if (t < 2 || (u32)t + 2u >= PRM(n_time)) fl |= 2u;
      if (qc == 1023u) fl |= 4u;
      c0 = make_uint4(Q, (u32)Sp, (u32)St, Spp);
      c1 = make_uint4(Stt, qc | ((u32)t << 16), pad | (row << 8) | (sector << 16) | (fl << 24), 0u);
    };
    auto cog_sums = [&](u32 e, uint4& c0, uint4& c1) { cog_int(e, c0, c1); k6_finalise(c0, c1); };
    auto emit = [&](u64 slot, const uint4& c0, const uint4& c1) {
      if (MODE == TPC_MODE_DET_TEMP) {
        if (slot < a.temp_cap) { a.temp[slot * 2u] = c0; a.temp[slot * 2u + 1u] = c1; }
      } else {
        if (slot < a.capacity) { a.out[slot * 2u] = c0; a.out[slot * 2u + 1u] = c1; }
        else atomicOr(a.status, TPC_STATUS_OVERFLOW);
      }
    };
    if (MODE == TPC_MODE_FAST) {
      // FAST: the order of the output is free (Q15), so nothing is ranked: every warp tests its peaks,
      // reserves the places of its survivors with one global atomic -- in flight while the 5x5 sums
      // are taken -- and writes them.  No survivor mask, no rank scan, no barrier before the emission.
      const u32 lane = lane_id(), lt = (1u << lane) - 1u;
      if (COG == 2) {   // Q10'': the survivor set of all listed rows first (the partners of the owned clusters), barrier F
        for (u32 i = tid; i < npk; i += TPC_K6_CONSUMERS) {
          const u32 e = s.peaks[i];
          if (!suppressed(e)) atomicOr(&s.rowmask[(e >> 8) * 8u + ((e & 0xFFu) >> 5)], 1u << (e & 31u));
        }
        csync();
      }
      if (total * 4u <= TPC_K6_CONSUMERS) {   // a sparse tile has at most one peak per thread: the clusters are written AFTER
        const u32 e = tid < npk ? s.peaks[tid] : 0u;   // barrier E, so that nobody waits there for the global atomic
        const bool keep = tid < npk && (COG == 2 ? owned(e) && survivor(e) : !suppressed(e));
        const u32 m = __ballot_sync(0xFFFFFFFFu, keep);
        u64 base = 0ull;
        u32 ridx = 0xFFFFFFFFu;   // this warp's first entry in the emitter's ring, if it has room
        if (EMIT && m) {
          if (lane == 0u) {
            const u32 n = (u32)__popc(m);
            for (;;) {
              const u32 h = *(volatile u32*)&s.rctl[0];
              if (h + n - *(volatile u32*)&s.rctl[1] > TPC_K6_RING) break;
              if (atomicCAS(&s.rctl[0], h, h + n) == h) { ridx = h; break; }
            }
          }
          ridx = __shfl_sync(0xFFFFFFFFu, ridx, 0);
        }
        const bool self = m != 0u && ridx == 0xFFFFFFFFu;   // warp-uniform
        if (lane == 0u && self) base = atomicAdd(a.n_clusters, (u64)__popc(m));
        if (keep) {
          cog_int(e, o0, o1);
          if (self) k6_finalise(o0, o1);
          else {
            const u32 i = ridx + __popc(m & lt), slot = i % TPC_K6_RING;
            o1.w = i / TPC_K6_RING + 1u;
            s.ring[2u * slot] = o0;
            __threadfence_block();
            s.ring[2u * slot + 1u] = o1;
          }
        }
        csync();   // E
        if (my_r != 0u) {
          const u32 tl = k6_row(my_r, sl), pad = my_r & 0xFFu;
          s.tile[tl * pitch + pad + TPC_PG] = 0;
          s.pmask[tl * TPC_K6_PMW + ((pad + TPC_PG) >> 5)] = 0u;
          if (COG == 2) s.rowmask[tl * 8u + (pad >> 5)] = 0u;
        }
        if (tid == 0) s.misc[0] = 0u;
        if (self) {
          base = __shfl_sync(0xFFFFFFFFu, base, 0);
          if (keep) emit(base + __popc(m & lt), o0, o1);
        }
        continue;
      }
      for (u32 i0 = (tid >> 5) * 32u; i0 < npk; i0 += TPC_K6_CONSUMERS) {
        const u32 i = i0 + lane;
        const u32 e = i < npk ? s.peaks[i] : 0u;
        const bool keep = i < npk && (COG == 2 ? owned(e) && survivor(e) : !suppressed(e));
        const u32 m = __ballot_sync(0xFFFFFFFFu, keep);
        if (!m) continue;
        u64 base = 0ull;
        if (lane == 0u) base = atomicAdd(a.n_clusters, (u64)__popc(m));
        if (keep) cog_sums(e, o0, o1);
        base = __shfl_sync(0xFFFFFFFFu, base, 0);
        if (keep) emit(base + __popc(m & lt), o0, o1);
      }
      // For the next tile (barrier A orders it before the scatter): barrier E -- nobody reads the map any
      // more -- then a sparse tile undoes its own writes (every cell and peak bit sits at a record, and
      // the thread that owns the record clears them) and any other tile is swept.
      csync();   // E
      if (total * 4u <= TPC_K6_CONSUMERS) {
        if (my_r != 0u) {
          const u32 tl = k6_row(my_r, sl), pad = my_r & 0xFFu;
          s.tile[tl * pitch + pad + TPC_PG] = 0;
          s.pmask[tl * TPC_K6_PMW + ((pad + TPC_PG) >> 5)] = 0u;
          if (COG == 2) s.rowmask[tl * 8u + (pad >> 5)] = 0u;
        }
        if (tid == 0) s.misc[0] = 0u;
      } else
        zero_tile();
      continue;
    }
    if (MODE == TPC_MODE_DET_TEMP && EMIT && total * 4u <= TPC_K6_CONSUMERS && npk <= 32u) {   // block-uniform
      // A sparse tile in deterministic mode: its peaks sit in the lanes of warp 0, which settles everything the
      // ordered output needs among its lanes -- the survivors (ballot), their ranks in (time, pad) order (the
      // keys compared by shuffle), the tile's run (cut from the CTA's block of the temporary buffer: a global
      // atomic per TPC_K6_BLK clusters, none per tile) -- and hands the clusters, with their places, to the
      // emitter warp.  No survivor mask, no rank scan over the 134 rows, barriers F and G gone.
      if (tid < 32u) {
        const u32 lane = tid, lt = (1u << lane) - 1u;
        const u32 e = lane < npk ? s.peaks[lane] : 0xFFFFu;
        const bool keep = lane < npk && !suppressed(e);
        const u32 m = __ballot_sync(0xFFFFFFFFu, keep);
        const u32 count = (u32)__popc(m);
        u32 rank = 0u;
        for (u32 mm = m; mm != 0u; mm &= mm - 1u) rank += __shfl_sync(0xFFFFFFFFu, e, __ffs((int)mm) - 1) < e ? 1u : 0u;
        u32 at = 0u, ridx = 0xFFFFFFFFu;
        if (lane == 0u) {
          u32 nx = s.misc[1], en = s.misc[2];
          if (count != 0u && nx + count > en) {   // a new block (what is left of the old one stays unused)
            const u64 g = atomicAdd(a.temp_cursor, (u64)TPC_K6_BLK);
            if (g + TPC_K6_BLK > a.temp_cap) atomicOr(a.det_flag, 1u);
            nx = (u32)(g < 0xFFFFFF00ull ? g : 0xFFFFFF00ull); en = nx + TPC_K6_BLK;   // (beyond the buffer: the flag is set, nothing is stored)
          }
          at = nx;
          s.misc[1] = nx + count; s.misc[2] = en;
          a.tile_base[tile] = at; a.tile_cnt[tile] = count;
          if (count != 0u)
            for (;;) {   // room in the emitter's ring?
              const u32 h = *(volatile u32*)&s.rctl[0];
              if (h + count - *(volatile u32*)&s.rctl[1] > TPC_K6_RING) break;
              if (atomicCAS(&s.rctl[0], h, h + count) == h) { ridx = h; break; }
            }
        }
        at = __shfl_sync(0xFFFFFFFFu, at, 0);
        ridx = __shfl_sync(0xFFFFFFFFu, ridx, 0);
        if (keep) {
          cog_int(e, o0, o1);
          if (ridx == 0xFFFFFFFFu) k6_finalise(o0, o1);   // the ring is full: this warp writes them itself, after barrier E
          else {
            const u32 i = ridx + __popc(m & lt), slot = i % TPC_K6_RING;
            o0 = make_uint4(o0.x | (o0.w << 15), o0.y, o0.z, at + rank);
            o1.w = i / TPC_K6_RING + 1u;
            s.ring[2u * slot] = o0;
            __threadfence_block();
            s.ring[2u * slot + 1u] = o1;
          }
        }
        csync();   // E
        if (keep && ridx == 0xFFFFFFFFu) emit((u64)(at + rank), o0, o1);
      } else
        csync();   // E
      if (my_r != 0u) {
        const u32 tl = k6_row(my_r, sl), pad = my_r & 0xFFu;
        s.tile[tl * pitch + pad + TPC_PG] = 0;
        s.pmask[tl * TPC_K6_PMW + ((pad + TPC_PG) >> 5)] = 0u;
      }
      if (tid == 0) s.misc[0] = 0u;
      continue;
    }
    bool survived = false;
    for (u32 i = tid; i < npk; i += TPC_K6_CONSUMERS) {
      const u32 e = s.peaks[i];
      if (!suppressed(e)) { atomicOr(&s.rowmask[(e >> 8) * 8u + ((e & 0xFFu) >> 5)], 1u << (e & 31u)); if (owned(e)) survived = true; }
    }
    // F: survivor set complete.  With at most one peak per thread (the usual case) the barrier
    // itself counts the survivors, so the tile's base can be requested before the rank scan.
    const u32 fcount = csync_popc(survived);
    const bool early = npk <= TPC_K6_CONSUMERS;   // block-uniform

    // ---- rank (last warp) || O3 + O4 (everyone else first) ------------------------------------
    // rowpre[tl] = survivors in rows < tl, which ranks every cluster in (time, pad) order inside
    // the tile without a sort.  The last warp computes it and fetches the tile's base (FAST: one
    // atomic; DET: the chained scan) while the other warps already do the 5x5 arithmetic; the
    // results meet at barrier G.
    if (tid >= TPC_K6_CONSUMERS - 32u) {
      const u32 lane = lane_id();
      u64 at = 0ull;   // FAST / DET_TEMP: the tile's place, one global atomic (in flight during the scan below)
      if (early && lane == 31u) {
        if (MODE == TPC_MODE_FAST) at = atomicAdd(a.n_clusters, (u64)fcount);
        if (MODE == TPC_MODE_DET_TEMP) at = atomicAdd(a.temp_cursor, (u64)fcount);
      }
      __syncwarp();   // keeps the atomic ahead of the loads below (ptxas sinks it otherwise)
      u32 cnt[5], t = 0u;
      {   // a lane counts 5 consecutive rows: ten 128-bit loads issued together, no branches
        const uint4* rm = (const uint4*)s.rowmask;
        uint4 v[10];
#pragma unroll
        for (int k = 0; k < 5; ++k) {
          const u32 tl = lane * 5u + (u32)k, tc = tl < TPC_TT ? tl : TPC_TT - 1u;
          v[2 * k] = rm[tc * 2u]; v[2 * k + 1] = rm[tc * 2u + 1u];
        }
#pragma unroll
        for (int k = 0; k < 5; ++k) {
          const uint4 x = v[2 * k], y = v[2 * k + 1];
          const u32 n = (__popc(x.x) + __popc(x.y)) + (__popc(x.z) + __popc(x.w)) + ((__popc(y.x) + __popc(y.y)) + (__popc(y.z) + __popc(y.w)));
          cnt[k] = (lane * 5u + (u32)k >= TPC_HALO && lane * 5u + (u32)k < TPC_TS + TPC_HALO) ? n : 0u; t += cnt[k];   // survivors only sit in listed rows, clusters in owned ones
        }
      }
      u32 inc = t;
#pragma unroll
      for (int d = 1; d < 32; d <<= 1) { u32 o = __shfl_up_sync(0xFFFFFFFFu, inc, d); if ((int)lane >= d) inc += o; }
      u32 ex = inc - t;
#pragma unroll
      for (int k = 0; k < 5; ++k) { const u32 tl = lane * 5u + (u32)k; if (tl < TPC_TT) s.rowpre[tl] = ex; ex += cnt[k]; }
      const u32 count = __shfl_sync(0xFFFFFFFFu, inc, 31);
      if (MODE == TPC_MODE_FAST) { if (lane == 31u) s.base[0] = early ? at : atomicAdd(a.n_clusters, (u64)count); }
      if (MODE == TPC_MODE_DET_TEMP) {
        if (lane == 31u) {
          if (!early) at = atomicAdd(a.temp_cursor, (u64)count);
          a.tile_base[tile] = at; a.tile_cnt[tile] = count; s.base[0] = at;
          if (at + count > a.temp_cap) atomicOr(a.det_flag, 1u);
        }
      }
      if (MODE == TPC_MODE_DET) {
        const u64 ex = k6_chain(a.tile_state, tile, count);
        if (lane == 0u) { s.base[0] = ex; if (tile == n_tiles - 1u) *a.n_clusters = ex + (u64)count; }
      }
    }
    // one cluster per thread held in registers across barrier G (further ones, npk > threads, after it)
    u32 inrow = 0xFFFFFFFFu, my_tl = 0u;
    auto cog = [&](u32 e, uint4& c0, uint4& c1, u32& rk) -> bool {
      const u32 tl = e >> 8, pad = e & 0xFFu;
      const u32 w = pad >> 5, bitpos = pad & 31u;
      const u32 mword = s.rowmask[tl * 8u + w];
      if (!((mword >> bitpos) & 1u) || !owned(e)) return false;   // suppressed, or a partner in a halo row
      rk = __popc(mword & ((1u << bitpos) - 1u));
      for (u32 k = 0; k < w; ++k) rk += __popc(s.rowmask[tl * 8u + k]);
      cog_sums(e, c0, c1);
      return true;
    };
    if (tid < npk) {
      const u32 e = s.peaks[tid];
      my_tl = e >> 8;
      u32 rk;
      if (cog(e, o0, o1, rk)) inrow = rk;
    }
    csync();   // G: rowpre and base are there; nobody reads the map of this tile's first 256 peaks any more
    {
      const u64 base = s.base[0];
      if (inrow != 0xFFFFFFFFu) emit(base + s.rowpre[my_tl] + inrow, o0, o1);
      for (u32 i = tid + TPC_K6_CONSUMERS; i < npk; i += TPC_K6_CONSUMERS) {   // dense tiles only
        const u32 e = s.peaks[i];
        u32 rk;
        if (cog(e, o0, o1, rk)) emit(base + s.rowpre[e >> 8] + rk, o0, o1);
      }
      if (npk > TPC_K6_CONSUMERS) csync();   // block-uniform: the extra clusters still read the map
    }
    // for the next tile (barrier A orders it before the scatter).  A sparse tile undoes its own
    // writes instead of sweeping 50 KB: every cell, peak bit and survivor bit sits at a record,
    // and the thread that owns the record clears the three words.
    if (total * 4u <= TPC_K6_CONSUMERS) {   // block-uniform (the condition of the sparse scatter)
      if (my_r != 0u) {
        const u32 tl = k6_row(my_r, sl), pad = my_r & 0xFFu;
        s.tile[tl * pitch + pad + TPC_PG] = 0;
        s.pmask[tl * TPC_K6_PMW + ((pad + TPC_PG) >> 5)] = 0u;
        s.rowmask[tl * 8u + (pad >> 5)] = 0u;
      }
      if (tid == 0) s.misc[0] = 0u;
    } else
      zero_tile();
   }
  }
  if (EMIT) {   // every entry of the ring is written: tell the emitter warp
    csync();
    if (tid == 0) { __threadfence_block(); *(volatile u32*)&s.rctl[2] = 1u; }
  }
}

#define TPC_K6_ENTRY(name, MODE, COG, EMIT, GUARD)                                                      \
  extern "C" __global__ void __launch_bounds__((EMIT) ? TPC_K6_THREADS_E : TPC_K6_THREADS, TPC_K6_CTAS) name(K6Args a) { \
    extern __shared__ __align__(128) u32 smem_u32[];                                                    \
    GUARD                                                                                               \
    k6_body<MODE, COG, EMIT>(a, smem_u32);                                                            \
  }
// the chained-scan variants only run when K7-K9 could not deliver the ordered output (flag set)
#define TPC_K6_IF_FLAG if (*a.det_flag == 0u) return;
#if TPC_UNITS & TPC_U_TILES_FAST
TPC_K6_ENTRY(k_cluster_tiles_fast, TPC_MODE_FAST, 0, false, )
TPC_K6_ENTRY(k_cluster_tiles_fast_e, TPC_MODE_FAST, 0, true, )
#endif
#if TPC_UNITS & TPC_U_TILES_DET
TPC_K6_ENTRY(k_cluster_tiles_det, TPC_MODE_DET, 0, false, TPC_K6_IF_FLAG)
TPC_K6_ENTRY(k_cluster_tiles_det_temp, TPC_MODE_DET_TEMP, 0, false, )
TPC_K6_ENTRY(k_cluster_tiles_det_temp_e, TPC_MODE_DET_TEMP, 0, true, )
#endif
#if TPC_UNITS & TPC_U_TILES_DUMP
TPC_K6_ENTRY(k_cluster_tiles_dump_map, TPC_MODE_DUMP_MAP, 0, false, )
#endif
// reading Q10' (TPCCLUS_COG_GATED)
#if TPC_UNITS & TPC_U_TILES_FAST_G
TPC_K6_ENTRY(k_cluster_tiles_fast_gated, TPC_MODE_FAST, 1, false, )
TPC_K6_ENTRY(k_cluster_tiles_fast_gated_e, TPC_MODE_FAST, 1, true, )
#endif
#if TPC_UNITS & TPC_U_TILES_DET_G
TPC_K6_ENTRY(k_cluster_tiles_det_gated, TPC_MODE_DET, 1, false, TPC_K6_IF_FLAG)
TPC_K6_ENTRY(k_cluster_tiles_det_temp_gated, TPC_MODE_DET_TEMP, 1, false, )
TPC_K6_ENTRY(k_cluster_tiles_det_temp_gated_e, TPC_MODE_DET_TEMP, 1, true, )
#endif
// reading Q10'' (TPCCLUS_COG_SHARED): these units -- and the partition units of such a handle -- are compiled with TPC_HALO = 5
#if TPC_UNITS & TPC_U_TILES_FAST_S
TPC_K6_ENTRY(k_cluster_tiles_fast_shared, TPC_MODE_FAST, 2, false, )
#endif
#if TPC_UNITS & TPC_U_TILES_DET_S
TPC_K6_ENTRY(k_cluster_tiles_det_shared, TPC_MODE_DET, 2, false, TPC_K6_IF_FLAG)
TPC_K6_ENTRY(k_cluster_tiles_det_temp_shared, TPC_MODE_DET_TEMP, 2, false, )
#endif
#endif   // TPC_UNITS != 0u
