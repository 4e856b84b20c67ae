// librlxpp: RANLUX++ stream generation for B200 (sm_100a).  C ABI in include/rlxpp.h; this file is the host side
// (tables, caches, launch logic, the extern "C" entry points) and the one translation unit of the library.
//
// Hot path, one thread per stream, the 576-bit state as 18 x 32-bit limbs in registers.  Per LCG advance
// (PAPER.md lines 29, 33, 39):
//   multiply9x9 + mod_m -> UMMA engine (default): one u8 x u8 -> s32 tcgen05.mma tile per 128 streams against the byte
//                   matrix of A 2^(8k) mod m, then a 72-column carry normalisation and a 15-bit fold
//                   (include/rlxpp_tile.cuh, umma_path.cuh, kernels_umma.cuh);
//                   IMAD engine: 324 IMAD.WIDE.U32.X with the multiplier as immediates, rows pre-reduced mod m
//                   (include/rlxpp_rows.cuh, state.cuh, kernels_imad.cuh)
//   to_ranlux    -> 8-limb add + carry decision (to_ranlux_fast; exact fallback)
//   12 doubles   -> byte permutes + one exact DADD each (emit.cuh); coalesced 64-bit stores (interleaved layout), TMA
//                   boxes staged in shared memory (stream-major: stages.cuh) or DADD / DFMA accumulation in registers
//                   (fused reduce).
#include <cuda.h>
#include <cuda_runtime.h>

#include <atomic>
#include <functional>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <mutex>
#include <string>
#include <vector>

#include "../../include/rlxpp.h"
#include "arith.cuh"
#include "normal_coeffs.cuh"
#include "host_bigint.h"

namespace rlx {

// ----------------------------------------------------------------------------- errors
static thread_local std::string g_last_error;
static std::atomic<uint64_t> g_launches{0};

static int fail(int code, const char* fmt, ...) {
  char buf[512];
  va_list ap;
  va_start(ap, fmt);
  vsnprintf(buf, sizeof(buf), fmt, ap);
  va_end(ap);
  g_last_error = buf;
  return code;
}
#define CUDA_TRY(expr)                                                                         \
  do {                                                                                         \
    cudaError_t _e = (expr);                                                                   \
    if (_e != cudaSuccess)                                                                     \
      return fail(_e == cudaErrorMemoryAllocation ? RLXPP_ENOMEM : RLXPP_ECUDA, "%s: %s", #expr, \
                  cudaGetErrorString(_e));                                                     \
  } while (0)
#define LAUNCH_CHECK()        \
  do {                        \
    g_launches++;             \
    CUDA_TRY(cudaGetLastError()); \
  } while (0)

}  // namespace rlx

#include "state.cuh"
#include "emit.cuh"
#include "kernels_imad.cuh"
#include "umma_path.cuh"
#include "stages.cuh"
#include "kernels_umma.cuh"
#include "kernels_misc.cuh"

namespace rlx {

// ----------------------------------------------------------------------------- host side
struct Tables {
  uint32_t p = 0;
  Limbs18 A;
  std::vector<uint32_t> tabA, tabG;  // [64][18]: A^(2^b), G^(2^b) with G = A^(2^96)
};

static void build_tables(uint32_t p, Tables& t, bool with_pow_tables) {
  t.p = p;
  host::Big A = host::multiplier_ap(p);
  A.to_u32x18(t.A.v);
  if (!with_pow_tables) return;
  t.tabA.resize(64 * 18);
  t.tabG.resize(64 * 18);
  host::Big cur = A;
  for (int b = 0; b < 64; b++) {
    cur.to_u32x18(&t.tabA[b * 18]);
    cur = host::mulmod(cur, cur);
  }
  cur = host::pow2k(A, 96);
  for (int b = 0; b < 64; b++) {
    cur.to_u32x18(&t.tabG[b * 18]);
    cur = host::mulmod(cur, cur);
  }
}

// The tables depend on p only (about 230 host modular products): built once per luxury level and process.
static const Tables& cached_tables(uint32_t p) {
  static std::mutex mu;
  static std::vector<Tables*> cache;  // never freed: handles keep references
  std::lock_guard<std::mutex> lock(mu);
  for (const Tables* t : cache)
    if (t->p == p) return *t;
  Tables* t = new Tables();
  build_tables(p, *t, true);
  cache.push_back(t);
  return *t;
}

// Shared-memory image of the byte matrix B of the UMMA engine: B[n][k] = byte n of
// R_k = A 2^(8k) mod m (k, n < 72), zero padding up to 80 x 96, laid out as tc::b_offset says.
static void build_bmatrix(uint32_t p, std::vector<uint8_t>& img) {
  img.assign(tc::kBBytes, 0);
  host::Big R = host::multiplier_ap(p);
  for (int k = 0; k < tc::kKUsed; k++) {  // 72 bytes of a state + the two bytes an unreduced product has above 2^576
    uint32_t w[18];
    R.to_u32x18(w);
    for (int n = 0; n < 72; n++) img[tc::b_offset(n, k)] = (uint8_t)(w[n / 4] >> (8 * (n % 4)));
    R = host::reduce(host::Big::shl(R, 8));
  }
}

// Device copies of B, one per (device, p), kept for the life of the process (7.5 KB each).
struct BmatEntry { int dev; uint32_t p; uint4* ptr; };
static std::mutex g_bmat_mutex;
static std::vector<BmatEntry> g_bmat_cache;
static int get_bmatrix(uint32_t p, const uint4** out) {
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lock(g_bmat_mutex);
  for (const BmatEntry& e : g_bmat_cache)
    if (e.dev == dev && e.p == p) { *out = e.ptr; return RLXPP_OK; }
  std::vector<uint8_t> img;
  build_bmatrix(p, img);
  uint4* d = nullptr;
  CUDA_TRY(cudaMalloc(&d, tc::kBBytes));
  cudaError_t e = cudaMemcpy(d, img.data(), tc::kBBytes, cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(d);
    return fail(RLXPP_ECUDA, "uploading the UMMA byte matrix: %s", cudaGetErrorString(e));
  }
  g_bmat_cache.push_back({dev, p, d});
  *out = d;
  return RLXPP_OK;
}

// Images of the byte matrices of A^1 .. A^kMaxLanes (time-parallel path), one set per (device, p), built on first use.
static std::vector<BmatEntry> g_bmat_pow_cache;
static int get_bmatrix_powers(uint32_t p, const uint4** out) {
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  std::lock_guard<std::mutex> lock(g_bmat_mutex);
  for (const BmatEntry& e : g_bmat_pow_cache)
    if (e.dev == dev && e.p == p) { *out = e.ptr; return RLXPP_OK; }
  std::vector<uint8_t> all((size_t)kMaxLanes * tc::kBBytes, 0);
  const host::Big A = host::multiplier_ap(p);
  host::Big R0 = A;  // A^(k + 1)
  for (u32 k = 0; k < kMaxLanes; k++) {
    host::Big R = R0;
    uint8_t* img = all.data() + (size_t)k * tc::kBBytes;
    for (int col = 0; col < tc::kKUsed; col++) {
      uint32_t w[18];
      R.to_u32x18(w);
      for (int n = 0; n < 72; n++) img[tc::b_offset(n, col)] = (uint8_t)(w[n / 4] >> (8 * (n % 4)));
      R = host::reduce(host::Big::shl(R, 8));
    }
    R0 = host::mulmod(R0, A);
  }
  uint4* d = nullptr;
  CUDA_TRY(cudaMalloc(&d, all.size()));
  cudaError_t e = cudaMemcpy(d, all.data(), all.size(), cudaMemcpyHostToDevice);
  if (e != cudaSuccess) {
    cudaFree(d);
    return fail(RLXPP_ECUDA, "uploading the byte matrices of A^k: %s", cudaGetErrorString(e));
  }
  g_bmat_pow_cache.push_back({dev, p, d});
  *out = d;
  return RLXPP_OK;
}

// engine used by advance_states / generate_*: the tensor-core path unless told otherwise
static std::atomic<int> g_engine{RLXPP_ENGINE_UMMA};
// > 0: cut every tile into this many chunks whatever plan_items says (rlxpp_set_chunks; tests)
static std::atomic<int> g_force_chunks{0};

template <int P>
static bool fixed_matches(const Limbs18& A) {
  for (int j = 0; j < 18; j++)
    if (FixedMultiplier<P>::kA[j] != A.v[j]) return false;
  return true;
}
// which baked-in multiplier serves p (0 = none): the generated constants must equal the
// host's own a^p, otherwise the header is stale and we refuse to use it
static int fixed_level(uint32_t p, const Limbs18& A) {
#define RLXPP_CASE(P) \
  if (p == P) return fixed_matches<P>(A) ? P : -1;
  RLXPP_FOR_EACH_FIXED_P(RLXPP_CASE)
#undef RLXPP_CASE
  return 0;
}

}  // namespace rlx

using namespace rlx;

struct rlxpp {
  uint64_t n = 0;
  uint32_t p = 0;
  int fixed = 0;
  cudaStream_t stream = nullptr;
  cudaStream_t copy_stream = nullptr;
  uint4* st = nullptr;
  uint32_t* tabA = nullptr;
  uint32_t* tabG = nullptr;
  const uint4* bmat = nullptr;  // owned by the process-wide cache
  uint32_t* sched = nullptr;    // scheduler words of the persistent UMMA kernel: 1 + ceil(n / 128)
  uint32_t* lane_sync = nullptr;  // time-parallel path: one reader counter per tile, zero between launches
  double* scratch_q = nullptr;  // sum of squares when the caller passes none (chunked reduce carries it)
  Tables tables;
  bool aligned = true;  // every cursor is known to be 12
  uint32_t uniform_pos = 12;
  bool pos_uniform = true;
  // staging for the *_host variants
  double* stage[2] = {nullptr, nullptr};
  size_t stage_bytes = 0;
  cudaEvent_t ev_kernel[2] = {nullptr, nullptr};
  cudaEvent_t ev_copy[2] = {nullptr, nullptr};
};

static inline unsigned grid_for(uint64_t n) { return (unsigned)((n + kThreads - 1) / kThreads); }

template <class Mult, int MODE>
static int launch_generate_mode(const GenArgs& a, bool aligned, cudaStream_t s) {
  if (aligned) generate_kernel<Mult, MODE, true><<<grid_for(a.count), kThreads, 0, s>>>(a);
  else generate_kernel<Mult, MODE, false><<<grid_for(a.count), kThreads, 0, s>>>(a);
  LAUNCH_CHECK();
  return RLXPP_OK;
}
template <class Mult>
static int launch_generate_mult(const GenArgs& a, int mode, bool aligned, cudaStream_t s) {
  switch (mode) {
    case kStoreStreamMajor: return launch_generate_mode<Mult, kStoreStreamMajor>(a, aligned, s);
    case kStoreInterleaved: return launch_generate_mode<Mult, kStoreInterleaved>(a, aligned, s);
    default: return launch_generate_mode<Mult, kReduce>(a, aligned, s);
  }
}
// Work items of the persistent UMMA kernel: how many chunks to cut every tile's n_per draws into.  One chunk unless the
// tiles alone fill the resident CTAs badly; a chunk is never shorter than 16 advances (state I/O and pipeline fill).
//   Store kernels (hbm_bound): the CTAs of a wave start together and, all waiting on the same HBM, stay in step, so every
//   wave boundary is a bubble in the write stream that no other CTA fills, while a ragged last wave costs little (the
//   CTAs still running get the bandwidth of those that finished).  Fewest chunks that give >= 6.5 items per resident
//   CTA (items of two tiles; 13 where an item is one tile): measured round 3 (profiles/ab_r03_chunks.md) cfg3 787 -> 827 G doubles/s with 1 chunk instead of 2; within 2 %
//   of the best chunk count on every shape tried (2^18 .. 2^21 streams x 768 .. 6,144 draws).
//   Fused reduce (ALU-bound): CTAs run at their own pace and the last wave counts in full: >= 97 % fill and >= 12 waves.
static void plan_items(uint64_t n_tiles, uint64_t n_per, unsigned slots, uint32_t* n_chunks, uint64_t* chunk_len, bool hbm_bound,
                       bool pairs) {
  *n_chunks = 1;
  *chunk_len = n_per;
  const uint64_t blocks = n_per / 12;
  if (n_tiles <= slots || blocks < 32) return;
  uint64_t best_c = 1;
  if (hbm_bound) {
    const uint64_t want = pairs ? ((uint64_t)slots * 13 + 1) / 2 : (uint64_t)slots * 13;  // 6.5 items of two tiles per resident CTA, or 13 of one
    best_c = (want + n_tiles - 1) / n_tiles;
    if (best_c > 16) best_c = 16;
    while (best_c > 1 && blocks / best_c < 16) best_c--;
  } else {
    double best = 0.0;
    for (uint64_t c = 1; c <= 16 && blocks / c >= 16; c++) {
      const uint64_t items = n_tiles * c, waves = (items + slots - 1) / slots;
      const double eff = (double)items / (double)(waves * slots);
      const double score = eff - (waves < 12 ? 0.05 : 0.0);
      if (score > best + 1e-9) { best = score; best_c = c; }
      if (eff >= 0.97 && waves >= 12) break;
    }
  }
  if (best_c == 1) return;
  const uint64_t len = ((blocks + best_c - 1) / best_c + 7) / 8 * 96;  // whole cycles of 8 blocks (StreamMajorStage)
  *chunk_len = len;
  *n_chunks = (uint32_t)((n_per + len - 1) / len);
}

static unsigned tc_slots() {  // resident CTAs of the persistent UMMA kernels on the CURRENT device
  static std::atomic<unsigned> cache[64];
  int dev = 0, sms = 148;
  if (cudaGetDevice(&dev) != cudaSuccess) dev = 0;
  if (dev >= 0 && dev < 64 && cache[dev].load()) return cache[dev].load();
  cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
  const unsigned slots = (unsigned)sms * tc::kCtasPerSm;
  if (dev >= 0 && dev < 64) cache[dev].store(slots);
  return slots;
}

// cuTensorMapEncodeTiled from the driver through the runtime (no link against libcuda); looked up once.
typedef CUresult (*TensorMapEncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                      const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                      CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
static int tensor_map_encoder(TensorMapEncodeFn* out) {
  static std::atomic<void*> cached{nullptr};
  void* fn = cached.load();
  if (!fn) {
    cudaDriverEntryPointQueryResult q;
    CUDA_TRY(cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &q));
    if (q != cudaDriverEntryPointSuccess || !fn) return fail(RLXPP_ECUDA, "cuTensorMapEncodeTiled is not available");
    cached.store(fn);
  }
  *out = (TensorMapEncodeFn)fn;
  return RLXPP_OK;
}

// Opt-in shared memory of a kernel above the 48 KB default, set once per (kernel, device).
template <class Kernel>
static int allow_dynamic_smem(Kernel kernel, std::atomic<uint64_t>& done, int bytes) {
  int dev = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 64 && (done.load() >> dev & 1)) return RLXPP_OK;
  CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, bytes));
  CUDA_TRY(cudaFuncSetAttribute(kernel, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
  if (dev < 64) done.fetch_or(1ull << dev);
  return RLXPP_OK;
}

// Tensor map of a stream-major output (UMMA engine, aligned): out[count][n_per] doubles viewed as
// [count][n_per / 16][16], box 32 x 2 x 16, 128-byte swizzle (StreamMajorStage).  n_per >= 16.
static int encode_stream_major_map(CUtensorMap* map, double* out, uint64_t count, uint64_t n_per, uint64_t pitch) {
  TensorMapEncodeFn encode = nullptr;
  const int erc = tensor_map_encoder(&encode);
  if (erc) return erc;
  if (n_per >= (1ull << 31) || count >= (1ull << 31))
    return fail(RLXPP_EINVAL, "stream-major output: n_per_stream and the stream count must be below 2^31");
  const cuuint64_t dims[3] = {16, n_per / 16, count};
  const cuuint64_t strides[2] = {16 * sizeof(double), pitch * sizeof(double)};
  const cuuint32_t box[3] = {16, 2, 32};
  const cuuint32_t estr[3] = {1, 1, 1};
  const CUresult r = encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 3, out, dims, strides, box, estr,
                            CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE,
                            CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(RLXPP_ECUDA, "cuTensorMapEncodeTiled failed (%d)", (int)r);
  return RLXPP_OK;
}

// Tensor map of an interleaved float output (F32RowStage): float rows of `ld` floats, `count` of them written by this
// launch, 2 n_per rows; box = 128 streams x 24 rows.  ld must be a multiple of 4 (16-byte row pitch).
static int encode_f32_rows_map(CUtensorMap* map, float* out, uint64_t count, uint64_t ld, uint64_t rows) {
  TensorMapEncodeFn encode = nullptr;
  const int erc = tensor_map_encoder(&encode);
  if (erc) return erc;
  const cuuint64_t dims[2] = {count, rows};
  const cuuint64_t strides[1] = {ld * sizeof(float)};
  const cuuint32_t box[2] = {128, 24};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT32, 2, out, dims, strides, box, estr,
                                    CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_NONE,
                                    CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(RLXPP_ECUDA, "cuTensorMapEncodeTiled (float rows) failed (%d)", (int)r);
  return RLXPP_OK;
}

// Tensor map of a stream-major output whose rows are written through RingStage (cursors not at a block boundary):
// out[count][n_per] doubles with a row pitch of `pitch` doubles (even), box = 16 doubles x 32 rows, 128-byte swizzle.
static int encode_ring_map(CUtensorMap* map, double* out, uint64_t count, uint64_t n_per, uint64_t pitch) {
  TensorMapEncodeFn encode = nullptr;
  const int erc = tensor_map_encoder(&encode);
  if (erc) return erc;
  const cuuint64_t dims[2] = {n_per, count};
  const cuuint64_t strides[1] = {pitch * sizeof(double)};
  const cuuint32_t box[2] = {16, 32};
  const cuuint32_t estr[2] = {1, 1};
  const CUresult r = encode(map, CU_TENSOR_MAP_DATA_TYPE_FLOAT64, 2, out, dims, strides, box, estr, CU_TENSOR_MAP_INTERLEAVE_NONE,
                            CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_NONE, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
  if (r != CUDA_SUCCESS) return fail(RLXPP_ECUDA, "cuTensorMapEncodeTiled (ring rows) failed (%d)", (int)r);
  return RLXPP_OK;
}

template <int MODE, int OUT = kF64>
static int launch_tc_generate_mode(GenArgs a, bool aligned, cudaStream_t s) {
  if (MODE == kStoreInterleaved && OUT == kF32 && aligned && a.ld % 4 == 0 && a.count < (1ull << 31) && a.n_per < (1ull << 30)) {
    const int rc = encode_f32_rows_map(&a.tmap, reinterpret_cast<float*>(a.out), a.count, a.ld, 2 * a.n_per);
    if (rc) return rc;
    a.f32_boxes = 1;
  }
  if (MODE == kStoreStreamMajor && aligned && a.n_per >= kStageCycle) {  // shorter rows never reach the TMA path
    const int rc = encode_stream_major_map(&a.tmap, a.out, a.count, a.n_per, a.pitch ? a.pitch : a.n_per);
    if (rc) return rc;
  }
  // the fused reduce and the interleaved stores run two tiles per CTA (tc_pair_kernel): their work items are pairs of
  // tiles.  (Interleaved floats keep the one-tile kernel with its row boxes, stream-major its staged TMA path.)
  constexpr bool kPairs = MODE == kReduce || (MODE == kStoreInterleaved && OUT != kF32);
  const uint64_t n_tiles = kPairs ? (a.count + 2 * tc::kTile - 1) / (2 * tc::kTile) : (a.count + tc::kTile - 1) / tc::kTile;
  // stream-major rows shifted against each other go through per-lane rings and TMA boxes when the rows are 16-byte
  // aligned (even pitch; RingStage: 57 KB of shared memory, three CTAs per SM), else through the warp's row stage
  const uint64_t row_pitch = a.pitch ? a.pitch : a.n_per;
  const bool ring = MODE == kStoreStreamMajor && !aligned && row_pitch % 2 == 0 && (uintptr_t)a.out % 16 == 0 &&
                    a.count < (1ull << 31) && a.n_per < (1ull << 31);
  const unsigned slots = ring ? tc_slots() / tc::kCtasPerSm * 3 : tc_slots();  // (a fourth CTA per SM fits since the A operands left shared memory: measured, no gain)
  a.n_tiles = (u32)n_tiles;
  if constexpr (MODE != kReduce) {
    // Short calls that leave most of the grid empty: K lanes per tile, each reaching its blocks with the matrices of
    // A^(j+1) and A^K (tc_generate_lanes_kernel).  All CTAs must be co-resident (the last lane waits for its tile's
    // readers): n_tiles K <= slots.  rlxpp_set_chunks(c > 0) keeps the persistent path.
    const uint64_t nblk = a.n_per / 12, tiles1 = (a.count + tc::kTile - 1) / tc::kTile;  // lanes work on single tiles
    uint64_t K = nblk < kMaxLanes ? nblk : kMaxLanes;
    uint64_t lane_slots = slots;
    if (aligned && a.lane_sync && g_force_chunks.load() == 0 && K >= 4 && tiles1 * 4 <= slots) {
      // what the runtime will accept as a cooperative grid: queried once per (kernel, device)
      static std::atomic<int> cached[64];
      int dev = 0, per_sm = 0;
      CUDA_TRY(cudaGetDevice(&dev));
      if (dev < 64) per_sm = cached[dev].load();
      if (per_sm == 0) {
        CUDA_TRY(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&per_sm, tc_generate_lanes_kernel<MODE, OUT>, tc::kTile, 0));
        if (dev < 64) cached[dev].store(per_sm);
      }
      lane_slots = (uint64_t)(slots / tc::kCtasPerSm) * (uint64_t)(per_sm < tc::kCtasPerSm ? per_sm : tc::kCtasPerSm);
    }
    if (K > lane_slots / tiles1) K = lane_slots / tiles1;
    if (aligned && a.lane_sync && K >= 4 && g_force_chunks.load() == 0) {
      int rc = get_bmatrix_powers(a.p, &a.bmat_pow);
      if (rc) return rc;
      a.lanes = (u32)K;
      // A cooperative launch: the lane that writes a tile's new state waits for the tile's other lanes to have read the
      // old one, so all CTAs must be resident together -- the runtime guarantees it (and holds the launch back while other
      // work occupies the SMs) instead of the grid size merely allowing it.
      void* params[] = {&a};
      CUDA_TRY(cudaLaunchCooperativeKernel(reinterpret_cast<const void*>(&tc_generate_lanes_kernel<MODE, OUT>),
                                           dim3((unsigned)(tiles1 * K)), dim3(tc::kTile), params, 0, s));
      g_launches++;
      return RLXPP_OK;
    }
  }
  plan_items(n_tiles, a.n_per, slots, &a.n_chunks, &a.chunk_len, MODE != kReduce, kPairs);
  if (g_force_chunks.load() > 0 && a.n_per / 12 >= (uint64_t)g_force_chunks.load()) {  // test hook
    const uint64_t c = (uint64_t)g_force_chunks.load(), blocks = a.n_per / 12;
    a.chunk_len = ((blocks + c - 1) / c + 7) / 8 * 96;
    a.n_chunks = (u32)((a.n_per + a.chunk_len - 1) / a.chunk_len);
  }
  const uint64_t items = n_tiles * a.n_chunks;
  const unsigned grid = (unsigned)(items < slots ? items : slots);
  CUDA_TRY(cudaMemsetAsync(a.sched, 0, sizeof(u32) * (1 + (a.n_chunks > 1 ? n_tiles : 0)), s));
  if constexpr (kPairs) {
    // (Row boxes through the TMA instead of the direct stores were tried for the 8-byte outputs: same burst rate, and
    // under the power cap NOT better -- doubles 663 vs 662, 48-bit integers 676 vs 704 G/s sustained; profiles/ab_r02_pairs.md.)
    if (aligned) tc_pair_kernel<true, MODE, OUT><<<grid, tc::kTile, 0, s>>>(a);
    else tc_pair_kernel<false, MODE, OUT><<<grid, tc::kTile, 0, s>>>(a);
  } else if (aligned) {
    constexpr bool kStaged = MODE == kStoreStreamMajor;  // the kernel's kStaged
    // 8 KB static + 33 KB (stream-major boxes) or 36 KB (float-row boxes): the function attribute is needed above 48 KB in all; 4 CTAs per SM fit
    if (kStaged || a.f32_boxes) {
      static std::atomic<uint64_t> done{0};  // one bit per device: function attributes are per device
      const int rc = allow_dynamic_smem(tc_generate_kernel<MODE, true, OUT>, done, (int)(kStaged ? kStageCtaBytes : kF32StageBytes));
      if (rc) return rc;
    }
    tc_generate_kernel<MODE, true, OUT><<<grid, tc::kTile, kStaged ? kStageCtaBytes : (a.f32_boxes ? kF32StageBytes : 0), s>>>(a);
  } else if (MODE == kStoreStreamMajor) {
    unsigned dyn = 4 * kRowStageWarpBytes;
    if (ring) {
      int rc = encode_ring_map(&a.tmap, a.out, a.count, a.n_per, row_pitch);
      if (rc) return rc;
      static std::atomic<uint64_t> done{0};  // 8 KB static + 49 KB of rings
      rc = allow_dynamic_smem(tc_generate_kernel<MODE, false, OUT>, done, (int)kRingCtaBytes);
      if (rc) return rc;
      a.ring = 1;
      dyn = kRingCtaBytes;
    }
    tc_generate_kernel<MODE, false, OUT><<<grid, tc::kTile, dyn, s>>>(a);
  } else {
    tc_generate_kernel<MODE, false, OUT><<<grid, tc::kTile, 0, s>>>(a);
  }
  LAUNCH_CHECK();
  return RLXPP_OK;
}
static int launch_generate(int fixed, const GenArgs& a, int mode, bool aligned, cudaStream_t s) {
  if (g_engine.load() == RLXPP_ENGINE_UMMA) {
    switch (mode) {
      case kStoreStreamMajor: return launch_tc_generate_mode<kStoreStreamMajor>(a, aligned, s);
      case kStoreInterleaved: return launch_tc_generate_mode<kStoreInterleaved>(a, aligned, s);
      default: return launch_tc_generate_mode<kReduce>(a, aligned, s);
    }
  }
#define RLXPP_CASE(P) \
  if (fixed == P) return launch_generate_mult<Fixed<P>>(a, mode, aligned, s);
  RLXPP_FOR_EACH_FIXED_P(RLXPP_CASE)
#undef RLXPP_CASE
  return launch_generate_mult<Generic>(a, mode, aligned, s);
}

template <class Mult>
static int launch_advance_mult(uint64_t* states, uint64_t n, uint32_t reps, int layout, const Limbs18& A,
                               cudaStream_t s) {
  if (layout == RLXPP_AOS) advance_states_kernel<Mult, RLXPP_AOS><<<grid_for(n), kThreads, 0, s>>>(states, n, reps, A);
  else advance_states_kernel<Mult, RLXPP_SOA><<<grid_for(n), kThreads, 0, s>>>(states, n, reps, A);
  LAUNCH_CHECK();
  return RLXPP_OK;
}

static int check_device() {
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  return RLXPP_OK;
}

// ----------------------------------------------------------------------------- rlxpp_generate_doubles_static
// The scratch of the one entry point that allocates nothing (include/rlxpp.h says who needs that and why).  It is
// part of the library's device image: each GPU gets its own copy when the image is loaded there and keeps it until
// the process ends.  Layout, all offsets multiples of 256 bytes:
//   [kStaticBmat,  + 8 KB)   byte matrix of the luxury level last used on this device (tc::kBBytes = 7,680)
//   [kStaticSched, + 4 KB)   scheduler words of the persistent kernel: ticket + one chunk counter per tile (<= 513)
//   [kStaticState, + 5 MB)   the five state planes of up to RLXPP_STATIC_MAX_STREAMS streams (80 bytes each)
// In HOST code `g_static_scratch` is only a stand-in the runtime knows the symbol by -- not a device address; handing
// it to a kernel would fault, or quietly use the wrong memory.  static_scratch_base() asks the runtime for the real
// address, once per device, with that device current.
constexpr size_t kStaticBmat = 0, kStaticSched = 8192, kStaticState = 12288;
constexpr size_t kStaticBytes = kStaticState + 5 * sizeof(uint4) * RLXPP_STATIC_MAX_STREAMS;
static_assert(kStaticBytes == RLXPP_STATIC_SCRATCH_BYTES, "rlxpp.h states the size of the static scratch");
static_assert(tc::kBBytes <= kStaticSched - kStaticBmat, "byte matrix does not fit its slot");
static_assert((1 + (RLXPP_STATIC_MAX_STREAMS + tc::kTile - 1) / tc::kTile) * sizeof(uint32_t) <= kStaticState - kStaticSched,
              "scheduler words do not fit their slot");
static __device__ __align__(256) unsigned char g_static_scratch[kStaticBytes];

struct StaticDev {
  unsigned char* base = nullptr;  // device address of g_static_scratch on this device
  uint32_t p_loaded = 0;          // luxury level whose byte matrix sits at kStaticBmat (0 = none yet)
};
static std::mutex g_static_mutex;
static StaticDev g_static_dev[64];

// Host images of the byte matrices, one per p, never freed: the upload below reads them asynchronously.
static const std::vector<uint8_t>& static_bmatrix_image(uint32_t p) {
  static std::vector<std::pair<uint32_t, std::vector<uint8_t>*>> cache;  // under g_static_mutex
  for (const auto& e : cache)
    if (e.first == p) return *e.second;
  std::vector<uint8_t>* img = new std::vector<uint8_t>();
  build_bmatrix(p, *img);
  cache.emplace_back(p, img);
  return *img;
}

// Set-up of the static scratch for the CURRENT device and luxury level p: address look-up on the device's first call,
// matrix upload (stream-ordered on s) whenever p changes.  No device allocation.
static int static_scratch_base(uint32_t p, cudaStream_t s, unsigned char** out) {
  int dev = -1;
  CUDA_TRY(cudaGetDevice(&dev));
  if (dev < 0 || dev >= 64) return fail(RLXPP_EINVAL, "rlxpp_generate_doubles_static: device ordinal %d not in [0, 64)", dev);
  std::lock_guard<std::mutex> lock(g_static_mutex);
  StaticDev& d = g_static_dev[dev];
  if (!d.base) {
    unsigned char* ptr = nullptr;
    const cudaError_t e = cudaGetSymbolAddress((void**)&ptr, g_static_scratch);
    if (e != cudaSuccess || !ptr)
      return fail(RLXPP_ECUDA, "rlxpp_generate_doubles_static: cudaGetSymbolAddress on device %d: %s", dev, cudaGetErrorString(e));
    d.base = ptr;
  }
  if (d.p_loaded != p) {
    const std::vector<uint8_t>& img = static_bmatrix_image(p);
    d.p_loaded = 0;  // unknown contents if the copy fails half way
    CUDA_TRY(cudaMemcpyAsync(d.base + kStaticBmat, img.data(), tc::kBBytes, cudaMemcpyHostToDevice, s));
    d.p_loaded = p;
  }
  *out = d.base;
  return RLXPP_OK;
}

extern "C" {

const char* rlxpp_last_error(void) { return g_last_error.c_str(); }
const char* rlxpp_version(void) { return "rlxpp 0.1 (sm_100a)"; }
uint64_t rlxpp_launch_count(void) { return g_launches.load(); }
uint64_t rlxpp_n_streams(const rlxpp_t* h) { return h ? h->n : 0; }

int rlxpp_set_engine(int engine) {
  if (engine != RLXPP_ENGINE_UMMA && engine != RLXPP_ENGINE_IMAD)
    return fail(RLXPP_EINVAL, "rlxpp_set_engine: unknown engine %d", engine);
  g_engine.store(engine);
  return RLXPP_OK;
}
int rlxpp_get_engine(void) { return g_engine.load(); }
int rlxpp_set_chunks(int n_chunks) {
  if (n_chunks < 0 || n_chunks > 4096) return fail(RLXPP_EINVAL, "rlxpp_set_chunks: %d not in [0, 4096]", n_chunks);
  g_force_chunks.store(n_chunks);
  return RLXPP_OK;
}

int rlxpp_rare_counts(uint64_t* out_host, int reset) {
  static_assert(RLXPP_RARE_KINDS == kRareKinds, "rlxpp.h and arith.cuh disagree on the rare-path counters");
  int rc = check_device();
  if (rc) return rc;
  CUDA_TRY(cudaDeviceSynchronize());
  if (out_host) {
    unsigned long long tmp[kRareKinds];
    CUDA_TRY(cudaMemcpyFromSymbol(tmp, g_rare_counts, sizeof(tmp)));
    for (int k = 0; k < kRareKinds; k++) out_host[k] = tmp[k];
  }
  if (reset) {
    const unsigned long long zero[kRareKinds] = {};
    CUDA_TRY(cudaMemcpyToSymbol(g_rare_counts, zero, sizeof(zero)));
  }
  return RLXPP_OK;
}

int rlxpp_has_fixed_multiplier(uint32_t p) {
#define RLXPP_CASE(P) \
  if (p == P) return 1;
  RLXPP_FOR_EACH_FIXED_P(RLXPP_CASE)
#undef RLXPP_CASE
  return 0;
}

int rlxpp_multiplier(uint32_t p, uint64_t* out_host) {
  if (!out_host || p == 0) return fail(RLXPP_EINVAL, "rlxpp_multiplier: null output or p == 0");
  host::multiplier_ap(p).to_u64x9(out_host);
  return RLXPP_OK;
}
int rlxpp_umma_matrix(uint32_t p, uint8_t* out_host) {
  if (!out_host || p == 0) return fail(RLXPP_EINVAL, "rlxpp_umma_matrix: null output or p == 0");
  std::vector<uint8_t> img;
  build_bmatrix(p, img);
  for (int n = 0; n < 72; n++)
    for (int k = 0; k < 72; k++) out_host[n * 72 + k] = img[tc::b_offset(n, k)];
  return RLXPP_OK;
}
int rlxpp_seed_state(uint64_t seed, uint32_t p, uint64_t* out_host) {
  if (!out_host || p == 0) return fail(RLXPP_EINVAL, "rlxpp_seed_state: null output or p == 0");
  host::Big G = host::pow2k(host::multiplier_ap(p), 96);
  host::powmod(G, seed).to_u64x9(out_host);
  return RLXPP_OK;
}

int rlxpp_create(rlxpp_t** hout, uint64_t n_streams, uint64_t seed, uint32_t p, void* cuda_stream) {
  if (!hout) return fail(RLXPP_EINVAL, "rlxpp_create: null handle pointer");
  *hout = nullptr;
  if (n_streams == 0) return fail(RLXPP_EINVAL, "rlxpp_create: n_streams == 0");
  if (p == 0) return fail(RLXPP_EINVAL, "rlxpp_create: p == 0");
  if (n_streams > (1ull << 31) * kThreads) return fail(RLXPP_EINVAL, "rlxpp_create: too many streams");
  int rc = check_device();
  if (rc) return rc;
  rlxpp* h = new (std::nothrow) rlxpp();
  if (!h) return fail(RLXPP_ENOMEM, "rlxpp_create: host allocation failed");
  h->n = n_streams;
  h->p = p;
  h->stream = (cudaStream_t)cuda_stream;
  h->tables = cached_tables(p);
  h->fixed = fixed_level(p, h->tables.A);
  if (h->fixed < 0) {
    delete h;
    return fail(RLXPP_EINVAL, "rlxpp_create: include/rlxpp_rows.cuh is stale for p = %u (rebuild)", p);
  }
  rc = get_bmatrix(p, &h->bmat);
  if (rc) {
    delete h;
    return rc;
  }
  cudaError_t e = cudaMalloc(&h->st, sizeof(uint4) * 5 * n_streams);
  if (e == cudaSuccess) e = cudaMalloc(&h->sched, sizeof(uint32_t) * (1 + (n_streams + tc::kTile - 1) / tc::kTile));
  const size_t lane_words = (n_streams + tc::kTile - 1) / tc::kTile;
  if (e == cudaSuccess) e = cudaMalloc(&h->lane_sync, sizeof(uint32_t) * lane_words);
  if (e == cudaSuccess) e = cudaMemsetAsync(h->lane_sync, 0, sizeof(uint32_t) * lane_words, h->stream);
  if (e == cudaSuccess) e = cudaMalloc(&h->tabA, 64 * 18 * sizeof(uint32_t));
  if (e == cudaSuccess) e = cudaMalloc(&h->tabG, 64 * 18 * sizeof(uint32_t));
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(h->tabA, h->tables.tabA.data(), 64 * 18 * sizeof(uint32_t), cudaMemcpyHostToDevice, h->stream);
  if (e == cudaSuccess)
    e = cudaMemcpyAsync(h->tabG, h->tables.tabG.data(), 64 * 18 * sizeof(uint32_t), cudaMemcpyHostToDevice, h->stream);
  if (e != cudaSuccess) {
    int code = e == cudaErrorMemoryAllocation ? RLXPP_ENOMEM : RLXPP_ECUDA;
    fail(code, "rlxpp_create: %s", cudaGetErrorString(e));
    rlxpp_destroy(h);
    return code;
  }
  seed_kernel<<<grid_for(n_streams), kThreads, 0, h->stream>>>(h->st, n_streams, seed, h->tabG);
  g_launches++;
  e = cudaGetLastError();
  if (e != cudaSuccess) {
    fail(RLXPP_ECUDA, "rlxpp_create: seed kernel: %s", cudaGetErrorString(e));
    rlxpp_destroy(h);
    return RLXPP_ECUDA;
  }
  *hout = h;
  return RLXPP_OK;
}

int rlxpp_destroy(rlxpp_t* h) {
  if (!h) return RLXPP_OK;
  if (h->stream || h->st) cudaStreamSynchronize(h->stream);
  cudaFree(h->st);
  cudaFree(h->sched);
  cudaFree(h->lane_sync);
  cudaFree(h->scratch_q);
  cudaFree(h->tabA);
  cudaFree(h->tabG);
  for (int b = 0; b < 2; b++) {
    cudaFree(h->stage[b]);
    if (h->ev_kernel[b]) cudaEventDestroy(h->ev_kernel[b]);
    if (h->ev_copy[b]) cudaEventDestroy(h->ev_copy[b]);
  }
  if (h->copy_stream) cudaStreamDestroy(h->copy_stream);
  delete h;
  return RLXPP_OK;
}

int rlxpp_skip(rlxpp_t* h, uint64_t n) {
  if (!h) return fail(RLXPP_EINVAL, "rlxpp_skip: null handle");
  if (n == 0) return RLXPP_OK;
  skip_kernel<<<grid_for(h->n), kThreads, 0, h->stream>>>(h->st, h->n, n, nullptr, h->tabA);
  LAUNCH_CHECK();
  if (h->pos_uniform) {
    const uint64_t t = n - 1;
    const uint32_t total = (uint32_t)(t % 12) + h->uniform_pos;
    h->uniform_pos = total % 12 + 1;
  }
  h->aligned = h->pos_uniform && h->uniform_pos == 12;
  return RLXPP_OK;
}

int rlxpp_skip_each(rlxpp_t* h, const uint64_t* n_dev) {
  if (!h || !n_dev) return fail(RLXPP_EINVAL, "rlxpp_skip_each: null argument");
  skip_kernel<<<grid_for(h->n), kThreads, 0, h->stream>>>(h->st, h->n, 0, n_dev, h->tabA);
  LAUNCH_CHECK();
  h->pos_uniform = false;
  h->aligned = false;
  return RLXPP_OK;
}

int rlxpp_advance_states(uint64_t* states_dev, uint64_t n_states, uint32_t p, uint32_t reps, int layout,
                         void* cuda_stream) {
  if (p == 0) return fail(RLXPP_EINVAL, "rlxpp_advance_states: p == 0");
  if (layout != RLXPP_AOS && layout != RLXPP_SOA) return fail(RLXPP_EINVAL, "rlxpp_advance_states: unknown layout %d", layout);
  if (n_states == 0) return RLXPP_OK;
  if (!states_dev) return fail(RLXPP_EINVAL, "rlxpp_advance_states: null states");
  if ((uintptr_t)states_dev % 16) return fail(RLXPP_EINVAL, "rlxpp_advance_states: states must be 16-byte aligned");
  int rc = check_device();
  if (rc) return rc;
  const Tables& t = cached_tables(p);
  const int fixed = fixed_level(p, t.A);
  if (fixed < 0) return fail(RLXPP_EINVAL, "rlxpp_advance_states: include/rlxpp_rows.cuh is stale for p = %u", p);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (g_engine.load() == RLXPP_ENGINE_UMMA) {
    const uint4* bmat = nullptr;
    rc = get_bmatrix(p, &bmat);
    if (rc) return rc;
    {  // one CTA per SM with tc::kGroups groups (cfg2: 1,180 with pairs in four CTAs, 1,228 with 5 groups, 1,320 with 6)
      const size_t smem_bytes = ((sizeof(tc::GroupsSmem) + 127) & ~(size_t)127) +
                                (layout == RLXPP_AOS ? (size_t)tc::kGroups * kRawStageWords * sizeof(uint4) : 0);
      const unsigned ctas = tc_slots() / tc::kCtasPerSm;
      static std::atomic<uint64_t> done_aos{0}, done_soa{0};
      if (layout == RLXPP_AOS) {
        rc = allow_dynamic_smem(tc_advance_states_group_kernel<RLXPP_AOS>, done_aos, (int)smem_bytes);
        if (rc) return rc;
        tc_advance_states_group_kernel<RLXPP_AOS><<<ctas, tc::kGroups * tc::kTile, smem_bytes, s>>>(states_dev, n_states, reps, bmat);
      } else {
        rc = allow_dynamic_smem(tc_advance_states_group_kernel<RLXPP_SOA>, done_soa, (int)smem_bytes);
        if (rc) return rc;
        tc_advance_states_group_kernel<RLXPP_SOA><<<ctas, tc::kGroups * tc::kTile, smem_bytes, s>>>(states_dev, n_states, reps, bmat);
      }
      LAUNCH_CHECK();
      return RLXPP_OK;
    }
  }
#define RLXPP_CASE(P) \
  if (fixed == P) return launch_advance_mult<Fixed<P>>(states_dev, n_states, reps, layout, t.A, s);
  RLXPP_FOR_EACH_FIXED_P(RLXPP_CASE)
#undef RLXPP_CASE
  return launch_advance_mult<Generic>(states_dev, n_states, reps, layout, t.A, s);
}

static void after_generate(rlxpp_t* h, uint64_t n) {
  if (h->pos_uniform && n > 0) {
    const uint64_t t = n - 1;
    const uint32_t total = (uint32_t)(t % 12) + h->uniform_pos;
    h->uniform_pos = total % 12 + 1;
  }
  h->aligned = h->pos_uniform && h->uniform_pos == 12;
}

// STREAM_MAJOR, UMMA engine, ONE cursor common to all streams, but the call does not consist of whole blocks (the
// cursor is inside a block, or the draw count is not a multiple of 12): the rows are still aligned with each
// other, so the call is cut into  head (up to the block boundary) + whole blocks + tail  and the whole blocks take the
// aligned path (TMA stores, 780 G doubles/s) with the full rows' pitch; head and tail (< 12 draws each) take the
// general path.  The aligned path needs 16-byte aligned row pieces: an even pitch and an even head.  Returns -1 if
// the call does not qualify (the caller then launches it whole).
static int launch_stream_major_split(const rlxpp_t* h, const GenArgs& a,
                                     const std::function<int(const GenArgs&, bool)>& launch) {
  const uint64_t n = a.n_per;
  if (g_engine.load() != RLXPP_ENGINE_UMMA || !h->pos_uniform || n % 2 || h->uniform_pos % 2) return -1;
  const uint64_t to_boundary = 12 - h->uniform_pos;  // 0 at a block boundary
  uint64_t head = to_boundary < n ? to_boundary : n;
  // rows that are 256-byte multiples: a head of 32 j doubles keeps the aligned path's boxes on the 256-byte granules
  // the memory system wants (780 instead of 590 G doubles/s for the whole blocks); head = to_boundary + 12 k
  if (head && n % 32 == 0)
    for (uint64_t k = 0; k < 8; k++)
      if ((to_boundary + 12 * k) % 32 == 0 && to_boundary + 12 * k + kStageCycle <= n) {
        head = to_boundary + 12 * k;
        break;
      }
  const uint64_t mid = (n - head) / 12 * 12, tail = n - head - mid;
  if (mid < kStageCycle || (head == 0 && tail == 0)) return -1;
  GenArgs b = a;
  b.pitch = n;
  int rc = RLXPP_OK;
  if (head) {
    b.n_per = head;
    rc = launch(b, false);
  }
  if (rc == RLXPP_OK) {
    b.out = a.out + head;
    b.n_per = mid;
    rc = launch(b, true);
  }
  if (rc == RLXPP_OK && tail) {
    b.out = a.out + head + mid;
    b.n_per = tail;
    rc = launch(b, false);
  }
  return rc;
}

int rlxpp_generate_doubles(rlxpp_t* h, double* out_dev, uint64_t n_per_stream, int layout) {
  if (!h) return fail(RLXPP_EINVAL, "rlxpp_generate_doubles: null handle");
  if (layout != RLXPP_STREAM_MAJOR && layout != RLXPP_INTERLEAVED)
    return fail(RLXPP_EINVAL, "rlxpp_generate_doubles: unknown layout %d", layout);
  if (n_per_stream == 0) return RLXPP_OK;
  if (!out_dev) return fail(RLXPP_EINVAL, "rlxpp_generate_doubles: null output");
  if ((uintptr_t)out_dev % 16) return fail(RLXPP_EINVAL, "rlxpp_generate_doubles: output must be 16-byte aligned");
  GenArgs a;
  a.st = h->st; a.n_total = h->n; a.first = 0; a.count = h->n; a.out = out_dev; a.ld = h->n;
  a.n_per = n_per_stream; a.sum = nullptr; a.sumsq = nullptr; a.A = h->tables.A; a.bmat = h->bmat; a.sched = h->sched;
  a.lane_sync = h->lane_sync; a.p = h->p;  // whole-handle call: short ones may run time-parallel
  const bool aligned = h->aligned && n_per_stream % 12 == 0;
  int rc = -1;
  if (layout == RLXPP_STREAM_MAJOR && !aligned)
    rc = launch_stream_major_split(h, a, [&](const GenArgs& b, bool al) {
      return launch_generate(h->fixed, b, kStoreStreamMajor, al, h->stream);
    });
  if (rc == -1)
    rc = launch_generate(h->fixed, a, layout == RLXPP_STREAM_MAJOR ? kStoreStreamMajor : kStoreInterleaved, aligned,
                         h->stream);
  if (rc) return rc;
  after_generate(h, n_per_stream);
  return RLXPP_OK;
}

int rlxpp_generate_reduce(rlxpp_t* h, double* sum_dev, double* sumsq_dev, uint64_t n_per_stream) {
  if (!h || !sum_dev) return fail(RLXPP_EINVAL, "rlxpp_generate_reduce: null argument");
  if (!sumsq_dev && g_engine.load() == RLXPP_ENGINE_UMMA) {
    if (!h->scratch_q) CUDA_TRY(cudaMalloc(&h->scratch_q, sizeof(double) * h->n));
    sumsq_dev = h->scratch_q;
  }
  GenArgs a;
  a.st = h->st; a.n_total = h->n; a.first = 0; a.count = h->n; a.out = nullptr; a.ld = 0;
  a.n_per = n_per_stream; a.sum = sum_dev; a.sumsq = sumsq_dev; a.A = h->tables.A; a.bmat = h->bmat; a.sched = h->sched;
  const bool aligned = h->aligned && n_per_stream % 12 == 0;
  int rc = launch_generate(h->fixed, a, kReduce, aligned, h->stream);
  if (rc) return rc;
  after_generate(h, n_per_stream);
  return RLXPP_OK;
}

// 48-bit integers and 24-bit floats (S8 f-2): always the UMMA engine's kernels.
static int generate_other(rlxpp_t* h, void* out_dev, uint64_t n_draws, int layout, int kind, const char* who) {
  if (!h) return fail(RLXPP_EINVAL, "%s: null handle", who);
  if (layout != RLXPP_STREAM_MAJOR && layout != RLXPP_INTERLEAVED) return fail(RLXPP_EINVAL, "%s: unknown layout %d", who, layout);
  if (n_draws == 0) return RLXPP_OK;
  if (!out_dev) return fail(RLXPP_EINVAL, "%s: null output", who);
  if ((uintptr_t)out_dev % 16) return fail(RLXPP_EINVAL, "%s: output must be 16-byte aligned", who);
  GenArgs a;
  a.st = h->st; a.n_total = h->n; a.first = 0; a.count = h->n; a.out = (double*)out_dev; a.ld = h->n;
  a.n_per = n_draws; a.sum = nullptr; a.sumsq = nullptr; a.A = h->tables.A; a.bmat = h->bmat; a.sched = h->sched;
  a.lane_sync = h->lane_sync; a.p = h->p;
  const bool aligned = h->aligned && n_draws % 12 == 0;
  int rc = -1;
  if (layout == RLXPP_STREAM_MAJOR && !aligned)
    rc = launch_stream_major_split(h, a, [&](const GenArgs& b, bool al) {
      return kind == kU48      ? launch_tc_generate_mode<kStoreStreamMajor, kU48>(b, al, h->stream)
             : kind == kNormal ? launch_tc_generate_mode<kStoreStreamMajor, kNormal>(b, al, h->stream)
                               : launch_tc_generate_mode<kStoreStreamMajor, kF32>(b, al, h->stream);
    });
  if (rc != -1) {
    if (rc) return rc;
    after_generate(h, n_draws);
    return RLXPP_OK;
  }
  if (kind == kU48)
    rc = layout == RLXPP_STREAM_MAJOR ? launch_tc_generate_mode<kStoreStreamMajor, kU48>(a, aligned, h->stream)
                                      : launch_tc_generate_mode<kStoreInterleaved, kU48>(a, aligned, h->stream);
  else if (kind == kNormal)
    rc = layout == RLXPP_STREAM_MAJOR ? launch_tc_generate_mode<kStoreStreamMajor, kNormal>(a, aligned, h->stream)
                                      : launch_tc_generate_mode<kStoreInterleaved, kNormal>(a, aligned, h->stream);
  else
    rc = layout == RLXPP_STREAM_MAJOR ? launch_tc_generate_mode<kStoreStreamMajor, kF32>(a, aligned, h->stream)
                                      : launch_tc_generate_mode<kStoreInterleaved, kF32>(a, aligned, h->stream);
  if (rc) return rc;
  after_generate(h, n_draws);
  return RLXPP_OK;
}

int rlxpp_generate_u48(rlxpp_t* h, uint64_t* out_dev, uint64_t n_per_stream, int layout) {
  return generate_other(h, out_dev, n_per_stream, layout, kU48, "rlxpp_generate_u48");
}

int rlxpp_generate_floats(rlxpp_t* h, float* out_dev, uint64_t n_per_stream, int layout) {
  if (n_per_stream % 2) return fail(RLXPP_EINVAL, "rlxpp_generate_floats: n_per_stream must be even (two floats per 48-bit draw)");
  return generate_other(h, out_dev, n_per_stream / 2, layout, kF32, "rlxpp_generate_floats");
}

int rlxpp_generate_normal(rlxpp_t* h, double* out_dev, uint64_t n_per_stream, int layout) {
  return generate_other(h, out_dev, n_per_stream, layout, kNormal, "rlxpp_generate_normal");
}

// Generation for callers that must not allocate on the device (include/rlxpp.h has the contract and the reasons): the
// same import -> persistent tensor-core kernel -> export sequence a handle would run, with the handle's device buffers
// replaced by slices of g_static_scratch.  Nothing below may call cudaMalloc / cudaFree or a routine that does --
// which rules out get_bmatrix(), cached_tables()'s device copies and the time-parallel path (lane_sync stays null).
int rlxpp_generate_doubles_static(uint64_t* lcg_dev, uint64_t n_streams, uint32_t p, double* out_dev, uint64_t n_per_stream,
                                  int layout, void* cuda_stream) {
  const char* who = "rlxpp_generate_doubles_static";
  if (p == 0) return fail(RLXPP_EINVAL, "%s: p == 0", who);
  if (layout != RLXPP_STREAM_MAJOR && layout != RLXPP_INTERLEAVED) return fail(RLXPP_EINVAL, "%s: unknown layout %d", who, layout);
  if (n_streams > RLXPP_STATIC_MAX_STREAMS)
    return fail(RLXPP_EINVAL, "%s: %llu streams exceeds the static scratch, which holds at most %llu (use rlxpp_create for more)", who,
                (unsigned long long)n_streams, (unsigned long long)RLXPP_STATIC_MAX_STREAMS);
  if (n_per_stream % 12)
    return fail(RLXPP_EINVAL, "%s: n_per_stream = %llu is not a multiple of 12 (whole blocks only)", who, (unsigned long long)n_per_stream);
  if (n_streams == 0 || n_per_stream == 0) return RLXPP_OK;
  if (!lcg_dev || !out_dev) return fail(RLXPP_EINVAL, "%s: null states or output", who);
  if ((uintptr_t)lcg_dev % 8 || (uintptr_t)out_dev % 16) return fail(RLXPP_EINVAL, "%s: states must be 8-byte, output 16-byte aligned", who);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  unsigned char* base = nullptr;
  int rc = static_scratch_base(p, s, &base);  // first call on this device: address look-up; new p: matrix upload
  if (rc) return rc;
  uint4* planes = reinterpret_cast<uint4*>(base + kStaticState);
  // every word of the planes that the kernels read is rewritten here, so the last call's states never show through
  import_kernel<<<grid_for(n_streams), kThreads, 0, s>>>(planes, n_streams, lcg_dev, nullptr);
  LAUNCH_CHECK();
  GenArgs a;
  a.st = planes; a.n_total = n_streams; a.first = 0; a.count = n_streams; a.out = out_dev; a.ld = n_streams;
  a.n_per = n_per_stream; a.sum = nullptr; a.sumsq = nullptr; a.p = p;
  host::multiplier_ap(p).to_u32x18(a.A.v);
  a.bmat = reinterpret_cast<const uint4*>(base + kStaticBmat);
  a.sched = reinterpret_cast<uint32_t*>(base + kStaticSched);  // zeroed by the launch below (cudaMemsetAsync), every call
  rc = layout == RLXPP_STREAM_MAJOR ? launch_tc_generate_mode<kStoreStreamMajor>(a, true, s)
                                    : launch_tc_generate_mode<kStoreInterleaved>(a, true, s);
  if (rc) return rc;
  export_kernel<<<grid_for(n_streams), kThreads, 0, s>>>(planes, n_streams, nullptr, nullptr, nullptr, lcg_dev);
  LAUNCH_CHECK();
  return RLXPP_OK;
}

static int ensure_staging(rlxpp_t* h, size_t bytes_each) {
  if (!h->copy_stream) CUDA_TRY(cudaStreamCreateWithFlags(&h->copy_stream, cudaStreamNonBlocking));
  for (int b = 0; b < 2; b++) {
    if (!h->ev_kernel[b]) CUDA_TRY(cudaEventCreateWithFlags(&h->ev_kernel[b], cudaEventDisableTiming));
    if (!h->ev_copy[b]) CUDA_TRY(cudaEventCreateWithFlags(&h->ev_copy[b], cudaEventDisableTiming));
  }
  if (h->stage_bytes < bytes_each) {
    for (int b = 0; b < 2; b++) {
      cudaFree(h->stage[b]);
      h->stage[b] = nullptr;
    }
    h->stage_bytes = 0;
    for (int b = 0; b < 2; b++) CUDA_TRY(cudaMalloc(&h->stage[b], bytes_each));
    h->stage_bytes = bytes_each;
  }
  return RLXPP_OK;
}

int rlxpp_generate_doubles_host(rlxpp_t* h, double* out_host, uint64_t n_per_stream, int layout) {
  if (!h) return fail(RLXPP_EINVAL, "rlxpp_generate_doubles_host: null handle");
  if (layout != RLXPP_STREAM_MAJOR && layout != RLXPP_INTERLEAVED)
    return fail(RLXPP_EINVAL, "rlxpp_generate_doubles_host: unknown layout %d", layout);
  if (n_per_stream == 0) return RLXPP_OK;
  if (!out_host) return fail(RLXPP_EINVAL, "rlxpp_generate_doubles_host: null output");
  // chunks of streams, at most 512 MiB of doubles each, double-buffered: the kernel of chunk
  // c+1 overlaps the device->host copy of chunk c
  const uint64_t max_doubles = (512ull << 20) / 8;
  uint64_t chunk = max_doubles / n_per_stream;
  chunk = chunk / 1024 * 1024;
  if (chunk == 0) chunk = kThreads;
  if (chunk > h->n) chunk = h->n;
  int rc = ensure_staging(h, chunk * n_per_stream * sizeof(double));
  if (rc) return rc;
  const bool aligned = h->aligned && n_per_stream % 12 == 0;
  const int mode = layout == RLXPP_STREAM_MAJOR ? kStoreStreamMajor : kStoreInterleaved;
  // A failure inside the loop leaves earlier stream ranges advanced and copies possibly in flight: drain both streams
  // and stop trusting the cursor bookkeeping (the handle stays usable through the general path, or can be re-imported).
  auto run = [&]() -> int {
    int buf = 0;
    uint64_t done = 0;
    for (uint64_t first = 0; first < h->n; first += chunk, buf ^= 1, done++) {
      const uint64_t count = h->n - first < chunk ? h->n - first : chunk;
      if (done >= 2) CUDA_TRY(cudaStreamWaitEvent(h->stream, h->ev_copy[buf], 0));  // buffer free again
      GenArgs a;
      a.st = h->st; a.n_total = h->n; a.first = first; a.count = count; a.out = h->stage[buf]; a.ld = count;
      a.n_per = n_per_stream; a.sum = nullptr; a.sumsq = nullptr; a.A = h->tables.A; a.bmat = h->bmat; a.sched = h->sched;
      const int lrc = launch_generate(h->fixed, a, mode, aligned, h->stream);
      if (lrc) return lrc;
      CUDA_TRY(cudaEventRecord(h->ev_kernel[buf], h->stream));
      CUDA_TRY(cudaStreamWaitEvent(h->copy_stream, h->ev_kernel[buf], 0));
      if (layout == RLXPP_STREAM_MAJOR) {
        CUDA_TRY(cudaMemcpyAsync(out_host + first * n_per_stream, h->stage[buf], count * n_per_stream * sizeof(double),
                                 cudaMemcpyDeviceToHost, h->copy_stream));
      } else {
        CUDA_TRY(cudaMemcpy2DAsync(out_host + first, h->n * sizeof(double), h->stage[buf], count * sizeof(double),
                                   count * sizeof(double), n_per_stream, cudaMemcpyDeviceToHost, h->copy_stream));
      }
      CUDA_TRY(cudaEventRecord(h->ev_copy[buf], h->copy_stream));
    }
    CUDA_TRY(cudaStreamSynchronize(h->copy_stream));
    CUDA_TRY(cudaStreamSynchronize(h->stream));
    return RLXPP_OK;
  };
  rc = run();
  if (rc) {
    const std::string why = g_last_error;
    cudaStreamSynchronize(h->copy_stream);
    cudaStreamSynchronize(h->stream);
    h->pos_uniform = false;
    h->aligned = false;
    g_last_error = why;
    return rc;
  }
  after_generate(h, n_per_stream);
  return RLXPP_OK;
}

int rlxpp_generate_reduce_host(rlxpp_t* h, double* sum_host, double* sumsq_host, uint64_t n_per_stream) {
  if (!h || !sum_host) return fail(RLXPP_EINVAL, "rlxpp_generate_reduce_host: null argument");
  int rc = ensure_staging(h, 2 * h->n * sizeof(double));
  if (rc) return rc;
  double* s = h->stage[0];
  double* q = h->stage[0] + h->n;
  rc = rlxpp_generate_reduce(h, s, q, n_per_stream);
  if (rc) return rc;
  CUDA_TRY(cudaMemcpyAsync(sum_host, s, h->n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  if (sumsq_host) CUDA_TRY(cudaMemcpyAsync(sumsq_host, q, h->n * sizeof(double), cudaMemcpyDeviceToHost, h->stream));
  CUDA_TRY(cudaStreamSynchronize(h->stream));
  return RLXPP_OK;
}

int rlxpp_get_state(rlxpp_t* h, uint64_t* ranlux_dev, uint32_t* carry_dev, uint32_t* pos_dev, uint64_t* lcg_dev) {
  if (!h) return fail(RLXPP_EINVAL, "rlxpp_get_state: null handle");
  export_kernel<<<grid_for(h->n), kThreads, 0, h->stream>>>(h->st, h->n, ranlux_dev, carry_dev, pos_dev, lcg_dev);
  LAUNCH_CHECK();
  return RLXPP_OK;
}

int rlxpp_set_state(rlxpp_t* h, const uint64_t* lcg_dev, const uint32_t* pos_dev) {
  if (!h || !lcg_dev) return fail(RLXPP_EINVAL, "rlxpp_set_state: null argument");
  import_kernel<<<grid_for(h->n), kThreads, 0, h->stream>>>(h->st, h->n, lcg_dev, pos_dev);
  LAUNCH_CHECK();
  h->pos_uniform = pos_dev == nullptr;
  h->uniform_pos = 12;
  h->aligned = h->pos_uniform;
  return RLXPP_OK;
}

int rlxpp_set_state_ranlux(rlxpp_t* h, const uint64_t* ranlux_dev, const uint32_t* carry_dev, const uint32_t* pos_dev) {
  if (!h || !ranlux_dev) return fail(RLXPP_EINVAL, "rlxpp_set_state_ranlux: null argument");
  import_ranlux_kernel<<<grid_for(h->n), kThreads, 0, h->stream>>>(h->st, h->n, ranlux_dev, carry_dev, pos_dev);
  LAUNCH_CHECK();
  h->pos_uniform = pos_dev == nullptr;
  h->uniform_pos = 12;
  h->aligned = h->pos_uniform;
  return RLXPP_OK;
}

// ---- host engine (S8 f-3; the same sequence on the host, so that control can move
// between host and device mid-stream).  Plain host code on csrc/host_bigint.h; no device needed.
int rlxpp_host_generate(uint64_t* lcg_inout, uint32_t* pos_inout, uint32_t p, uint64_t skip, uint64_t n,
                        double* out_host) {
  if (!lcg_inout || !pos_inout || p == 0 || (n > 0 && !out_host))
    return fail(RLXPP_EINVAL, "rlxpp_host_generate: null argument or p == 0");
  if (*pos_inout > 12) return fail(RLXPP_EINVAL, "rlxpp_host_generate: cursor %u > 12", *pos_inout);
  const host::Big A = host::multiplier_ap(p);
  host::Big X = host::reduce(host::from_u64x9(lcg_inout));
  uint32_t pos = *pos_inout;
  if (skip > 0) {  // D8: k = floor((pos + skip - 1) / 12) without 64-bit overflow
    const uint64_t t = skip - 1;
    const uint32_t total = (uint32_t)(t % 12) + pos;
    const uint64_t k = t / 12 + total / 12;
    X = host::mulmod(host::powmod(A, k), X);
    pos = total % 12 + 1;
  }
  uint32_t v[18];
  bool have_block = false;
  for (uint64_t t = 0; t < n; t++) {
    if (pos == 12) {
      X = host::mulmod(A, X);
      pos = 0;
      have_block = false;
    }
    if (!have_block) {
      host::to_ranlux(X, v, nullptr);
      have_block = true;
    }
    const uint32_t w = (3 * pos) >> 1;
    const uint64_t k = (pos & 1) ? ((uint64_t)v[w] >> 16) | ((uint64_t)v[w + 1] << 16)
                                 : (uint64_t)v[w] | ((uint64_t)(v[w + 1] & 0xFFFFu) << 32);
    out_host[t] = (double)(int64_t)k * 0x1p-48;
    pos++;
  }
  X.to_u64x9(lcg_inout);
  *pos_inout = pos;
  return RLXPP_OK;
}

int rlxpp_device_view(rlxpp_t* h, struct rlxpp_view* out_host) {
  if (!h || !out_host) return fail(RLXPP_EINVAL, "rlxpp_device_view: null argument");
  out_host->st = h->st;
  out_host->n = h->n;
  out_host->A = h->tabA;  // entry 0 of the power table is A itself
  out_host->bmat = h->bmat;
  // kernels of the caller may move the cursors: the library no longer knows them
  h->pos_uniform = false;
  h->aligned = false;
  return RLXPP_OK;
}

static int launch_ragged(rlxpp_t* h, const uint32_t* counts_dev, double* out, uint64_t ld, double* sum, double* sumsq,
                         int coop, bool reduce) {
  rlxpp_view_t view;
  int rc = rlxpp_device_view(h, &view);
  if (rc) return rc;
  const unsigned grid = grid_for(h->n);
  if (coop == 3) {
    if (reduce) ragged_tile_kernel<true><<<grid, tc::kTile, 0, h->stream>>>(view, counts_dev, out, ld, sum, sumsq);
    else ragged_tile_kernel<false><<<grid, tc::kTile, 0, h->stream>>>(view, counts_dev, out, ld, sum, sumsq);
    LAUNCH_CHECK();
    return RLXPP_OK;
  }
  // the per-thread generator with the handle's luxury level baked in when it is one of the generated ones
#define RLXPP_RAGGED(COOP, RED, P) ragged_kernel<COOP, RED, P><<<grid, kThreads, 0, h->stream>>>(view, counts_dev, out, ld, sum, sumsq)
#define RLXPP_CASE(P)                                      \
  if (h->fixed == P && coop != 2) {                        \
    if (reduce) { if (coop) RLXPP_RAGGED(1, true, P); else RLXPP_RAGGED(0, true, P); }   \
    else { if (coop) RLXPP_RAGGED(1, false, P); else RLXPP_RAGGED(0, false, P); }        \
    LAUNCH_CHECK();                                        \
    return RLXPP_OK;                                       \
  }
  RLXPP_FOR_EACH_FIXED_P(RLXPP_CASE)
#undef RLXPP_CASE
  if (reduce) {
    if (coop == 2) RLXPP_RAGGED(2, true, 0);
    else if (coop) RLXPP_RAGGED(1, true, 0);
    else RLXPP_RAGGED(0, true, 0);
  } else {
    if (coop == 2) RLXPP_RAGGED(2, false, 0);
    else if (coop) RLXPP_RAGGED(1, false, 0);
    else RLXPP_RAGGED(0, false, 0);
  }
#undef RLXPP_RAGGED
  LAUNCH_CHECK();
  return RLXPP_OK;
}

int rlxpp_generate_ragged(rlxpp_t* h, const uint32_t* counts_dev, double* out_dev, uint64_t ld, int cooperative) {
  if (!h || !counts_dev || !out_dev) return fail(RLXPP_EINVAL, "rlxpp_generate_ragged: null argument");
  return launch_ragged(h, counts_dev, out_dev, ld, nullptr, nullptr, cooperative, false);
}

int rlxpp_generate_ragged_reduce(rlxpp_t* h, const uint32_t* counts_dev, double* sum_dev, double* sumsq_dev,
                                 int cooperative) {
  if (!h || !counts_dev || !sum_dev) return fail(RLXPP_EINVAL, "rlxpp_generate_ragged_reduce: null argument");
  return launch_ragged(h, counts_dev, nullptr, 0, sum_dev, sumsq_dev, cooperative, true);
}

// device buffer and event pair of a probe, released on every return path
struct ProbeScratch {
  void* buf = nullptr;
  cudaEvent_t e0 = nullptr, e1 = nullptr;
  ~ProbeScratch() {
    if (e0) cudaEventDestroy(e0);
    if (e1) cudaEventDestroy(e1);
    cudaFree(buf);
  }
};

int rlxpp_measure_imad_peak(int iters, double* imad_per_s, void* cuda_stream) {
  if (!imad_per_s || iters <= 0) return fail(RLXPP_EINVAL, "rlxpp_measure_imad_peak: bad argument");
  int rc = check_device();
  if (rc) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  ProbeScratch ps;
  CUDA_TRY(cudaMalloc(&ps.buf, 64));
  CUDA_TRY(cudaEventCreate(&ps.e0));
  CUDA_TRY(cudaEventCreate(&ps.e1));
  u64* out = static_cast<u64*>(ps.buf);
  const cudaEvent_t e0 = ps.e0, e1 = ps.e1;
  const unsigned blocks = (unsigned)sms * 8;  // 8 x 128 threads per SM = 8 warps per scheduler
  const u32 loop = 4096;
  double best = 0.0;
  for (int it = 0; it < iters + 2; it++) {
    CUDA_TRY(cudaEventRecord(e0, s));
    imad_peak_kernel<<<blocks, kThreads, 0, s>>>(out, loop, 12345u + it);
    g_launches++;
    CUDA_TRY(cudaEventRecord(e1, s));
    CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
    const double rate = (double)blocks * kThreads * loop * kImadPerIter / (ms * 1e-3);
    if (it >= 2 && rate > best) best = rate;
  }
  *imad_per_s = best;
  return RLXPP_OK;
}

int rlxpp_measure_hbm_write_peak(uint64_t bytes, int iters, double* bytes_per_s, void* cuda_stream) {
  if (!bytes_per_s || iters <= 0 || bytes < 16) return fail(RLXPP_EINVAL, "rlxpp_measure_hbm_write_peak: bad argument");
  int rc = check_device();
  if (rc) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  int dev = 0, sms = 0;
  CUDA_TRY(cudaGetDevice(&dev));
  CUDA_TRY(cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev));
  ProbeScratch ps;
  CUDA_TRY(cudaMalloc(&ps.buf, bytes));
  CUDA_TRY(cudaEventCreate(&ps.e0));
  CUDA_TRY(cudaEventCreate(&ps.e1));
  uint4* buf = static_cast<uint4*>(ps.buf);
  const cudaEvent_t e0 = ps.e0, e1 = ps.e1;
  double best = 0.0;
  for (int it = 0; it < iters + 2; it++) {
    CUDA_TRY(cudaEventRecord(e0, s));
    hbm_write_kernel<<<sms * 8, 256, 0, s>>>(buf, bytes / 16);
    g_launches++;
    CUDA_TRY(cudaEventRecord(e1, s));
    CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
    const double rate = (double)(bytes / 16 * 16) / (ms * 1e-3);
    if (it >= 2 && rate > best) best = rate;
  }
  // second pattern: rows of 2^18 doubles written strip by strip as the interleaved generate kernels write them
  // (hbm_write_rows_kernel); the result is the better of the two
  const u64 ld = 1ull << 18, n_rows = bytes / (ld * sizeof(double));
  if (n_rows >= 768) {
    for (int it = 0; it < iters + 2; it++) {
      CUDA_TRY(cudaEventRecord(e0, s));
      hbm_write_rows_kernel<<<tc_slots(), 128, 0, s>>>(reinterpret_cast<double*>(buf), ld, n_rows, 768u);
      g_launches++;
      CUDA_TRY(cudaEventRecord(e1, s));
      CUDA_TRY(cudaEventSynchronize(e1));
      float ms = 0.f;
      CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
      const double rate = (double)(n_rows * ld * sizeof(double)) / (ms * 1e-3);
      if (it >= 2 && rate > best) best = rate;
    }
  }
  *bytes_per_s = best;
  return RLXPP_OK;
}

int rlxpp_measure_hbm_write_pieces(uint64_t rows, uint64_t pitch_bytes, uint32_t piece_bytes, int iters, double* bytes_per_s,
                                   void* cuda_stream) {
  if (!bytes_per_s || iters <= 0 || rows < 32 || rows % 32 || piece_bytes < 16 || piece_bytes % 16 || pitch_bytes % 16 ||
      pitch_bytes < piece_bytes)
    return fail(RLXPP_EINVAL, "rlxpp_measure_hbm_write_pieces: rows must be a multiple of 32, piece and pitch multiples of 16 bytes");
  int rc = check_device();
  if (rc) return rc;
  cudaStream_t s = (cudaStream_t)cuda_stream;
  ProbeScratch ps;
  CUDA_TRY(cudaMalloc(&ps.buf, rows * pitch_bytes));
  CUDA_TRY(cudaEventCreate(&ps.e0));
  CUDA_TRY(cudaEventCreate(&ps.e1));
  uint4* buf = static_cast<uint4*>(ps.buf);
  const cudaEvent_t e0 = ps.e0, e1 = ps.e1;
  const uint64_t written = rows * (pitch_bytes / piece_bytes) * piece_bytes;
  double best = 0.0;
  for (int it = 0; it < iters + 2; it++) {
    CUDA_TRY(cudaEventRecord(e0, s));
    hbm_write_pieces_kernel<<<tc_slots(), 128, 0, s>>>(buf, rows, pitch_bytes / 16, piece_bytes / 16);
    g_launches++;
    CUDA_TRY(cudaEventRecord(e1, s));
    CUDA_TRY(cudaEventSynchronize(e1));
    float ms = 0.f;
    CUDA_TRY(cudaEventElapsedTime(&ms, e0, e1));
    const double rate = (double)written / (ms * 1e-3);
    if (it >= 2 && rate > best) best = rate;
  }
  *bytes_per_s = best;
  return RLXPP_OK;
}

}  // extern "C"
