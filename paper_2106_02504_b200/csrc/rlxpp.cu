// librlxpp: RANLUX++ stream generation for B200 (sm_100a).  C ABI in include/rlxpp.h.
//
// Hot path: one thread per stream, the 576-bit state as 18 x 32-bit
// limbs in registers.  Per LCG advance:
//   multiply9x9  -> 324 IMAD.WIDE.U32.X with the fixed multiplier as immediates, rows
//                   pre-reduced mod m (rows_generated.cuh)
//   mod_m        -> fold of the top 37 bits (fold_fast; exact fallback mod_m20)
//   to_ranlux    -> 8-limb add + carry decision (to_ranlux_fast; exact fallback)
//   12 doubles   -> byte permutes + one exact DADD each; coalesced 64-bit stores
//                   (interleaved layout), 128-bit stores (stream-major) or DADD/DFMA
//                   accumulation in registers (fused reduce).
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
#include "rows_generated.cuh"

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

constexpr int kThreads = 128;

// ----------------------------------------------------------------------------- state I/O
// Stream state in HBM: 5 planes of uint4, plane g holds limbs 4g .. 4g+3 of every stream
// (plane 4: limbs 16, 17, pos, 0).  Thread i reads st[g * n + i]: a warp moves 512 contiguous
// bytes per 128-bit access.  80 B per stream.
__device__ __forceinline__ void load_state(const uint4* __restrict__ st, u64 n, u64 i, u32 (&x)[18], u32& pos) {
#pragma unroll
  for (int g = 0; g < 4; g++) {
    const uint4 q = __ldcg(st + (u64)g * n + i);  // L2: another CTA may have written it (chunked items)
    x[4 * g] = q.x; x[4 * g + 1] = q.y; x[4 * g + 2] = q.z; x[4 * g + 3] = q.w;
  }
  const uint4 q = __ldcg(st + 4 * n + i);
  x[16] = q.x; x[17] = q.y; pos = q.z;
}
__device__ __forceinline__ void store_state(uint4* __restrict__ st, u64 n, u64 i, const u32 (&x)[18], u32 pos) {
#pragma unroll
  for (int g = 0; g < 4; g++) st[(u64)g * n + i] = make_uint4(x[4 * g], x[4 * g + 1], x[4 * g + 2], x[4 * g + 3]);
  st[4 * n + i] = make_uint4(x[16], x[17], pos, 0u);
}

struct Limbs18 { u32 v[18]; };

// ----------------------------------------------------------------------------- slow paths
// Exact recomputation from the unreduced 20-limb product; reached with probability ~2^-16
// per advance (carry out of the 8-limb addition in to_ranlux_fast), far less for the rest.
__device__ __noinline__ void exact_fold(const u32* zin, u32* xout) {
  u32 z[20], x[18];
#pragma unroll
  for (int j = 0; j < 20; j++) z[j] = zin[j];
  mod_m20(z, x);
#pragma unroll
  for (int j = 0; j < 18; j++) xout[j] = x[j];
}
__device__ __noinline__ void exact_fold_to_ranlux(const u32* zin, u32* xout, u32* vout, u32* cout) {
  u32 z[20], x[18], v[18], c;
#pragma unroll
  for (int j = 0; j < 20; j++) z[j] = zin[j];
  mod_m20(z, x);
  to_ranlux_exact(x, v, c);
#pragma unroll
  for (int j = 0; j < 18; j++) { xout[j] = x[j]; vout[j] = v[j]; }
  *cout = c;
}

__device__ __noinline__ void exact_to_ranlux(const u32* xin, u32* vout, u32* cout) {
  u32 x[18], v[18], c;
#pragma unroll
  for (int j = 0; j < 18; j++) x[j] = xin[j];
  to_ranlux_exact(x, v, c);
#pragma unroll
  for (int j = 0; j < 18; j++) vout[j] = v[j];
  *cout = c;
}

// ----------------------------------------------------------------------------- advance
// Multiplier policy: Fixed<P> bakes A = a^P into the instruction stream; Generic carries A
// as 18 runtime limbs (kernel parameter -> uniform registers) and runs the full-width
// multiply9x9 + mod_m.
template <int P>
struct Fixed {
  static constexpr bool kFixed = true;
  __device__ __forceinline__ Fixed(const Limbs18&) {}
  // x <- A x mod m (canonical)
  __device__ __forceinline__ void advance(u32 (&x)[18]) const {
    u64 E[9], O[9];
    u32 e9, o9, z[20], rare = 0;
    FixedMultiplier<P>::mul(x, E, e9, O, o9);
    merge_eo(E, e9, O, o9, z);
    fold_fast(z, x, rare);
    if (__builtin_expect(rare != 0, 0)) {
      count_rare(fold_rare_mask(z[0], z[1], z[7], z[8], z[9], z[17], z[18], z[19]));
      exact_fold(z, x);
    }
  }
  // x <- A x mod m and v, c <- to_ranlux(x)
  __device__ __forceinline__ void advance_block(u32 (&x)[18], u32 (&v)[18], u32& c) const {
    u64 E[9], O[9];
    u32 e9, o9, z[20], rare = 0;
    FixedMultiplier<P>::mul(x, E, e9, O, o9);
    merge_eo(E, e9, O, o9, z);
    fold_fast(z, x, rare);
    to_ranlux_fast(x, v, c, rare);
    if (__builtin_expect(rare != 0, 0)) {
      // to_ranlux_fast saw the right x only if the fold was exact: its conditions count only then
      const u32 fm = fold_rare_mask(z[0], z[1], z[7], z[8], z[9], z[17], z[18], z[19]);
      exact_fold_to_ranlux(z, x, v, &c);
      const u32 rm = ranlux_rare_mask(x, v, c);
      count_rare(fm ? fm | (rm & (1u << kRareRanluxThird)) : rm);
    }
  }
};
struct Generic {
  static constexpr bool kFixed = false;
  u32 a[18];
  __device__ __forceinline__ Generic(const Limbs18& A) {
#pragma unroll
    for (int j = 0; j < 18; j++) a[j] = A.v[j];
  }
  __device__ __forceinline__ void advance(u32 (&x)[18]) const {
    u32 r[18];
    mulmod_generic(x, a, r);
#pragma unroll
    for (int j = 0; j < 18; j++) x[j] = r[j];
  }
  __device__ __forceinline__ void advance_block(u32 (&x)[18], u32 (&v)[18], u32& c) const {
    advance(x);
    to_ranlux_exact(x, v, c);
  }
};

// ----------------------------------------------------------------------------- kernels
// Raw uint64[9] states (cfg2).  AoS: the block's 128 states are 9216 contiguous bytes: 128-bit
// coalesced accesses to/from shared memory, each thread picks up its 72 bytes there (stride 18
// words: 2-way bank conflict).  SoA: limb-major planes, coalesced directly.
constexpr int kRawStageWords = kThreads * 72 / 16;
// tid = thread within the 128 that own the tile, sync() = barrier over them (a CTA, or one group of a larger CTA)
struct CtaSync {
  __device__ __forceinline__ void operator()() const { __syncthreads(); }
};
template <int LAYOUT, class SYNC = CtaSync>
__device__ __forceinline__ void load_raw(const u64* __restrict__ states, u64 n, uint4* stage, u32 (&x)[18], u64 blk,
                                         u32 tid = threadIdx.x, SYNC sync = SYNC()) {
  const u64 base = blk * kThreads;
  const u64 i = base + tid;
#pragma unroll
  for (int j = 0; j < 18; j++) x[j] = 0;
  if (LAYOUT == RLXPP_AOS) {
    const u64 cnt = (n - base < (u64)kThreads ? n - base : (u64)kThreads) * 72 / 8;  // u64 words
    const uint4* src = reinterpret_cast<const uint4*>(states + base * 9);
    for (u32 q = tid; q < (cnt + 1) / 2; q += kThreads) {
      if (2 * (u64)q + 1 < cnt) stage[q] = src[q];
      else {  // odd tail: last 8 bytes
        const u64 lastw = states[base * 9 + 2 * (u64)q];
        stage[q] = make_uint4((u32)lastw, (u32)(lastw >> 32), 0u, 0u);
      }
    }
    sync();
    const u32* sw = reinterpret_cast<const u32*>(stage);
    if (i < n) {
#pragma unroll
      for (int j = 0; j < 18; j++) x[j] = sw[tid * 18 + j];
    }
  } else if (i < n) {
#pragma unroll
    for (int l = 0; l < 9; l++) {
      const u64 w = states[(u64)l * n + i];
      x[2 * l] = (u32)w;
      x[2 * l + 1] = (u32)(w >> 32);
    }
  }
}
template <int LAYOUT, class SYNC = CtaSync>
__device__ __forceinline__ void store_raw(u64* __restrict__ states, u64 n, uint4* stage, const u32 (&x)[18], u64 blk,
                                          u32 tid = threadIdx.x, SYNC sync = SYNC()) {
  const u64 base = blk * kThreads;
  const u64 i = base + tid;
  if (LAYOUT == RLXPP_AOS) {
    sync();
    u32* sw = reinterpret_cast<u32*>(stage);
    if (i < n) {
#pragma unroll
      for (int j = 0; j < 18; j++) sw[tid * 18 + j] = x[j];
    }
    sync();
    const u64 cnt = (n - base < (u64)kThreads ? n - base : (u64)kThreads) * 72 / 8;
    uint4* dst = reinterpret_cast<uint4*>(states + base * 9);
    for (u32 q = tid; q < (cnt + 1) / 2; q += kThreads) {
      if (2 * (u64)q + 1 < cnt) dst[q] = stage[q];
      else states[base * 9 + 2 * (u64)q] = (u64)stage[q].x | ((u64)stage[q].y << 32);
    }
  } else if (i < n) {
#pragma unroll
    for (int l = 0; l < 9; l++) states[(u64)l * n + i] = (u64)x[2 * l] | ((u64)x[2 * l + 1] << 32);
  }
}
__device__ __forceinline__ void canonicalise(u32 (&x)[18]) {
  u32 z[20], r[18];
#pragma unroll
  for (int j = 0; j < 20; j++) z[j] = j < 18 ? x[j] : 0u;
  exact_fold(z, r);
#pragma unroll
  for (int j = 0; j < 18; j++) x[j] = r[j];
}

// cfg2: x <- A^reps x mod m on raw uint64[9] states, in place (IMAD engine).
template <class Mult, int LAYOUT>
__global__ void __launch_bounds__(kThreads) advance_states_kernel(u64* __restrict__ states, u64 n, u32 reps,
                                                                  const __grid_constant__ Limbs18 A) {
  __shared__ uint4 stage[LAYOUT == RLXPP_AOS ? kRawStageWords : 1];
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  u32 x[18];
  load_raw<LAYOUT>(states, n, stage, x, blockIdx.x);
  if (i < n) {
    const Mult mult(A);
    if (reps == 0) canonicalise(x);
#pragma unroll 1
    for (u32 r = 0; r < reps; r++) mult.advance(x);
  }
  store_raw<LAYOUT>(states, n, stage, x, blockIdx.x);
}

struct GenArgs {
  uint4* st;     // state planes of the whole handle
  u64 n_total;   // streams in the handle (plane stride)
  u64 first;     // first stream of this launch
  u64 count;     // streams in this launch
  double* out;   // output of this launch (already offset to its first stream)
  u64 ld;        // INTERLEAVED: doubles between consecutive draws of one stream
  u64 n_per;     // draws per stream
  u64 pitch = 0; // STREAM_MAJOR: doubles between the rows of consecutive streams (0 = n_per: dense rows)
  u32 f32_boxes = 0;  // INTERLEAVED floats, aligned: tmap describes the float rows (F32RowStage)
  u32 ring = 0;       // STREAM_MAJOR, unaligned, even pitch: tmap describes the rows (RingStage)
  double* sum;   // REDUCE: per-stream outputs of this launch (already offset)
  double* sumsq;
  Limbs18 A;
  const uint4* bmat;  // UMMA engine: shared-memory image of the byte matrix B (umma_path.cuh)
  // UMMA engine, persistent scheduler: sched[0] = ticket counter, sched[1 + tile] = finished chunks
  u32* sched;
  u32 n_tiles, n_chunks;
  u64 chunk_len;      // draws per chunk (a multiple of 96 = 8 blocks when n_chunks > 1)
  u32 kexp = kExp16;  // see arith.cuh: a launch parameter on purpose
  // time-parallel path of short calls (tc_generate_lanes_kernel): images of the byte matrices of A^1 .. A^kMaxLanes,
  // lanes per tile, and one reader counter per tile
  const uint4* bmat_pow = nullptr;
  u32 lanes = 0;
  u32* lane_sync = nullptr;
  u32 p = 0;  // luxury level (selects the cached matrices)
  // UMMA engine, aligned stream-major stores: tensor map of out (StreamMajorStage)
  alignas(64) CUtensorMap tmap;
};

enum { kStoreStreamMajor = 0, kStoreInterleaved = 1, kReduce = 2 };
// What a 48-bit draw is written as (S8 f-2): the double k 2^-48; the integer k as uint64; or its two
// 24-bit RANLUX numbers as floats x 2^-24 (low number first).  Every form is 8 bytes per draw, carried
// through the emission code as the bit pattern of a double.
// kNormal (reading N-1 in DESIGN.md): a standard normal deviate per draw position, Box-Muller on the draw pair
// (2i, 2i + 1) of the block -- fp64 log / sqrt / sincospi, the only output form that is not exact (<= 6 ulp).
enum { kF64 = 0, kU48 = 1, kF32 = 2, kNormal = 3 };

template <int OUT, int J>
__device__ __forceinline__ double draw_value(const u32 (&v)[18], u32 kexp) {
  if (OUT == kF64) return draw_double<J>(v, kexp);
  u32 lo, hi;  // bits 0..31 and 32..47 of the draw
  if (J % 2 == 0) {
    lo = v[3 * J / 2];
    hi = v[3 * J / 2 + 1] & 0xFFFFu;
  } else {
    lo = __byte_perm(v[(3 * J - 1) / 2], v[(3 * J + 1) / 2], 0x5432);
    hi = v[(3 * J + 1) / 2] >> 16;
  }
  if (OUT == kU48) return __hiloint2double((int)hi, (int)lo);
  const float f0 = __uint2float_rn(lo & 0xFFFFFFu) * 0x1p-24f;               // RANLUX number 2J (exact)
  const float f1 = __uint2float_rn(__byte_perm(lo, hi, 0x6543)) * 0x1p-24f;  // number 2J + 1 = bits 24..47
  return __hiloint2double(__float_as_int(f1), __float_as_int(f0));
}

// The transcendental part of reading N-1, written for the arguments that occur (CUDA's log / sincospi cost 175
// instructions per pair with their range checks and general reductions; these cost about half).  Polynomial
// coefficients: normal_coeffs.cuh (csrc/gen_normal_coeffs.py).  Error against the exact values: ln <= 1 ulp,
// sin / cos <= 1 ulp, so a deviate is within ~3 ulp (tests: 6 ulp against the long-double oracle).
namespace nrm {
// ln(x) for x = 1 - k 2^-48 in [2^-48, 1]: x = 2^e m with m in [sqrt(1/2), sqrt(2)), f = m - 1 (exact),
// s = f / (2 + f), ln m = 2 s + s z P(z) = f - s (f - z P(z)) with z = s^2: f is exact and dominates, so the rounding
// of s only enters at second order.  e ln2 is added as hi (32 bits, e hi exact) + lo.  N arguments at once, step by
// step, so that every constant is set up once per N uses (normal_coeffs.cuh).
template <int N>
__device__ __forceinline__ void log_unit(const double (&x)[N], double (&r)[N]) {
  double f[N], s[N], z[N], p[N], ed[N];
#pragma unroll
  for (int i = 0; i < N; i++) {
    int hx = __double2hiint(x[i]) + (0x3ff00000 - 0x3fe6a09e);  // 0x3fe6a09e: high word of sqrt(1/2)
    ed[i] = (double)((hx >> 20) - 0x3ff);
    hx = (hx & 0x000fffff) + 0x3fe6a09e;
    f[i] = __hiloint2double(hx, __double2loint(x[i])) - 1.0;
  }
#pragma unroll
  for (int i = 0; i < N; i++) {
    const double d = 2.0 + f[i];
    double y;
    asm("rcp.approx.ftz.f64 %0, %1;" : "=d"(y) : "d"(d));  // ~20 bits; two Newton steps, then one correction of s
    double t = fma(-d, y, 1.0);
    y = fma(y, t, y);
    t = fma(-d, y, 1.0);
    y = fma(y, t, y);
    double q = f[i] * y;
    q = fma(fma(-d, q, f[i]), y, q);
    s[i] = q;
    z[i] = q * q;
  }
  poly_atanh<N>(z, p);
#pragma unroll
  for (int i = 0; i < N; i++) r[i] = fma(ed[i], kLn2Hi, f[i]) - fma(-ed[i], kLn2Lo, s[i] * fma(-z[i], p[i], f[i]));
}
// sin and cos of u turns, u = k 2^-48 in [0, 1): x = 2 u (angle pi x), n = round(2 x) in 0 .. 4, r = x - n / 2 exact in
// [-1/4, 1/4]; the quarter turns are exact sign changes and swaps, so the exact zeros of sin and cos stay exact.
template <int N>
__device__ __forceinline__ void sincos_turn(const double (&u)[N], double (&sn)[N], double (&cs)[N]) {
  double r[N], z[N], ps[N], pc[N];
  u32 n[N];
#pragma unroll
  for (int i = 0; i < N; i++) {
    const double x = u[i] + u[i];
    const double j = fma(x, 2.0, 0x1.8p52);  // the integer nearest to 2 x sits in the low mantissa bits
    n[i] = (u32)__double2loint(j);
    r[i] = fma(j - 0x1.8p52, -0.5, x);
    z[i] = r[i] * r[i];
  }
  poly_sinpi<N>(z, ps);
  poly_cospi<N>(z, pc);
#pragma unroll
  for (int i = 0; i < N; i++) {
    const double s = fma(z[i] * r[i], ps[i], r[i] * kPi);
    const double c = fma(z[i], pc[i], 1.0);
    const bool odd = n[i] & 1u;
    const double so = odd ? c : s, co = odd ? s : c;  // sin(n pi/2 + t), cos(n pi/2 + t) up to sign
    sn[i] = __hiloint2double(__double2hiint(so) ^ (int)((n[i] & 2u) << 30), __double2loint(so));
    cs[i] = __hiloint2double(__double2hiint(co) ^ (int)(((n[i] + 1u) & 2u) << 30), __double2loint(co));
  }
}
}  // namespace nrm

// draws J (even) and J + 1 of the block in output form OUT
template <int OUT, int J>
__device__ __forceinline__ void draw_pair(const u32 (&v)[18], u32 kexp, double& a, double& b) {
  static_assert(J % 2 == 0, "pairs start at even draws");
  if constexpr (OUT == kNormal) {
    const double x[1] = {1.0 - draw_double<J>(v, kexp)}, u1[1] = {draw_double<J + 1>(v, kexp)};  // 1 - u0: exact, in (0, 1]
    double l[1], sn[1], cs[1];
    nrm::log_unit<1>(x, l);
    nrm::sincos_turn<1>(u1, sn, cs);
    const double r = sqrt(-2.0 * l[0]);
    a = r * cs[0];
    b = r * sn[0];
  } else {
    a = draw_value<OUT, J>(v, kexp);
    b = draw_value<OUT, J + 1>(v, kexp);
  }
}

// kNormal: the 12 deviates of a block, its six pairs evaluated side by side
template <int... I>
__device__ __forceinline__ void draws_of_block(const u32 (&v)[18], u32 kexp, double (&d)[12]) {
  ((d[I] = draw_double<I>(v, kexp)), ...);
}
__device__ __forceinline__ void normal_block(const u32 (&v)[18], u32 kexp, double (&zn)[12]) {
  double d[12];
  draws_of_block<0, 1, 2, 3, 4, 5, 6, 7, 8, 9, 10, 11>(v, kexp, d);
  double x[6], u1[6], l[6], sn[6], cs[6];
#pragma unroll
  for (int i = 0; i < 6; i++) {
    x[i] = 1.0 - d[2 * i];  // exact, in (0, 1]
    u1[i] = d[2 * i + 1];
  }
  nrm::log_unit<6>(x, l);
  nrm::sincos_turn<6>(u1, sn, cs);
#pragma unroll
  for (int i = 0; i < 6; i++) {
    const double r = sqrt(-2.0 * l[i]);
    zn[2 * i] = r * cs[i];
    zn[2 * i + 1] = r * sn[i];
  }
}

template <int MODE, int OUT = kF64>
struct Sink {
  double* p;      // STREAM_MAJOR: &out[i_local * n_per]; INTERLEAVED: &out[i_local] (kF32: float index i_local)
  u64 ld;
  double S, Q;
  u32 kexp;       // exp16()
  __device__ __forceinline__ void emit(u64 t, double d) {
    if (MODE == kStoreStreamMajor) p[t] = d;
    else if (MODE == kStoreInterleaved && OUT == kF32) {  // floats 2t and 2t + 1 of the stream: rows of 4-byte elements
      float* pf = reinterpret_cast<float*>(p);
      __stcs(pf + (2 * t) * ld, __int_as_float(__double2loint(d)));
      __stcs(pf + (2 * t + 1) * ld, __int_as_float(__double2hiint(d)));
    } else if (MODE == kStoreInterleaved) __stcs(p + t * ld, d);
    else { S = S + d; Q = __fma_rn(d, d, Q); }
  }
};

template <int J, int MODE, int OUT = kF64>
struct EmitBlock {
  // all 12 draws of block v go to output indices t0 .. t0 + 11 (VEC: t0 is even and p is 16-byte aligned)
  template <bool VEC = true>
  static __device__ __forceinline__ void all(Sink<MODE, OUT>& s, const u32 (&v)[18], u64 t0) {
    if constexpr (OUT == kNormal && J == 0) {
      double z[12];
      normal_block(v, s.kexp, z);
#pragma unroll
      for (int j = 0; j < 12; j += 2) {
        if (MODE == kStoreStreamMajor && VEC) __stcs(reinterpret_cast<double2*>(s.p + t0 + j), make_double2(z[j], z[j + 1]));
        else { s.emit(t0 + j, z[j]); s.emit(t0 + j + 1, z[j + 1]); }
      }
      return;
    }
    if constexpr (MODE == kStoreStreamMajor && VEC) {
      if constexpr (J % 2 == 0) {  // two draws per 128-bit store (p + t0 is 16-byte aligned: n_per % 12 == 0)
        double2 d2;
        draw_pair<OUT, J>(v, s.kexp, d2.x, d2.y);
        __stcs(reinterpret_cast<double2*>(s.p + t0 + J), d2);
      }
    } else if constexpr (OUT == kNormal) {
      if constexpr (J % 2 == 0) {
        double a, b;
        draw_pair<OUT, J>(v, s.kexp, a, b);
        s.emit(t0 + J, a);
        s.emit(t0 + J + 1, b);
      }
    } else {
      s.emit(t0 + J, draw_value<OUT, J>(v, s.kexp));
    }
    EmitBlock<J + 1, MODE, OUT>::template all<VEC>(s, v, t0);
  }
  // draw J of the block at absolute draw position q0 + J is output index q0 + J - pos if in [0, n)
  static __device__ __forceinline__ void masked(Sink<MODE, OUT>& s, const u32 (&v)[18], u64 q0, u32 pos, u64 n) {
    const u64 t = q0 + J - pos;  // wraps when q0 + J < pos: then t >= n
    if constexpr (OUT == kNormal) {
      if constexpr (J % 2 == 0) {  // the deviate of a draw position depends on both draws of its pair
        if (t < n || t + 1 < n) {
          double a, b;
          draw_pair<OUT, J>(v, s.kexp, a, b);
          if (t < n) s.emit(t, a);
          if (t + 1 < n) s.emit(t + 1, b);
        }
      }
    } else {
      const bool valid = t < n;
      const double d = draw_value<OUT, J>(v, s.kexp);
      if (MODE == kReduce) s.emit(t, valid ? d : 0.0);  // + 0.0 and fma(0, 0, Q) are exact no-ops
      else if (valid) s.emit(t, d);
    }
    EmitBlock<J + 1, MODE, OUT>::masked(s, v, q0, pos, n);
  }
};
template <int MODE, int OUT>
struct EmitBlock<12, MODE, OUT> {
  template <bool VEC = true>
  static __device__ __forceinline__ void all(Sink<MODE, OUT>&, const u32 (&)[18], u64) {}
  static __device__ __forceinline__ void masked(Sink<MODE, OUT>&, const u32 (&)[18], u64, u32, u64) {}
};

// ALIGNED: every cursor is 12 and n_per % 12 == 0: n_per / 12 advances, no masks.
// General: draw t of a stream sits at absolute position q = pos + t counted from the start of
// its current block; block s = q / 12 needs s advances (D8).  All threads run the same trip
// count; a thread skips an advance only when it lies beyond its own last block.
template <class Mult, int MODE, bool ALIGNED>
__global__ void __launch_bounds__(kThreads) generate_kernel(const __grid_constant__ GenArgs a) {
  const u64 il = (u64)blockIdx.x * kThreads + threadIdx.x;
  if (il >= a.count) return;
  const u64 i = a.first + il;
  u32 x[18], v[18], pos, c;
  load_state(a.st, a.n_total, i, x, pos);
  const Mult mult(a.A);
  Sink<MODE> sink;
  sink.ld = a.ld;
  sink.S = 0.0;
  sink.Q = 0.0;
  sink.kexp = MODE == kReduce ? a.kexp : kExp16;
  sink.p = MODE == kStoreStreamMajor ? a.out + il * (a.pitch ? a.pitch : a.n_per) : (MODE == kStoreInterleaved ? a.out + il : nullptr);
  const u64 n = a.n_per;
  if (ALIGNED) {
    const u64 nblk = n / 12;
#pragma unroll 1
    for (u64 b = 0; b < nblk; b++) {
      mult.advance_block(x, v, c);
      EmitBlock<0, MODE>::all(sink, v, b * 12);
    }
  } else if (n > 0) {
    const u64 last = ((u64)pos + (n - 1)) / 12;  // own last block (n >= 1)
    // pos + n - 1 can exceed 64 bits only for n near 2^64, which no output buffer can hold
    const u64 smax = (12 + (n - 1)) / 12;                                                // last block of any thread
    if (pos < 12) {  // block 0 = the current block
      to_ranlux_exact(x, v, c);
      EmitBlock<0, MODE>::masked(sink, v, 0, pos, n);
    }
#pragma unroll 1
    for (u64 s = 1; s <= smax; s++) {
      if (s <= last) {
        mult.advance_block(x, v, c);
        EmitBlock<0, MODE>::masked(sink, v, s * 12, pos, n);
      }
    }
    pos = (u32)((u64)pos + n - 12 * last);
  }
  store_state(a.st, a.n_total, i, x, pos);
  if (MODE == kReduce) {
    a.sum[il] = sink.S;
    if (a.sumsq) a.sumsq[il] = sink.Q;
  }
}

}  // namespace rlx
#include "umma_path.cuh"
namespace rlx {

// Stream-major stores through shared memory and the TMA (S8 a-7a; north_star: "shared-memory
// staging, or TMA bulk stores, so HBM writes are fully coalesced").  A thread's block is 96
// contiguous bytes of ITS stream's row, so direct stores make every warp instruction touch 32 rows
// (measured 287 G doubles/s, 36 % of the HBM peak).  What the memory system wants is measured in
// profiles/ab_r01_stream_major.md: row pieces that are 256 bytes long, 256-byte aligned and written by ONE
// operation reach the interleaved layout's bandwidth; 96-, 128- or 192-byte pieces (or two 128-byte
// halves from two operations) stop at 4.7 - 5.8 TB/s however they are fenced or buffered.
// So each warp owns ONE box of [32 streams][32 doubles] in shared memory.  The 96 bytes of an advance
// go where they fall in a cycle of 8 advances = 768 bytes = 3 boxes; an advance that straddles a box
// end (phases 2 and 5) fills the box, one lane hands it to the TMA (cp.async.bulk.tensor.3d, SASS
// UTMASTG) and the thread keeps the limbs of its remaining 4 or 8 draws in registers until the next
// advance, which first waits for the copy to have read the box (cp.async.bulk.wait_group.read: one
// whole advance of slack) and then stores them at the start of the box.
// Tensor map: out[count][n_per] viewed as [count][n_per / 16][16 doubles] with a {16, 2, 32} box and
// SWIZZLE_128B, so that one operation writes 32 x 256 contiguous bytes while the 16-byte chunks of a
// row are XOR-swizzled in shared memory (2-way instead of 8-way bank conflicts on the st.shared.v2.f64;
// a 2-D box with a 256-byte inner extent cannot be swizzled).  Rows past the end of the launch are
// clipped by the tensor map.  Only whole cycles are staged: the last (n_per / 12) % 8 blocks of a row
// are stored directly.
constexpr u32 kStageWarpBytes = 32u * 256u;                    // one box
constexpr u32 kStageCtaBytes = 4u * kStageWarpBytes + 1024u;   // dynamic shared memory of the staged kernels (+ alignment)
constexpr u64 kStageCycle = 96;                                // draws per cycle of 8 advances
struct StreamMajorStage {
  u32 box;        // shared address of this warp's box (1,024-byte aligned: the swizzle works on address bits)
  u32 rowbase;    // ... of this lane's 256-byte row
  u32 rs;         // swizzle term of the row: ((2 lane) & 6) << 4
  u32 q;          // phase: advance within the cycle
  int col16;      // tensor coordinate (in units of 16 doubles) of the box being filled
  int c1;         // tensor row of the warp's first stream
  const void* tmap;
  u32 kexp;       // exp16()
  u32 cv[18];     // limbs of the block whose last draws wait for the next box (only [6, 18) are ever live)
  double cz[8];   // kNormal: the waiting deviates themselves
  __device__ __forceinline__ void init(uint8_t* stage, const void* tensor_map, u64 tile_first, u32 kexp_, u64 t0) {
    const u32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    box = ((umma::smem_u32(stage) + 1023u) & ~1023u) + warp * kStageWarpBytes;
    rowbase = box + lane * 256u;
    rs = ((2u * lane) & 6u) << 4;
    q = 0;
    col16 = (int)(t0 / 16);
    c1 = (int)(tile_first + warp * 32u);
    tmap = tensor_map;
    kexp = kexp_;
  }
  // draws J, J + 1 of v to byte offset O of the lane's row.  The box is 64 lines of 128 bytes (line 2 r + h
  // = half h of row r); SWIZZLE_128B stores 16-byte chunk c of a line at c ^ (line & 7) = c ^ h ^ ((2 r) & 6).
  template <int OUT, int J, int O>
  __device__ __forceinline__ void put2(const u32 (&v)[18]) {
    constexpr u32 h = (u32)O >> 7, K = ((((u32)O >> 4) & 7u) ^ h) << 4;
    double a, b;
    draw_pair<OUT, J>(v, kexp, a, b);
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"((rowbase | (rs ^ K)) + h * 128u), "d"(a), "d"(b) : "memory");
  }
  // doubles z[J0 .. J1) to byte offset O of the lane's row
  template <int J0, int J1, int O>
  __device__ __forceinline__ void putd(const double* z) {
    if constexpr (J0 < J1) {
      constexpr u32 h = (u32)O >> 7, K = ((((u32)O >> 4) & 7u) ^ h) << 4;
      asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"((rowbase | (rs ^ K)) + h * 128u), "d"(z[J0]), "d"(z[J0 + 1])
                   : "memory");
      putd<J0 + 2, J1, O + 16>(z);
    }
  }
  template <int OUT, int J0, int J1, int O>
  struct Put {
    static __device__ __forceinline__ void all(StreamMajorStage& st, const u32 (&v)[18]) {
      st.put2<OUT, J0, O>(v);
      Put<OUT, J0 + 2, J1, O + 16>::all(st, v);
    }
  };
  __device__ __forceinline__ void wait_box() {  // whole warp: the last copy has read the box
    if ((threadIdx.x & 31u) == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncwarp();
  }
  __device__ __forceinline__ void send() {  // whole warp: the box is full
    umma::fence_proxy_async_smem();
    __syncwarp();
    if ((threadIdx.x & 31u) == 0) {
      asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(tmap), "r"(0),
                   "r"(col16), "r"(c1), "r"(box)
                   : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    col16 += 2;
  }
  template <int FROM>
  __device__ __forceinline__ void keep(const u32 (&v)[18]) {
#pragma unroll
    for (int j = FROM; j < 18; j++) cv[j] = v[j];
  }
  // whole-warp call: the next block of the item (blocks come in whole cycles of 8)
  template <int OUT>
  __device__ __forceinline__ void emit(const u32 (&v)[18]) {
    if constexpr (OUT == kNormal) {
      // the transform is too long to sit in all eight phases (instruction cache): evaluate the block first, then
      // place it; straddling deviates are carried as doubles (cz[j - 4] = z[j])
      double z[12];
      normal_block(v, kexp, z);
      switch (q) {
        case 0: wait_box(); putd<0, 12, 0>(z); break;
        case 1: putd<0, 12, 96>(z); break;
        case 2: putd<0, 8, 192>(z); send(); cz[4] = z[8]; cz[5] = z[9]; cz[6] = z[10]; cz[7] = z[11]; break;
        case 3: wait_box(); putd<4, 8, 0>(cz); putd<0, 12, 32>(z); break;
        case 4: putd<0, 12, 128>(z); break;
        case 5:
          putd<0, 4, 224>(z);
          send();
#pragma unroll
          for (int j = 0; j < 8; j++) cz[j] = z[j + 4];
          break;
        case 6: wait_box(); putd<0, 8, 0>(cz); putd<0, 12, 64>(z); break;
        default: putd<0, 12, 160>(z); send(); break;
      }
      q = (q + 1u) & 7u;
      return;
    }
    switch (q) {
      case 0: wait_box(); Put<OUT, 0, 12, 0>::all(*this, v); break;
      case 1: Put<OUT, 0, 12, 96>::all(*this, v); break;
      case 2: Put<OUT, 0, 8, 192>::all(*this, v); send(); keep<12>(v); break;
      case 3: wait_box(); Put<OUT, 8, 12, 0>::all(*this, cv); Put<OUT, 0, 12, 32>::all(*this, v); break;
      case 4: Put<OUT, 0, 12, 128>::all(*this, v); break;
      case 5: Put<OUT, 0, 4, 224>::all(*this, v); send(); keep<6>(v); break;
      case 6: wait_box(); Put<OUT, 4, 12, 0>::all(*this, cv); Put<OUT, 0, 12, 64>::all(*this, v); break;
      default: Put<OUT, 0, 12, 160>::all(*this, v); send(); break;
    }
    q = (q + 1u) & 7u;
  }
  // before the box is reused by another item or the CTA exits
  __device__ __forceinline__ void drain() {
    if ((threadIdx.x & 31u) == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    __syncwarp();
  }
};
template <int OUT, int J1, int O>
struct StreamMajorStage::Put<OUT, J1, J1, O> {
  static __device__ __forceinline__ void all(StreamMajorStage&, const u32 (&)[18]) {}
};

// Stream-major stores when the cursors are not all at a block boundary (per-stream skips, draw counts that are
// not multiples of 12): the rows are shifted against each other by up to 11 doubles, so no TMA box fits, and a thread
// storing its own 8-byte pieces makes every warp instruction touch 32 rows (measured 100 G doubles/s at the cfg3
// shape).  Instead the warp parks the block as [32 streams][12 + 1 doubles] in shared memory and copies it out
// element by element in row order: 32 consecutive lanes write 32 consecutive doubles of 2.67 rows, each lane with the
// cursor of its element's stream (one shuffle) for the output index and the range mask.
constexpr u32 kRowStagePitch = 13;                                // doubles; odd: conflict-free 8-byte accesses
constexpr u32 kRowStageWarpBytes = 32u * kRowStagePitch * 8u;     // 3,328
struct UnalignedRowStage {
  u32 buf;        // shared address of this warp's buffer
  double* row0;   // &out[first stream of the warp][first draw of the item]
  u64 pitch;      // doubles between rows
  u32 rows;       // streams of the warp that exist (0 .. 32)
  u32 kexp;
  __device__ __forceinline__ void init(uint8_t* stage, double* out_item, u64 warp_first, u64 count, u64 n_per, u32 kexp_) {
    buf = umma::smem_u32(stage) + (threadIdx.x >> 5) * kRowStageWarpBytes;
    row0 = out_item + warp_first * n_per;
    pitch = n_per;
    rows = warp_first >= count ? 0u : (count - warp_first < 32 ? (u32)(count - warp_first) : 32u);
    kexp = kexp_;
  }
  template <int OUT, int J>
  __device__ __forceinline__ void park(u32 dst, const u32 (&v)[18]) {
    if constexpr (J < 12) {
      double a, b;
      draw_pair<OUT, J>(v, kexp, a, b);
      asm volatile("st.shared.f64 [%0], %1;" ::"r"(dst + J * 8), "d"(a) : "memory");
      asm volatile("st.shared.f64 [%0], %1;" ::"r"(dst + J * 8 + 8), "d"(b) : "memory");
      park<OUT, J + 2>(dst, v);
    }
  }
  // whole-warp call: block v holds the draws at positions q0 .. q0 + 11 counted from the start of each stream's
  // current block; position q of a stream with cursor pos is output index q - pos of the item if that is in [0, n)
  template <int OUT>
  __device__ __forceinline__ void emit(const u32 (&v)[18], u64 q0, u32 pos, u64 n) {
    const u32 lane = threadIdx.x & 31u;
    __syncwarp();  // the copy loop of the previous block has read the buffer
    park<OUT, 0>(buf + lane * (kRowStagePitch * 8u), v);
    __syncwarp();
#pragma unroll 4  // fully unrolled: spills, no faster; hoisting the shuffles out of the loop changes nothing either
    for (u32 k = 0; k < 12; k++) {
      const u32 e = 32u * k + lane;         // element of the [32][12] block in row order
      const u32 r = (e * 2731u) >> 15;      // e / 12 for e < 384
      const u32 c = e - 12u * r;
      const u32 pr = __shfl_sync(0xFFFFFFFFu, pos, r);
      const u64 t = q0 + c - pr;            // wraps when the draw lies before the stream's cursor: then t >= n
      if (r < rows && t < n) {
        double d;
        asm volatile("ld.shared.f64 %0, [%1];" : "=d"(d) : "r"(buf + (e + r) * 8u) : "memory");
        __stcs(row0 + (u64)r * pitch + t, d);
      }
    }
  }
};

// The same case (stream-major, cursors not all at a block boundary) when the row pitch is even, i.e. every row starts
// 16-byte aligned: the aligned path's store pattern -- boxes of 32 rows handed to the TMA -- survives if the
// misalignment is moved into shared memory.  Output index q of a row is the same column for all 32 rows of a warp; what
// differs per lane is only how far it has got: after block step s lane i holds columns up to 12 (s + 1) - pos_i.  So every
// lane writes its 12 doubles at ITS OWN columns of a ring of three granules (16 doubles = 128 bytes per row, 32 rows:
// one 4 KB box with SWIZZLE_128B, 2-way bank conflicts at worst), and when the slowest lane (largest cursor of the warp)
// has completed a granule, lane 0 sends it as one box {16 doubles, 32 rows}.  The lanes are at most 12 doubles apart, so
// the columns in flight span less than three granules, and the granule written now was sent two steps ago
// (cp.async.bulk.wait_group.read makes sure it has been read).  Row ends and rows past the launch are clipped by the
// tensor map: no masked direct stores at all.  12 KB per warp; with the 20 KB of the tile three CTAs per SM.
constexpr u32 kRingBoxBytes = 32u * 128u;
constexpr u32 kRingWarpBytes = 3u * kRingBoxBytes;
constexpr u32 kRingCtaBytes = 4u * kRingWarpBytes + 1024u;  // dynamic shared memory (+ alignment)
struct RingStage {
  u32 row;      // shared address of this lane's row in granule slot 0 of its warp's ring
  u32 rx;       // swizzle term of the row: (lane & 7) << 4
  u32 p0;       // ring position (0 .. 47) of the first draw of the next block
  u32 sent;     // granules handed to the TMA (warp-uniform)
  u32 pmax;     // largest cursor in the warp (warp-uniform): the slowest lane
  u32 ring;     // shared address of the warp's ring
  int c1;       // tensor row of the warp's first stream
  u64 col0;     // tensor column of the item's first draw
  const void* tmap;
  u32 kexp;
  __device__ __forceinline__ void init(uint8_t* stage, const void* tensor_map, u64 tile_first, u64 t0, u32 pos, u32 kexp_) {
    const u32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    ring = ((umma::smem_u32(stage) + 1023u) & ~1023u) + warp * kRingWarpBytes;
    row = ring + lane * 128u;
    rx = (lane & 7u) << 4;
    p0 = pos ? 48u - pos : 0u;  // block 0 starts pos columns before the item's first draw
    sent = 0;
    pmax = __reduce_max_sync(0xFFFFFFFFu, pos);
    c1 = (int)(tile_first + warp * 32u);
    col0 = t0;
    tmap = tensor_map;
    kexp = kexp_;
  }
  // shared address of ring position p (0 .. 47) of this lane's row: slot p / 16, 16-byte chunk (p % 16) / 2 XOR-swizzled
  // with the row, half p % 2
  __device__ __forceinline__ u32 at(u32 p) const {
    const u32 ps = p << 3;
    return row + ((ps & 0x180u) << 5) + ((ps & 0x78u) ^ rx);
  }
  template <int OUT, int J, bool MASKED>
  __device__ __forceinline__ void put(const u32 (&v)[18], u64 q0, u64 n) {
    if constexpr (J < 12) {
      double a, b;
      draw_pair<OUT, J>(v, kexp, a, b);
      u32 pa = p0 + J, pb = p0 + J + 1;
      pa = pa >= 48u ? pa - 48u : pa;
      pb = pb >= 48u ? pb - 48u : pb;
      if (!MASKED || q0 + J < n) asm volatile("st.shared.f64 [%0], %1;" ::"r"(at(pa)), "d"(a) : "memory");
      if (!MASKED || q0 + J + 1 < n) asm volatile("st.shared.f64 [%0], %1;" ::"r"(at(pb)), "d"(b) : "memory");
      put<OUT, J + 2, MASKED>(v, q0, n);
    }
  }
  // whole-warp call: block step s (0 = the current block).  Draw j of the block is output index q = 12 s + j - pos of the
  // item if that is in [0, n) (it wraps below zero for draws before the cursor: then q >= n).
  template <int OUT, bool MASKED>
  __device__ __forceinline__ void emit(const u32 (&v)[18], u64 s, u32 pos, u64 n) {
    if ((threadIdx.x & 31u) == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncwarp();
    put<OUT, 0, MASKED>(v, 12 * s - pos, n);
    p0 = p0 + 12u >= 48u ? p0 - 36u : p0 + 12u;
    umma::fence_proxy_async_smem();
    __syncwarp();
    // granules every lane has completed: the slowest lane holds columns up to 12 (s + 1) - pmax
    const u64 have = 12 * (s + 1) >= pmax ? 12 * (s + 1) - pmax : 0;
    const u32 done = (u32)(have >= n ? (n + 15) / 16 : have / 16);
    if ((threadIdx.x & 31u) == 0 && done > sent) {
      for (u32 g = sent; g < done; g++)
        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(tmap),
                     "r"((int)(col0 + 16ull * g)), "r"(c1), "r"(ring + (g % 3u) * kRingBoxBytes)
                     : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    sent = done > sent ? done : sent;
  }
  __device__ __forceinline__ void drain() {  // before the ring serves another item or the CTA exits
    if ((threadIdx.x & 31u) == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    __syncwarp();
  }
};

// Interleaved 24-bit floats (rlxpp_generate_floats, aligned cursors).  A float row holds 4 bytes per stream: direct
// stores are 24 instructions of 128 bytes per warp and advance (measured 700 G draws/s).  Instead the CTA parks a
// block as [24 float rows][128 streams] in shared memory and ONE thread of the MMA-issuing warp hands it to the TMA
// as a box of 24 rows x 512 bytes.  No new barrier: the box of block b - 1 is sent from Tile::issue() of advance
// b + 1, where every thread has fenced its stores and arrived at the hand-off barrier anyway.  Ring of three boxes:
// block b is written after collect() of advance b, i.e. after the MMA-done mbarrier that the issuing thread committed
// AFTER waiting (cp.async.bulk.wait_group.read) for the copy of block b - 3.
constexpr u32 kF32BoxBytes = 24u * 128u * 4u;               // 12,288
constexpr u32 kF32StageBytes = 3u * kF32BoxBytes + 128u;    // dynamic shared memory (+ alignment)
struct F32RowStage {
  u32 base;        // shared address of the ring
  u32 col;         // this thread's byte offset in a row
  u32 nfilled;     // blocks parked so far (the same in all threads)
  u32 nsent;       // blocks handed to the TMA (meaningful in the sending thread only)
  bool sender;     // lane 0 of the MMA-issuing warp
  int c0, r0;      // tensor coordinates of the tile's first stream and of the item's first float row
  const void* tmap;
  __device__ __forceinline__ void init(uint8_t* stage, const void* tensor_map, u64 tile_first, u64 t0, u32 issuer_warp) {
    base = (umma::smem_u32(stage) + 127u) & ~127u;
    col = threadIdx.x * 4u;
    nfilled = 0;
    nsent = 0;
    sender = (threadIdx.x >> 5) == issuer_warp && (threadIdx.x & 31u) == 0;
    c0 = (int)tile_first;
    r0 = (int)(2 * t0);
    tmap = tensor_map;
  }
  template <int J>
  __device__ __forceinline__ void park(u32 dst, const u32 (&v)[18]) {
    if constexpr (J < 12) {
      const double d = draw_value<kF32, J>(v, 0u);
      asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst + (2 * J) * 512u), "r"(__double2loint(d)) : "memory");
      asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst + (2 * J + 1) * 512u), "r"(__double2hiint(d)) : "memory");
      park<J + 1>(dst, v);
    }
  }
  __device__ __forceinline__ void emit(const u32 (&v)[18]) {
    park<0>(base + (nfilled % 3u) * kF32BoxBytes + col, v);
    nfilled++;
  }
  // issuing warp, before the MMAs: the boxes sent so far have been read
  __device__ __forceinline__ void before_mma() {
    if (sender) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncwarp();
  }
  // the CTA's stores to the parked blocks are fenced and handed over: send what is parked and unsent
  __device__ __forceinline__ void send_parked() {
    if (sender) {
      while (nsent < nfilled) {
        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(tmap), "r"(c0),
                     "r"(r0 + 24 * (int)nsent), "r"(base + (nsent % 3u) * kF32BoxBytes)
                     : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        nsent++;
      }
    }
  }
  // CTA-collective, after the item's last block
  __device__ __forceinline__ void drain() {
    umma::fence_proxy_async_smem();
    __syncthreads();
    send_parked();
    if (sender) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  }
};

// ----------------------------------------------------------------------------- UMMA engine
// Same contract as generate_kernel / advance_states_kernel, with multiply9x9 + mod_m done by
// the tensor core (umma_path.cuh).  One CTA = 128 streams; every thread of the CTA runs the same
// number of issue()/collect() pairs (they contain CTA barriers), rows past `count` carry x = 0.
__device__ __forceinline__ void to_ranlux_hot(const u32 (&x)[18], u32 (&v)[18], u32& c) {
  u32 rare = 0;
  to_ranlux_fast(x, v, c, rare);
  if (__builtin_expect(rare != 0, 0)) {
    to_ranlux_exact(x, v, c);  // inline: a call would force x, v into local memory
    count_rare(ranlux_rare_mask(x, v, c));
  }
}

// Persistent grid with a ticket scheduler.  A work item = (tile of 128 streams, chunk of
// chunk_len draws); ticket w is item (w % n_tiles, w / n_tiles), so the chunks of one tile are
// handed out in order and sched[1 + tile] counts the chunks of it that are finished (state written
// back).  With n_chunks == 1 this is a plain grid-stride loop over tiles; with more, the grid's last
// partial wave shrinks from a whole tile's work to one chunk's (cfg4 / cfg5: 2,048 tiles over
// 148 x 4 CTAs).  A CTA that waits for chunk c - 1 of its tile waits for an EARLIER ticket, which a
// resident CTA holds: no deadlock whatever the number of resident CTAs.
template <int MODE, bool ALIGNED, int OUT = kF64>
__global__ void __launch_bounds__(tc::kTile, tc::kCtasPerSm) tc_generate_kernel(const __grid_constant__ GenArgs a) {
  __shared__ tc::Smem smem;
  constexpr bool kStaged = MODE == kStoreStreamMajor && ALIGNED;
  extern __shared__ __align__(128) uint8_t stage[];  // kStageCtaBytes when kStaged; float row boxes; row stage or ring; else none
  constexpr bool kRowStaged = MODE == kStoreStreamMajor && !ALIGNED;
  const bool ring = kRowStaged && a.ring != 0;
  tc::Tile<MODE == kReduce ? tc::kSyncCta : tc::kSyncArrive> tile;
  tile.setup(smem, a.bmat);
  // the parameter form saves 12 instructions per advance and helps the ALU-bound fused kernel (+5 %); the
  // HBM-bound store kernels measured 4.5 % SLOWER with it (different store scheduling) and keep the literal
  const u32 kexp = MODE == kReduce ? a.kexp : kExp16;
  const u64 n_items = (u64)a.n_tiles * a.n_chunks;
  for (;;) {
    if (threadIdx.x == 0) smem.ticket = atomicAdd(a.sched, 1u);
    __syncthreads();
    const u64 w = smem.ticket;
    if (w >= n_items) break;
    const u32 tidx = (u32)(w % a.n_tiles), chunk = (u32)(w / a.n_tiles);
    if (chunk > 0) {
      if (threadIdx.x == 0) {
        u32 done;
        do {
          asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(done) : "l"(a.sched + 1 + tidx) : "memory");
        } while (done < chunk);
      }
      __syncthreads();
    }
    const u64 il = (u64)tidx * tc::kTile + threadIdx.x;
    const bool live = il < a.count;
    const u64 i = a.first + il;
    const u64 t0 = (u64)chunk * a.chunk_len;                               // first draw of this item
    const u64 n = a.n_per - t0 < a.chunk_len ? a.n_per - t0 : a.chunk_len;  // its draws
    u32 x[18], v[18], pos = 12, c;
#pragma unroll
    for (int j = 0; j < 18; j++) x[j] = 0;
    if (live) load_state(a.st, a.n_total, i, x, pos);
    Sink<MODE, OUT> sink;
    sink.ld = a.ld;
    sink.S = 0.0;
    sink.Q = 0.0;
    sink.kexp = kexp;
    if (MODE == kReduce && chunk > 0 && live) {
      sink.S = __ldcg(a.sum + il);
      sink.Q = __ldcg(a.sumsq + il);
    }
    const u64 pitch = a.pitch ? a.pitch : a.n_per;
    if (MODE == kStoreStreamMajor) sink.p = a.out + il * pitch + t0;
    else if (MODE == kStoreInterleaved && OUT == kF32)  // 4-byte elements: float il of float row 2 t0
      sink.p = reinterpret_cast<double*>(reinterpret_cast<float*>(a.out) + il + 2 * t0 * a.ld);
    else if (MODE == kStoreInterleaved) sink.p = a.out + il + t0 * a.ld;
    else sink.p = nullptr;
    if (ALIGNED) {
      const u64 nblk = n / 12;
      StreamMajorStage sm;
      if (kStaged) sm.init(stage, &a.tmap, (u64)tidx * tc::kTile, kexp, t0);
      const u64 nstaged = nblk & ~(u64)7;  // whole cycles go through the TMA, the rest of a row is stored directly
      constexpr bool kF32Rows = MODE == kStoreInterleaved && OUT == kF32;
      const bool f32_boxes = kF32Rows && a.f32_boxes != 0;
      F32RowStage fs;
      if (f32_boxes) fs.init(stage, &a.tmap, (u64)tidx * tc::kTile, t0, tile.issuer);
      if (nblk > 0) tile.issue(x);
#pragma unroll 1
      for (u64 b = 0; b < nblk; b++) {
        u32 z[20];
        tile.collect(z);
        tc::reduce_z(z, x);
        // the tensor core works on advance b + 2 while block b + 1 is emitted
        if (b + 1 < nblk) {
          if (f32_boxes) tile.issue(x, [&] { fs.before_mma(); }, [&] { fs.send_parked(); });
          else tile.issue(x);
        }
        to_ranlux_hot(x, v, c);
        if (kStaged && b < nstaged) sm.emit<OUT>(v);
        else if (f32_boxes) fs.emit(v);
        else if (live) EmitBlock<0, MODE, OUT>::all(sink, v, b * 12);
      }
      if (kStaged) sm.drain();
      if (f32_boxes) fs.drain();
    } else if (n > 0) {
      const u64 last = ((u64)pos + (n - 1)) / 12;  // own last block
      const u64 smax = (12 + (n - 1)) / 12;        // last block of any thread (uniform)
      UnalignedRowStage rs;
      RingStage rg;
      if (kRowStaged) {
#pragma unroll
        for (int j = 0; j < 18; j++) v[j] = 0;  // lanes without a current block still take part in the warp's copy
        if (ring) rg.init(stage, &a.tmap, (u64)tidx * tc::kTile, t0, pos, kexp);
        else rs.init(stage, a.out + t0, (u64)tidx * tc::kTile + (threadIdx.x & ~31u), a.count, pitch, kexp);
      }
      if (pos < 12) {
        to_ranlux_exact(x, v, c);
        if (!kRowStaged && live) EmitBlock<0, MODE, OUT>::masked(sink, v, 0, pos, n);
      }
      if (kRowStaged) {  // cursor 12: every position lies before the cursor, nothing is stored
        if (ring) rg.emit<OUT, true>(v, 0, pos, n);
        else rs.emit<OUT>(v, 0, pos, n);
      }
      tile.issue(x);
      // blocks 1 .. smax - 2 lie wholly inside [0, n) for every cursor (last >= smax - 1): no masks
      u64 s = 1;
#pragma unroll 1
      for (; s + 2 <= smax; s++) {
        u32 z[20];
        tile.collect(z);
        tc::reduce_z(z, x);
        tile.issue(x);
        to_ranlux_hot(x, v, c);
        if (kRowStaged) {
          if (ring) rg.emit<OUT, false>(v, s, pos, n);
          else rs.emit<OUT>(v, s * 12, pos, n);
        } else if (live) EmitBlock<0, MODE, OUT>::template all<false>(sink, v, s * 12 - pos);
      }
#pragma unroll 1
      for (; s <= smax; s++) {
        u32 z[20], xn[18];
        tile.collect(z);
        tc::reduce_z(z, xn);
        const bool take = s <= last;  // false only at s == smax for streams that end one block early
        if (take) {
#pragma unroll
          for (int j = 0; j < 18; j++) x[j] = xn[j];
        }
        if (s < smax) tile.issue(x);
        if (take) {
          to_ranlux_hot(x, v, c);
          if (!kRowStaged && live) EmitBlock<0, MODE, OUT>::masked(sink, v, s * 12, pos, n);
        }
        if (kRowStaged) {  // a stream that ended a block early has all of it past n
          if (ring) rg.emit<OUT, true>(v, s, pos, n);
          else rs.emit<OUT>(v, s * 12, pos, n);
        }
      }
      if (ring) rg.drain();
      pos = (u32)((u64)pos + n - 12 * last);
    }
    if (live) {
      store_state(a.st, a.n_total, i, x, pos);
      if (MODE == kReduce) {
        a.sum[il] = sink.S;
        if (a.sumsq) a.sumsq[il] = sink.Q;
      }
    }
    if (a.n_chunks > 1) {  // publish: state (and partial sums) of this tile are in global memory
      __threadfence();
      __syncthreads();
      if (threadIdx.x == 0)
        asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(a.sched + 1 + tidx), "r"(chunk + 1u) : "memory");
    } else {
      __syncthreads();  // smem.ticket is rewritten at the top of the loop
    }
  }
  tile.teardown();
}

// Short calls (cfg1: 8 tiles x 32 blocks, S8d "launch-latency dominated"): a tile's blocks are a serial chain only if
// they are computed one from the other.  Block b of a stream is to_ranlux(A^(b+1) X) (D7; "fast exponentiation"),
// so with the byte matrices of A^1 .. A^K at hand, K CTAs ("lanes") work on ONE tile at once: lane j reads the stored
// state, reaches block j with ONE pass against the matrix of A^(j+1), and then strides through blocks j + K, j + 2K, ...
// with the matrix of A^K.  cfg1 becomes 256 CTAs of one pass each instead of 8 CTAs of 32 passes.  The lane that
// computes the last block holds A^nblk X = the new state; it writes it in place once all K lanes of the tile have
// read the old one (one counter per tile, left at zero again; all CTAs of the grid are co-resident by construction).
// Aligned cursors, whole blocks, every store mode and output form (direct stores: the outputs are L2-sized).
constexpr u32 kMaxLanes = 32;
template <int MODE, int OUT>
__global__ void __launch_bounds__(tc::kTile, tc::kCtasPerSm) tc_generate_lanes_kernel(const __grid_constant__ GenArgs a) {
  static_assert(MODE != kReduce, "the fused sums are sequential in the draw index");
  __shared__ tc::Smem smem;
  __shared__ __align__(128) uint8_t bstride[tc::kBBytes];  // matrix of A^lanes: every pass after a lane's first
  const u32 K = a.lanes, tidx = blockIdx.x / K, lane = blockIdx.x % K;
  const u64 nblk = a.n_per / 12;
  const bool strides = lane + K < nblk;  // this lane makes more than one pass
  if (strides) {
    const uint4* src = a.bmat_pow + (u64)(K - 1) * (tc::kBBytes / 16);
    uint4* dst = reinterpret_cast<uint4*>(bstride);
    for (u32 q = threadIdx.x; q < tc::kBBytes / 16; q += tc::kTile) dst[q] = __ldg(src + q);
  }
  tc::Tile<tc::kSyncCta> tile;
  tile.setup(smem, a.bmat_pow + (u64)lane * (tc::kBBytes / 16));  // the matrix of A^(lane + 1)
  const u64 il = (u64)tidx * tc::kTile + threadIdx.x;
  const bool live = il < a.count;
  u32 x[18], v[18], pos = 12, c;
#pragma unroll
  for (int j = 0; j < 18; j++) x[j] = 0;
  if (live) load_state(a.st, a.n_total, a.first + il, x, pos);
  Sink<MODE, OUT> sink;
  sink.ld = a.ld;
  sink.S = 0.0;
  sink.Q = 0.0;
  sink.kexp = kExp16;
  if (MODE == kStoreStreamMajor) sink.p = a.out + il * (a.pitch ? a.pitch : a.n_per);
  else if (OUT == kF32) sink.p = reinterpret_cast<double*>(reinterpret_cast<float*>(a.out) + il);
  else sink.p = a.out + il;
  tile.issue(x);  // (CTA barrier inside: every thread's state now sits in shared memory)
  if (threadIdx.x == 0) {
    __threadfence();
    atomicAdd(a.lane_sync + tidx, 1u);  // this lane has read the tile's state
  }
  if (strides) tile.bdesc = umma::smem_desc(umma::smem_u32(bstride), tc::kBChunk, 128u);
#pragma unroll 1
  for (u64 b = lane; b < nblk; b += K) {
    u32 z[20];
    tile.collect(z);
    tc::reduce_z(z, x);
    if (b + K < nblk) tile.issue(x);
    to_ranlux_hot(x, v, c);
    if (live) EmitBlock<0, MODE, OUT>::all(sink, v, b * 12);
    if (b + 1 == nblk) {  // uniform: this lane ends on the tile's last block
      if (threadIdx.x == 0) {
        u32 readers;
        do {
          asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(readers) : "l"(a.lane_sync + tidx) : "memory");
        } while (readers < K);
        a.lane_sync[tidx] = 0;
      }
      __syncthreads();
      if (live) store_state(a.st, a.n_total, a.first + il, x, 12u);
    }
  }
  tile.teardown();
}

// Fused sum / sum of squares (S8 a-7b, cfg5) and interleaved stores (cfg3 / cfg4) with TWO tiles per CTA on one
// accumulator (tc::PairTile): a tile is a chain of advances, and interleaving two chains hides the tensor pipe's round
// trip behind the other tile's integer work.  Work item = (PAIR of adjacent tiles, chunk of draws); n_tiles counts pairs.
// Same contract and the same per-stream arithmetic as tc_generate_kernel.
// Hand-off (profiles/ab_r02_pairs.md): the fused reduce is indifferent (CTA barrier 1,228, named barrier 1,223 G doubles/s);
// the store kernels want the named barrier (cfg3 727 vs 759 burst, 633 vs 655 sustained).
// The work loop of the 128 threads that own pairs of tiles, written against the tile policy TILE (tc::PairTile): tile.tid =
// thread within the 128, tile.sync() = barrier over them, tile.ticket = their shared scheduler word, tile.collect() = one
// half-step.  (The same loop on tc::GroupTile -- 5 groups of 128 threads in one CTA per SM, 80 registers -- was measured
// for the fused reduce: 1,128 vs 1,230 G doubles/s.  More warps do not help: the ALU pipe binds; profiles/ab_r02_pairs.md.)
template <bool ALIGNED, int MODE, int OUT, class TILE>
__device__ __forceinline__ void pair_items(TILE& tile, const GenArgs& a) {
  static_assert(MODE == kReduce || MODE == kStoreInterleaved, "pairs: fused reduce or interleaved stores");
  const u32 kexp = a.kexp;  // a launch parameter: the PRMT selectors become immediates (arith.cuh)
  const u64 n_items = (u64)a.n_tiles * a.n_chunks;
  for (;;) {
    if (tile.tid == 0) *tile.ticket = atomicAdd(a.sched, 1u);
    tile.sync();
    const u64 w = *reinterpret_cast<volatile u32*>(tile.ticket);
    if (w >= n_items) break;
    const u32 pidx = (u32)(w % a.n_tiles), chunk = (u32)(w / a.n_tiles);
    if (chunk > 0) {
      if (tile.tid == 0) {
        u32 done;
        do {
          asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(done) : "l"(a.sched + 1 + pidx) : "memory");
        } while (done < chunk);
      }
      tile.sync();
    }
    const u64 t0 = (u64)chunk * a.chunk_len;
    const u64 n = a.n_per - t0 < a.chunk_len ? a.n_per - t0 : a.chunk_len;
    const u64 smax = n ? (12 + (n - 1)) / 12 : 0;  // unaligned: last block of any thread (uniform)
    u64 il[2];
    bool live[2], early[2];
    u32 pos[2], newpos[2];
    Sink<MODE, OUT> sink[2];
    u32 x[18], v[18], c;
#pragma unroll
    for (int t = 0; t < 2; t++) {
      il[t] = ((u64)pidx * 2 + t) * tc::kTile + tile.tid;
      live[t] = il[t] < a.count;
      pos[t] = 12;
#pragma unroll
      for (int j = 0; j < 18; j++) x[j] = 0;
      if (live[t]) load_state(a.st, a.n_total, a.first + il[t], x, pos[t]);
      if (MODE == kStoreInterleaved && OUT == kF32)
        sink[t].p = reinterpret_cast<double*>(reinterpret_cast<float*>(a.out) + il[t] + 2 * t0 * a.ld);
      else sink[t].p = MODE == kStoreInterleaved ? a.out + il[t] + t0 * a.ld : nullptr;
      sink[t].ld = a.ld;
      sink[t].kexp = kexp;
      sink[t].S = 0.0;
      sink[t].Q = 0.0;
      if (MODE == kReduce && chunk > 0 && live[t]) {
        sink[t].S = __ldcg(a.sum + il[t]);
        sink[t].Q = __ldcg(a.sumsq + il[t]);
      }
      const u64 last = n ? ((u64)pos[t] + (n - 1)) / 12 : 0;  // own last block
      early[t] = last < smax;
      newpos[t] = (u32)((u64)pos[t] + n - 12 * last);
      if (!ALIGNED && n > 0 && pos[t] < 12) {  // block 0 = the current block
        to_ranlux_exact(x, v, c);
        if (live[t]) EmitBlock<0, MODE, OUT>::masked(sink[t], v, 0, pos[t], n);
      }
      tile.stash(t, x);
    }
    if (ALIGNED) {
      const u64 nblk = n / 12;
      if (nblk > 0) tile.start(0);
#pragma unroll 1
      for (u64 b = 0; b < nblk; b++) {
#pragma unroll
        for (int t = 0; t < 2; t++) {
          u32 z[20];
          tile.collect(z, t == 0 || b + 1 < nblk, t ^ 1);  // the other tile's MMA runs under this tile's integer work
          tc::reduce_z(z, x);
          if (b + 1 < nblk) tile.stash(t, x);
          else if (live[t]) store_state(a.st, a.n_total, a.first + il[t], x, 12u);
          to_ranlux_hot(x, v, c);
          if (live[t]) EmitBlock<0, MODE, OUT>::all(sink[t], v, b * 12);
        }
      }
    } else if (n > 0) {
      tile.start(0);
      // blocks 1 .. smax - 2 lie wholly inside [0, n) for every cursor: no masks
      u64 s = 1;
#pragma unroll 1
      for (; s + 2 <= smax; s++) {
#pragma unroll
        for (int t = 0; t < 2; t++) {
          u32 z[20];
          tile.collect(z, true, t ^ 1);
          tc::reduce_z(z, x);
          tile.stash(t, x);
          to_ranlux_hot(x, v, c);
          if (live[t]) EmitBlock<0, MODE, OUT>::template all<false>(sink[t], v, s * 12 - pos[t]);
        }
      }
      // the last two blocks carry per-draw masks; a stream that ends one block early (early[t]) discards the last
      // product.  Every stream takes block smax - 1 (if there is one), so the state is written there and again at smax.
#pragma unroll 1
      for (; s <= smax; s++) {
#pragma unroll
        for (int t = 0; t < 2; t++) {
          u32 z[20];
          tile.collect(z, t == 0 || s < smax, t ^ 1);
          tc::reduce_z(z, x);
          if (s < smax) tile.stash(t, x);
          if (!(s == smax && early[t])) {
            if (live[t]) store_state(a.st, a.n_total, a.first + il[t], x, newpos[t]);
            to_ranlux_hot(x, v, c);
            if (live[t]) EmitBlock<0, MODE, OUT>::masked(sink[t], v, s * 12, pos[t], n);
          }
        }
      }
    }
#pragma unroll
    for (int t = 0; t < 2; t++) {
      if (!live[t]) continue;
      if (!ALIGNED && n > 0 && smax == 1 && early[t]) {  // never advanced: only the cursor moves
        uint4 q = __ldcg(a.st + 4 * a.n_total + a.first + il[t]);
        q.z = newpos[t];
        a.st[4 * a.n_total + a.first + il[t]] = q;
      }
      if (MODE == kReduce) {
        a.sum[il[t]] = sink[t].S;
        if (a.sumsq) a.sumsq[il[t]] = sink[t].Q;
      }
    }
    if (a.n_chunks > 1) {  // publish: state and partial sums of this pair are in global memory
      __threadfence();
      tile.sync();
      if (tile.tid == 0)
        asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(a.sched + 1 + pidx), "r"(chunk + 1u) : "memory");
    } else {
      tile.sync();  // the ticket word is rewritten at the top of the loop
    }
  }
}

template <bool ALIGNED, int MODE = kReduce, int OUT = kF64>
__global__ void __launch_bounds__(tc::kTile, tc::kCtasPerSm) tc_pair_kernel(const __grid_constant__ GenArgs a) {
  __shared__ tc::PairSmem smem;
  tc::PairTile<MODE == kReduce ? tc::kSyncCta : tc::kSyncArrive> tile;
  tile.setup(smem, a.bmat);
  pair_items<ALIGNED, MODE, OUT>(tile, a);
  tile.teardown();
}
// Raw advance (cfg2; S8 a-3 / a-4 alone): x <- A^reps x on raw uint64[9] states, in place.  Two tiles per accumulator
// (the other tile's MMA runs under this tile's normalisation, as in tc_pair_kernel) and tc::kGroups groups of 128
// threads in one CTA per SM (tc::GroupTile): six accumulators per SM instead of four.  Persistent: group (CTA c, group g)
// strides over the pairs of tiles.  Measured at cfg2 (G doubles-equivalent/s): one tile per CTA 1,160; pairs in four
// CTAs 1,180; 5 groups 1,228; 6 groups 1,320.
struct GroupSync {
  u32 barid;
  __device__ __forceinline__ void operator()() const { asm volatile("bar.sync %0, 128;" ::"r"(barid) : "memory"); }
};
template <int LAYOUT>
__global__ void __launch_bounds__(tc::kGroups * tc::kTile, 1) tc_advance_states_group_kernel(u64* __restrict__ states, u64 n, u32 reps,
                                                                                          const uint4* __restrict__ bmat) {
  extern __shared__ __align__(128) uint8_t group_smem[];
  tc::GroupsSmem& smem = *reinterpret_cast<tc::GroupsSmem*>(group_smem);
  uint4* stage_all = reinterpret_cast<uint4*>(group_smem + ((sizeof(tc::GroupsSmem) + 127) & ~(size_t)127));
  tc::GroupTile tile;
  tile.setup(smem, bmat);
  const u32 gid = threadIdx.x / tc::kTile;
  uint4* stage = stage_all + (size_t)gid * kRawStageWords;
  const GroupSync gsync{tile.barid};
  const u64 n_tiles = (n + kThreads - 1) / kThreads, n_pairs = (n_tiles + 1) / 2;
#pragma unroll 1
  for (u64 pair = (u64)blockIdx.x * tc::kGroups + gid; pair < n_pairs; pair += (u64)gridDim.x * tc::kGroups) {
    u32 x[18];
#pragma unroll
    for (int t = 0; t < 2; t++) {
      const u64 blk = 2 * pair + t;
#pragma unroll
      for (int j = 0; j < 18; j++) x[j] = 0;
      if (blk < n_tiles) {  // uniform over the group
        load_raw<LAYOUT>(states, n, stage, x, blk, tile.tid, gsync);
        if (reps == 0) {
          canonicalise(x);
          store_raw<LAYOUT>(states, n, stage, x, blk, tile.tid, gsync);
        }
        gsync();  // the staging buffer is reused
      }
      tile.stash(t, x);
    }
    if (reps > 0) tile.start(0);
#pragma unroll 1
    for (u32 r = 0; r < reps; r++) {
#pragma unroll
      for (int t = 0; t < 2; t++) {
        u32 z[20];
        tile.collect(z, t == 0 || r + 1 < reps, t ^ 1);
        tc::reduce_z(z, x);
        if (r + 1 < reps) tile.stash(t, x);
        else if (2 * pair + t < n_tiles) {
          store_raw<LAYOUT>(states, n, stage, x, 2 * pair + t, tile.tid, gsync);
          gsync();
        }
      }
    }
  }
  tile.teardown();
}

// Seeding and skip-ahead ("fast exponentiation by squaring"): x <- x * prod_b T[b]^(bit b of e)
// with T[b] = base^(2^b) precomputed on the host (64 entries of 18 limbs).  A bit is processed by
// the whole warp if any lane has it set; lanes without it keep their value.
__device__ __forceinline__ void pow_table_mul(u32 (&x)[18], u64 e, const u32* __restrict__ table) {
#pragma unroll 1
  for (int b = 0; b < 64; b++) {
    const bool bit = (e >> b) & 1;
    if (!__any_sync(0xFFFFFFFFu, bit)) continue;
    u32 t[18], r[18];
#pragma unroll
    for (int j = 0; j < 18; j++) t[j] = __ldg(table + b * 18 + j);
    mulmod_generic(x, t, r);
#pragma unroll
    for (int j = 0; j < 18; j++) x[j] = bit ? r[j] : x[j];
  }
}

__global__ void __launch_bounds__(kThreads) seed_kernel(uint4* __restrict__ st, u64 n, u64 seed0,
                                                        const u32* __restrict__ tableG) {
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  const bool live = i < n;
  u32 x[18];
#pragma unroll
  for (int j = 0; j < 18; j++) x[j] = j == 0 ? 1u : 0u;
  pow_table_mul(x, live ? seed0 + i : 0ull, tableG);  // D7: X = G^seed, start state 1
  if (live) store_state(st, n, i, x, 12u);
}

__global__ void __launch_bounds__(kThreads) skip_kernel(uint4* __restrict__ st, u64 n, u64 n_uniform,
                                                        const u64* __restrict__ n_each,
                                                        const u32* __restrict__ tableA) {
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  const bool live = i < n;
  u32 x[18], pos = 12;
#pragma unroll
  for (int j = 0; j < 18; j++) x[j] = 0;
  if (live) load_state(st, n, i, x, pos);
  const u64 nn = live ? (n_each ? n_each[i] : n_uniform) : 0ull;
  u64 k = 0;
  u32 newpos = pos;
  if (nn > 0) {  // D8: k = floor((pos + nn - 1) / 12) without 64-bit overflow
    const u64 t = nn - 1;
    const u32 total = (u32)(t % 12) + pos;  // <= 23
    k = t / 12 + total / 12;
    newpos = total % 12 + 1;
  }
  pow_table_mul(x, k, tableA);
  if (live) store_state(st, n, i, x, newpos);
}

// get_state: the paper's stored form: packed RANLUX numbers + carry, cursor, LCG state
__global__ void __launch_bounds__(kThreads) export_kernel(const uint4* __restrict__ st, u64 n, u64* __restrict__ ranlux,
                                                          u32* __restrict__ carry, u32* __restrict__ pos_out,
                                                          u64* __restrict__ lcg) {
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  u32 x[18], v[18], pos, c;
  load_state(st, n, i, x, pos);
  to_ranlux_exact(x, v, c);
#pragma unroll
  for (int l = 0; l < 9; l++) {
    if (ranlux) ranlux[i * 9 + l] = (u64)v[2 * l] | ((u64)v[2 * l + 1] << 32);
    if (lcg) lcg[i * 9 + l] = (u64)x[2 * l] | ((u64)x[2 * l + 1] << 32);
  }
  if (carry) carry[i] = c;
  if (pos_out) pos_out[i] = pos;
}

__global__ void __launch_bounds__(kThreads) import_kernel(uint4* __restrict__ st, u64 n, const u64* __restrict__ lcg,
                                                          const u32* __restrict__ pos_in) {
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  u32 z[20], x[18];
#pragma unroll
  for (int l = 0; l < 9; l++) {
    const u64 w = lcg[i * 9 + l];
    z[2 * l] = (u32)w;
    z[2 * l + 1] = (u32)(w >> 32);
  }
  z[18] = 0; z[19] = 0;
  mod_m20(z, x);
  u32 pos = pos_in ? pos_in[i] : 12u;
  store_state(st, n, i, x, pos > 12u ? 12u : pos);
}

// S8 a-2 / D3: the paper's stored form -> LCG state, X = V - (V >> 336) + c, and X == m -> 0
// (V = 2^576 - 1 with c = 1, the one combination that reaches m).  Cold path: the kernels keep the LCG form.
__device__ __forceinline__ void to_lcg(const u32 (&v)[18], u32 c, u32 (&x)[18]) {
  u32 z[20];
  u64 borrow = 0;
#pragma unroll
  for (int j = 0; j < 18; j++) {
    const u32 hi = j + 11 < 18 ? v[j + 11] : 0u, lo = j + 10 < 18 ? v[j + 10] : 0u;
    const u64 d = (u64)v[j] - (u64)((lo >> 16) | (hi << 16)) - borrow;  // limb j of V >> 336
    z[j] = (u32)d;
    borrow = d >> 63;
  }
  u64 carry = c & 1u;
#pragma unroll
  for (int j = 0; j < 18; j++) {
    const u64 t = (u64)z[j] + carry;
    z[j] = (u32)t;
    carry = t >> 32;
  }
  z[18] = 0; z[19] = 0;  // V >= V >> 336 and the sum is <= m: no borrow, no carry out
  mod_m20(z, x);
}

__global__ void __launch_bounds__(kThreads) import_ranlux_kernel(uint4* __restrict__ st, u64 n, const u64* __restrict__ ranlux,
                                                                 const u32* __restrict__ carry, const u32* __restrict__ pos_in) {
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  if (i >= n) return;
  u32 v[18], x[18];
#pragma unroll
  for (int l = 0; l < 9; l++) {
    const u64 w = ranlux[i * 9 + l];
    v[2 * l] = (u32)w;
    v[2 * l + 1] = (u32)(w >> 32);
  }
  to_lcg(v, carry ? carry[i] : 0u, x);
  u32 pos = pos_in ? pos_in[i] : 12u;
  store_state(st, n, i, x, pos > 12u ? 12u : pos);
}

// ----------------------------------------------------------------------------- device API (S8 f-1)
// rlxpp_generate_ragged[_reduce]: every stream draws ITS OWN number of doubles -- the paper's GPU use
// (one state per thread, threads consume numbers at their own pace).  Written entirely
// with the public per-thread API of include/rlxpp_device.cuh, of which it is the reference use:
// COOP = draw_coop() (one advance pass per warp and 12 draws whatever the cursors), else draw()
// (the paper's per-thread advance, which diverges); COOP = 2 alternates the two from draw to draw on the same Stream
// (they mix freely: a spare block made by draw_coop() is entered by draw()).
template <int COOP, bool REDUCE>
__global__ void __launch_bounds__(kThreads) ragged_kernel(const rlxpp_view_t view, const u32* __restrict__ counts,
                                                          double* __restrict__ out, u64 ld, double* __restrict__ sum,
                                                          double* __restrict__ sumsq) {
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  const bool live = i < view.n;
  rlxpp_dev::Stream g;
  if (live) g.load(view, i);
  const u32 cnt = live ? counts[i] : 0u;
  double S = 0.0, Q = 0.0;
  double* row = REDUCE ? nullptr : out + i * ld;
  if (COOP) {
    const u32 maxc = __reduce_max_sync(0xFFFFFFFFu, cnt);
#pragma unroll 1
    for (u32 t = 0; t < maxc; t++) {
      const unsigned mask = __ballot_sync(0xFFFFFFFFu, t < cnt);
      if (t < cnt) {
        const double d = (COOP == 2 && (t & 1u)) ? g.draw() : g.draw_coop(mask);
        if (REDUCE) { S = S + d; Q = __fma_rn(d, d, Q); }
        else row[t] = d;
      }
    }
  } else {
#pragma unroll 1
    for (u32 t = 0; t < cnt; t++) {
      const double d = g.draw();
      if (REDUCE) { S = S + d; Q = __fma_rn(d, d, Q); }
      else row[t] = d;
    }
  }
  if (live) {
    g.store(view, i);
    if (REDUCE) {
      sum[i] = S;
      if (sumsq) sumsq[i] = Q;
    }
  }
}

// The same ragged generation with the block-cooperative tensor-core advance of include/rlxpp_tile.cuh
// (rlxpp_dev::TileStream, cooperative = 3): a CTA of 128 threads = one tile; when some thread is out of numbers the CTA
// makes one UMMA pass for every thread that holds no spare block.  Reference use of that public API.
template <bool REDUCE>
__global__ void __launch_bounds__(tc::kTile, tc::kCtasPerSm) ragged_tile_kernel(const rlxpp_view_t view, const u32* __restrict__ counts,
                                                                               double* __restrict__ out, u64 ld,
                                                                               double* __restrict__ sum, double* __restrict__ sumsq) {
  __shared__ rlxpp_dev::TileShared sh;
  __shared__ u32 max_count;
  rlxpp_dev::TileStream g;
  g.begin(sh, view);
  const u64 i = (u64)blockIdx.x * tc::kTile + threadIdx.x;
  const bool live = i < view.n;
  g.load(view, i, live);
  const u32 cnt = live ? counts[i] : 0u;
  if (threadIdx.x == 0) max_count = 0;
  __syncthreads();
  const u32 wmax = __reduce_max_sync(0xFFFFFFFFu, cnt);
  if ((threadIdx.x & 31u) == 0) atomicMax(&max_count, wmax);
  __syncthreads();
  const u32 maxc = max_count;
  double S = 0.0, Q = 0.0;
  double* row = REDUCE ? nullptr : out + i * ld;
#pragma unroll 4
  for (u32 t = 0; t < maxc; t++) {
    const double d = g.draw(t < cnt);
    if (t < cnt) {
      if (REDUCE) { S = S + d; Q = __fma_rn(d, d, Q); }
      else row[t] = d;
    }
  }
  if (live) {
    g.store(view, i);
    if (REDUCE) {
      sum[i] = S;
      if (sumsq) sumsq[i] = Q;
    }
  }
  g.end();
}

// ----------------------------------------------------------------------------- roofline probes
// IMAD peak: 8 independent carry chains of IMAD.WIDE.U32.X per thread, nothing else in the loop.
__global__ void __launch_bounds__(kThreads) imad_peak_kernel(u64* out, u32 iters, u32 seed) {
  u64 acc[8];
  u32 x = seed + threadIdx.x;
#pragma unroll
  for (int j = 0; j < 8; j++) acc[j] = (u64)seed * (j + 1);
#pragma unroll 1
  for (u32 it = 0; it < iters; it++) {
#pragma unroll
    for (int rep = 0; rep < 8; rep++) {
      asm("{\n\t.reg .u64 t;\n\t"
          "mul.wide.u32 t, %8, 0x9e3779b9; add.cc.u64  %0, %0, t;\n\t"
          "mul.wide.u32 t, %8, 0x7f4a7c15; addc.cc.u64 %1, %1, t;\n\t"
          "mul.wide.u32 t, %8, 0xbf58476d; addc.cc.u64 %2, %2, t;\n\t"
          "mul.wide.u32 t, %8, 0x1ce4e5b9; addc.cc.u64 %3, %3, t;\n\t"
          "mul.wide.u32 t, %8, 0x94d049bb; add.cc.u64  %4, %4, t;\n\t"
          "mul.wide.u32 t, %8, 0x133111eb; addc.cc.u64 %5, %5, t;\n\t"
          "mul.wide.u32 t, %8, 0xe220a839; addc.cc.u64 %6, %6, t;\n\t"
          "mul.wide.u32 t, %8, 0x7b1dcdaf; addc.cc.u64 %7, %7, t;\n\t"
          "}"
          : "+l"(acc[0]), "+l"(acc[1]), "+l"(acc[2]), "+l"(acc[3]), "+l"(acc[4]), "+l"(acc[5]), "+l"(acc[6]), "+l"(acc[7])
          : "r"(x));
    }
  }
  u64 r = 0;
#pragma unroll
  for (int j = 0; j < 8; j++) r ^= acc[j];
  if (r == 0x1234567u) out[0] = r;  // never true in practice; keeps the chains alive
}
constexpr int kImadPerIter = 64;

__global__ void __launch_bounds__(256) hbm_write_kernel(uint4* __restrict__ out, u64 n16) {
  const u64 stride = (u64)gridDim.x * blockDim.x;
  const uint4 val = make_uint4(threadIdx.x, blockIdx.x, 0x3ff00000u, 0u);
  for (u64 q = (u64)blockIdx.x * blockDim.x + threadIdx.x; q < n16; q += stride) __stcs(out + q, val);
}

// Store-pattern probe (rlxpp_measure_hbm_write_pieces): what a stream-major output looks like to the
// memory system.  Every warp of a persistent grid owns 32 rows at a time and walks along them, writing
// one piece of `piece16` x 16 bytes of each of its rows per step with full 128-bit stores.
__global__ void __launch_bounds__(128, 4) hbm_write_pieces_kernel(uint4* __restrict__ out, u64 rows, u64 pitch16, u32 piece16) {
  const u32 lane = threadIdx.x & 31u;
  const u64 warp = (u64)blockIdx.x * 4 + (threadIdx.x >> 5), n_warps = (u64)gridDim.x * 4;
  const uint4 v = make_uint4(0x3c3c3c3cu, 0x5a5a5a5au, (u32)warp, lane);
  for (u64 g = warp; g < rows / 32; g += n_warps) {
    uint4* base = out + g * 32 * pitch16;
    for (u64 c = 0; c + piece16 <= pitch16; c += piece16)
      for (u32 u = lane; u < 32u * piece16; u += 32u) __stcs(base + (u64)(u / piece16) * pitch16 + c + u % piece16, v);
  }
}

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
  for (int k = 0; k < 72; k++) {
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
    for (int col = 0; col < 72; col++) {
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
// Work items of the persistent UMMA kernel: how many chunks to cut every tile's n_per draws into so
// that the last, partial wave of the grid is short.  One chunk unless the tiles alone fill the
// resident CTAs badly; a chunk is never shorter than 16 advances (state I/O and pipeline fill).
static void plan_items(uint64_t n_tiles, uint64_t n_per, unsigned slots, uint32_t* n_chunks, uint64_t* chunk_len) {
  *n_chunks = 1;
  *chunk_len = n_per;
  const uint64_t blocks = n_per / 12;
  if (n_tiles <= slots || blocks < 32) return;
  // a good plan fills >= 97 % of its last wave AND has >= 12 waves: CTAs do not run at equal speed when the
  // kernel is HBM-bound, and finer items even that out (cfg4: 2 chunks 764, 4 chunks 793 G doubles/s at the
  // same 98.8 % fill; profiles/ab_r01_sync.md)
  double best = 0.0;
  uint64_t best_c = 1;
  for (uint64_t c = 1; c <= 16 && blocks / c >= 16; c++) {
    const uint64_t items = n_tiles * c, waves = (items + slots - 1) / slots;
    const double eff = (double)items / (double)(waves * slots);
    const double score = eff - (waves < 12 ? 0.05 : 0.0);
    if (score > best + 1e-9) { best = score; best_c = c; }
    if (eff >= 0.97 && waves >= 12) break;
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
  // aligned (even pitch; RingStage: 69 KB of shared memory, three CTAs per SM), else through the warp's row stage
  const uint64_t row_pitch = a.pitch ? a.pitch : a.n_per;
  const bool ring = MODE == kStoreStreamMajor && !aligned && row_pitch % 2 == 0 && (uintptr_t)a.out % 16 == 0 &&
                    a.count < (1ull << 31) && a.n_per < (1ull << 31);
  const unsigned slots = ring ? tc_slots() / tc::kCtasPerSm * 3 : tc_slots();
  a.n_tiles = (u32)n_tiles;
  if constexpr (MODE != kReduce) {
    // Short calls that leave most of the grid empty: K lanes per tile, each reaching its blocks with the matrices of
    // A^(j+1) and A^K (tc_generate_lanes_kernel).  All CTAs must be co-resident (the last lane waits for its tile's
    // readers): n_tiles K <= slots.  rlxpp_set_chunks(c > 0) keeps the persistent path.
    const uint64_t nblk = a.n_per / 12, tiles1 = (a.count + tc::kTile - 1) / tc::kTile;  // lanes work on single tiles
    uint64_t K = nblk < kMaxLanes ? nblk : kMaxLanes;
    if (K > slots / tiles1) K = slots / tiles1;
    if (aligned && a.lane_sync && K >= 4 && g_force_chunks.load() == 0) {
      int rc = get_bmatrix_powers(a.p, &a.bmat_pow);
      if (rc) return rc;
      a.lanes = (u32)K;
      tc_generate_lanes_kernel<MODE, OUT><<<(unsigned)(tiles1 * K), tc::kTile, 0, s>>>(a);
      LAUNCH_CHECK();
      return RLXPP_OK;
    }
  }
  plan_items(n_tiles, a.n_per, slots, &a.n_chunks, &a.chunk_len);
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
    // 20 KB static + 33 KB (stream-major boxes) or 36 KB (float-row boxes): above the 48 KB default, 4 CTAs per SM fit
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
      static std::atomic<uint64_t> done{0};  // 20 KB static + 49 KB of rings: three CTAs per SM
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
    return fail(RLXPP_EINVAL, "rlxpp_create: rows_generated.cuh is stale for p = %u (rebuild)", p);
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
  if (fixed < 0) return fail(RLXPP_EINVAL, "rlxpp_advance_states: rows_generated.cuh is stale for p = %u", p);
  cudaStream_t s = (cudaStream_t)cuda_stream;
  if (g_engine.load() == RLXPP_ENGINE_UMMA) {
    const uint4* bmat = nullptr;
    rc = get_bmatrix(p, &bmat);
    if (rc) return rc;
    const uint64_t tiles = (n_states + tc::kTile - 1) / tc::kTile;
    // one CTA per tile: measured faster than a persistent grid here (1,050 vs 946 G doubles-equivalent/s at
    // cfg2: with 16 advances per tile the load / compute / store phases of co-resident CTAs overlap better when
    // the CTAs are not in lock step); the kernel's tile loop serves grids smaller than the tile count
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
  if (reduce) {
    if (coop == 2) ragged_kernel<2, true><<<grid, kThreads, 0, h->stream>>>(view, counts_dev, out, ld, sum, sumsq);
    else if (coop) ragged_kernel<1, true><<<grid, kThreads, 0, h->stream>>>(view, counts_dev, out, ld, sum, sumsq);
    else ragged_kernel<0, true><<<grid, kThreads, 0, h->stream>>>(view, counts_dev, out, ld, sum, sumsq);
  } else {
    if (coop == 2) ragged_kernel<2, false><<<grid, kThreads, 0, h->stream>>>(view, counts_dev, out, ld, sum, sumsq);
    else if (coop) ragged_kernel<1, false><<<grid, kThreads, 0, h->stream>>>(view, counts_dev, out, ld, sum, sumsq);
    else ragged_kernel<0, false><<<grid, kThreads, 0, h->stream>>>(view, counts_dev, out, ld, sum, sumsq);
  }
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
