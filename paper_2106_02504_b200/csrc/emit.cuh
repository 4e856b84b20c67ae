// Launch arguments of the generate kernels and the emission of a block: output forms (double, u48, f32 pair, normal deviate), sinks (stores, fused sums).
// Part of librlxpp (included by rlxpp.cu, one translation unit); see DESIGN.md 5.
#pragma once

#include <cuda.h>
#include "arith.cuh"
#include "normal_coeffs.cuh"

namespace rlx {

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


}  // namespace rlx
