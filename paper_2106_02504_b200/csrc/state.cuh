// Stream state in HBM, the exact slow paths, and the multiplier policies of the IMAD engine (Fixed<P> / Generic).
// Part of librlxpp (included by rlxpp.cu, one translation unit); see DESIGN.md 5.
#pragma once

#include "arith.cuh"
#include "../../include/rlxpp_rows.cuh"

namespace rlx {

using rlxpp_dev::FixedMultiplier;
constexpr int kThreads = 128;  // threads per CTA of the one-thread-per-stream kernels = streams per UMMA tile

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


}  // namespace rlx
