// Device arithmetic of the RANLUX++ hot path on 18 little-endian 32-bit limbs.
//
//   m = 2^576 - 2^240 + 1                                   (sec. 2.2)
//   limbs of m: [0] = 1, [1..6] = 0, [7] = 0xFFFF0000, [8..17] = 0xFFFFFFFF
//
// Two families:
//   * generic, exact, branch-light code (mul18x18, mod_m36, to_ranlux_exact): used by the
//     cold paths (seeding, skip-ahead, arbitrary luxury levels, state export) and as the
//     slow path of the hot kernels;
//   * the hot-path fast forms (fold_fast, to_ranlux_fast) that assume the overwhelmingly
//     likely case and raise a `rare` flag otherwise; the caller then recomputes with the
//     exact functions.  Every rare condition is derived in DESIGN.md ("Kernel: advance").
#pragma once
#include <cstdint>

#include "../../include/rlxpp_tile.cuh"  // the generic, exact arithmetic, the fast forms, the tile geometry (public device API)

namespace rlx {

// the PTX wrappers of the tensor-core path (tcgen05 / TMEM / mbarrier / proxy fences) live in the public header too,
// shared by the library's kernels and by rlxpp_dev::TileStream
namespace umma = rlxpp_dev::umma;

using rlxpp_dev::detail::u32;
using rlxpp_dev::detail::u64;
using rlxpp_dev::detail::i64;
using rlxpp_dev::detail::m_limb;
using rlxpp_dev::detail::k240_limb;
using rlxpp_dev::detail::mul18x18;
using rlxpp_dev::detail::ge_m;
using rlxpp_dev::detail::sub_m;
using rlxpp_dev::detail::mod_m36;
using rlxpp_dev::detail::mod_m20;
using rlxpp_dev::detail::mulmod_generic;
using rlxpp_dev::detail::to_ranlux_exact;
using rlxpp_dev::detail::fold_fast;
using rlxpp_dev::detail::to_ranlux_fast;
using rlxpp_dev::detail::merge_eo;

// ------------------------------------------------------------------ rare-path counters
// Which condition sent an advance of the hot kernels to the exact code (rlxpp_rare_counts, include/rlxpp.h).  The
// conditions are re-derived HERE, in the cold path, from z (the unreduced product) and x (the canonical state), so the
// fast forms above stay as they are: a test that crafts a state for one condition can assert that exactly that
// branch fired.  Indices = RLXPP_RARE_* of rlxpp.h.
enum {
  kRareFoldBorrow = 0,  // fold_fast: the borrow of "- hi" leaves limb 1
  kRareFoldCarry = 1,   // fold_fast: the carry of "+ hi 2^240" leaves limb 9
  kRareFoldTop = 2,     // fold_fast: top limb all ones (the folded value may be >= m)
  kRareRanluxCarry = 3, // to_ranlux_fast: carry out of the 8-limb addition X + (X >> 336)
  kRareRanluxNear = 4,  // to_ranlux_fast: |u - w| <= 1 (the two leading words do not decide the sign of D)
  kRareRanluxUMax = 5,  // to_ranlux_fast: u = 2^32 - 1 (Xl + Xh may cross 2^336)
  kRareRanluxV0 = 6,    // to_ranlux_fast: the "- c" would borrow out of limb 0
  kRareRanluxThird = 7, // exact result was D4's third combination (T = Xh, c = 1)
  kRareKinds = 8
};
__device__ unsigned long long g_rare_counts[kRareKinds];

__device__ __noinline__ void count_rare(u32 mask) {
#pragma unroll 1
  for (int k = 0; k < kRareKinds; k++)
    if (mask >> k & 1u) atomicAdd(&g_rare_counts[k], 1ull);
}
// fold_fast's conditions from the limbs of z it looks at (scalars: taking z's address would move it to local memory)
__device__ __forceinline__ u32 fold_rare_mask(u32 z0, u32 z1, u32 z7, u32 z8, u32 z9, u32 z17, u32 z18, u32 z19) {
  const u64 hi = (u64)z18 | ((u64)z19 << 32);  // < 2^37
  const u64 lo = (u64)z0 | ((u64)z1 << 32);
  const u64 mid = (u64)z7 | ((u64)z8 << 32), sum = mid + (hi << 16);
  const bool cry = sum < mid && z9 == 0xFFFFFFFFu;  // hi 2^16 < 2^53: limb 9 only receives the carry of limbs 7, 8
  return (lo < hi ? 1u << kRareFoldBorrow : 0u) | (cry ? 1u << kRareFoldCarry : 0u) |
         (z17 == 0xFFFFFFFFu ? 1u << kRareFoldTop : 0u);
}
// to_ranlux_fast's conditions from the canonical x, and whether the exact result (v, c) is the third combination
__device__ __forceinline__ u32 ranlux_rare_mask(const u32 (&x)[18], const u32 (&v)[18], u32 c) {
  const u32 u = __funnelshift_r(x[9], x[10], 16), w = x[17];
  u64 cy = 0;
  u32 s0 = 0;
#pragma unroll
  for (int j = 0; j < 8; j++) {
    const u32 xh = j < 7 ? __funnelshift_r(x[10 + j], x[11 + j], 16) : x[17] >> 16;
    const u64 t = (u64)x[j] + xh + cy;
    if (j == 0) s0 = (u32)t;
    cy = t >> 32;
  }
  const u32 cfast = u < w ? 1u : 0u;
  return (cy ? 1u << kRareRanluxCarry : 0u) | (u - w + 1u <= 2u ? 1u << kRareRanluxNear : 0u) |
         (u == 0xFFFFFFFFu ? 1u << kRareRanluxUMax : 0u) | (s0 < cfast ? 1u << kRareRanluxV0 : 0u) |
         (c == 1u && v[0] == s0 ? 1u << kRareRanluxThird : 0u);
}

// D6 (c-5, c-11): draw j of a block = bits [48 j, 48 j + 48) of V, as the double k 2^-48.
// The 48 bits are placed in the mantissa of 2^4 (value 16 + k 2^-48, exact) and 16.0 is
// subtracted (exact): one PRMT or two, one DADD; no int->float conversion instruction.
// kexp = the high word of 16.0 (0x40300000), handed to the kernels as a launch PARAMETER so that it
// sits in a register and the PRMT selectors are immediates: with both as literals ptxas puts the
// selector in a register and re-materialises it for every draw (12 extra instructions per advance).
constexpr u32 kExp16 = 0x40300000u;
template <int J>
__device__ __forceinline__ double draw_double(const u32 (&v)[18], u32 kexp) {
  u32 lo, hi;
  if (J % 2 == 0) {  // bits 48J.. start on a limb boundary: limbs 3J/2, 3J/2 + 1 (low half)
    lo = v[3 * J / 2];
    hi = __byte_perm(v[3 * J / 2 + 1], kexp, 0x7610);
  } else {  // start in the middle of limb (3J - 1)/2
    lo = __byte_perm(v[(3 * J - 1) / 2], v[(3 * J + 1) / 2], 0x5432);
    hi = __byte_perm(v[(3 * J + 1) / 2], kexp, 0x7632);
  }
  return __hiloint2double((int)hi, (int)lo) - 16.0;
}

}  // namespace rlx
