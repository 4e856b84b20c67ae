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

namespace rlx {

typedef uint32_t u32;
typedef uint64_t u64;
typedef int64_t i64;

__host__ __device__ __forceinline__ constexpr u32 m_limb(int j) {
  return j == 0 ? 1u : (j < 7 ? 0u : (j == 7 ? 0xFFFF0000u : 0xFFFFFFFFu));
}
// limbs of 2^240 - 1  (2^576 == 2^240 - 1 mod m)
__host__ __device__ __forceinline__ constexpr u32 k240_limb(int j) {
  return j < 7 ? 0xFFFFFFFFu : (j == 7 ? 0x0000FFFFu : 0u);
}

// ------------------------------------------------------------------ generic product
// multiply9x9 (sec. 2.1) on 32-bit limbs, column by column: "For every 64 bit in the
// output, there are up to 9 contributing pairs ... The lower 64 bits of the sum constitutes
// one entry of the output, while the rest is propagated to the next entry" -- here with
// 32-bit entries and up to 18 pairs per column (device code multiplies 32-bit values).
__device__ __forceinline__ void mul18x18(const u32 (&x)[18], const u32 (&y)[18], u32 (&z)[36]) {
  u64 acc = 0;  // low 64 bits of the running column sum
  u32 ovf = 0;  // bits 64.. of it
#pragma unroll
  for (int k = 0; k < 35; k++) {
#pragma unroll
    for (int i = 0; i < 18; i++) {
      const int j = k - i;
      if (j >= 0 && j < 18) {
        const u64 p = (u64)x[i] * y[j];
        acc += p;
        ovf += (acc < p);  // P:134-137 Listing 4: branch-free carry
      }
    }
    z[k] = (u32)acc;
    acc = (acc >> 32) | ((u64)ovf << 32);
    ovf = 0;
  }
  z[35] = (u32)acc;
}

// x >= m ?
__device__ __forceinline__ bool ge_m(const u32 (&x)[18]) {
  u32 all = x[8];
#pragma unroll
  for (int j = 9; j < 18; j++) all &= x[j];
  u32 low = x[0] | x[1] | x[2] | x[3] | x[4] | x[5] | x[6] | (x[7] & 0xFFFFu);
  return all == 0xFFFFFFFFu && (x[7] >> 16) == 0xFFFFu && low != 0;
}
// x -= m for x in [m, 2^576): the top 336 bits are all ones, so x - m = (x mod 2^240) - 1
__device__ __forceinline__ void sub_m(u32 (&x)[18]) {
  i64 c = -1;
#pragma unroll
  for (int j = 0; j < 8; j++) {
    const i64 s = (i64)(j == 7 ? (x[7] & 0xFFFFu) : x[j]) + c;
    x[j] = (u32)s;
    c = s >> 32;
  }
#pragma unroll
  for (int j = 8; j < 18; j++) x[j] = 0;
}

// mod_m (sec. 2.2): remainder of a 1152-bit value modulo m "using additions,
// subtractions, and bit shifts" plus the "fix to ensure that the result is smaller than m
// in all cases".  Reading c-9:  z = lo + hi 2^576, hi = t1 2^336 + t0, u = t0 + t1,
//   z == lo - hi - t1 + (u mod 2^336) 2^240 + (u >> 336)(2^240 - 1)   (mod m)
// summed limb by limb with a signed carry; the final carry k is folded again as
// k (2^240 - 1), and m is subtracted once if the result is still >= m.
__device__ __forceinline__ void mod_m36(const u32 (&z)[36], u32 (&r)[18]) {
  u32 t1[8];
#pragma unroll
  for (int j = 0; j < 7; j++) t1[j] = (z[28 + j] >> 16) | (z[29 + j] << 16);
  t1[7] = z[35] >> 16;
  u32 u[11];
  u64 c = 0;
#pragma unroll
  for (int j = 0; j < 11; j++) {
    const u64 s = (u64)(j < 10 ? z[18 + j] : (z[28] & 0xFFFFu)) + (j < 8 ? t1[j] : 0u) + c;
    u[j] = (u32)s;
    c = s >> 32;
  }
  const u32 ubit = u[10] >> 16;  // u >> 336
  u[10] &= 0xFFFFu;              // u mod 2^336
  i64 carry = 0;
#pragma unroll
  for (int j = 0; j < 18; j++) {
    u32 ush = 0;  // limb j of (u mod 2^336) << 240
    if (j == 7) ush = u[0] << 16;
    else if (j > 7) ush = (u[j - 7] << 16) | (u[j - 8] >> 16);
    const i64 s = (i64)z[j] - (i64)z[18 + j] - (i64)(j < 8 ? t1[j] : 0u) + (i64)ush +
                  (i64)(ubit ? k240_limb(j) : 0u) + carry;
    r[j] = (u32)s;
    carry = s >> 32;
  }
  // value = r + carry 2^576 == r + carry (2^240 - 1); by the bound in c-9 |carry| <= 1 and one
  // fold suffices; a second pass (normally with 0) keeps this exact even if it did not.
#pragma unroll
  for (int pass = 0; pass < 2; pass++) {
    const i64 k = carry;
    carry = 0;
#pragma unroll
    for (int j = 0; j < 18; j++) {
      const i64 s = (i64)r[j] + k * (i64)k240_limb(j) + carry;
      r[j] = (u32)s;
      carry = s >> 32;
    }
  }
  if (ge_m(r)) sub_m(r);  // the fix: result < m
}

// canonical representative of a 640-bit value given as 20 limbs (what the row-reduced
// product leaves): zero-extend and reduce
__device__ __forceinline__ void mod_m20(const u32 (&z)[20], u32 (&r)[18]) {
  u32 zz[36];
#pragma unroll
  for (int j = 0; j < 36; j++) zz[j] = j < 20 ? z[j] : 0u;
  mod_m36(zz, r);
}

__device__ __forceinline__ void mulmod_generic(const u32 (&x)[18], const u32 (&y)[18], u32 (&r)[18]) {
  u32 z[36];
  mul18x18(x, y, z);
  mod_m36(z, r);
}

// ------------------------------------------------------------------ LCG -> RANLUX numbers
// P:39 (sec. 2.3): "converts the LCG state back to RANLUX numbers".  Reading D4 (c-4), exact:
//   Xh = X >> 336, Xl = X mod 2^336, S = Xl + Xh, D = S 2^240 - S - Xh 2^336 (signed)
//   T = Xh - [D < 0]   (D >= m is impossible: D <= (2^336 - 1)(2^240 - 1) < m)
//   V = X + T,  c = (V >> 336) - T
// X must be canonical (< m).  V = the 24 RANLUX numbers packed, oldest in the low bits.
__device__ __forceinline__ void to_ranlux_exact(const u32 (&x)[18], u32 (&v)[18], u32& c_out) {
  u32 xh[8];
#pragma unroll
  for (int j = 0; j < 7; j++) xh[j] = (x[10 + j] >> 16) | (x[11 + j] << 16);
  xh[7] = x[17] >> 16;
  u32 s[11];  // S = Xl + Xh, up to 337 bits
  u64 c = 0;
#pragma unroll
  for (int j = 0; j < 11; j++) {
    const u64 t = (u64)(j < 10 ? x[j] : (x[10] & 0xFFFFu)) + (j < 8 ? xh[j] : 0u) + c;
    s[j] = (u32)t;
    c = t >> 32;
  }
  // sign of D = (S << 240) - S - (Xh << 336), limbs 0..18
  i64 carry = 0;
#pragma unroll
  for (int j = 0; j < 19; j++) {
    u32 ssh = 0;  // limb j of S << 240
    if (j == 7) ssh = s[0] << 16;
    else if (j > 7 && j < 18) ssh = (s[j - 7] << 16) | (s[j - 8] >> 16);
    else if (j == 18) ssh = s[10] >> 16;
    u32 xsh = 0;  // limb j of Xh << 336 = the bits of X at and above 336
    if (j == 10) xsh = x[10] & 0xFFFF0000u;
    else if (j > 10 && j < 18) xsh = x[j];
    const i64 t = (i64)ssh - (i64)(j < 11 ? s[j] : 0u) - (i64)xsh + carry;
    carry = t >> 32;
  }
  const u32 neg = carry < 0 ? 1u : 0u;  // D < 0
  // V = X + Xh - neg
  i64 cy = -(i64)neg;
#pragma unroll
  for (int j = 0; j < 18; j++) {
    const i64 t = (i64)x[j] + (i64)(j < 8 ? xh[j] : 0u) + cy;
    v[j] = (u32)t;
    cy = t >> 32;
  }
  // c = (V >> 336) - Xh + neg; (V >> 336) - Xh is 0 or 1, so its low limb decides
  const u32 vh0 = (v[10] >> 16) | (v[11] << 16);
  c_out = (vh0 - xh[0]) + neg;
}

// ------------------------------------------------------------------ hot-path fast forms
// Row-reduced product: Z = sum_i x_i R_i < 2^613 arrives as E/O accumulators (see
// rows_generated.cuh).  merge_eo adds the two interleaved sets into 20 limbs.
__device__ __forceinline__ void merge_eo(const u64 (&E)[9], u32 e9, const u64 (&O)[9], u32 o9, u32 (&z)[20]) {
  u32 el[19], ol[19];
#pragma unroll
  for (int w = 0; w < 9; w++) {
    el[2 * w] = (u32)E[w];
    el[2 * w + 1] = (u32)(E[w] >> 32);
    ol[2 * w] = (u32)O[w];
    ol[2 * w + 1] = (u32)(O[w] >> 32);
  }
  el[18] = e9;
  ol[18] = o9;
  z[0] = el[0];
  asm("add.cc.u32 %0, %19, %37;\n\t"
      "addc.cc.u32 %1, %20, %38;\n\t"
      "addc.cc.u32 %2, %21, %39;\n\t"
      "addc.cc.u32 %3, %22, %40;\n\t"
      "addc.cc.u32 %4, %23, %41;\n\t"
      "addc.cc.u32 %5, %24, %42;\n\t"
      "addc.cc.u32 %6, %25, %43;\n\t"
      "addc.cc.u32 %7, %26, %44;\n\t"
      "addc.cc.u32 %8, %27, %45;\n\t"
      "addc.cc.u32 %9, %28, %46;\n\t"
      "addc.cc.u32 %10, %29, %47;\n\t"
      "addc.cc.u32 %11, %30, %48;\n\t"
      "addc.cc.u32 %12, %31, %49;\n\t"
      "addc.cc.u32 %13, %32, %50;\n\t"
      "addc.cc.u32 %14, %33, %51;\n\t"
      "addc.cc.u32 %15, %34, %52;\n\t"
      "addc.cc.u32 %16, %35, %53;\n\t"
      "addc.cc.u32 %17, %36, %54;\n\t"
      "addc.u32 %18, %55, 0;"
      : "=r"(z[1]), "=r"(z[2]), "=r"(z[3]), "=r"(z[4]), "=r"(z[5]), "=r"(z[6]), "=r"(z[7]), "=r"(z[8]), "=r"(z[9]), "=r"(z[10]), "=r"(z[11]), "=r"(z[12]), "=r"(z[13]), "=r"(z[14]), "=r"(z[15]), "=r"(z[16]), "=r"(z[17]), "=r"(z[18]), "=r"(z[19])
      : "r"(el[1]), "r"(el[2]), "r"(el[3]), "r"(el[4]), "r"(el[5]), "r"(el[6]), "r"(el[7]), "r"(el[8]), "r"(el[9]), "r"(el[10]), "r"(el[11]), "r"(el[12]), "r"(el[13]), "r"(el[14]), "r"(el[15]), "r"(el[16]), "r"(el[17]), "r"(el[18]), "r"(ol[0]), "r"(ol[1]), "r"(ol[2]), "r"(ol[3]), "r"(ol[4]), "r"(ol[5]), "r"(ol[6]), "r"(ol[7]), "r"(ol[8]), "r"(ol[9]), "r"(ol[10]), "r"(ol[11]), "r"(ol[12]), "r"(ol[13]), "r"(ol[14]), "r"(ol[15]), "r"(ol[16]), "r"(ol[17]), "r"(ol[18]));
}

// Fast fold of z (20 limbs, hi = z[18] + z[19] 2^32 < 2^37) to x = z mod 2^576 - hi + hi 2^240.
// Exact iff `rare` stays 0:  rare is raised when the borrow of "- hi" leaves limb 1, when the
// carry of "+ hi 2^240" leaves limb 9, or when the top limb is all ones (x might be >= m).
__device__ __forceinline__ void fold_fast(const u32 (&z)[20], u32 (&x)[18], u32& rare) {
  const u32 h0 = z[18], h1 = z[19];
  const u32 s0 = h0 << 16;
  const u32 s1 = __funnelshift_l(h0, h1, 16);  // bits 16..47 of hi
  const u32 s2 = h1 >> 16;
  u32 brw, cry;
  asm("sub.cc.u32 %0, %3, %5;\n\t"
      "subc.cc.u32 %1, %4, %6;\n\t"
      "subc.u32 %2, 0, 0;"
      : "=r"(x[0]), "=r"(x[1]), "=r"(brw)
      : "r"(z[0]), "r"(z[1]), "r"(h0), "r"(h1));
  asm("add.cc.u32 %0, %4, %7;\n\t"
      "addc.cc.u32 %1, %5, %8;\n\t"
      "addc.cc.u32 %2, %6, %9;\n\t"
      "addc.u32 %3, 0, 0;"
      : "=r"(x[7]), "=r"(x[8]), "=r"(x[9]), "=r"(cry)
      : "r"(z[7]), "r"(z[8]), "r"(z[9]), "r"(s0), "r"(s1), "r"(s2));
#pragma unroll
  for (int j = 2; j < 7; j++) x[j] = z[j];
#pragma unroll
  for (int j = 10; j < 18; j++) x[j] = z[j];
  // borrow out of limb 1 is harmless only if it is absorbed below limb 7: we do not track
  // that here -- any borrow or carry goes to the exact path.
  rare |= brw | cry | (x[17] == 0xFFFFFFFFu ? 1u : 0u);
}

// Fast to_ranlux.  With u = bits 304..335 of X and w = bits 544..575 of X (the leading
// 32 bits of the middle and of the top 240-bit field):
//   u >= w + 2 and u != 2^32 - 1  =>  D > 0, no overflow of Xl + Xh:  V = X + Xh,     c = 0
//   u + 2 <= w                    =>  D < 0:                          V = X + Xh - 1, c = 1
// (derivation in DESIGN.md).  Otherwise, or if the 8-limb addition carries out of limb 7,
// or if the "- c" would borrow, `rare` is raised.  Limbs 8..17 of V equal those of X.
__device__ __forceinline__ void to_ranlux_fast(const u32 (&x)[18], u32 (&v)[18], u32& c_out, u32& rare) {
  const u32 u = __funnelshift_r(x[9], x[10], 16);
  const u32 w = x[17];
  const u32 c = u < w ? 1u : 0u;
  const u32 d = u - w + 1u;  // in {0, 1, 2}  <=>  |u - w| <= 1
  u32 xh[8];
#pragma unroll
  for (int j = 0; j < 7; j++) xh[j] = __funnelshift_r(x[10 + j], x[11 + j], 16);
  xh[7] = x[17] >> 16;
  u32 cry;
  asm("add.cc.u32 %0, %9, %17;\n\t"
      "addc.cc.u32 %1, %10, %18;\n\t"
      "addc.cc.u32 %2, %11, %19;\n\t"
      "addc.cc.u32 %3, %12, %20;\n\t"
      "addc.cc.u32 %4, %13, %21;\n\t"
      "addc.cc.u32 %5, %14, %22;\n\t"
      "addc.cc.u32 %6, %15, %23;\n\t"
      "addc.cc.u32 %7, %16, %24;\n\t"
      "addc.u32 %8, 0, 0;"
      : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(cry)
      : "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]), "r"(x[6]), "r"(x[7]), "r"(xh[0]),
        "r"(xh[1]), "r"(xh[2]), "r"(xh[3]), "r"(xh[4]), "r"(xh[5]), "r"(xh[6]), "r"(xh[7]));
  rare |= cry | (d <= 2u ? 1u : 0u) | (u == 0xFFFFFFFFu ? 1u : 0u) | (v[0] < c ? 1u : 0u);
  v[0] -= c;
#pragma unroll
  for (int j = 8; j < 18; j++) v[j] = x[j];
  c_out = c;
}

// D6 (c-5, c-11): draw j of a block = bits [48 j, 48 j + 48) of V, as the double k 2^-48.
// The 48 bits are placed in the mantissa of 2^4 (value 16 + k 2^-48, exact) and 16.0 is
// subtracted (exact): one PRMT or two, one DADD; no int->float conversion instruction.
template <int J>
__device__ __forceinline__ double draw_double(const u32 (&v)[18]) {
  u32 lo, hi;
  if (J % 2 == 0) {  // bits 48J.. start on a limb boundary: limbs 3J/2, 3J/2 + 1 (low half)
    lo = v[3 * J / 2];
    hi = __byte_perm(v[3 * J / 2 + 1], 0x40300000u, 0x7610);
  } else {  // start in the middle of limb (3J - 1)/2
    lo = __byte_perm(v[(3 * J - 1) / 2], v[(3 * J + 1) / 2], 0x5432);
    hi = __byte_perm(v[(3 * J + 1) / 2], 0x40300000u, 0x7632);
  }
  return __hiloint2double((int)hi, (int)lo) - 16.0;
}

}  // namespace rlx
