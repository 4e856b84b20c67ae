// rlxpp_device.cuh -- header-only DEVICE API of RANLUX++ for use inside your own CUDA kernels
// (the paper's GPU use is "one state per thread", every
// thread drawing numbers where it needs them).
//
//   #include "rlxpp_device.cuh"
//   __global__ void my_kernel(rlxpp_view_t view, ...) {
//     rlxpp_dev::Stream g;
//     g.load(view, i);                 // stream i of a handle made by rlxpp_create (rlxpp_device_view)
//     double u = g.draw_coop();        // or g.draw(); next double in [0, 1) on the 2^-48 lattice
//     ...
//     g.store(view, i);                // the handle can go on with rlxpp_generate_* / rlxpp_get_state
//   }
//
// The sequence is the one rlxpp_generate_doubles produces for the same stream (same cursor
// semantics, reading D8): draws made here and draws made by the library interleave freely.
//
// draw():      the paper's scheme -- a thread advances its LCG state when its own block of 12 draws is used
//              up.  Threads of a warp whose cursors differ then advance at different calls and the warp
//              pays for up to 12 advances per 12 draws (the "7x slower" of PAPER.md line 176).
// draw_coop(): warp-cooperative.  Every lane of the (converged) warp calls it together.  When ANY lane has
//              used up its block and holds no spare one, EVERY lane without a spare computes its next
//              block in the same pass (state and spare block live in local memory / registers).  Each
//              lane uses its spare when its own block runs out, so the warp pays one advance pass per
//              12 draws per lane whatever the cursors are.
// The two mix freely on one Stream (draw_coop() in converged code, draw() inside a divergent branch): draw()
// enters a spare block that draw_coop() has made instead of advancing again.
//
// The advance here is the paper's own formulation (multiply9x9, then mod_m) on 32-bit
// limbs with the multiplier a^p as 18 runtime limbs, any luxury level p.  (The library's bulk kernels
// use a tensor-core formulation that needs a CTA per 128 streams; this header needs nothing but the
// calling thread.)
#ifndef RLXPP_DEVICE_CUH
#define RLXPP_DEVICE_CUH
#include <cuda_runtime.h>
#include <stdint.h>

/* What rlxpp_device_view() fills in (include/rlxpp.h).  Plain device pointers, owned by the handle. */
typedef struct rlxpp_view {
  uint4* st;          /* state planes: st[g * n + i], g = 0..4 (limbs 4g..4g+3; plane 4: limbs 16, 17, pos, 0) */
  uint64_t n;         /* streams in the handle */
  const uint32_t* A;  /* the 18 little-endian 32-bit limbs of a^p mod m */
  const uint4* bmat;  /* shared-memory image of the byte matrix of a^p (rlxpp_tile.cuh: TileStream) */
} rlxpp_view_t;

namespace rlxpp_dev {
namespace detail {

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
// multiply9x9 (sec. 2.1): the 1152-bit schoolbook product, here on 32-bit limbs
// (device code multiplies 32-bit values): 18 x 18 = 324 products 32x32->64.
// Row by row with two interleaved sets of 64-bit accumulators, E[w] at 32-bit columns (2w, 2w + 1)
// and O[w] at columns (2w + 1, 2w + 2): the product x_i y_j belongs to column i + j, so row i feeds
// nine consecutive accumulators of each set through one carry chain (ptxas fuses every
// mul.wide.u32 + add(c).cc.u64 into ONE IMAD.WIDE.U32.X: 324 instructions for the 324 products).
// After rows 0..i each set is < 2^(32 (i + 19)): the carry out of a chain either lands in an
// accumulator that holds less than 2^32 (added, cannot overflow) or is zero (chain already ends at
// that bound) -- no carry ever ripples further.
template <int I, bool ODD>  // one chain of row I: the products at even (ODD = false) or odd columns
struct MulChain {
  static constexpr int kJ0 = ODD ? ((I + 1) & 1) : (I & 1);  // first j of the chain (j advances by 2)
  static constexpr int kW0 = ODD ? (I + kJ0 - 1) / 2 : (I + kJ0) / 2;
  static constexpr bool kTail = kJ0 == 0;                     // carry out goes to accumulator kW0 + 9
  static __device__ __forceinline__ void run(u64 (&acc)[18], u32 xi, const u32 (&y)[18]) {
    if (kTail) {
      asm("{\n\t.reg .u64 t;\n\t"
          "mul.wide.u32 t, %10, %11; add.cc.u64  %0, %0, t;\n\t"
          "mul.wide.u32 t, %10, %12; addc.cc.u64 %1, %1, t;\n\t"
          "mul.wide.u32 t, %10, %13; addc.cc.u64 %2, %2, t;\n\t"
          "mul.wide.u32 t, %10, %14; addc.cc.u64 %3, %3, t;\n\t"
          "mul.wide.u32 t, %10, %15; addc.cc.u64 %4, %4, t;\n\t"
          "mul.wide.u32 t, %10, %16; addc.cc.u64 %5, %5, t;\n\t"
          "mul.wide.u32 t, %10, %17; addc.cc.u64 %6, %6, t;\n\t"
          "mul.wide.u32 t, %10, %18; addc.cc.u64 %7, %7, t;\n\t"
          "mul.wide.u32 t, %10, %19; addc.cc.u64 %8, %8, t;\n\t"
          "addc.u64 %9, %9, 0;\n\t"
          "}"
          : "+l"(acc[kW0]), "+l"(acc[kW0 + 1]), "+l"(acc[kW0 + 2]), "+l"(acc[kW0 + 3]), "+l"(acc[kW0 + 4]),
            "+l"(acc[kW0 + 5]), "+l"(acc[kW0 + 6]), "+l"(acc[kW0 + 7]), "+l"(acc[kW0 + 8]),
            "+l"(acc[kW0 + 9 < 18 ? kW0 + 9 : 17])
          : "r"(xi), "r"(y[kJ0]), "r"(y[kJ0 + 2]), "r"(y[kJ0 + 4]), "r"(y[kJ0 + 6]), "r"(y[kJ0 + 8]), "r"(y[kJ0 + 10]),
            "r"(y[kJ0 + 12]), "r"(y[kJ0 + 14]), "r"(y[kJ0 + 16]));
    } else {
      asm("{\n\t.reg .u64 t;\n\t"
          "mul.wide.u32 t, %9, %10; add.cc.u64  %0, %0, t;\n\t"
          "mul.wide.u32 t, %9, %11; addc.cc.u64 %1, %1, t;\n\t"
          "mul.wide.u32 t, %9, %12; addc.cc.u64 %2, %2, t;\n\t"
          "mul.wide.u32 t, %9, %13; addc.cc.u64 %3, %3, t;\n\t"
          "mul.wide.u32 t, %9, %14; addc.cc.u64 %4, %4, t;\n\t"
          "mul.wide.u32 t, %9, %15; addc.cc.u64 %5, %5, t;\n\t"
          "mul.wide.u32 t, %9, %16; addc.cc.u64 %6, %6, t;\n\t"
          "mul.wide.u32 t, %9, %17; addc.cc.u64 %7, %7, t;\n\t"
          "mul.wide.u32 t, %9, %18; addc.u64    %8, %8, t;\n\t"
          "}"
          : "+l"(acc[kW0]), "+l"(acc[kW0 + 1]), "+l"(acc[kW0 + 2]), "+l"(acc[kW0 + 3]), "+l"(acc[kW0 + 4]),
            "+l"(acc[kW0 + 5]), "+l"(acc[kW0 + 6]), "+l"(acc[kW0 + 7]), "+l"(acc[kW0 + 8])
          : "r"(xi), "r"(y[kJ0]), "r"(y[kJ0 + 2]), "r"(y[kJ0 + 4]), "r"(y[kJ0 + 6]), "r"(y[kJ0 + 8]), "r"(y[kJ0 + 10]),
            "r"(y[kJ0 + 12]), "r"(y[kJ0 + 14]), "r"(y[kJ0 + 16]));
    }
  }
};
template <int I>
struct MulRows {
  static __device__ __forceinline__ void run(u64 (&E)[18], u64 (&O)[18], const u32 (&x)[18], const u32 (&y)[18]) {
    MulChain<I, false>::run(E, x[I], y);
    MulChain<I, true>::run(O, x[I], y);
    MulRows<I + 1>::run(E, O, x, y);
  }
};
template <>
struct MulRows<18> {
  static __device__ __forceinline__ void run(u64 (&)[18], u64 (&)[18], const u32 (&)[18], const u32 (&)[18]) {}
};

__device__ __forceinline__ void mul18x18(const u32 (&x)[18], const u32 (&y)[18], u32 (&z)[36]) {
  u64 E[18], O[18];
#pragma unroll
  for (int w = 0; w < 18; w++) { E[w] = 0; O[w] = 0; }
  MulRows<0>::run(E, O, x, y);
  // Z = E + (O << 32): T[w] = columns (2w, 2w + 1) of O << 32 = (high half of O[w - 1], low half of O[w])
  u64 T[18], Z[18];
  T[0] = O[0] << 32;
#pragma unroll
  for (int w = 1; w < 18; w++) T[w] = (O[w - 1] >> 32) | (O[w] << 32);
  asm("add.cc.u64 %0, %18, %36;\n\t"
      "addc.cc.u64 %1, %19, %37;\n\t"
      "addc.cc.u64 %2, %20, %38;\n\t"
      "addc.cc.u64 %3, %21, %39;\n\t"
      "addc.cc.u64 %4, %22, %40;\n\t"
      "addc.cc.u64 %5, %23, %41;\n\t"
      "addc.cc.u64 %6, %24, %42;\n\t"
      "addc.cc.u64 %7, %25, %43;\n\t"
      "addc.cc.u64 %8, %26, %44;\n\t"
      "addc.cc.u64 %9, %27, %45;\n\t"
      "addc.cc.u64 %10, %28, %46;\n\t"
      "addc.cc.u64 %11, %29, %47;\n\t"
      "addc.cc.u64 %12, %30, %48;\n\t"
      "addc.cc.u64 %13, %31, %49;\n\t"
      "addc.cc.u64 %14, %32, %50;\n\t"
      "addc.cc.u64 %15, %33, %51;\n\t"
      "addc.cc.u64 %16, %34, %52;\n\t"
      "addc.u64 %17, %35, %53;"
      : "=l"(Z[0]), "=l"(Z[1]), "=l"(Z[2]), "=l"(Z[3]), "=l"(Z[4]), "=l"(Z[5]), "=l"(Z[6]), "=l"(Z[7]), "=l"(Z[8]),
        "=l"(Z[9]), "=l"(Z[10]), "=l"(Z[11]), "=l"(Z[12]), "=l"(Z[13]), "=l"(Z[14]), "=l"(Z[15]), "=l"(Z[16]), "=l"(Z[17])
      : "l"(E[0]), "l"(E[1]), "l"(E[2]), "l"(E[3]), "l"(E[4]), "l"(E[5]), "l"(E[6]), "l"(E[7]), "l"(E[8]), "l"(E[9]),
        "l"(E[10]), "l"(E[11]), "l"(E[12]), "l"(E[13]), "l"(E[14]), "l"(E[15]), "l"(E[16]), "l"(E[17]), "l"(T[0]),
        "l"(T[1]), "l"(T[2]), "l"(T[3]), "l"(T[4]), "l"(T[5]), "l"(T[6]), "l"(T[7]), "l"(T[8]), "l"(T[9]), "l"(T[10]),
        "l"(T[11]), "l"(T[12]), "l"(T[13]), "l"(T[14]), "l"(T[15]), "l"(T[16]), "l"(T[17]));
#pragma unroll
  for (int w = 0; w < 18; w++) {
    z[2 * w] = (u32)Z[w];
    z[2 * w + 1] = (u32)(Z[w] >> 32);
  }
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

// value = r + k 2^576 (k small, signed)  ->  r + k (2^240 - 1), returned again as (r, new k).
// k (2^240 - 1) as an 18-limb two's-complement constant: limb 0 = -k, limbs 1..6 = all ones if k > 0,
// limb 7 = (k << 16) - [k > 0], limbs 8..17 = all ones if k < 0 (sign extension).
__device__ __forceinline__ int fold_carry(u32 (&r)[18], int k) {
  const u32 c0 = (u32)(-k), sp = k > 0 ? 0xFFFFFFFFu : 0u, c7 = ((u32)k << 16) - (k > 0 ? 1u : 0u),
            ng = k < 0 ? 0xFFFFFFFFu : 0u;
  u32 cout;
  asm(
      "add.cc.u32 %0, %0, %19;\n\t"
      "addc.cc.u32 %1, %1, %20;\n\t"
      "addc.cc.u32 %2, %2, %20;\n\t"
      "addc.cc.u32 %3, %3, %20;\n\t"
      "addc.cc.u32 %4, %4, %20;\n\t"
      "addc.cc.u32 %5, %5, %20;\n\t"
      "addc.cc.u32 %6, %6, %20;\n\t"
      "addc.cc.u32 %7, %7, %21;\n\t"
      "addc.cc.u32 %8, %8, %22;\n\t"
      "addc.cc.u32 %9, %9, %22;\n\t"
      "addc.cc.u32 %10, %10, %22;\n\t"
      "addc.cc.u32 %11, %11, %22;\n\t"
      "addc.cc.u32 %12, %12, %22;\n\t"
      "addc.cc.u32 %13, %13, %22;\n\t"
      "addc.cc.u32 %14, %14, %22;\n\t"
      "addc.cc.u32 %15, %15, %22;\n\t"
      "addc.cc.u32 %16, %16, %22;\n\t"
      "addc.cc.u32 %17, %17, %22;\n\t"
      "addc.u32 %18, 0, 0;"
      : "+r"(r[0]), "+r"(r[1]), "+r"(r[2]), "+r"(r[3]), "+r"(r[4]), "+r"(r[5]), "+r"(r[6]), "+r"(r[7]), "+r"(r[8]), "+r"(r[9]), "+r"(r[10]), "+r"(r[11]), "+r"(r[12]), "+r"(r[13]), "+r"(r[14]), "+r"(r[15]), "+r"(r[16]), "+r"(r[17]), "=r"(cout)
      : "r"(c0), "r"(sp), "r"(c7), "r"(ng));
  return (int)cout - (k < 0 ? 1 : 0);
}

// mod_m (sec. 2.2): remainder of a 1152-bit value modulo m "using additions,
// subtractions, and bit shifts" plus the "fix to ensure that the result is smaller than m
// in all cases".  Reading c-9:  z = lo + hi 2^576, hi = t1 2^336 + t0, u = t0 + t1 (337 bits),
//   z == lo + u 2^240 - hi - t1   (mod m)        [hi 2^576 == hi (2^240 - 1), t1 2^576 likewise]
// evaluated as P - N with P = lo + u 2^240 and N = hi + t1 (19 limbs each, PTX carry chains); what
// lies above 2^576 is a small signed k, folded again as k (2^240 - 1); m is subtracted once if the
// result is still >= m.
__device__ __forceinline__ void mod_m36(const u32 (&z)[36], u32 (&r)[18]) {
  u32 t1[8];  // hi >> 336
#pragma unroll
  for (int j = 0; j < 7; j++) t1[j] = __funnelshift_r(z[28 + j], z[29 + j], 16);
  t1[7] = z[35] >> 16;
  u32 u[11];  // u = t0 + t1 < 2^337 (u[10] < 2^17)
  asm(
      "add.cc.u32 %0, %11, %22;\n\t"
      "addc.cc.u32 %1, %12, %23;\n\t"
      "addc.cc.u32 %2, %13, %24;\n\t"
      "addc.cc.u32 %3, %14, %25;\n\t"
      "addc.cc.u32 %4, %15, %26;\n\t"
      "addc.cc.u32 %5, %16, %27;\n\t"
      "addc.cc.u32 %6, %17, %28;\n\t"
      "addc.cc.u32 %7, %18, %29;\n\t"
      "addc.cc.u32 %8, %19, 0;\n\t"
      "addc.cc.u32 %9, %20, 0;\n\t"
      "addc.u32 %10, %21, 0;"
      : "=r"(u[0]), "=r"(u[1]), "=r"(u[2]), "=r"(u[3]), "=r"(u[4]), "=r"(u[5]), "=r"(u[6]), "=r"(u[7]), "=r"(u[8]), "=r"(u[9]), "=r"(u[10])
      : "r"(z[18]), "r"(z[19]), "r"(z[20]), "r"(z[21]), "r"(z[22]), "r"(z[23]), "r"(z[24]), "r"(z[25]), "r"(z[26]), "r"(z[27]), "r"(z[28] & 0xFFFFu), "r"(t1[0]), "r"(t1[1]), "r"(t1[2]), "r"(t1[3]), "r"(t1[4]), "r"(t1[5]), "r"(t1[6]), "r"(t1[7]));
  // P = lo + u 2^240 (19 limbs: limbs 0..6 are lo's), N = hi + t1 (19 limbs)
  u32 ush[12];  // limbs 7..18 of u << 240
  ush[0] = u[0] << 16;
#pragma unroll
  for (int j = 1; j < 11; j++) ush[j] = __funnelshift_l(u[j - 1], u[j], 16);
  ush[11] = u[10] >> 16;
  u32 pp[18], p18, nn[18], n18, bw;
#pragma unroll
  for (int j = 0; j < 7; j++) pp[j] = z[j];
  asm(
      "add.cc.u32 %0, %12, %23;\n\t"
      "addc.cc.u32 %1, %13, %24;\n\t"
      "addc.cc.u32 %2, %14, %25;\n\t"
      "addc.cc.u32 %3, %15, %26;\n\t"
      "addc.cc.u32 %4, %16, %27;\n\t"
      "addc.cc.u32 %5, %17, %28;\n\t"
      "addc.cc.u32 %6, %18, %29;\n\t"
      "addc.cc.u32 %7, %19, %30;\n\t"
      "addc.cc.u32 %8, %20, %31;\n\t"
      "addc.cc.u32 %9, %21, %32;\n\t"
      "addc.cc.u32 %10, %22, %33;\n\t"
      "addc.u32 %11, %34, 0;"
      : "=r"(pp[7]), "=r"(pp[8]), "=r"(pp[9]), "=r"(pp[10]), "=r"(pp[11]), "=r"(pp[12]), "=r"(pp[13]), "=r"(pp[14]), "=r"(pp[15]), "=r"(pp[16]), "=r"(pp[17]), "=r"(p18)
      : "r"(z[7]), "r"(z[8]), "r"(z[9]), "r"(z[10]), "r"(z[11]), "r"(z[12]), "r"(z[13]), "r"(z[14]), "r"(z[15]), "r"(z[16]), "r"(z[17]), "r"(ush[0]), "r"(ush[1]), "r"(ush[2]), "r"(ush[3]), "r"(ush[4]), "r"(ush[5]), "r"(ush[6]), "r"(ush[7]), "r"(ush[8]), "r"(ush[9]), "r"(ush[10]), "r"(ush[11]));
  asm(
      "add.cc.u32 %0, %19, %37;\n\t"
      "addc.cc.u32 %1, %20, %38;\n\t"
      "addc.cc.u32 %2, %21, %39;\n\t"
      "addc.cc.u32 %3, %22, %40;\n\t"
      "addc.cc.u32 %4, %23, %41;\n\t"
      "addc.cc.u32 %5, %24, %42;\n\t"
      "addc.cc.u32 %6, %25, %43;\n\t"
      "addc.cc.u32 %7, %26, %44;\n\t"
      "addc.cc.u32 %8, %27, 0;\n\t"
      "addc.cc.u32 %9, %28, 0;\n\t"
      "addc.cc.u32 %10, %29, 0;\n\t"
      "addc.cc.u32 %11, %30, 0;\n\t"
      "addc.cc.u32 %12, %31, 0;\n\t"
      "addc.cc.u32 %13, %32, 0;\n\t"
      "addc.cc.u32 %14, %33, 0;\n\t"
      "addc.cc.u32 %15, %34, 0;\n\t"
      "addc.cc.u32 %16, %35, 0;\n\t"
      "addc.cc.u32 %17, %36, 0;\n\t"
      "addc.u32 %18, 0, 0;"
      : "=r"(nn[0]), "=r"(nn[1]), "=r"(nn[2]), "=r"(nn[3]), "=r"(nn[4]), "=r"(nn[5]), "=r"(nn[6]), "=r"(nn[7]), "=r"(nn[8]), "=r"(nn[9]), "=r"(nn[10]), "=r"(nn[11]), "=r"(nn[12]), "=r"(nn[13]), "=r"(nn[14]), "=r"(nn[15]), "=r"(nn[16]), "=r"(nn[17]), "=r"(n18)
      : "r"(z[18]), "r"(z[19]), "r"(z[20]), "r"(z[21]), "r"(z[22]), "r"(z[23]), "r"(z[24]), "r"(z[25]), "r"(z[26]), "r"(z[27]), "r"(z[28]), "r"(z[29]), "r"(z[30]), "r"(z[31]), "r"(z[32]), "r"(z[33]), "r"(z[34]), "r"(z[35]), "r"(t1[0]), "r"(t1[1]), "r"(t1[2]), "r"(t1[3]), "r"(t1[4]), "r"(t1[5]), "r"(t1[6]), "r"(t1[7]));
  asm(
      "sub.cc.u32 %0, %19, %37;\n\t"
      "subc.cc.u32 %1, %20, %38;\n\t"
      "subc.cc.u32 %2, %21, %39;\n\t"
      "subc.cc.u32 %3, %22, %40;\n\t"
      "subc.cc.u32 %4, %23, %41;\n\t"
      "subc.cc.u32 %5, %24, %42;\n\t"
      "subc.cc.u32 %6, %25, %43;\n\t"
      "subc.cc.u32 %7, %26, %44;\n\t"
      "subc.cc.u32 %8, %27, %45;\n\t"
      "subc.cc.u32 %9, %28, %46;\n\t"
      "subc.cc.u32 %10, %29, %47;\n\t"
      "subc.cc.u32 %11, %30, %48;\n\t"
      "subc.cc.u32 %12, %31, %49;\n\t"
      "subc.cc.u32 %13, %32, %50;\n\t"
      "subc.cc.u32 %14, %33, %51;\n\t"
      "subc.cc.u32 %15, %34, %52;\n\t"
      "subc.cc.u32 %16, %35, %53;\n\t"
      "subc.cc.u32 %17, %36, %54;\n\t"
      "subc.u32 %18, 0, 0;"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(bw)
      : "r"(pp[0]), "r"(pp[1]), "r"(pp[2]), "r"(pp[3]), "r"(pp[4]), "r"(pp[5]), "r"(pp[6]), "r"(pp[7]), "r"(pp[8]), "r"(pp[9]), "r"(pp[10]), "r"(pp[11]), "r"(pp[12]), "r"(pp[13]), "r"(pp[14]), "r"(pp[15]), "r"(pp[16]), "r"(pp[17]), "r"(nn[0]), "r"(nn[1]), "r"(nn[2]), "r"(nn[3]), "r"(nn[4]), "r"(nn[5]), "r"(nn[6]), "r"(nn[7]), "r"(nn[8]), "r"(nn[9]), "r"(nn[10]), "r"(nn[11]), "r"(nn[12]), "r"(nn[13]), "r"(nn[14]), "r"(nn[15]), "r"(nn[16]), "r"(nn[17]));
  // z == r + k 2^576 with k = p18 - n18 - borrow in [-2, 2];  2^576 == 2^240 - 1:  fold k, then the
  // carry of that fold (|k'| <= 1; by the bound in c-9 a second fold leaves none)
  int k = (int)p18 - (int)n18 - (int)(bw & 1u);
  k = fold_carry(r, k);
  if (k != 0) k = fold_carry(r, k);
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
// Row-reduced product of a FIXED multiplier (include/rlxpp_rows.cuh): Z = sum_i x_i R_i < 2^613 arrives as two
// interleaved sets of 64-bit accumulators E / O; merge_eo adds them into 20 limbs.
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

// mod_m and to_ranlux as the hot paths run them: the overwhelmingly likely case, a `rare` flag otherwise;
// the caller then recomputes with the exact functions above (mod_m20, to_ranlux_exact).
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

}  // namespace detail

// The multiplier rows of a luxury level baked into the instruction stream: defined by include/rlxpp_rows.cuh for
// P in {24, 389, 1024, 2048} (include it after this header to use StreamT<P> with P != 0).
template <int P>
struct FixedMultiplier;

// P = 0 (rlxpp_dev::Stream): the multiplier a^p is read from the view at run time, any luxury level: the paper's
// multiply9x9 + mod_m.  P != 0: the luxury level is fixed at compile time and MUST be the handle's; the 324 products
// take the pre-reduced rows of include/rlxpp_rows.cuh as immediates and mod_m shrinks to a 37-bit fold.
template <int P = 0>
class StreamT {
 public:
  // Stream i of the handle behind `view`.
  __device__ __forceinline__ void load(const rlxpp_view_t& view, uint64_t i) {
#pragma unroll
    for (int g = 0; g < 4; g++) {
      const uint4 q = __ldcg(view.st + (uint64_t)g * view.n + i);
      x_[4 * g] = q.x; x_[4 * g + 1] = q.y; x_[4 * g + 2] = q.z; x_[4 * g + 3] = q.w;
    }
    const uint4 q = __ldcg(view.st + 4 * view.n + i);
    x_[16] = q.x; x_[17] = q.y;
    pos_ = q.z > 12u ? 12u : q.z;
    if (P == 0) {
#pragma unroll
      for (int j = 0; j < 18; j++) a_[j] = __ldg(view.A + j);
    }
    spare_ = 0;
    if (pos_ < 12u) {  // draws left in the current block: rebuild it from the state
      uint32_t c;
      detail::to_ranlux_exact(x_, v_, c);
    }
  }
  // Writes (state of the current block, cursor) back; a spare block that was computed but not yet
  // entered is dropped (it is recomputed from the state when needed again).
  __device__ __forceinline__ void store(const rlxpp_view_t& view, uint64_t i) const {
#pragma unroll
    for (int g = 0; g < 4; g++)
      view.st[(uint64_t)g * view.n + i] = make_uint4(x_[4 * g], x_[4 * g + 1], x_[4 * g + 2], x_[4 * g + 3]);
    view.st[4 * view.n + i] = make_uint4(x_[16], x_[17], pos_, 0u);
  }

  // Next 48-bit integer of the stream (reading D6), per-thread advance.
  __device__ __forceinline__ uint64_t draw_u48() {
    if (pos_ == 12u) {
      if (spare_) {  // draw_coop() already made the next block: enter it (draw and draw_coop mix freely)
#pragma unroll
        for (int j = 0; j < 18; j++) { x_[j] = xs_[j]; v_[j] = vs_[j]; }
        spare_ = 0;
      } else {
        advance(x_, v_);
      }
      pos_ = 0;
    }
    return take();
  }
  __device__ __forceinline__ double draw() { return to_double(draw_u48()); }

  // Warp-cooperative: all lanes named in `mask` call it together (default: the full warp).
  __device__ __forceinline__ uint64_t draw_u48_coop(unsigned mask = 0xFFFFFFFFu) {
    const bool starving = pos_ == 12u && !spare_;
    if (__any_sync(mask, starving)) {
      if (!spare_) {  // x_ is the state of the current block; the spare block's state goes to xs_
#pragma unroll
        for (int j = 0; j < 18; j++) xs_[j] = x_[j];
        advance(xs_, vs_);
        spare_ = 1;
      }
    }
    if (pos_ == 12u) {  // enter the spare block (it exists: either older, or made just now)
#pragma unroll
      for (int j = 0; j < 18; j++) { x_[j] = xs_[j]; v_[j] = vs_[j]; }
      spare_ = 0;
      pos_ = 0;
    }
    return take();
  }
  __device__ __forceinline__ double draw_coop(unsigned mask = 0xFFFFFFFFu) { return to_double(draw_u48_coop(mask)); }

  __device__ __forceinline__ uint32_t cursor() const { return pos_; }

  // k 2^-48, exact (48 <= 53 mantissa bits)
  static __device__ __forceinline__ double to_double(uint64_t k) { return (double)(long long)k * 0x1p-48; }

 private:
  // x <- A x mod m, v <- the 24 RANLUX numbers of the new state
  __device__ __forceinline__ void advance(uint32_t (&x)[18], uint32_t (&v)[18]) const {
    uint32_t c;
    if constexpr (P != 0) {
      uint64_t E[9], O[9];
      uint32_t e9, o9, z[20], r[18], rf = 0;
      FixedMultiplier<P>::mul(x, E, e9, O, o9);
      detail::merge_eo(E, e9, O, o9, z);
      detail::fold_fast(z, r, rf);
      if (__builtin_expect(rf != 0, 0)) detail::mod_m20(z, r);
#pragma unroll
      for (int j = 0; j < 18; j++) x[j] = r[j];
    } else {
      uint32_t r[18];
      detail::mulmod_generic(x, a_, r);
#pragma unroll
      for (int j = 0; j < 18; j++) x[j] = r[j];
    }
    uint32_t rare = 0;
    detail::to_ranlux_fast(x, v, c, rare);  // decides the carry from two leading words; exact form otherwise (~2^-16)
    if (__builtin_expect(rare != 0, 0)) detail::to_ranlux_exact(x, v, c);
  }
  // draw number pos_ of the current block: bits [48 pos, 48 pos + 48) of V.  v_[w] with a run-time w keeps the block in
  // local memory (L1-resident: 18 stores per advance, two loads per draw).  A 12-way switch with compile-time indices
  // keeps it in registers (0 bytes of stack) but measured SLOWER in round 3: aligned draw 245 -> 233, draw_coop
  // 209 -> 186, draw_coop with random cursors 116 -> 76 G doubles/s (up to 30 more registers, and the switch diverges
  // when the cursors differ) -- the indexed form stays.
  __device__ __forceinline__ uint64_t take() {
    const uint32_t w = (3u * pos_) >> 1;  // 32-bit word holding bit 48 pos
    uint64_t k;
    if (pos_ & 1u) k = ((uint64_t)v_[w] >> 16) | ((uint64_t)v_[w + 1] << 16);
    else k = (uint64_t)v_[w] | ((uint64_t)(v_[w + 1] & 0xFFFFu) << 32);
    pos_++;
    return k;
  }

  uint32_t x_[18];   // LCG state of the current block
  uint32_t v_[18];   // current block: packed RANLUX numbers
  uint32_t xs_[18];  // spare block (draw_coop): its state ...
  uint32_t vs_[18];  // ... and its numbers
  uint32_t a_[18];   // a^p (P = 0 only)
  uint32_t pos_;     // draws already taken from the current block, 0..12
  uint32_t spare_;
};
typedef StreamT<0> Stream;

}  // namespace rlxpp_dev
#endif  // RLXPP_DEVICE_CUH
