// Cold kernels and probes: seeding, skip-ahead, state export / import, the ragged kernels written with the public device headers, roofline probes.
// Part of librlxpp (included by rlxpp.cu, one translation unit); see DESIGN.md 5.
#pragma once

#include "state.cuh"
#include "kernels_imad.cuh"  // load_raw / store_raw: the AoS stage of the raw states

namespace rlx {

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

// get_state: the paper's stored form: packed RANLUX numbers + carry, cursor, LCG state.  The [n][9] uint64 arrays
// are AoS with a 72-byte stride per stream: 16-byte aligned arrays go through the raw-state stage of kernels_imad.cuh (the
// CTA's 128 states are 9,216 contiguous bytes: 128-bit coalesced accesses, each thread picks up its 72 bytes in shared
// memory); other alignments keep the direct per-thread accesses.
__device__ __forceinline__ bool aligned16(const void* p) { return (reinterpret_cast<uintptr_t>(p) & 15u) == 0; }
__device__ __forceinline__ void store_u64x9(u64* __restrict__ dst, u64 i, const u32 (&w)[18]) {
#pragma unroll
  for (int l = 0; l < 9; l++) dst[i * 9 + l] = (u64)w[2 * l] | ((u64)w[2 * l + 1] << 32);
}
__global__ void __launch_bounds__(kThreads) export_kernel(const uint4* __restrict__ st, u64 n, u64* __restrict__ ranlux,
                                                          u32* __restrict__ carry, u32* __restrict__ pos_out,
                                                          u64* __restrict__ lcg) {
  __shared__ uint4 stage[kRawStageWords];
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  const bool live = i < n;
  u32 x[18], v[18], pos = 12, c = 0;
#pragma unroll
  for (int j = 0; j < 18; j++) { x[j] = 0; v[j] = 0; }
  if (live) {
    load_state(st, n, i, x, pos);
    to_ranlux_exact(x, v, c);
  }
  if (ranlux) {  // uniform branches: the staged stores are CTA-collective
    if (aligned16(ranlux)) store_raw<RLXPP_AOS>(ranlux, n, stage, v, blockIdx.x);
    else if (live) store_u64x9(ranlux, i, v);
  }
  if (lcg) {
    if (aligned16(lcg)) store_raw<RLXPP_AOS>(lcg, n, stage, x, blockIdx.x);
    else if (live) store_u64x9(lcg, i, x);
  }
  if (live && carry) carry[i] = c;
  if (live && pos_out) pos_out[i] = pos;
}

__global__ void __launch_bounds__(kThreads) import_kernel(uint4* __restrict__ st, u64 n, const u64* __restrict__ lcg,
                                                          const u32* __restrict__ pos_in) {
  __shared__ uint4 stage[kRawStageWords];
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  u32 w[18], z[20], x[18];
  if (aligned16(lcg)) {
    load_raw<RLXPP_AOS>(lcg, n, stage, w, blockIdx.x);
  } else if (i < n) {
#pragma unroll
    for (int l = 0; l < 9; l++) {
      const u64 q = lcg[i * 9 + l];
      w[2 * l] = (u32)q;
      w[2 * l + 1] = (u32)(q >> 32);
    }
  }
  if (i >= n) return;
#pragma unroll
  for (int j = 0; j < 18; j++) z[j] = w[j];
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
// P = the handle's luxury level when it is one of the baked ones (rlxpp_dev::StreamT<P>: rows as immediates), else 0.
template <int COOP, bool REDUCE, int P = 0>
__global__ void __launch_bounds__(kThreads) ragged_kernel(const rlxpp_view_t view, const u32* __restrict__ counts,
                                                          double* __restrict__ out, u64 ld, double* __restrict__ sum,
                                                          double* __restrict__ sumsq) {
  const u64 i = (u64)blockIdx.x * kThreads + threadIdx.x;
  const bool live = i < view.n;
  rlxpp_dev::StreamT<P> g;
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

// The write-only ceiling for the pattern the interleaved generate kernels produce (tc_pair_kernel), without their
// arithmetic: a persistent grid of 128-thread CTAs, an item = a strip of 256 columns x `rows_per_item` rows of a row-major
// array of doubles with `ld` columns; per row the warp stores 256 contiguous bytes twice (the two tiles of a pair),
// streaming (st.global.cs), and walks down the rows.  Items are dealt round-robin: strips of one chunk of rows first.
__global__ void __launch_bounds__(128, 4) hbm_write_rows_kernel(double* __restrict__ out, u64 ld, u64 n_rows, u32 rows_per_item) {
  const u64 strips = ld / 256, chunks = (n_rows + rows_per_item - 1) / rows_per_item;
  const double v = __longlong_as_double(0x3ff0000000000000ll | (long long)threadIdx.x);
  for (u64 w = blockIdx.x; w < strips * chunks; w += gridDim.x) {
    const u64 strip = w % strips, r0 = (w / strips) * rows_per_item;
    const u64 r1 = r0 + rows_per_item < n_rows ? r0 + rows_per_item : n_rows;
    double* p = out + r0 * ld + strip * 256 + threadIdx.x;
    for (u64 r = r0; r < r1; r++, p += ld) {
      __stcs(p, v);
      __stcs(p + 128, v);
    }
  }
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


}  // namespace rlx
