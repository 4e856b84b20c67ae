// IMAD engine kernels: raw state I/O (also used by the UMMA raw advance), advance_states_kernel, generate_kernel.
// Part of librlxpp (included by rlxpp.cu, one translation unit); see DESIGN.md 5.
#pragma once

#include "state.cuh"
#include "emit.cuh"

namespace rlx {

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
