// UMMA engine kernels: tc_generate_kernel (one tile per CTA), tc_generate_lanes_kernel (short calls, time-parallel), tc_pair_kernel (two tiles per CTA), tc_advance_states_group_kernel (raw advance, six groups per SM).
// Part of librlxpp (included by rlxpp.cu, one translation unit); see DESIGN.md 5.
#pragma once

#include "state.cuh"
#include "stages.cuh"
#include "kernels_imad.cuh"  // load_raw / store_raw / canonicalise

namespace rlx {

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
    umma::fence_proxy_async_smem();  // read by tcgen05.mma (async proxy) after the CTA barrier in tile.setup()
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
  tile.issue(x);  // (CTA barrier inside: every thread has read its state and written it to the A operand in tensor memory)
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
        // back to zero for the next launch: a plain store is enough, the only later reader is a later launch on the
        // handle's stream (kernel boundaries order it); no CTA of THIS grid touches the word after its own atomicAdd
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
  tc::PairTile<tc::kSyncArrive> tile;  // (the fused reduce too since the A operands are in tensor memory: 1,245 -> 1,337)
  tile.setup(smem, a.bmat);
  pair_items<ALIGNED, MODE, OUT>(tile, a);
  tile.teardown();
}
// Raw advance (cfg2; S8 a-3 / a-4 alone): x <- A^reps x on raw uint64[9] states, in place.  Two tiles per accumulator
// (the other tile's MMA runs under this tile's normalisation, as in tc_pair_kernel) and tc::kGroups groups of 128
// threads in one CTA per SM (tc::GroupTile): six accumulators per SM instead of four.  Persistent: group (CTA c, group g)
// strides over the pairs of tiles.  Between repetitions the state stays an UNREDUCED product (19 limbs): mod_m is
// linear-algebra-free to defer because A z == A (z mod m), so only the last repetition pays the fold.  Measured at cfg2
// (G doubles-equivalent/s): one tile per CTA 1,160; pairs in four CTAs 1,180; 5 groups 1,228; 6 groups 1,320.
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
        if (r + 1 < reps) {
          // mod_m deferred: the product (< 2^591) is the next operand as it is -- the byte matrix has columns for
          // its two bytes above 2^576 (A z == A (z mod m); the next product is < 2^591 again) -- and only the last
          // repetition is folded to the canonical value ("smaller than m in all cases")
          tile.stash19(t, z);
        } else {
          tc::reduce_z(z, x);
          if (2 * pair + t < n_tiles) {
            store_raw<LAYOUT>(states, n, stage, x, 2 * pair + t, tile.tid, gsync);
            gsync();
          }
        }
      }
    }
  }
  tile.teardown();
}


}  // namespace rlx
