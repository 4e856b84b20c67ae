// Tensor-core form of the fixed-multiplier LCG advance (SURVEY f-4 "int8-limb Toeplitz
// formulation"; BASELINE.json north_star: "Use tensor cores only if an int8-limb Toeplitz
// formulation of the fixed-multiplier product is shown by ncu to beat the IMAD path").
//
// multiply9x9 + most of mod_m for a FIXED multiplier A = a^p:
//
//     A X  ==  sum_{k=0}^{71} xb_k R_k   (mod m),   R_k = A 2^(8k) mod m,   xb_k = byte k of X
//
// so with the byte matrix B[n][k] = byte n of R_k (72 x 72, host-computed for any p) the 72
// column sums  acc_n = sum_k xb_k B[n][k] < 72 * 255^2 < 2^23  are ONE u8 x u8 -> s32 GEMM
// tile:  D[128 streams][80] = Xbytes[128][96] * B[80][96]^T  (K padded 72 -> 96, N 72 -> 80 with
// zeros), three tcgen05.mma.kind::i8 of K = 32 per 128 advances.  The value
// Z = sum_n acc_n 2^(8n) < 72 * 255 * m < 2^591 is then carry-normalised per thread (one thread
// = one TMEM lane = one stream), the 15 bits above 2^576 are folded with 2^576 == 2^240 - 1
// (fold_fast / exact mod_m20 on the rare path) and the result is the canonical LCG state.
//
// Per advance and stream this replaces 324 IMAD.WIDE.U32.X (4 issue cycles each on the
// fma-heavy pipe) by ~75 plain integer instructions.
//
// Protocol per CTA (128 threads = 128 streams = UMMA M = the 128 TMEM lanes), per advance:
//   issue():   every thread stores its 72 state bytes as 18 columns of its own TENSOR-MEMORY lane (tcgen05.st: the A
//              operand is read from tensor memory, lane = row, 8 columns = the 32 K bytes of one MMA) ->
//              tcgen05.wait::st -> tcgen05.fence::before_thread_sync -> hand-off barrier -> one thread:
//              tcgen05.fence::after_thread_sync, 3 x tcgen05.mma, tcgen05.commit -> mbarrier
//   (the threads convert and emit the PREVIOUS block's doubles while the tensor core works)
//   collect(): mbarrier wait -> tcgen05.fence::after_thread_sync -> tcgen05.ld of 72 columns ->
//              tcgen05.wait::ld -> normalise.
// The next issue() orders the TMEM reads before the next MMA's TMEM writes (fence + barrier),
// and the mbarrier wait orders the MMA's reads of the A columns before the next tcgen05.st to them.
// (Round 1 and most of round 2 kept the A tile in shared memory: five st.shared.v4 and a fence.proxy.async -- SASS
// MEMBAR.ALL.CTA + FENCE.VIEW.ASYNC -- per advance and thread, and 12 KB of operand reads per MMA.  An allocation of
// 128 columns holds the accumulator (80) AND two operands (24 each); same results, less energy:
// profiles/ab_r02_pairs.md section 6.  GroupTile below still uses shared memory: six accumulators leave no columns.)
#pragma once
#include "arith.cuh"

namespace rlx {
namespace tc {

using rlxpp_dev::tile::kTile;
using rlxpp_dev::tile::kN;
using rlxpp_dev::tile::kKChunks;
using rlxpp_dev::tile::kAChunk;
using rlxpp_dev::tile::kBChunk;
using rlxpp_dev::tile::kABytes;
using rlxpp_dev::tile::kBBytes;
using rlxpp_dev::tile::kTmemCols;
using rlxpp_dev::tile::kCtasPerSm;
using rlxpp_dev::tile::kIdesc;
using rlxpp_dev::tile::b_offset;
using rlxpp_dev::tile::normalise;
// K columns of the byte matrix that are filled: the 72 bytes of a state, and bytes 72, 73 for operands that are products
// not yet folded (Z < 2^591: the raw advance keeps its state unreduced between repetitions, GroupTile::stash19)
constexpr int kKUsed = 74;
// A operands in tensor memory: operand t of an allocation at columns kACol + t kACols .. (96 K bytes = 24 columns)
constexpr u32 kACol = (u32)kN;
constexpr u32 kACols = 24;
static_assert(kACol + 2 * kACols <= kTmemCols, "accumulator + two A operands in one allocation");

// How the CTA hands the freshly written A operand to the thread that issues the MMAs.
//   kSyncCta:    __syncthreads, warp 0 issues.  Every warp waits for the slowest one.
//   kSyncArrive: named barrier 1 -- three warps `bar.arrive` and go straight on to their doubles, only the
//                issuing warp `bar.sync`s (asleep, no polling).  The issuing warp is rotated over the
//                SM's co-resident CTAs (warp w always runs on scheduler w % 4; the TMEM column base
//                0 / 128 / 256 / 384 is unique per resident CTA), so the four schedulers share the
//                issue work.  Measured (profiles/ab_r01_sync.md): +14 % on the store kernels; on the fused
//                reduce -6 % in round 1 (A tile in shared memory: the hand-off sat behind a MEMBAR.ALL.CTA
//                anyway) and +7 % now that the operand is in tensor memory (profiles/ab_r02_pairs.md section 6).
//                kSyncCta is left for the time-parallel lanes kernel (one pass per CTA and a CTA barrier of its own).
enum { kSyncCta = 0, kSyncArrive = 2 };

struct Smem {
  __align__(128) uint8_t b[kBBytes];
  __align__(8) u64 bar;        // MMA done (tcgen05.commit)
  u32 tmem_slot;
  u32 ticket;                  // work item of the persistent scheduler (rlxpp.cu)
};

template <int SYNC>
struct Tile {
  u32 bar;
  u32 phase;
  u32 tmem;    // TMEM base address of the accumulator (lane 0, first column)
  u32 tld;     // the same with this warp's lane quarter in bits [16,32)
  u32 issuer;         // the warp that issues this CTA's MMAs
  u64 bdesc;

  // CTA-collective.  bmat: device pointer to the kBBytes image of B.
  __device__ __forceinline__ void setup(Smem& s, const uint4* __restrict__ bmat) {
    const u32 tid = threadIdx.x;
    uint4* sb = reinterpret_cast<uint4*>(s.b);
    for (u32 q = tid; q < kBBytes / 16; q += kTile) sb[q] = __ldg(bmat + q);
    // B was written with ordinary (generic-proxy) stores and tcgen05.mma reads it through its shared-memory descriptor,
    // i.e. through the async proxy: every thread fences what it wrote, the barrier below hands it to the issuing thread
    umma::fence_proxy_async_smem();
    bar = umma::smem_u32(&s.bar);
    phase = 0;
    if (tid == 0) {
      umma::mbar_init(bar, 1);
      umma::fence_mbar_init();
    }
    if (tid < 32) {
      umma::tmem_alloc(umma::smem_u32(&s.tmem_slot), kTmemCols);
      umma::tmem_relinquish();
    }
    umma::fence_before_sync();
    __syncthreads();
    umma::fence_after_sync();
    tmem = *reinterpret_cast<volatile u32*>(&s.tmem_slot);
    issuer = SYNC == kSyncArrive ? ((tmem & 0xFFFFu) / kTmemCols) & 3u : 0u;
    tld = tmem + (((tid >> 5) & 3u) << 21);  // lane 32 (warp % 4) in bits [16,32)
    umma::tmem_st_zero8(tld + kACol + 16u);  // K bytes 72..95 of every row stay zero (issue() rewrites columns 16, 17)
    bdesc = umma::smem_desc(umma::smem_u32(s.b), kBChunk, 128u);
  }

  // CTA-collective: start  D = Xbytes * B^T  for the 128 states x (any value < 2^576).
  __device__ __forceinline__ void issue(const u32 (&x)[18]) {
    issue(x, [] {}, [] {});
  }
  // before() / after() run in the ISSUING warp (all of its lanes), after the hand-off barrier, right before and right
  // after the MMAs are issued and committed: the place for other async-proxy work on the CTA's shared memory that must be
  // ordered with the MMA-done mbarrier (F32RowStage).  The A operand lives in tensor memory, so issue() itself executes
  // NO proxy fence: a caller whose after() lets the TMA read shared memory must have had every writing thread execute
  // fence.proxy.async.shared::cta BEFORE calling issue() (F32RowStage::emit does, right after parking its floats); the
  // hand-off barrier then orders those fenced writes before the sender's cp.async.bulk.
  template <class Before, class After>
  __device__ __forceinline__ void issue(const u32 (&x)[18], Before&& before, After&& after) {
    umma::tmem_st18(tld + kACol, x);
    umma::tmem_wait_st();
    umma::fence_before_sync();
    if (SYNC == kSyncArrive) {
      if ((threadIdx.x >> 5) == issuer) {
        asm volatile("bar.sync 1, 128;" ::: "memory");
        before();
        if (umma::elect_one()) issue_mma();
        __syncwarp();
        after();
      } else {
        asm volatile("bar.arrive 1, 128;" ::: "memory");
      }
    } else {
      __syncthreads();
      if (threadIdx.x == 0) issue_mma();  // (elect.sync here measured 6 % slower on the fused kernel)
      __syncwarp();
    }
  }

  // One thread: D = Xbytes * B^T as three K steps of 32 bytes (A: 8 columns each; B: two 16-byte chunks each).
  __device__ __forceinline__ void issue_mma() {
    umma::fence_after_sync();
#pragma unroll
    for (u32 k = 0; k < 3; k++)
      umma::mma_i8_ts(tmem, tmem + kACol + 8u * k, bdesc + (u64)((2u * k * kBChunk) >> 4), kIdesc, k);
    umma::commit(bar);
  }

  // Waits for the product and returns Z = sum_n acc_n 2^(8n) as 19 limbs (z[18] < 2^15).
  __device__ __forceinline__ void collect(u32 (&z)[20]) {
    umma::mbar_wait(bar, phase);
    phase ^= 1u;
    __syncwarp();
    umma::fence_after_sync();
    u32 c[72];
    umma::tmem_ld72_wait(tld, tld + 64u, c);
    normalise(c, z);
  }

  // CTA-collective, after the last collect().
  __device__ __forceinline__ void teardown() {
    umma::fence_before_sync();
    __syncthreads();
    if (threadIdx.x < 32) umma::tmem_dealloc(tmem, kTmemCols);
  }
};

// ---------------------------------------------------------------------------------------------------------------
// Two tiles per CTA on ONE accumulator (the kernels no store path binds: fused reduce, raw advance).
// A tile's advances are a serial chain  MMA -> tcgen05.ld -> normalise + fold -> A-operand store -> MMA ..., and with one
// tile per CTA the threads sit idle for the MMA + commit + mbarrier round trip of every advance; TMEM (4 x 128
// allocated columns) caps the SM at four such chains.  The accumulator, however, is only live between the MMA and
// the tcgen05.ld that empties it into registers.  So a CTA of 128 threads owns TWO tiles (thread r = stream r of
// both), each with its own A operand in tensor memory, sharing the 80 accumulator columns in time:
//
//     load(t):   wait for MMA(t)  ->  tcgen05.ld + wait::ld                  (accumulator now free)
//     start(t'): hand-off barrier ->  issuing thread: MMA(t') + commit       (t' = the other tile; its A operand was
//                                                                             stored in the previous half-step)
//     normalise + fold tile t, stash(t) its new state for the next MMA(t), convert and consume its block
//
// MMA(t') runs under the ~250 instructions per warp of tile t's integer work: 8 chains per SM with the same 16 warps,
// same TMEM, and no thread ever waits for the tensor pipe's round trip.  Ordering: every thread's tcgen05.ld of
// the accumulator is complete (wait::ld, fence::before_thread_sync) before the hand-off barrier that precedes the next
// MMA; MMA(t)'s reads of A operand t are complete (mbarrier) before stash(t) overwrites it; one mbarrier serves both
// tiles because at most one commit is ever outstanding.
struct PairSmem {
  __align__(128) uint8_t b[kBBytes];
  __align__(8) u64 bar;
  u32 tmem_slot;
  u32 ticket;
};

template <int SYNC>
struct PairTile {
  u32 bar, phase, tmem, tld, issuer;
  u64 bdesc;
  u32 tid;           // thread within the tile (= stream within each of the two tiles)
  u32* ticket;       // shared word of the persistent scheduler

  __device__ __forceinline__ void sync() { __syncthreads(); }  // all 128 threads that share the tiles

  __device__ __forceinline__ void setup(PairSmem& s, const uint4* __restrict__ bmat) {
    tid = threadIdx.x;
    ticket = &s.ticket;
    uint4* sb = reinterpret_cast<uint4*>(s.b);
    for (u32 q = tid; q < kBBytes / 16; q += kTile) sb[q] = __ldg(bmat + q);
    // B was written with ordinary (generic-proxy) stores and tcgen05.mma reads it through its shared-memory descriptor,
    // i.e. through the async proxy: every thread fences what it wrote, the barrier below hands it to the issuing thread
    umma::fence_proxy_async_smem();
    bar = umma::smem_u32(&s.bar);
    phase = 0;
    if (tid == 0) {
      umma::mbar_init(bar, 1);
      umma::fence_mbar_init();
    }
    if (tid < 32) {
      umma::tmem_alloc(umma::smem_u32(&s.tmem_slot), kTmemCols);
      umma::tmem_relinquish();
    }
    umma::fence_before_sync();
    __syncthreads();
    umma::fence_after_sync();
    tmem = *reinterpret_cast<volatile u32*>(&s.tmem_slot);
    issuer = SYNC == kSyncArrive ? ((tmem & 0xFFFFu) / kTmemCols) & 3u : 0u;
    tld = tmem + (((tid >> 5) & 3u) << 21);
#pragma unroll
    for (u32 t = 0; t < 2; t++)  // K bytes 72..95 of every row stay zero (stash() rewrites columns 16, 17)
      umma::tmem_st_zero8(tld + kACol + t * kACols + 16u);
    bdesc = umma::smem_desc(umma::smem_u32(s.b), kBChunk, 128u);
  }

  // this thread's state of tile t -> A operand t (any value < 2^576), visible to the tensor core after the next start(t)
  __device__ __forceinline__ void stash(u32 t, const u32 (&x)[18]) { umma::tmem_st18(tld + kACol + t * kACols, x); }

  // CTA-collective: every thread has stashed tile t and emptied the accumulator; D = Xbytes(t) * B^T starts
  __device__ __forceinline__ void start(u32 t) {
    umma::tmem_wait_st();
    umma::fence_before_sync();
    if (SYNC == kSyncArrive) {
      if ((threadIdx.x >> 5) == issuer) {
        asm volatile("bar.sync 1, 128;" ::: "memory");
        if (umma::elect_one()) issue_mma(t);
        __syncwarp();
      } else {
        asm volatile("bar.arrive 1, 128;" ::: "memory");
      }
    } else {
      __syncthreads();
      if (threadIdx.x == 0) issue_mma(t);
      __syncwarp();
    }
  }
  __device__ __forceinline__ void issue_mma(u32 t) {
    umma::fence_after_sync();
#pragma unroll
    for (u32 k = 0; k < 3; k++)
      umma::mma_i8_ts(tmem, tmem + kACol + t * kACols + 8u * k, bdesc + (u64)((2u * k * kBChunk) >> 4), kIdesc, k);
    umma::commit(bar);
  }

  // waits for the MMA in flight and empties the accumulator into this thread's registers
  __device__ __forceinline__ void load(u32 (&c)[72]) {
    umma::mbar_wait(bar, phase);
    phase ^= 1u;
    __syncwarp();
    umma::fence_after_sync();
    umma::tmem_ld72_wait(tld, tld + 64u, c);
  }
  // one half-step: the product in flight -> Z (19 limbs), and the other tile's MMA started as soon as the
  // accumulator is empty
  __device__ __forceinline__ void collect(u32 (&z)[20], bool start_next, u32 next) {
    u32 cols[72];
    load(cols);
    if (start_next) start(next);
    normalise(cols, z);
  }

  __device__ __forceinline__ void teardown() {
    umma::fence_before_sync();
    __syncthreads();
    if (threadIdx.x < 32) umma::tmem_dealloc(tmem, kTmemCols);
  }
};

// ---------------------------------------------------------------------------------------------------------------
// More accumulators per SM than four (raw advance, cfg2: its 161 instructions per advance leave the tile waiting for
// the tensor pipe's round trip even with two tiles per accumulator).  Four CTAs of 128 threads fill the SM's 512 TMEM
// columns with four 128-column allocations although an accumulator needs 80.  So ONE CTA per SM allocates all 512
// columns and runs kGroups = 6 groups of 128 threads; a group is what a CTA is in PairTile -- two tiles, one accumulator
// (80 columns at an 80-column stride: measured, an accumulator may start at any multiple of 16 columns), its own A
// tiles, mbarrier and named barrier -- and the groups never synchronise with each other.  Registers: 65,536 / 768 = 85,
// so the accumulator is read in three pieces of 24 columns (6 limbs), each normalised before the next is loaded: at
// most 24 accumulator registers are live instead of 72 (the kernel needs 79).
constexpr int kGroups = 6;
constexpr u32 kGroupCols = 80;
struct GroupSmem {
  __align__(128) uint8_t a[2][kABytes];
  __align__(8) u64 bar;
};
struct GroupsSmem {
  __align__(128) uint8_t b[kBBytes];
  u32 tmem_slot;
  GroupSmem g[kGroups];
};

// 24 accumulator columns starting at taddr, then tcgen05.wait::ld -- one asm block, so that no use can be scheduled early
__device__ __forceinline__ void tmem_ld24_wait(u32 taddr, u32 (&r)[24]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%24];\n\t"
      "tcgen05.ld.sync.aligned.32x32b.x8.b32 {%16, %17, %18, %19, %20, %21, %22, %23}, [%25];\n\t"
      "tcgen05.wait::ld.sync.aligned;"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]), "=r"(r[9]),
        "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]), "=r"(r[17]), "=r"(r[18]),
        "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23])
      : "r"(taddr), "r"(taddr + 16u)
      : "memory");
}
// Piece P of three: columns 24 P .. 24 P + 23 -> limbs 6 P .. 6 P + 5 of Z (see normalise); o_prev = o_(6P-1), cy = the
// carry of the chain, both handed from piece to piece.
template <int P>
__device__ __forceinline__ void normalise_piece(const u32 (&c)[24], u32 (&z)[20], u32& o_prev, u32& cy) {
  u32 e[6], o[6], t[6];
#pragma unroll
  for (int k = 0; k < 6; k++) {
    e[k] = c[4 * k] + (c[4 * k + 1] << 8);
    o[k] = c[4 * k + 2] + (c[4 * k + 3] << 8);
  }
  t[0] = P == 0 ? o[0] << 16 : __byte_perm(o_prev, o[0], 0x5432);
#pragma unroll
  for (int k = 1; k < 6; k++) t[k] = __byte_perm(o[k - 1], o[k], 0x5432);
  // cy + 0xFFFFFFFF carries out exactly when cy == 1: the chain's carry flag is restored, then saved again
  asm("{\n\t.reg .u32 scratch;\n\t"
      "add.cc.u32 scratch, %6, 0xFFFFFFFF;\n\t"
      "addc.cc.u32 %0, %7, %13;\n\t"
      "addc.cc.u32 %1, %8, %14;\n\t"
      "addc.cc.u32 %2, %9, %15;\n\t"
      "addc.cc.u32 %3, %10, %16;\n\t"
      "addc.cc.u32 %4, %11, %17;\n\t"
      "addc.cc.u32 %5, %12, %18;\n\t"
      "addc.u32 %6, 0, 0;\n\t}"
      : "=&r"(z[6 * P]), "=&r"(z[6 * P + 1]), "=&r"(z[6 * P + 2]), "=&r"(z[6 * P + 3]), "=&r"(z[6 * P + 4]), "=&r"(z[6 * P + 5]),
        "+r"(cy)
      : "r"(e[0]), "r"(e[1]), "r"(e[2]), "r"(e[3]), "r"(e[4]), "r"(e[5]), "r"(t[0]), "r"(t[1]), "r"(t[2]), "r"(t[3]), "r"(t[4]),
        "r"(t[5]));
  o_prev = o[5];
}

struct GroupTile {
  u32 a_row, bar, phase, tmem, tld, barid;
  u64 adesc, bdesc;
  u32 tid;      // thread within the group

  __device__ __forceinline__ void sync() { asm volatile("bar.sync %0, 128;" ::"r"(barid) : "memory"); }

  // CTA-collective (all kGroups x 128 threads)
  __device__ __forceinline__ void setup(GroupsSmem& s, const uint4* __restrict__ bmat) {
    const u32 gid = threadIdx.x / kTile;
    tid = threadIdx.x % kTile;
    barid = 1u + gid;
    GroupSmem& g = s.g[gid];
    uint4* sb = reinterpret_cast<uint4*>(s.b);
    for (u32 q = threadIdx.x; q < kBBytes / 16; q += kGroups * kTile) sb[q] = __ldg(bmat + q);
    a_row = umma::smem_u32(g.a[0]) + tid * 16u;
#pragma unroll
    for (u32 t = 0; t < 2; t++)
      asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(a_row + t * kABytes + 5u * kAChunk), "r"(0u) : "memory");
    bar = umma::smem_u32(&g.bar);
    phase = 0;
    if (tid == 0) {
      umma::mbar_init(bar, 1);
      umma::fence_mbar_init();
    }
    if (threadIdx.x < 32) {
      umma::tmem_alloc(umma::smem_u32(&s.tmem_slot), 512u);
      umma::tmem_relinquish();
    }
    umma::fence_before_sync();
    __syncthreads();
    umma::fence_after_sync();
    tmem = *reinterpret_cast<volatile u32*>(&s.tmem_slot) + gid * kGroupCols;
    tld = tmem + (((tid >> 5) & 3u) << 21);  // this warp's lane quarter (warp index % 4: groups are whole warpgroups)
    adesc = umma::smem_desc(umma::smem_u32(g.a[0]), kAChunk, 128u);
    bdesc = umma::smem_desc(umma::smem_u32(s.b), kBChunk, 128u);
  }
  __device__ __forceinline__ void stash(u32 t, const u32 (&x)[18]) {
    const u32 row = a_row + t * kABytes;
#pragma unroll
    for (int g = 0; g < 4; g++)
      asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(row + (u32)g * kAChunk), "r"(x[4 * g]), "r"(x[4 * g + 1]),
                   "r"(x[4 * g + 2]), "r"(x[4 * g + 3])
                   : "memory");
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %3};" ::"r"(row + 4u * kAChunk), "r"(x[16]), "r"(x[17]), "r"(0u) : "memory");
    umma::fence_proxy_async_smem();
  }
  // the same for an unreduced product z (19 limbs, z[18] < 2^15): A z == A (z mod m), so the fold can wait
  __device__ __forceinline__ void stash19(u32 t, const u32 (&z)[20]) {
    const u32 row = a_row + t * kABytes;
#pragma unroll
    for (int g = 0; g < 4; g++)
      asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(row + (u32)g * kAChunk), "r"(z[4 * g]), "r"(z[4 * g + 1]),
                   "r"(z[4 * g + 2]), "r"(z[4 * g + 3])
                   : "memory");
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(row + 4u * kAChunk), "r"(z[16]), "r"(z[17]), "r"(z[18]), "r"(0u)
                 : "memory");
    umma::fence_proxy_async_smem();
  }
  __device__ __forceinline__ void start(u32 t) {
    umma::fence_before_sync();
    // (All 128 threads bar.sync.  An arrive-and-run-on hand-off as in PairTile needs a barrier of its own -- on the one
    // that also serves the raw state staging a warp that ran on arrives twice in one phase: deadlock -- and, with ids
    // 7 .. 12 and the issuing warps spread over the schedulers, measured the same: 1,467 vs 1,469.)
    sync();
    if (tid < 32) {
      if (umma::elect_one()) {
        umma::fence_after_sync();
        const u64 ad = adesc + (u64)((t * kABytes) >> 4);
#pragma unroll
        for (u32 k = 0; k < 3; k++)
          umma::mma_i8(tmem, ad + (u64)((2u * k * kAChunk) >> 4), bdesc + (u64)((2u * k * kBChunk) >> 4), kIdesc, k);
        umma::commit(bar);
      }
      __syncwarp();
    }
  }
  __device__ __forceinline__ void collect(u32 (&z)[20], bool start_next, u32 next) {
    umma::mbar_wait(bar, phase);
    phase ^= 1u;
    __syncwarp();
    umma::fence_after_sync();
    u32 c[24], o_prev = 0, cy = 0;
    tmem_ld24_wait(tld, c);
    normalise_piece<0>(c, z, o_prev, cy);
    tmem_ld24_wait(tld + 24u, c);
    normalise_piece<1>(c, z, o_prev, cy);
    tmem_ld24_wait(tld + 48u, c);
    if (start_next) start(next);  // the accumulator is empty
    normalise_piece<2>(c, z, o_prev, cy);
    z[18] = (o_prev >> 16) + cy;
    z[19] = 0;
  }
  // CTA-collective
  __device__ __forceinline__ void teardown() {
    umma::fence_before_sync();
    __syncthreads();
    // the allocation's own base (group 0's `tmem` happens to equal it, but the dealloc must not depend on that)
    if (threadIdx.x < 32) umma::tmem_dealloc(tmem - (threadIdx.x / kTile) * kGroupCols, 512u);
  }
};

// x <- canonical (Z mod m) for the Z of collect()
__device__ __forceinline__ void reduce_z(u32 (&z)[20], u32 (&x)[18]) {
  u32 rare = 0;
  fold_fast(z, x, rare);
  if (__builtin_expect(rare != 0, 0)) {
    count_rare(fold_rare_mask(z[0], z[1], z[7], z[8], z[9], z[17], z[18], z[19]));
    mod_m20(z, x);  // inline: a call would force z, x into local memory
  }
}

}  // namespace tc
}  // namespace rlx
