// rlxpp_tile.cuh -- the tensor-core form of the RANLUX++ advance for use inside your own CUDA kernels, and the
// building blocks the library's own kernels share with it.
//
// rlxpp_device.cuh gives every THREAD its own generator and advances it with the paper's 324 products 32x32 (P:29,
// P:109), which is what the paper's GPU test does and costs one IMAD.WIDE per product.  For a FIXED multiplier
// A = a^p the advance of 128 streams is instead one u8 x u8 -> s32 GEMM tile on the tcgen05 tensor cores:
//
//     A X  ==  sum_k xb_k (A 2^(8k) mod m)   (mod m),      xb_k = byte k of X
//
// rlxpp_dev::TileStream is that form as a device API: a CTA of exactly 128 threads (one warpgroup, blockDim.x == 128),
// every thread its own stream and its own cursor, draws where the thread needs them.
//
//   #include "rlxpp_tile.cuh"
//   __global__ void __launch_bounds__(128) my_kernel(rlxpp_view_t view, ...) {
//     __shared__ rlxpp_dev::TileShared sh;
//     rlxpp_dev::TileStream g;
//     g.begin(sh, view);                          // CTA-collective: tensor memory, byte matrix of the luxury level
//     g.load(view, i, i < view.n);                // stream i (threads past the end pass live = false)
//     for (...) { double u = g.draw(want); ... }  // CTA-collective: EVERY thread calls it, want = this thread takes a number
//     g.store(view, i);
//     g.end();                                    // CTA-collective
//   }
//
// draw() is called by all 128 threads together (like __syncthreads: not inside divergent code); a thread that needs no
// number at this call passes want = false.  When some thread has used up its block of 12 draws and holds no spare, the CTA
// makes ONE tensor-core pass that gives every thread without a spare its next block; threads enter their spare when
// their own block runs out.  So the CTA pays one pass per 12 draws per thread whatever the cursors are -- the paper's
// divergence penalty does not exist here -- and the CTA only synchronises once per pass, not per draw: after a
// vote the threads know how many calls nobody can starve in.  The sequence is the one rlxpp_generate_doubles gives
// (cursor semantics D8): draws made here and by the library interleave freely.
#ifndef RLXPP_TILE_CUH
#define RLXPP_TILE_CUH
#include "rlxpp_device.cuh"

namespace rlxpp_dev {

// ---------------------------------------------------------------------------------------------------- PTX wrappers
// One-to-one wrappers of the sm_100a instructions of the tensor-core path: tcgen05.mma kind::i8 (SASS UTCIMMA), tensor
// memory allocation and loads (LDTM), mbarrier completion, proxy fences.
namespace umma {

typedef uint32_t u32;
typedef uint64_t u64;

__device__ __forceinline__ u32 smem_u32(const void* p) { return (u32)__cvta_generic_to_shared(p); }

// Shared-memory matrix descriptor, K-major, no swizzle ("interleave"): the operand is a grid of
// core matrices of 8 rows x 16 bytes stored as 128 contiguous bytes (row r of the core matrix at
// byte 16 r).  lbo = byte distance between core matrices adjacent along K, sbo = byte distance
// between core matrices adjacent along M/N.  Bits: [0,14) address >> 4, [16,30) lbo >> 4,
// [32,46) sbo >> 4, [46,48) descriptor version = 1 (Blackwell), [61,64) swizzle mode = 0.
__device__ __forceinline__ u64 smem_desc(u32 saddr, u32 lbo_bytes, u32 sbo_bytes) {
  return (u64)((saddr & 0x3FFFFu) >> 4) | ((u64)(lbo_bytes >> 4) << 16) | ((u64)(sbo_bytes >> 4) << 32) | (1ull << 46);
}

// Instruction descriptor of kind::i8 with unsigned 8-bit A and B (format 0), 32-bit integer
// accumulator (c_format 2 at bits [4,6)), both operands K-major, N >> 3 at [17,23), M >> 4 at [24,29).
__host__ __device__ constexpr u32 idesc_u8u8_s32(int M, int N) {
  return (2u << 4) | ((u32)(N >> 3) << 17) | ((u32)(M >> 4) << 24);
}

// One lane of the (converged) warp: true for exactly one of the lanes in the mask.
__device__ __forceinline__ bool elect_one() {
  u32 pred;
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "elect.sync _|p, 0xFFFFFFFF;\n\t"
      "selp.u32 %0, 1, 0, p;\n\t"
      "}"
      : "=r"(pred));
  return pred != 0;
}

// D[tmem] (+)= A[smem] * B[smem]^T, one CTA; issued by ONE thread on behalf of the CTA.
__device__ __forceinline__ void mma_i8(u32 d_tmem, u64 adesc, u64 bdesc, u32 idesc, u32 accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], %1, %2, %3, p;\n\t"
      "}"
      :
      : "r"(d_tmem), "l"(adesc), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// The same with A read from tensor memory (lane = row, 8 columns of 32 bits = the 32 K bytes of one MMA).
__device__ __forceinline__ void mma_i8_ts(u32 d_tmem, u32 a_tmem, u64 bdesc, u32 idesc, u32 accumulate) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "setp.ne.b32 p, %4, 0;\n\t"
      "tcgen05.mma.cta_group::1.kind::i8 [%0], [%1], %2, %3, p;\n\t"
      "}"
      :
      : "r"(d_tmem), "r"(a_tmem), "l"(bdesc), "r"(idesc), "r"(accumulate)
      : "memory");
}
// tcgen05.st 32x32b: thread t of warp w writes N consecutive 32-bit columns of TMEM lane 32 (w % 4) + t.
__device__ __forceinline__ void tmem_st18(u32 taddr, const u32 (&x)[18]) {
  asm volatile(
      "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17};\n\t"
      "tcgen05.st.sync.aligned.32x32b.x2.b32 [%1], {%18, %19};"
      :
      : "r"(taddr), "r"(taddr + 16u), "r"(x[0]), "r"(x[1]), "r"(x[2]), "r"(x[3]), "r"(x[4]), "r"(x[5]), "r"(x[6]), "r"(x[7]),
        "r"(x[8]), "r"(x[9]), "r"(x[10]), "r"(x[11]), "r"(x[12]), "r"(x[13]), "r"(x[14]), "r"(x[15]), "r"(x[16]), "r"(x[17])
      : "memory");
}
__device__ __forceinline__ void tmem_st_zero8(u32 taddr) {
  asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1, %1, %1, %1, %1, %1, %1, %1};" ::"r"(taddr), "r"(0u) : "memory");
}
__device__ __forceinline__ void tmem_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
// ... and back: 18 columns, then tcgen05.wait::ld
__device__ __forceinline__ void tmem_ld18_wait(u32 taddr, u32 (&x)[18]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%18];\n\t"
      "tcgen05.ld.sync.aligned.32x32b.x2.b32 {%16, %17}, [%19];\n\t"
      "tcgen05.wait::ld.sync.aligned;"
      : "=r"(x[0]), "=r"(x[1]), "=r"(x[2]), "=r"(x[3]), "=r"(x[4]), "=r"(x[5]), "=r"(x[6]), "=r"(x[7]), "=r"(x[8]), "=r"(x[9]),
        "=r"(x[10]), "=r"(x[11]), "=r"(x[12]), "=r"(x[13]), "=r"(x[14]), "=r"(x[15]), "=r"(x[16]), "=r"(x[17])
      : "r"(taddr), "r"(taddr + 16u)
      : "memory");
}
// arrive on the mbarrier once every tcgen05.mma issued so far by this thread has completed
// (implies tcgen05.fence::before_thread_sync)
__device__ __forceinline__ void commit(u32 bar) {
  asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void fence_before_sync() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void fence_after_sync() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// generic-proxy shared-memory writes -> visible to the async proxy (the tensor core's operand reads)
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }

__device__ __forceinline__ void mbar_init(u32 bar, u32 count) {
  asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void fence_mbar_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void mbar_wait(u32 bar, u32 parity) {
  asm volatile(
      "{\n\t"
      ".reg .pred p;\n\t"
      "WAIT_%=:\n\t"
      "mbarrier.try_wait.parity.shared::cta.b64 p, [%0], %1;\n\t"
      "@p bra DONE_%=;\n\t"
      "bra WAIT_%=;\n\t"
      "DONE_%=:\n\t"
      "}"
      :
      : "r"(bar), "r"(parity)
      : "memory");
}

// Tensor memory: whole-warp calls.  ncols: power of two >= 32.  The base address is written to smem.
__device__ __forceinline__ void tmem_alloc(u32 smem_dst, u32 ncols) {
  asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_dst), "r"(ncols) : "memory");
}
// after the CTA's last allocation
__device__ __forceinline__ void tmem_relinquish() {
  asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(u32 taddr, u32 ncols) {
  asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
__device__ __forceinline__ void tmem_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// tcgen05.ld 32x32b: thread t of warp w receives, from TMEM lane 32 (w % 4) + t, N consecutive
// 32-bit columns starting at the column in taddr (lane in bits [16,32), column in bits [0,16)).
// All 72 accumulator columns of this thread's TMEM lane, then tcgen05.wait::ld -- ONE asm block, so
// that no use of the registers can be scheduled before the wait.
// taddr_lo: columns 0..63, taddr_hi: columns 64..71 (they may sit in different allocations).
__device__ __forceinline__ void tmem_ld72_wait(u32 taddr_lo, u32 taddr_hi, u32 (&r)[72]) {
  asm volatile(
      "tcgen05.ld.sync.aligned.32x32b.x64.b32 {%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32, %33, %34, %35, %36, %37, %38, %39, %40, %41, %42, %43, %44, %45, %46, %47, %48, %49, %50, %51, %52, %53, %54, %55, %56, %57, %58, %59, %60, %61, %62, %63}, [%72];\n\t"
      "tcgen05.ld.sync.aligned.32x32b.x8.b32 {%64, %65, %66, %67, %68, %69, %70, %71}, [%73];\n\t"
      "tcgen05.wait::ld.sync.aligned;"
      : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), 
        "=r"(r[8]), "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), 
        "=r"(r[16]), "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), 
        "=r"(r[24]), "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31]), 
        "=r"(r[32]), "=r"(r[33]), "=r"(r[34]), "=r"(r[35]), "=r"(r[36]), "=r"(r[37]), "=r"(r[38]), "=r"(r[39]), 
        "=r"(r[40]), "=r"(r[41]), "=r"(r[42]), "=r"(r[43]), "=r"(r[44]), "=r"(r[45]), "=r"(r[46]), "=r"(r[47]), 
        "=r"(r[48]), "=r"(r[49]), "=r"(r[50]), "=r"(r[51]), "=r"(r[52]), "=r"(r[53]), "=r"(r[54]), "=r"(r[55]), 
        "=r"(r[56]), "=r"(r[57]), "=r"(r[58]), "=r"(r[59]), "=r"(r[60]), "=r"(r[61]), "=r"(r[62]), "=r"(r[63]), 
        "=r"(r[64]), "=r"(r[65]), "=r"(r[66]), "=r"(r[67]), "=r"(r[68]), "=r"(r[69]), "=r"(r[70]), "=r"(r[71])
      : "r"(taddr_lo), "r"(taddr_hi)
      : "memory");
}

}  // namespace umma

// ---------------------------------------------------------------------------------------------------- tile geometry
namespace tile {
using umma::u32;
using umma::u64;

constexpr int kTile = 128;                    // streams per CTA = UMMA M
constexpr int kN = 80;                        // UMMA N (72 byte columns, padded to a multiple of 16)
constexpr int kKChunks = 6;                   // 16-byte K chunks: 96 bytes of K = 3 MMAs of K = 32
constexpr u32 kAChunk = kTile * 16;           // bytes of one K chunk of a shared-memory A tile (16 row groups x 128 B):
                                              // TileStream and the library's group kernel; its other kernels keep A in TMEM
constexpr u32 kBChunk = kN * 16;              // same for B (10 row groups x 128 B)
constexpr u32 kABytes = kKChunks * kAChunk;   // 12,288
constexpr u32 kBBytes = kKChunks * kBChunk;   // 7,680
constexpr u32 kTmemCols = 128;                // power of two >= kN (the library: kN + two A operands of 24 columns)
constexpr int kCtasPerSm = 4;                 // 4 x 128 = the SM's 512 TMEM columns
constexpr u32 kIdesc = umma::idesc_u8u8_s32(kTile, kN);

// Shared-memory image of B (what rlxpp_create uploads, see build_bmatrix on the host side):
// element (n, k) at byte (k / 16) * kBChunk + (n / 8) * 128 + (n % 8) * 16 + (k % 16).
__host__ __device__ constexpr u32 b_offset(int n, int k) {
  return (u32)(k / 16) * kBChunk + (u32)(n / 8) * 128u + (u32)(n % 8) * 16u + (u32)(k % 16);
}

// The 72 accumulator columns of one stream -> Z = sum_n acc_n 2^(8n) as 19 limbs (z[18] < 2^15, z[19] = 0).
__device__ __forceinline__ void normalise(const u32 (&c)[72], u32 (&z)[20]) {
  // limb k gets columns 4k .. 4k+3 at byte offsets 0, 8, 16, 24.  e_k = c0 + (c1 << 8) and
  // o_k = c2 + (c3 << 8) are both < 2^23 + 2^31 < 2^32, so  Z = E + (O << 16)  with E, O the
  // 18-limb numbers of limbs e_k, o_k: 36 shift-adds, 19 byte permutes, one 19-limb carry chain.
  u32 e[18], o[18], t[19];
#pragma unroll
  for (int k = 0; k < 18; k++) {
    e[k] = c[4 * k] + (c[4 * k + 1] << 8);
    o[k] = c[4 * k + 2] + (c[4 * k + 3] << 8);
  }
  t[0] = o[0] << 16;
#pragma unroll
  for (int k = 1; k < 18; k++) t[k] = __byte_perm(o[k - 1], o[k], 0x5432);
  t[18] = o[17] >> 16;
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
      : "=r"(z[0]), "=r"(z[1]), "=r"(z[2]), "=r"(z[3]), "=r"(z[4]), "=r"(z[5]), "=r"(z[6]), "=r"(z[7]), "=r"(z[8]),
        "=r"(z[9]), "=r"(z[10]), "=r"(z[11]), "=r"(z[12]), "=r"(z[13]), "=r"(z[14]), "=r"(z[15]), "=r"(z[16]),
        "=r"(z[17]), "=r"(z[18])
      : "r"(e[0]), "r"(e[1]), "r"(e[2]), "r"(e[3]), "r"(e[4]), "r"(e[5]), "r"(e[6]), "r"(e[7]), "r"(e[8]), "r"(e[9]),
        "r"(e[10]), "r"(e[11]), "r"(e[12]), "r"(e[13]), "r"(e[14]), "r"(e[15]), "r"(e[16]), "r"(e[17]), "r"(t[0]),
        "r"(t[1]), "r"(t[2]), "r"(t[3]), "r"(t[4]), "r"(t[5]), "r"(t[6]), "r"(t[7]), "r"(t[8]), "r"(t[9]), "r"(t[10]),
        "r"(t[11]), "r"(t[12]), "r"(t[13]), "r"(t[14]), "r"(t[15]), "r"(t[16]), "r"(t[17]), "r"(t[18]));
  z[19] = 0;
}

}  // namespace tile

// ---------------------------------------------------------------------------------------------------- TileStream
// Shared memory of one CTA of 128 threads (declare it __shared__ in the kernel; 44 KB).
struct alignas(128) TileShared {
  uint8_t a[tile::kABytes];        // newest state of every thread, K-major UMMA operand: what the next pass advances
  uint8_t b[tile::kBBytes];        // byte matrix of the luxury level
  uint2 draws[2][13][tile::kTile]; // two blocks per thread (current, spare): draw j as the bit pattern of 16 + k 2^-48
                                   // (a 13th row so that a cursor at 12 still addresses the buffer)
  alignas(16) uint32_t vote[8];    // two alternating sets of per-warp minima (read as one 16-byte word each)
  unsigned long long bar;          // MMA done
  uint32_t tmem_slot;
};

class TileStream {
 public:
  // CTA-collective, blockDim.x == 128.  Allocates 128 columns of tensor memory (at most 4 such CTAs per SM).
  __device__ __forceinline__ void begin(TileShared& sh, const rlxpp_view_t& view) {
    const uint32_t tid = threadIdx.x;
    uint4* sb = reinterpret_cast<uint4*>(sh.b);
    for (uint32_t q = tid; q < tile::kBBytes / 16; q += tile::kTile) sb[q] = __ldg(view.bmat + q);
    a_row_ = umma::smem_u32(sh.a) + tid * 16u;
    draws_ = umma::smem_u32(sh.draws) + tid * 8u;
    vote_ = umma::smem_u32(sh.vote);
    // K bytes 80..95 of every row stay zero
    asm volatile("st.shared.v4.u32 [%0], {%1, %1, %1, %1};" ::"r"(a_row_ + 5u * tile::kAChunk), "r"(0u) : "memory");
    bar_ = umma::smem_u32(&sh.bar);
    phase_ = 0;
    if (tid == 0) {
      umma::mbar_init(bar_, 1);
      umma::fence_mbar_init();
    }
    if (tid < 32) {
      umma::tmem_alloc(umma::smem_u32(&sh.tmem_slot), tile::kTmemCols);
      umma::tmem_relinquish();
    }
    umma::fence_before_sync();
    __syncthreads();
    umma::fence_after_sync();
    tmem_ = *reinterpret_cast<volatile uint32_t*>(&sh.tmem_slot);
    tld_ = tmem_ + (((tid >> 5) & 3u) << 21);
    adesc_ = umma::smem_desc(umma::smem_u32(sh.a), tile::kAChunk, 128u);
    bdesc_ = umma::smem_desc(umma::smem_u32(sh.b), tile::kBChunk, 128u);
    budget_ = 0;
    votes_ = 0;
    spare_ = 0;
    ptr_ = draws_;
    pos_ = 0;
    dead_ = 1;
  }
  // CTA-collective, after the last draw / store.
  __device__ __forceinline__ void end() {
    umma::fence_before_sync();
    __syncthreads();
    if (threadIdx.x < 32) umma::tmem_dealloc(tmem_, tile::kTmemCols);
  }

  // CTA-collective, once after begin(): stream i of the handle behind `view`; a thread with nothing to do passes
  // live = false (it never asks for a pass, and must call draw() with want = false).
  __device__ __forceinline__ void load(const rlxpp_view_t& view, uint64_t i, bool live = true) {
    uint32_t x[18];
#pragma unroll
    for (int j = 0; j < 18; j++) x[j] = 0;
    pos_ = 0;
    dead_ = live ? 0u : 1u;
    if (live) {
#pragma unroll
      for (int g = 0; g < 4; g++) {
        const uint4 q = __ldcg(view.st + (uint64_t)g * view.n + i);
        x[4 * g] = q.x; x[4 * g + 1] = q.y; x[4 * g + 2] = q.z; x[4 * g + 3] = q.w;
      }
      const uint4 q = __ldcg(view.st + 4 * view.n + i);
      x[16] = q.x; x[17] = q.y;
      pos_ = q.z > 12u ? 12u : q.z;
    }
    put_state(a_row_, x);
    umma::fence_proxy_async_smem();
    spare_ = 0;
    budget_ = 0;
    ptr_ = draws_ + pos_ * (tile::kTile * 8u);  // the current block lives in buffer 0
    if (live && pos_ < 12u) {  // draws left in the current block: rebuild it from the state
      uint32_t v[18], c;
      detail::to_ranlux_exact(x, v, c);
      put_block<0>(draws_, v);
    }
  }
  // (state of the current block, cursor) back to the handle; a spare block is dropped and recomputed when needed again
  __device__ __forceinline__ void store(const rlxpp_view_t& view, uint64_t i) const {
    uint32_t x[18];
    get_state(a_row_, x);  // the newest state: the current block's unless a spare exists
    if (spare_) {
#pragma unroll
      for (int j = 0; j < 18; j++) x[j] = xc_[j];
    }
#pragma unroll
    for (int g = 0; g < 4; g++)
      view.st[(uint64_t)g * view.n + i] = make_uint4(x[4 * g], x[4 * g + 1], x[4 * g + 2], x[4 * g + 3]);
    view.st[4 * view.n + i] = make_uint4(x[16], x[17], pos_, 0u);
  }

  // CTA-collective: all 128 threads call it together; want = this thread takes a number (else the result is 0).
  __device__ __forceinline__ double draw(bool want = true) {
    uint32_t lo, hi;
    if (!next(want, lo, hi)) return 0.0;
    return __hiloint2double((int)hi, (int)lo) - 16.0;  // exact: 16 + k 2^-48 has the 48 bits in its mantissa
  }
  __device__ __forceinline__ uint64_t draw_u48(bool want = true) {
    uint32_t lo, hi;
    if (!next(want, lo, hi)) return 0;
    return (uint64_t)lo | ((uint64_t)(hi & 0xFFFFu) << 32);
  }
  __device__ __forceinline__ uint32_t cursor() const { return pos_; }

 private:
  static constexpr uint32_t kBlockBytes = 13u * tile::kTile * 8u;  // one buffer of draws
  __device__ __forceinline__ bool next(bool want, uint32_t& lo, uint32_t& hi) {
    if (budget_ == 0) {  // (uniform: every thread counts the same calls)
      const uint32_t have = dead_ ? 0xFFFFu : (12u - pos_) + 12u * spare_;
      if (__syncthreads_or(have == 0 && want)) {
        // somebody is out of numbers: the tensor-core pass gives every thread without a spare its next block, so that
        // every live thread then holds at least 12 draws: nobody can starve in the next 12 calls
        pass();
        budget_ = 12;
      } else {
        // how many calls from now can nobody starve in?  min over the CTA of the draws each thread holds; a thread
        // that holds none (and wants none now) counts as 1: asked again at the next call
        const uint32_t m = cta_min(have ? have : 1u);
        budget_ = m > 4096u ? 4096u : m;
      }
    }
    budget_--;
    if (want && pos_ == 12u) {  // enter the spare block (it exists: the vote above guarantees it)
      ptr_ = draws_ + (ptr_ < draws_ + kBlockBytes ? kBlockBytes : 0u);  // the other buffer
      spare_ = 0;
      pos_ = 0;
    }
    // (a thread that wants nothing may sit at 12: the buffers have a 13th row)
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(lo), "=r"(hi) : "r"(ptr_) : "memory");
    if (want) {
      ptr_ += tile::kTile * 8u;
      pos_++;
    }
    return want;
  }
  // the 12 draws of block v into the buffer at `dst` (this thread's column), as the words of 16 + k 2^-48
  template <int J>
  static __device__ __forceinline__ void put_block(uint32_t dst, const uint32_t (&v)[18]) {
    if constexpr (J < 12) {
      constexpr uint32_t kexp = 0x40300000u;
      uint32_t lo, hi;
      if (J % 2 == 0) {
        lo = v[3 * J / 2];
        hi = __byte_perm(v[3 * J / 2 + 1], kexp, 0x7610);
      } else {
        lo = __byte_perm(v[(3 * J - 1) / 2], v[(3 * J + 1) / 2], 0x5432);
        hi = __byte_perm(v[(3 * J + 1) / 2], kexp, 0x7632);
      }
      asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(dst + (uint32_t)J * (tile::kTile * 8u)), "r"(lo), "r"(hi) : "memory");
      put_block<J + 1>(dst, v);
    }
  }
  static __device__ __forceinline__ void put_state(uint32_t row, const uint32_t (&x)[18]) {
#pragma unroll
    for (int g = 0; g < 4; g++)
      asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(row + (uint32_t)g * tile::kAChunk), "r"(x[4 * g]),
                   "r"(x[4 * g + 1]), "r"(x[4 * g + 2]), "r"(x[4 * g + 3])
                   : "memory");
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %3};" ::"r"(row + 4u * tile::kAChunk), "r"(x[16]), "r"(x[17]), "r"(0u)
                 : "memory");
  }
  static __device__ __forceinline__ void get_state(uint32_t row, uint32_t (&x)[18]) {
#pragma unroll
    for (int g = 0; g < 4; g++)
      asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];"
                   : "=r"(x[4 * g]), "=r"(x[4 * g + 1]), "=r"(x[4 * g + 2]), "=r"(x[4 * g + 3])
                   : "r"(row + (uint32_t)g * tile::kAChunk)
                   : "memory");
    asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(x[16]), "=r"(x[17]) : "r"(row + 4u * tile::kAChunk) : "memory");
  }
  // min over the 128 threads (one barrier; the per-warp minima alternate between two sets of words)
  __device__ __forceinline__ uint32_t cta_min(uint32_t val) {
    const uint32_t wmin = __reduce_min_sync(0xFFFFFFFFu, val);
    const uint32_t set = vote_ + (votes_ & 1u) * 16u;
    votes_++;
    if ((threadIdx.x & 31u) == 0) asm volatile("st.shared.u32 [%0], %1;" ::"r"(set + (threadIdx.x >> 5) * 4u), "r"(wmin) : "memory");
    __syncthreads();
    uint32_t m0, m1, m2, m3;
    asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(m0), "=r"(m1), "=r"(m2), "=r"(m3) : "r"(set) : "memory");
    return min(min(m0, m1), min(m2, m3));
  }
  __device__ __forceinline__ void issue_mma() {  // one thread: D = (newest states) x B^T
    umma::fence_after_sync();
#pragma unroll
    for (uint32_t k = 0; k < 3; k++)
      umma::mma_i8(tmem_, adesc_ + (uint64_t)((2u * k * tile::kAChunk) >> 4), bdesc_ + (uint64_t)((2u * k * tile::kBChunk) >> 4),
                   tile::kIdesc, k);
    umma::commit(bar_);
  }
  // CTA-collective, right after the vote's CTA barrier (every thread's stores to the A tile are fenced and ordered by
  // it): D = (newest states) x B^T on the tensor core; every thread without a spare block takes its row as the next
  // block (state to the A tile, draws to the other buffer) and keeps the state of its current block in registers for
  // store(); the others discard theirs.  (Starting the next product at the end of a pass, to hide the tensor pipe's
  // round trip behind the next 12 draws, was measured: 415 vs 449 G doubles/s -- the extra barrier costs more.)
  __device__ __forceinline__ void pass() {
    if (threadIdx.x < 32) {
      if (umma::elect_one()) issue_mma();
      __syncwarp();
    }
    umma::mbar_wait(bar_, phase_);
    phase_ ^= 1u;
    __syncwarp();
    umma::fence_after_sync();
    uint32_t c[72], z[20], x[18];
    umma::tmem_ld72_wait(tld_, tld_ + 64u, c);
    tile::normalise(c, z);
    uint32_t rare = 0;
    detail::fold_fast(z, x, rare);
    if (__builtin_expect(rare != 0, 0)) detail::mod_m20(z, x);
    if (!spare_ && !dead_) {
      uint32_t v[18], cc;
      rare = 0;
      detail::to_ranlux_fast(x, v, cc, rare);
      if (__builtin_expect(rare != 0, 0)) detail::to_ranlux_exact(x, v, cc);
      get_state(a_row_, xc_);  // the state this product advanced is the current block's
      put_state(a_row_, x);
      put_block<0>(draws_ + (ptr_ < draws_ + kBlockBytes ? kBlockBytes : 0u), v);  // the buffer the cursor is not in
      spare_ = 1;
    }
    umma::fence_proxy_async_smem();
    umma::fence_before_sync();  // (orders this thread's tcgen05.ld before the barrier that precedes the next pass)
  }

  uint32_t xc_[18];  // state of the current block while a spare exists (otherwise the A tile holds it)
  uint32_t a_row_, draws_, vote_, bar_, phase_, tmem_, tld_;
  uint64_t adesc_, bdesc_;
  uint32_t ptr_;     // shared address of the next draw (this thread's column of one of the two buffers)
  uint32_t pos_, spare_, budget_, votes_, dead_;
};

}  // namespace rlxpp_dev
#endif  // RLXPP_TILE_CUH
