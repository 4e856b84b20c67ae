// Shared-memory staging of the UMMA engine's store paths: StreamMajorStage (aligned rows, TMA), UnalignedRowStage, RingStage (shifted rows, TMA), F32RowStage (float rows, TMA).
// Part of librlxpp (included by rlxpp.cu, one translation unit); see DESIGN.md 5.
#pragma once

#include "emit.cuh"
#include "umma_path.cuh"

namespace rlx {


// Stream-major stores through shared memory and the TMA (S8 a-7a; north_star: "shared-memory
// staging, or TMA bulk stores, so HBM writes are fully coalesced").  A thread's block is 96
// contiguous bytes of ITS stream's row, so direct stores make every warp instruction touch 32 rows
// (measured 287 G doubles/s, 36 % of the HBM peak).  What the memory system wants is measured in
// profiles/ab_r01_stream_major.md: row pieces that are 256 bytes long, 256-byte aligned and written by ONE
// operation reach the interleaved layout's bandwidth; 96-, 128- or 192-byte pieces (or two 128-byte
// halves from two operations) stop at 4.7 - 5.8 TB/s however they are fenced or buffered.
// So each warp owns ONE box of [32 streams][32 doubles] in shared memory.  The 96 bytes of an advance
// go where they fall in a cycle of 8 advances = 768 bytes = 3 boxes; an advance that straddles a box
// end (phases 2 and 5) fills the box, one lane hands it to the TMA (cp.async.bulk.tensor.3d, SASS
// UTMASTG) and the thread keeps the limbs of its remaining 4 or 8 draws in registers until the next
// advance, which first waits for the copy to have read the box (cp.async.bulk.wait_group.read: one
// whole advance of slack) and then stores them at the start of the box.
// Tensor map: out[count][n_per] viewed as [count][n_per / 16][16 doubles] with a {16, 2, 32} box and
// SWIZZLE_128B, so that one operation writes 32 x 256 contiguous bytes while the 16-byte chunks of a
// row are XOR-swizzled in shared memory (2-way instead of 8-way bank conflicts on the st.shared.v2.f64;
// a 2-D box with a 256-byte inner extent cannot be swizzled).  Rows past the end of the launch are
// clipped by the tensor map.  Only whole cycles are staged: the last (n_per / 12) % 8 blocks of a row
// are stored directly.
constexpr u32 kStageWarpBytes = 32u * 256u;                    // one box
constexpr u32 kStageCtaBytes = 4u * kStageWarpBytes + 1024u;   // dynamic shared memory of the staged kernels (+ alignment)
constexpr u64 kStageCycle = 96;                                // draws per cycle of 8 advances
struct StreamMajorStage {
  u32 box;        // shared address of this warp's box (1,024-byte aligned: the swizzle works on address bits)
  u32 rowbase;    // ... of this lane's 256-byte row
  u32 rs;         // swizzle term of the row: ((2 lane) & 6) << 4
  u32 q;          // phase: advance within the cycle
  int col16;      // tensor coordinate (in units of 16 doubles) of the box being filled
  int c1;         // tensor row of the warp's first stream
  const void* tmap;
  u32 kexp;       // exp16()
  u32 cv[18];     // limbs of the block whose last draws wait for the next box (only [6, 18) are ever live)
  double cz[8];   // kNormal: the waiting deviates themselves
  __device__ __forceinline__ void init(uint8_t* stage, const void* tensor_map, u64 tile_first, u32 kexp_, u64 t0) {
    const u32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    box = ((umma::smem_u32(stage) + 1023u) & ~1023u) + warp * kStageWarpBytes;
    rowbase = box + lane * 256u;
    rs = ((2u * lane) & 6u) << 4;
    q = 0;
    col16 = (int)(t0 / 16);
    c1 = (int)(tile_first + warp * 32u);
    tmap = tensor_map;
    kexp = kexp_;
  }
  // draws J, J + 1 of v to byte offset O of the lane's row.  The box is 64 lines of 128 bytes (line 2 r + h
  // = half h of row r); SWIZZLE_128B stores 16-byte chunk c of a line at c ^ (line & 7) = c ^ h ^ ((2 r) & 6).
  template <int OUT, int J, int O>
  __device__ __forceinline__ void put2(const u32 (&v)[18]) {
    constexpr u32 h = (u32)O >> 7, K = ((((u32)O >> 4) & 7u) ^ h) << 4;
    double a, b;
    draw_pair<OUT, J>(v, kexp, a, b);
    asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"((rowbase | (rs ^ K)) + h * 128u), "d"(a), "d"(b) : "memory");
  }
  // doubles z[J0 .. J1) to byte offset O of the lane's row
  template <int J0, int J1, int O>
  __device__ __forceinline__ void putd(const double* z) {
    if constexpr (J0 < J1) {
      constexpr u32 h = (u32)O >> 7, K = ((((u32)O >> 4) & 7u) ^ h) << 4;
      asm volatile("st.shared.v2.f64 [%0], {%1, %2};" ::"r"((rowbase | (rs ^ K)) + h * 128u), "d"(z[J0]), "d"(z[J0 + 1])
                   : "memory");
      putd<J0 + 2, J1, O + 16>(z);
    }
  }
  template <int OUT, int J0, int J1, int O>
  struct Put {
    static __device__ __forceinline__ void all(StreamMajorStage& st, const u32 (&v)[18]) {
      st.put2<OUT, J0, O>(v);
      Put<OUT, J0 + 2, J1, O + 16>::all(st, v);
    }
  };
  __device__ __forceinline__ void wait_box() {  // whole warp: the last copy has read the box
    if ((threadIdx.x & 31u) == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncwarp();
  }
  __device__ __forceinline__ void send() {  // whole warp: the box is full
    umma::fence_proxy_async_smem();
    __syncwarp();
    if ((threadIdx.x & 31u) == 0) {
      asm volatile("cp.async.bulk.tensor.3d.global.shared::cta.bulk_group [%0, {%1, %2, %3}], [%4];" ::"l"(tmap), "r"(0),
                   "r"(col16), "r"(c1), "r"(box)
                   : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    col16 += 2;
  }
  template <int FROM>
  __device__ __forceinline__ void keep(const u32 (&v)[18]) {
#pragma unroll
    for (int j = FROM; j < 18; j++) cv[j] = v[j];
  }
  // whole-warp call: the next block of the item (blocks come in whole cycles of 8)
  template <int OUT>
  __device__ __forceinline__ void emit(const u32 (&v)[18]) {
    if constexpr (OUT == kNormal) {
      // the transform is too long to sit in all eight phases (instruction cache): evaluate the block first, then
      // place it; straddling deviates are carried as doubles (cz[j - 4] = z[j])
      double z[12];
      normal_block(v, kexp, z);
      switch (q) {
        case 0: wait_box(); putd<0, 12, 0>(z); break;
        case 1: putd<0, 12, 96>(z); break;
        case 2: putd<0, 8, 192>(z); send(); cz[4] = z[8]; cz[5] = z[9]; cz[6] = z[10]; cz[7] = z[11]; break;
        case 3: wait_box(); putd<4, 8, 0>(cz); putd<0, 12, 32>(z); break;
        case 4: putd<0, 12, 128>(z); break;
        case 5:
          putd<0, 4, 224>(z);
          send();
#pragma unroll
          for (int j = 0; j < 8; j++) cz[j] = z[j + 4];
          break;
        case 6: wait_box(); putd<0, 8, 0>(cz); putd<0, 12, 64>(z); break;
        default: putd<0, 12, 160>(z); send(); break;
      }
      q = (q + 1u) & 7u;
      return;
    }
    switch (q) {
      case 0: wait_box(); Put<OUT, 0, 12, 0>::all(*this, v); break;
      case 1: Put<OUT, 0, 12, 96>::all(*this, v); break;
      case 2: Put<OUT, 0, 8, 192>::all(*this, v); send(); keep<12>(v); break;
      case 3: wait_box(); Put<OUT, 8, 12, 0>::all(*this, cv); Put<OUT, 0, 12, 32>::all(*this, v); break;
      case 4: Put<OUT, 0, 12, 128>::all(*this, v); break;
      case 5: Put<OUT, 0, 4, 224>::all(*this, v); send(); keep<6>(v); break;
      case 6: wait_box(); Put<OUT, 4, 12, 0>::all(*this, cv); Put<OUT, 0, 12, 64>::all(*this, v); break;
      default: Put<OUT, 0, 12, 160>::all(*this, v); send(); break;
    }
    q = (q + 1u) & 7u;
  }
  // before the box is reused by another item or the CTA exits
  __device__ __forceinline__ void drain() {
    if ((threadIdx.x & 31u) == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    __syncwarp();
  }
};
template <int OUT, int J1, int O>
struct StreamMajorStage::Put<OUT, J1, J1, O> {
  static __device__ __forceinline__ void all(StreamMajorStage&, const u32 (&)[18]) {}
};

// Stream-major stores when the cursors are not all at a block boundary (per-stream skips, draw counts that are
// not multiples of 12): the rows are shifted against each other by up to 11 doubles, so no TMA box fits, and a thread
// storing its own 8-byte pieces makes every warp instruction touch 32 rows (measured 100 G doubles/s at the cfg3
// shape).  Instead the warp parks the block as [32 streams][12 + 1 doubles] in shared memory and copies it out
// element by element in row order: 32 consecutive lanes write 32 consecutive doubles of 2.67 rows, each lane with the
// cursor of its element's stream (one shuffle) for the output index and the range mask.
constexpr u32 kRowStagePitch = 13;                                // doubles; odd: conflict-free 8-byte accesses
constexpr u32 kRowStageWarpBytes = 32u * kRowStagePitch * 8u;     // 3,328
struct UnalignedRowStage {
  u32 buf;        // shared address of this warp's buffer
  double* row0;   // &out[first stream of the warp][first draw of the item]
  u64 pitch;      // doubles between rows
  u32 rows;       // streams of the warp that exist (0 .. 32)
  u32 kexp;
  __device__ __forceinline__ void init(uint8_t* stage, double* out_item, u64 warp_first, u64 count, u64 n_per, u32 kexp_) {
    buf = umma::smem_u32(stage) + (threadIdx.x >> 5) * kRowStageWarpBytes;
    row0 = out_item + warp_first * n_per;
    pitch = n_per;
    rows = warp_first >= count ? 0u : (count - warp_first < 32 ? (u32)(count - warp_first) : 32u);
    kexp = kexp_;
  }
  template <int OUT, int J>
  __device__ __forceinline__ void park(u32 dst, const u32 (&v)[18]) {
    if constexpr (J < 12) {
      double a, b;
      draw_pair<OUT, J>(v, kexp, a, b);
      asm volatile("st.shared.f64 [%0], %1;" ::"r"(dst + J * 8), "d"(a) : "memory");
      asm volatile("st.shared.f64 [%0], %1;" ::"r"(dst + J * 8 + 8), "d"(b) : "memory");
      park<OUT, J + 2>(dst, v);
    }
  }
  // whole-warp call: block v holds the draws at positions q0 .. q0 + 11 counted from the start of each stream's
  // current block; position q of a stream with cursor pos is output index q - pos of the item if that is in [0, n)
  template <int OUT>
  __device__ __forceinline__ void emit(const u32 (&v)[18], u64 q0, u32 pos, u64 n) {
    const u32 lane = threadIdx.x & 31u;
    __syncwarp();  // the copy loop of the previous block has read the buffer
    park<OUT, 0>(buf + lane * (kRowStagePitch * 8u), v);
    __syncwarp();
#pragma unroll 4  // fully unrolled: spills, no faster; hoisting the shuffles out of the loop changes nothing either
    for (u32 k = 0; k < 12; k++) {
      const u32 e = 32u * k + lane;         // element of the [32][12] block in row order
      const u32 r = (e * 2731u) >> 15;      // e / 12 for e < 384
      const u32 c = e - 12u * r;
      const u32 pr = __shfl_sync(0xFFFFFFFFu, pos, r);
      const u64 t = q0 + c - pr;            // wraps when the draw lies before the stream's cursor: then t >= n
      if (r < rows && t < n) {
        double d;
        asm volatile("ld.shared.f64 %0, [%1];" : "=d"(d) : "r"(buf + (e + r) * 8u) : "memory");
        __stcs(row0 + (u64)r * pitch + t, d);
      }
    }
  }
};

// The same case (stream-major, cursors not all at a block boundary) when the row pitch is even, i.e. every row starts
// 16-byte aligned: the aligned path's store pattern -- boxes of 32 rows handed to the TMA -- survives if the
// misalignment is moved into shared memory.  Output index q of a row is the same column for all 32 rows of a warp; what
// differs per lane is only how far it has got: after block step s lane i holds columns up to 12 (s + 1) - pos_i.  So every
// lane writes its 12 doubles at ITS OWN columns of a ring of three granules (16 doubles = 128 bytes per row, 32 rows:
// one 4 KB box with SWIZZLE_128B, 2-way bank conflicts at worst), and when the slowest lane (largest cursor of the warp)
// has completed a granule, lane 0 sends it as one box {16 doubles, 32 rows}.  The lanes are at most 12 doubles apart, so
// the columns in flight span less than three granules, and the granule written now was sent two steps ago
// (cp.async.bulk.wait_group.read makes sure it has been read).  Row ends and rows past the launch are clipped by the
// tensor map: no masked direct stores at all.  12 KB per warp; with the 20 KB of the tile three CTAs per SM.
constexpr u32 kRingBoxBytes = 32u * 128u;
constexpr u32 kRingWarpBytes = 3u * kRingBoxBytes;
constexpr u32 kRingCtaBytes = 4u * kRingWarpBytes + 1024u;  // dynamic shared memory (+ alignment)
struct RingStage {
  u32 row;      // shared address of this lane's row in granule slot 0 of its warp's ring
  u32 rx;       // swizzle term of the row: (lane & 7) << 4
  u32 p0;       // ring position (0 .. 47) of the first draw of the next block
  u32 sent;     // granules handed to the TMA (warp-uniform)
  u32 pmax;     // largest cursor in the warp (warp-uniform): the slowest lane
  u32 ring;     // shared address of the warp's ring
  int c1;       // tensor row of the warp's first stream
  u64 col0;     // tensor column of the item's first draw
  const void* tmap;
  u32 kexp;
  __device__ __forceinline__ void init(uint8_t* stage, const void* tensor_map, u64 tile_first, u64 t0, u32 pos, u32 kexp_) {
    const u32 lane = threadIdx.x & 31u, warp = threadIdx.x >> 5;
    ring = ((umma::smem_u32(stage) + 1023u) & ~1023u) + warp * kRingWarpBytes;
    row = ring + lane * 128u;
    rx = (lane & 7u) << 4;
    p0 = pos ? 48u - pos : 0u;  // block 0 starts pos columns before the item's first draw
    sent = 0;
    pmax = __reduce_max_sync(0xFFFFFFFFu, pos);
    c1 = (int)(tile_first + warp * 32u);
    col0 = t0;
    tmap = tensor_map;
    kexp = kexp_;
  }
  // shared address of ring position p (0 .. 47) of this lane's row: slot p / 16, 16-byte chunk (p % 16) / 2 XOR-swizzled
  // with the row, half p % 2
  __device__ __forceinline__ u32 at(u32 p) const {
    const u32 ps = p << 3;
    return row + ((ps & 0x180u) << 5) + ((ps & 0x78u) ^ rx);
  }
  template <int OUT, int J, bool MASKED>
  __device__ __forceinline__ void put(const u32 (&v)[18], u64 q0, u64 n) {
    if constexpr (J < 12) {
      double a, b;
      draw_pair<OUT, J>(v, kexp, a, b);
      u32 pa = p0 + J, pb = p0 + J + 1;
      pa = pa >= 48u ? pa - 48u : pa;
      pb = pb >= 48u ? pb - 48u : pb;
      if (!MASKED || q0 + J < n) asm volatile("st.shared.f64 [%0], %1;" ::"r"(at(pa)), "d"(a) : "memory");
      if (!MASKED || q0 + J + 1 < n) asm volatile("st.shared.f64 [%0], %1;" ::"r"(at(pb)), "d"(b) : "memory");
      put<OUT, J + 2, MASKED>(v, q0, n);
    }
  }
  // whole-warp call: block step s (0 = the current block).  Draw j of the block is output index q = 12 s + j - pos of the
  // item if that is in [0, n) (it wraps below zero for draws before the cursor: then q >= n).
  template <int OUT, bool MASKED>
  __device__ __forceinline__ void emit(const u32 (&v)[18], u64 s, u32 pos, u64 n) {
    if ((threadIdx.x & 31u) == 0) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncwarp();
    put<OUT, 0, MASKED>(v, 12 * s - pos, n);
    p0 = p0 + 12u >= 48u ? p0 - 36u : p0 + 12u;
    umma::fence_proxy_async_smem();
    __syncwarp();
    // granules every lane has completed: the slowest lane holds columns up to 12 (s + 1) - pmax
    const u64 have = 12 * (s + 1) >= pmax ? 12 * (s + 1) - pmax : 0;
    const u32 done = (u32)(have >= n ? (n + 15) / 16 : have / 16);
    if ((threadIdx.x & 31u) == 0 && done > sent) {
      for (u32 g = sent; g < done; g++)
        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(tmap),
                     "r"((int)(col0 + 16ull * g)), "r"(c1), "r"(ring + (g % 3u) * kRingBoxBytes)
                     : "memory");
      asm volatile("cp.async.bulk.commit_group;" ::: "memory");
    }
    sent = done > sent ? done : sent;
  }
  __device__ __forceinline__ void drain() {  // before the ring serves another item or the CTA exits
    if ((threadIdx.x & 31u) == 0) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
    __syncwarp();
  }
};

// Interleaved 24-bit floats (rlxpp_generate_floats, aligned cursors).  A float row holds 4 bytes per stream: direct
// stores are 24 instructions of 128 bytes per warp and advance (measured 700 G draws/s).  Instead the CTA parks a
// block as [24 float rows][128 streams] in shared memory and ONE thread of the MMA-issuing warp hands it to the TMA
// as a box of 24 rows x 512 bytes.  No new barrier: the box of block b - 1 is sent from Tile::issue() of advance
// b + 1, after the hand-off barrier every thread arrives at anyway.  Tile::issue() no longer fences (its A operand
// moved to tensor memory), so emit() itself ends with fence.proxy.async.shared::cta in every thread: the floats a
// thread parked are ordered before the barrier, and through it before the sender's cp.async.bulk.  Ring of three boxes:
// block b is written after collect() of advance b, i.e. after the MMA-done mbarrier that the issuing thread committed
// AFTER waiting (cp.async.bulk.wait_group.read) for the copy of block b - 3.
constexpr u32 kF32BoxBytes = 24u * 128u * 4u;               // 12,288
constexpr u32 kF32StageBytes = 3u * kF32BoxBytes + 128u;    // dynamic shared memory (+ alignment)
struct F32RowStage {
  u32 base;        // shared address of the ring
  u32 col;         // this thread's byte offset in a row
  u32 nfilled;     // blocks parked so far (the same in all threads)
  u32 nsent;       // blocks handed to the TMA (meaningful in the sending thread only)
  bool sender;     // lane 0 of the MMA-issuing warp
  int c0, r0;      // tensor coordinates of the tile's first stream and of the item's first float row
  const void* tmap;
  __device__ __forceinline__ void init(uint8_t* stage, const void* tensor_map, u64 tile_first, u64 t0, u32 issuer_warp) {
    base = (umma::smem_u32(stage) + 127u) & ~127u;
    col = threadIdx.x * 4u;
    nfilled = 0;
    nsent = 0;
    sender = (threadIdx.x >> 5) == issuer_warp && (threadIdx.x & 31u) == 0;
    c0 = (int)tile_first;
    r0 = (int)(2 * t0);
    tmap = tensor_map;
  }
  template <int J>
  __device__ __forceinline__ void park(u32 dst, const u32 (&v)[18]) {
    if constexpr (J < 12) {
      const double d = draw_value<kF32, J>(v, 0u);
      asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst + (2 * J) * 512u), "r"(__double2loint(d)) : "memory");
      asm volatile("st.shared.b32 [%0], %1;" ::"r"(dst + (2 * J + 1) * 512u), "r"(__double2hiint(d)) : "memory");
      park<J + 1>(dst, v);
    }
  }
  __device__ __forceinline__ void emit(const u32 (&v)[18]) {
    park<0>(base + (nfilled % 3u) * kF32BoxBytes + col, v);
    umma::fence_proxy_async_smem();  // generic-proxy stores above -> async-proxy read by the TMA in send_parked()
    nfilled++;
  }
  // issuing warp, before the MMAs: the boxes sent so far have been read
  __device__ __forceinline__ void before_mma() {
    if (sender) asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory");
    __syncwarp();
  }
  // every thread fenced its parked floats in emit() and has passed the hand-off barrier: send what is parked and unsent
  __device__ __forceinline__ void send_parked() {
    if (sender) {
      while (nsent < nfilled) {
        asm volatile("cp.async.bulk.tensor.2d.global.shared::cta.bulk_group [%0, {%1, %2}], [%3];" ::"l"(tmap), "r"(c0),
                     "r"(r0 + 24 * (int)nsent), "r"(base + (nsent % 3u) * kF32BoxBytes)
                     : "memory");
        asm volatile("cp.async.bulk.commit_group;" ::: "memory");
        nsent++;
      }
    }
  }
  // CTA-collective, after the item's last block
  __device__ __forceinline__ void drain() {
    umma::fence_proxy_async_smem();
    __syncthreads();
    send_parked();
    if (sender) asm volatile("cp.async.bulk.wait_group 0;" ::: "memory");
  }
};


}  // namespace rlx
