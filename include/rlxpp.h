/* rlxpp.h -- C ABI of the B200-native RANLUX++ stream library (librlxpp.so).
 *
 * Implements the data-parallel hot path of arxiv 2106.02504, Hahnfeld & Moneta,
 * "A Portable Implementation of RANLUX++".  Citations "P:<n>" are line numbers of
 * /root/reference/PAPER.md with the section they fall in; "D<k>" / "c-<k>" are the
 * readings listed in DESIGN.md (the paper prints no algorithm bodies).
 *
 * Model.  N independent generator streams.  Stream i holds a 576-bit LCG state X_i
 * in [0, m), m = 2^576 - 2^240 + 1 (sec. 2.2), and a cursor pos_i in [0, 12]
 * = number of draws already taken from the block V_i = to_ranlux(X_i) (24 RANLUX
 * numbers of 24 bits + carry, sec. 2/2.3).  One LCG advance is
 * X <- A X mod m with A = a^p mod m, p the luxury level;
 * each advance yields 12 doubles k 2^-48, k = 48 consecutive bits of V.
 * A fresh stream has pos = 12, i.e. the first draw advances first (D8, c-6).  The paper does not say whether the
 * block of the seeded state itself is emitted (parity with the published engine unpinned): an engine
 * that starts at pos = 0 produces this library's sequence with one extra leading block, and
 * rlxpp_set_state(rlxpp_seed_state(seed, p), pos = 0) starts a stream there.
 *
 * Conventions.
 *   - Every function returns 0 on success and a negative RLXPP_E* code on error;
 *     rlxpp_last_error() then returns a thread-local, NUL-terminated description.
 *     No exception crosses the boundary.  There is NO CPU fallback: without a CUDA
 *     device every compute entry point fails with RLXPP_ECUDA.
 *   - Pointers named *_dev are DEVICE pointers, *_host are HOST pointers.  The caller
 *     owns every buffer it passes; the library owns the stream state behind a handle.
 *   - All work is enqueued on the `cuda_stream` given at creation (a cudaStream_t cast
 *     to void*, e.g. torch.cuda.current_stream().cuda_stream; NULL = default stream)
 *     and the calls return WITHOUT synchronising, except the *_host variants, which
 *     return after the host buffer is complete.
 *   - 576-bit integers cross the boundary as 9 little-endian uint64_t.
 *   - Threads and processes.  The library is built for ONE PROCESS PER GPU (streams are independent,
 *     a rank owns a contiguous range of them; no collective).  A handle belongs to the device that was current at
 *     rlxpp_create and is single-threaded: it owns one scheduler buffer and one pair of staging buffers, so two
 *     host threads must not call into the same handle at the same time (different handles are fine).
 *     rlxpp_set_engine, rlxpp_set_chunks and the rare-path counters are process-wide.  Caches keyed by
 *     (device, p) -- the byte matrices, the power tables -- live for the life of the process.
 *   - After a failed rlxpp_generate_*_host call the streams are in a defined but partly advanced state (earlier
 *     stream ranges have drawn, later ones have not); re-import states or destroy the handle.
 */
#ifndef RLXPP_H
#define RLXPP_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define RLXPP_OK 0
#define RLXPP_EINVAL (-1) /* bad argument (null pointer, n_streams == 0, p == 0, unknown layout ...) */
#define RLXPP_ECUDA (-2)  /* CUDA runtime error, including "no device" */
#define RLXPP_ENOMEM (-3) /* device or host allocation failed */

/* output layouts of rlxpp_generate_doubles (BASELINE.json configs 1 and 3) */
#define RLXPP_STREAM_MAJOR 0 /* out[i * n_per_stream + k] */
#define RLXPP_INTERLEAVED 1  /* out[k * n_streams + i]   : a warp writes 32 consecutive doubles */

/* state layouts of rlxpp_advance_states */
#define RLXPP_AOS 0 /* states[i * 9 + limb] */
#define RLXPP_SOA 1 /* states[limb * n_states + i] */

/* engines of the LCG advance (multiply9x9 + mod_m, P:29 / P:33) used by rlxpp_advance_states and
 * rlxpp_generate_*; both give bit-identical results:
 *   UMMA (default): u8 x u8 -> s32 tensor-core GEMM against the byte matrix of A 2^(8k) mod m
 *                   (tcgen05.mma kind::i8, 128 streams per CTA), any luxury level;
 *   IMAD:           324 IMAD.WIDE.U32.X per advance with the multiplier as immediates
 *                   (p in {24, 389, 1024, 2048}), generic 36-limb product otherwise. */
#define RLXPP_ENGINE_UMMA 0
#define RLXPP_ENGINE_IMAD 1

typedef struct rlxpp rlxpp_t;

/* Creates n_streams streams for luxury level p; stream i is seeded with seed + i
 * (mod 2^64) by X = (A^(2^96))^(seed + i) mod m, pos = 12 (sec. 2.4
 * "seed the generator ... fast exponentiation by squaring"; exponent: D7, c-7).
 * The host computes A = a^p and the square tables; a seeding kernel runs on
 * `cuda_stream`.  p in {24, 389, 1024, 2048} uses kernels with the multiplier baked
 * in as immediates; any other p >= 1 uses the generic-multiplier kernels.
 * Errors: EINVAL (h null, n_streams == 0, p == 0), ENOMEM, ECUDA. */
int rlxpp_create(rlxpp_t** h, uint64_t n_streams, uint64_t seed, uint32_t p, void* cuda_stream);
int rlxpp_destroy(rlxpp_t* h);

/* Skips n draws on every stream (rlxpp_skip) or n_dev[i] draws on stream i
 * (rlxpp_skip_each; n_dev: device pointer, n_streams entries) "without generating
 * them": X <- A^k X, k = floor((pos + n - 1) / 12), pos <- pos + n - 12 k
 * (D8, c-8).  Full 64-bit range; n == 0 is a no-op. */
int rlxpp_skip(rlxpp_t* h, uint64_t n);
int rlxpp_skip_each(rlxpp_t* h, const uint64_t* n_dev);

/* Handle-free raw LCG arithmetic (BASELINE.json configs[1]): every uint64[9] value
 * x in [0, 2^576) (non-canonical values >= m allowed) is replaced, in place, by
 * A^reps x mod m, A = a^p, canonical (< m "in all cases").  multiply9x9
 * + mod_m per repetition.  reps == 0 only canonicalises.
 * states_dev: device pointer, 9 * n_states uint64_t, 16-byte aligned, `layout`
 * RLXPP_AOS or RLXPP_SOA.  n_states == 0 is a no-op. */
int rlxpp_advance_states(uint64_t* states_dev, uint64_t n_states, uint32_t p, uint32_t reps, int layout,
                         void* cuda_stream);

/* The next n_per_stream draws of every stream as doubles in [0, 1) on the 2^-48
 * lattice ("uses only 48 bits for each floating point value"; P:174 one LCG
 * operation per 12 numbers), written to out_dev (>= n_streams * n_per_stream doubles,
 * 16-byte aligned) in `layout`.  Any n_per_stream >= 0; multiples of 12 on streams
 * whose cursors are all at 12 take the fast path.  The streams' states advance. */
int rlxpp_generate_doubles(rlxpp_t* h, double* out_dev, uint64_t n_per_stream, int layout);

/* Same draws, consumed in registers (sec. 4.2: "we sum all numbers per thread
 * and store them into global memory at the end"): per stream, in draw order,
 * S <- S + d and Q <- fma(d, d, Q) in IEEE fp64 round-to-nearest, both from +0.0
 * (c-14).  sum_dev / sumsq_dev: n_streams doubles each (sumsq_dev may be NULL). */
int rlxpp_generate_reduce(rlxpp_t* h, double* sum_dev, double* sumsq_dev, uint64_t n_per_stream);

/* End-to-end variants with HOST destination buffers: generation on the device in
 * chunks of streams, device->host copies overlapped on a second CUDA stream; they
 * return when out_host is complete.  Pinned host memory gives full PCIe rate. */
int rlxpp_generate_doubles_host(rlxpp_t* h, double* out_host, uint64_t n_per_stream, int layout);
int rlxpp_generate_reduce_host(rlxpp_t* h, double* sum_host, double* sumsq_host, uint64_t n_per_stream);

/* Exports the paper's stored state (24 RANLUX numbers packed in uint64[9] + carry)
 * and the cursor; optionally also the LCG form.  Any pointer may be NULL.
 * ranlux_dev, lcg_dev: [n_streams][9] uint64_t;  carry_dev, pos_dev: [n_streams] uint32_t. */
int rlxpp_get_state(rlxpp_t* h, uint64_t* ranlux_dev, uint32_t* carry_dev, uint32_t* pos_dev, uint64_t* lcg_dev);

/* Imports states (sec. 4.2: "the state can be copied between host and device"):
 * lcg_dev [n_streams][9] canonical LCG states (values >= m are reduced), pos_dev
 * [n_streams] cursors in [0, 12] (NULL = all 12).  Errors: EINVAL. */
int rlxpp_set_state(rlxpp_t* h, const uint64_t* lcg_dev, const uint32_t* pos_dev);
/* The same from the paper's stored form (SURVEY 8a-2 / reading D3 `to_lcg`): ranlux_dev
 * [n_streams][9] = the 24 RANLUX numbers of 24 bits, oldest lowest, carry_dev [n_streams] in {0, 1} (NULL = all
 * 0), as rlxpp_get_state exports them.  X = V - (V >> 336) + c on the device (V = 2^576 - 1 with c = 1 gives m,
 * stored as 0).  pos_dev as above.  Errors: EINVAL. */
int rlxpp_set_state_ranlux(rlxpp_t* h, const uint64_t* ranlux_dev, const uint32_t* carry_dev, const uint32_t* pos_dev);

/* Host-only helpers: A = a^p mod m as computed by the library's own host arithmetic,
 * and the seed state (A^(2^96))^seed mod m.  out: 9 uint64_t on the host. */
int rlxpp_multiplier(uint32_t p, uint64_t* out_host);
int rlxpp_seed_state(uint64_t seed, uint32_t p, uint64_t* out_host);
/* The byte matrix of the UMMA engine for luxury level p, as the host builds it:
 * out_host[n * 72 + k] = byte n of (A 2^(8k) mod m), n, k in [0, 72) (5,184 bytes), so that for
 * every x < 2^576 with bytes xb_k:  sum_n (sum_k xb_k out[n][k]) 2^(8n) == A x (mod m). */
int rlxpp_umma_matrix(uint32_t p, uint8_t* out_host);

/* Selects the engine for all later calls of this process (default RLXPP_ENGINE_UMMA).
 * Errors: EINVAL for an unknown engine. */
int rlxpp_set_engine(int engine);
int rlxpp_get_engine(void);
/* UMMA engine only.  The generate kernels run as a persistent grid over work items (128 streams x
 * one chunk of draws); the library cuts every tile's draws into chunks so that the grid's last
 * partial wave is short (DESIGN.md 5.1 "Scheduler").  n_chunks = 0 (default): the library decides;
 * n_chunks > 0: every call with at least n_chunks advances per stream uses that many chunks.
 * Results never depend on it.  Errors: EINVAL outside [0, 4096]. */
int rlxpp_set_chunks(int n_chunks);

/* ---- Other output forms of the same draws ("IntRndm") --------------
 * rlxpp_generate_u48: the 48-bit integers k themselves (the double is k 2^-48), one uint64_t each.
 * rlxpp_generate_floats: the 24-bit RANLUX numbers as floats x 2^-24 in [0, 1), exact; one 48-bit draw
 *   gives two floats, low number (the older one) first, so n_per_stream must be even and the cursor
 *   moves by n_per_stream / 2 draws.
 * Layouts as rlxpp_generate_doubles, in elements of the output type (INTERLEAVED floats:
 * out[k * n_streams + i], k = float index).  Same cursor, same sequence: calls of all generate
 * functions interleave freely.  Both always run on the UMMA engine's kernels.  Errors as
 * rlxpp_generate_doubles, plus EINVAL for an odd float count. */
int rlxpp_generate_u48(rlxpp_t* h, uint64_t* out_dev, uint64_t n_per_stream, int layout);
int rlxpp_generate_floats(rlxpp_t* h, float* out_dev, uint64_t n_per_stream, int layout);
/* rlxpp_generate_normal: standard normal deviates, fused into the generation kernel (SURVEY 8f-2 "a distribution
 *   on top (Gaussian)"; the paper stops at uniform numbers, so the transform is this
 *   library's: DESIGN.md reading N-1).  Box-Muller on the stream's draw pairs (2i, 2i + 1), counted from the
 *   stream's first draw: u0 = k[2i] 2^-48, u1 = k[2i+1] 2^-48, r = sqrt(-2 ln(1 - u0)); the deviate at draw
 *   position 2i is r cos(2 pi u1), at 2i + 1 r sin(2 pi u1).  One deviate per draw position: the call consumes
 *   n_per_stream draws of every stream, any cursor, any count, and interleaves freely with the other generate
 *   calls and with skips (a call that starts or ends inside a pair evaluates that pair twice).  The logarithm
 *   and the sine / cosine of a turn are the library's own fp64 polynomials (csrc/normal_coeffs.cuh), the square
 *   root is IEEE: within 6 ulp of the exact value (the only output form that is not bit-exact);
 *   |z| <= sqrt(96 ln 2) = 8.157.  Layouts, ownership and errors as rlxpp_generate_doubles; UMMA engine. */
int rlxpp_generate_normal(rlxpp_t* h, double* out_dev, uint64_t n_per_stream, int layout);

/* ---- Host engine ------------------------------------------
 * ONE stream continued on the host, with the library's own host arithmetic: the same sequence as the
 * device kernels, so a stream can move between host and device mid-stream through rlxpp_get_state /
 * rlxpp_set_state.  lcg_inout: 9 uint64_t (LCG form, any value < 2^576, canonical on return);
 * pos_inout: cursor 0..12; first `skip` draws are skipped (any 64-bit count), then `n` doubles are
 * written to out_host.  Needs no device.  Errors: EINVAL (null pointer, p == 0, cursor > 12). */
int rlxpp_host_generate(uint64_t* lcg_inout, uint32_t* pos_inout, uint32_t p, uint64_t skip, uint64_t n,
                        double* out_host);

/* ---- Device-side draw API -------------------------------
 * include/rlxpp_device.cuh is a header-only per-thread generator for use inside the caller's own
 * kernels (rlxpp_dev::Stream: load / draw / draw_coop / store); include/rlxpp_tile.cuh adds
 * rlxpp_dev::TileStream, the same for CTAs of 128 threads with the advance on the tensor cores.  rlxpp_device_view fills the plain
 * struct such kernels take (device pointers owned by the handle, valid until rlxpp_destroy); after it
 * the library assumes nothing about the cursors.  Kernels using the view must be ordered after the
 * handle's pending work (same CUDA stream, or an event). */
struct rlxpp_view;
int rlxpp_device_view(rlxpp_t* h, struct rlxpp_view* out_host);
/* Ragged generation, written with that device API: stream i draws counts_dev[i] doubles (uint32,
 * device pointer, n_streams entries).  out_dev[i * ld + t] = draw t of stream i (ld >= max count;
 * entries beyond a stream's count are left untouched); the _reduce form keeps S = S + d and
 * Q = fma(d, d, Q) per stream in draw order (sumsq_dev may be NULL).  cooperative = 1 uses the
 * warp-cooperative advance (draw_coop), 0 the paper's per-thread advance (draw), 2 alternates the two from
 * draw to draw on the same generator (they mix freely), 3 the block-cooperative tensor-core advance of
 * include/rlxpp_tile.cuh (rlxpp_dev::TileStream: one UMMA pass per CTA of 128 streams); results are identical.
 * State and cursors are updated; the draws are the ones rlxpp_generate_doubles would give. */
int rlxpp_generate_ragged(rlxpp_t* h, const uint32_t* counts_dev, double* out_dev, uint64_t ld, int cooperative);
int rlxpp_generate_ragged_reduce(rlxpp_t* h, const uint32_t* counts_dev, double* sum_dev, double* sumsq_dev,
                                 int cooperative);

/* ---- Generation for callers that must not allocate device memory -----------------------------------
 * Who this is for.  Every other way into the generator allocates on the device at some point: rlxpp_create
 * (state planes, scheduler words, power tables), the first use of a luxury level (its byte matrix), the host
 * variants (staging buffers).  Some callers cannot afford that, or are not allowed to:
 *   - code that runs after a framework's memory pool has taken the whole device, where a cudaMalloc from a
 *     third-party library either fails or goes behind the pool's back;
 *   - code with a latency budget (a serving loop, a simulation step inside a timed region): cudaMalloc and
 *     cudaFree synchronise the device and can take milliseconds;
 *   - code running under a fixed, audited memory plan, where every device byte is accounted for up front.
 * rlxpp_generate_doubles_static is the one entry point for them: it calls no cudaMalloc, no cudaFree and no
 * library routine that allocates on the device.  The caller passes the inputs and outputs; everything else the
 * kernels need -- the 80-byte-per-stream working copy of the states, the scheduler words of the persistent
 * kernel, the 7,680-byte byte matrix of the luxury level -- lives in ONE fixed array inside the library's
 * device image (RLXPP_STATIC_SCRATCH_BYTES = 5,255,168 bytes, about 5 MB).  Every GPU that loads librlxpp.so
 * holds that array from the moment the library's code is loaded on it until the process exits, used or not:
 * that is the price, and the reason the limit is modest.
 *
 * What it computes.  lcg_dev: n_streams LCG states, [n_streams][9] uint64_t (the form rlxpp_get_state exports as
 * `lcg_dev`; values >= m are reduced first), every stream at a block boundary (cursor 12).  Each stream makes
 * n_per_stream / 12 advances by A = a^p and its draws (line 39: 12 doubles of 48 bits
 * per advance) go to out_dev in `layout`, exactly as rlxpp_generate_doubles writes them for a handle holding the
 * same states; lcg_dev is then overwritten with the advanced states, so that the next call continues the
 * sequences.  Always the tensor-core kernels (rlxpp_set_engine does not apply); bit-identical with the handle path.
 *   n_streams <= RLXPP_STATIC_MAX_STREAMS (65,536), else RLXPP_EINVAL ("... exceeds the static scratch ...");
 *   n_per_stream a multiple of 12 (there is no cursor to keep a partial block in), else RLXPP_EINVAL;
 *   lcg_dev 8-byte, out_dev 16-byte aligned DEVICE pointers owned by the caller; n_streams == 0 or
 *   n_per_stream == 0 is a no-op.  Work is enqueued on cuda_stream; the call does not wait for it.
 *
 * Set-up.  The FIRST call on each device looks up the array's device address (with that device current) and
 * uploads the byte matrix; a later call with a DIFFERENT p uploads that level's matrix over it (a copy from
 * ordinary host memory, enqueued on cuda_stream).  Make the first call on a device -- and the first call for each
 * new p -- before any stream capture begins.
 *
 * Sharing.  There is one array per device and every call uses all of it; it keeps what the last call left there.
 * The call itself clears the words that must start at zero (scheduler ticket and chunk counters) and rewrites the
 * state copy from lcg_dev, so nothing carries over between calls.  But two calls that can overlap on the GPU
 * (different CUDA streams without an event between them, or two host threads) RACE on the array and give wrong
 * numbers: issue all calls for one device on one stream, or order them yourself.  Handles (rlxpp_create) do not
 * touch the array and may run alongside. */
#define RLXPP_STATIC_MAX_STREAMS 65536ull
#define RLXPP_STATIC_SCRATCH_BYTES 5255168ull
int rlxpp_generate_doubles_static(uint64_t* lcg_dev, uint64_t n_streams, uint32_t p, double* out_dev,
                                  uint64_t n_per_stream, int layout, void* cuda_stream);

/* ---- Rare-path counters (debug / test instrumentation of the hot kernels) ------------------------------
 * mod_m ("smaller than m in all cases") and the conversion back to RANLUX numbers (line 39)
 * run in the hot kernels as fast forms that take the overwhelmingly likely case and hand everything else to
 * the exact code.  Each condition that does so is counted per device, per advance of one stream,
 * in the cold path only:
 *   [RLXPP_RARE_FOLD_BORROW]   folding the bits above 2^576: the borrow of "- hi" leaves limb 1
 *   [RLXPP_RARE_FOLD_CARRY]    ... the carry of "+ hi 2^240" leaves limb 9
 *   [RLXPP_RARE_FOLD_TOP]      ... top limb all ones (the folded value may be >= m)
 *   [RLXPP_RARE_RANLUX_CARRY]  to_ranlux: carry out of the 8-limb addition X + (X >> 336)
 *   [RLXPP_RARE_RANLUX_NEAR]   to_ranlux: |u - w| <= 1, u = bits 304..335, w = bits 544..575 of X
 *   [RLXPP_RARE_RANLUX_UMAX]   to_ranlux: u = 2^32 - 1
 *   [RLXPP_RARE_RANLUX_V0]     to_ranlux: subtracting the carry would borrow out of limb 0
 *   [RLXPP_RARE_RANLUX_THIRD]  the exact conversion gave reading D4's third combination (T = Xh, c = 1)
 * rlxpp_rare_counts synchronises the current device, copies the RLXPP_RARE_KINDS counters to out_host (may be
 * NULL) and zeroes them if reset != 0.  Process-wide per device; not meant for concurrent use.  Errors: ECUDA. */
#define RLXPP_RARE_FOLD_BORROW 0
#define RLXPP_RARE_FOLD_CARRY 1
#define RLXPP_RARE_FOLD_TOP 2
#define RLXPP_RARE_RANLUX_CARRY 3
#define RLXPP_RARE_RANLUX_NEAR 4
#define RLXPP_RARE_RANLUX_UMAX 5
#define RLXPP_RARE_RANLUX_V0 6
#define RLXPP_RARE_RANLUX_THIRD 7
#define RLXPP_RARE_KINDS 8
int rlxpp_rare_counts(uint64_t* out_host, int reset);

uint64_t rlxpp_n_streams(const rlxpp_t* h);
/* 1 if the kernels with immediate multipliers serve this luxury level */
int rlxpp_has_fixed_multiplier(uint32_t p);
/* number of kernel launches this library has enqueued in this process (bench.py's gpu_launches) */
uint64_t rlxpp_launch_count(void);

/* Roofline denominators measured on the device the caller is on:
 *   imad: a dependency-free stream of IMAD.WIDE.U32.X (carry-chained, 64-bit accumulate)
 *         issued from every SM; returns multiply-accumulates per second.
 *   hbm_write: write-only kernels storing `bytes` bytes: a grid-stride sweep of 128-bit stores, and (for >= 1.5 GiB)
 *         the interleaved generate kernels' own pattern without their arithmetic -- strips of 256 doubles of 2 MB rows,
 *         256 contiguous bytes per warp store, walking down the rows; the better of the two in bytes/s.
 * Both time `iters` launches with CUDA events after a warm-up and report the best. */
int rlxpp_measure_imad_peak(int iters, double* imad_per_s, void* cuda_stream);
int rlxpp_measure_hbm_write_peak(uint64_t bytes, int iters, double* bytes_per_s, void* cuda_stream);
/* The stream-major store pattern as the memory system sees it (no passage of the paper: it
 * never writes draws to memory).  A persistent grid (the generate kernels' grid) in
 * which every warp owns 32 rows of `pitch_bytes` at a time and writes one piece of `piece_bytes` of each of
 * them per step; `rows` x pitch_bytes are allocated and freed inside the call.  rows: multiple of 32; piece
 * and pitch: multiples of 16 bytes.  Returns the bytes/s of the best of `iters` launches after a warm-up. */
int rlxpp_measure_hbm_write_pieces(uint64_t rows, uint64_t pitch_bytes, uint32_t piece_bytes, int iters, double* bytes_per_s,
                                   void* cuda_stream);

const char* rlxpp_last_error(void);
const char* rlxpp_version(void);

#ifdef __cplusplus
}
#endif
#endif /* RLXPP_H */
