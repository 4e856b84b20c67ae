// RANLUX++ CPU oracle  --  TEST INFRASTRUCTURE, NOT PRODUCT CODE.
//
// A plain, slow, obviously-correct CPU implementation of what the hot path of
// arxiv 2106.02504 (Hahnfeld & Moneta, "A Portable Implementation of RANLUX++")
// computes.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
// --impl reference legs may call it.  It shares no code, header, table or
// constant generator with the CUDA path (paper_2106_02504_b200/csrc) and
// neither includes the other.
//
// Citations "P:<n>" are line numbers of /root/reference/PAPER.md; "S8c-<k>" are
// the readings in SURVEY.md section 8(c), repeated in DESIGN.md.
//
// Where the paper fixes an algorithm the oracle follows it (multiply9x9 P:29,
// mod_m P:33); where it only fixes a result (X*A mod m; floor(2^576 X / m)) the
// plain definition is ALSO here (bitwise long division) and the tests assert
// both agree.  Everything is exact integer arithmetic except the fused
// sum / sum-of-squares, which is IEEE fp64 round-to-nearest in draw order
// (build with -ffp-contract=off; std::fma is a single rounding).
//
// Parity status:
//   * multiply9x9, mod_m, mulmod, powmod, multiplier a^p : pinned (Python big
//     integers: %, pow; identities a*b == 1 mod m).
//   * swb_step / to_lcg / to_ranlux / advance              : pinned (advance by
//     a^p == p direct subtract-with-borrow steps; closed form == long division
//     == digit formula; tiny-parameter exhaustive check of the state map).
//   * normals (SURVEY 8f-2 "a distribution on top (Gaussian)"; the paper names no
//     transform: reading N-1 in DESIGN.md, Box-Muller)   : pinned (Python math
//     functions; z0^2 + z1^2 and atan2(z1, z0); special arguments; sample moments).
//   * draw order / bit order inside uint64[9] (S8c-5), "advance first" (S8c-6),
//     seeding exponent 2^96 (S8c-7): conventions, PARITY UNPINNED against
//     ROOT's RanluxppEngine (no values are printed in the paper).
//
// Build: g++ -O2 -std=c++17 -ffp-contract=off -fPIC -shared -pthread
#include <cmath>
#include <cstdint>
#include <cstring>
#include <thread>
#include <vector>

typedef uint64_t u64;
typedef unsigned __int128 u128;

namespace {

// m = 2^576 - 2^240 + 1 as little-endian uint64[9]
const u64 kM[9] = {1ull, 0ull, 0ull, 0xFFFF000000000000ull, ~0ull, ~0ull, ~0ull, ~0ull, ~0ull};

// ---------------------------------------------------------------- helpers ---
// little-endian multi-limb helpers; n = number of 64-bit limbs
int cmp_n(const u64* a, const u64* b, int n) {
  for (int i = n - 1; i >= 0; i--) {
    if (a[i] < b[i]) return -1;
    if (a[i] > b[i]) return 1;
  }
  return 0;
}
u64 add_n(u64* r, const u64* a, const u64* b, int n) {  // r = a + b, returns carry
  u64 carry = 0;
  for (int i = 0; i < n; i++) {
    u128 t = (u128)a[i] + b[i] + carry;
    r[i] = (u64)t;
    carry = (u64)(t >> 64);
  }
  return carry;
}
u64 sub_n(u64* r, const u64* a, const u64* b, int n) {  // r = a - b, returns borrow
  u64 borrow = 0;
  for (int i = 0; i < n; i++) {
    u128 t = (u128)a[i] - b[i] - borrow;
    r[i] = (u64)t;
    borrow = (u64)(t >> 64) & 1;
  }
  return borrow;
}
// r (nr limbs, zero-extended) = (a >> sh), a has na limbs
void shr_bits(u64* r, int nr, const u64* a, int na, int sh) {
  int ws = sh / 64, bs = sh % 64;
  for (int i = 0; i < nr; i++) {
    u64 lo = (i + ws < na) ? a[i + ws] : 0;
    u64 hi = (i + ws + 1 < na) ? a[i + ws + 1] : 0;
    r[i] = bs ? (lo >> bs) | (hi << (64 - bs)) : lo;
  }
}
// r (nr limbs) = (a << sh) truncated to nr limbs, a has na limbs
void shl_bits(u64* r, int nr, const u64* a, int na, int sh) {
  int ws = sh / 64, bs = sh % 64;
  for (int i = 0; i < nr; i++) {
    int j = i - ws;
    u64 lo = (j >= 0 && j < na) ? a[j] : 0;
    u64 lower = (j - 1 >= 0 && j - 1 < na) ? a[j - 1] : 0;
    r[i] = bs ? (lo << bs) | (lower >> (64 - bs)) : lo;
  }
}
// keep the low `bits` bits of a (n limbs) in place
void mask_bits(u64* a, int n, int bits) {
  for (int i = 0; i < n; i++) {
    int lo = i * 64;
    if (lo >= bits) a[i] = 0;
    else if (lo + 64 > bits) a[i] &= (~0ull) >> (64 - (bits - lo));
  }
}

// ------------------------------------------------- the paper's arithmetic ---
// P:29 (sec. 2.1) multiply9x9: "For every 64 bit in the output, there are up to
// 9 contributing pairs of 64 bit numbers from the input. The code multiplies
// each of these pairs and sums their individual products. The lower 64 bits of
// the sum constitutes one entry of the output, while the rest is propagated to
// the next entry."  Products by unsigned __int128 (Listing 2).
void multiply9x9(const u64 in1[9], const u64 in2[9], u64 out[18]) {
  u64 next = 0;        // bits 64..127 of the running column sum
  u64 nextCarry = 0;   // bits 128.. of the running column sum
  for (int i = 0; i < 18; i++) {
    u64 current = next;
    u64 carry = nextCarry;
    next = 0;
    nextCarry = 0;
    for (int j = 0; j < 9; j++) {
      int k = i - j;
      if (k < 0 || k >= 9) continue;
      u128 prod = (u128)in1[j] * in2[k];
      u64 upper = (u64)(prod >> 64);
      u64 lower = (u64)prod;
      current += lower;
      carry += (current < lower);  // P:134-137 Listing 4
      next += upper;
      nextCarry += (next < upper);
    }
    next += carry;
    nextCarry += (next < carry);
    out[i] = current;
  }
}

// Definition of "remainder / quotient by m": bitwise restoring long division of
// an 18-limb (1152 bit) numerator by m.  q may be null.  Obviously correct,
// ~1152 iterations of a 10-limb shift/compare/subtract.
void divmod_m(const u64 num[18], u64 q[18], u64 rem[9]) {
  u64 r[10] = {0};  // running remainder, < 2m < 2^577
  u64 m10[10];
  for (int i = 0; i < 9; i++) m10[i] = kM[i];
  m10[9] = 0;
  if (q) memset(q, 0, 18 * sizeof(u64));
  for (int bit = 1151; bit >= 0; bit--) {
    // r = 2 r + bit
    for (int i = 9; i > 0; i--) r[i] = (r[i] << 1) | (r[i - 1] >> 63);
    r[0] = (r[0] << 1) | ((num[bit / 64] >> (bit % 64)) & 1);
    if (cmp_n(r, m10, 10) >= 0) {
      sub_n(r, r, m10, 10);
      if (q) q[bit / 64] |= 1ull << (bit % 64);
    }
  }
  for (int i = 0; i < 9; i++) rem[i] = r[i];
}

// P:33 (sec. 2.2) mod_m: remainder mod m = 2^576 - 2^240 + 1 "using additions,
// subtractions, and bit shifts", "with an additional fix to ensure that the
// result is smaller than m in all cases".  Reading S8c-9:
//   z = lo + hi 2^576,  hi = t1 2^336 + t0,  u = t0 + t1,  2^576 = 2^240 - 1 (mod m)
//   z = lo - hi - t1 + (u mod 2^336) 2^240 + (u >> 336)(2^240 - 1)      (mod m)
// evaluated in a 640-bit two's complement accumulator = r + k 2^576 with
// r in [0, 2^576), k in {-1, 0, 1}; then r += k (2^240 - 1); then the fix:
// subtract m while r >= m (the bound in S8c-9 says at most once).
void mod_m(const u64 z[18], u64 out[9]) {
  const u64* lo = z;
  const u64* hi = z + 9;
  u64 t0[10], t1[10], u[10], hi10[10], acc[10], tmp[10];
  for (int i = 0; i < 9; i++) { hi10[i] = hi[i]; t0[i] = hi[i]; }
  hi10[9] = 0; t0[9] = 0;
  mask_bits(t0, 10, 336);               // t0 = hi mod 2^336
  shr_bits(t1, 10, hi, 9, 336);         // t1 = hi >> 336  (< 2^240)
  add_n(u, t0, t1, 10);                 // u = t0 + t1     (< 2^337)
  for (int i = 0; i < 9; i++) acc[i] = lo[i];
  acc[9] = 0;
  sub_n(acc, acc, hi10, 10);            // - hi
  sub_n(acc, acc, t1, 10);              // - t1
  u64 ulow[10];
  memcpy(ulow, u, sizeof(ulow));
  mask_bits(ulow, 10, 336);
  shl_bits(tmp, 10, ulow, 10, 240);     // (u mod 2^336) 2^240  (< 2^576)
  add_n(acc, acc, tmp, 10);
  u64 twop240m1[10] = {~0ull, ~0ull, ~0ull, 0x0000FFFFFFFFFFFFull, 0, 0, 0, 0, 0, 0};  // 2^240 - 1
  u64 ubit = (u[5] >> 16) & 1;          // u >> 336 (0 or 1); 336 = 5*64 + 16
  if (ubit) add_n(acc, acc, twop240m1, 10);
  // acc = r + k 2^576 (two's complement): fold k once more
  int64_t k = (int64_t)acc[9];
  acc[9] = 0;
  if (k == 1) add_n(acc, acc, twop240m1, 10);
  else if (k == -1) sub_n(acc, acc, twop240m1, 10);
  // (|k| > 1 cannot happen: S8c-9 bound; the long-division cross-check in the
  // tests would expose it.)
  u64 m10[10];
  for (int i = 0; i < 9; i++) m10[i] = kM[i];
  m10[9] = 0;
  while (cmp_n(acc, m10, 10) >= 0) sub_n(acc, acc, m10, 10);  // the "fix": result < m
  for (int i = 0; i < 9; i++) out[i] = acc[i];
}

void mulmod(const u64 a[9], const u64 b[9], u64 out[9]) {
  u64 z[18];
  multiply9x9(a, b, z);
  mod_m(z, out);
}

// P:47 "fast exponentiation by squaring": base^e mod m, e given as ne 64-bit limbs
void powmod(const u64 base[9], const u64* e, int ne, u64 out[9]) {
  u64 result[9] = {1, 0, 0, 0, 0, 0, 0, 0, 0};
  u64 sq[9];
  memcpy(sq, base, sizeof(sq));
  for (int bit = 0; bit < 64 * ne; bit++) {
    if ((e[bit / 64] >> (bit % 64)) & 1) mulmod(result, sq, result);
    mulmod(sq, sq, sq);
  }
  memcpy(out, result, sizeof(result));
}

// S8c-2: the LCG multiplier a = b^-1 mod m = m - (m - 1)/b, b = 2^24
//        = 2^576 - 2^552 - 2^240 + 2^216 + 1          ("very large multiplier")
void multiplier_a(u64 a[9]) {
  // (m - 1) / 2^24 = 2^552 - 2^216
  u64 mm1[9], q[9];
  memcpy(mm1, kM, sizeof(mm1));
  mm1[0] -= 1;
  shr_bits(q, 9, mm1, 9, 24);
  sub_n(a, kM, q, 9);
}
void multiplier_ap(uint32_t p, u64 A[9]) {  // A = a^p mod m  (luxury level p)
  u64 a[9];
  multiplier_a(a);
  u64 e[1] = {p};
  powmod(a, e, 1, A);
}

// ------------------------------------------------------- RANLUX <-> LCG ---
// S8c-1 (D1): subtract-with-borrow step, base b = 2^24, lags r = 24, s = 10:
//   t = x[n-10] - x[n-24] - c;  c' = [t < 0];  x[n] = t + 2^24 c'
// V packs the 24 numbers, oldest in the least significant 24 bits (S8c-5).
void swb_steps(u64 V[9], unsigned* c, u64 nsteps) {
  int64_t x[24];
  for (int j = 0; j < 24; j++) {
    int bit = 24 * j;
    u64 w = V[bit / 64] >> (bit % 64);
    if (bit % 64 > 40) w |= V[bit / 64 + 1] << (64 - bit % 64);
    x[j] = (int64_t)(w & 0xFFFFFF);
  }
  int64_t carry = *c;
  for (u64 n = 0; n < nsteps; n++) {
    int64_t t = x[24 - 10] - x[0] - carry;
    carry = t < 0 ? 1 : 0;
    t += carry << 24;
    for (int j = 0; j < 23; j++) x[j] = x[j + 1];
    x[23] = t;
  }
  memset(V, 0, 9 * sizeof(u64));
  for (int j = 0; j < 24; j++) {
    int bit = 24 * j;
    V[bit / 64] |= (u64)x[j] << (bit % 64);
    if (bit % 64 > 40) V[bit / 64 + 1] |= (u64)x[j] >> (64 - bit % 64);
  }
  *c = (unsigned)carry;
}

// S8c-3 (D3): X = V - floor(V / 2^336) + c   (== m -> 0, degenerate only)
void to_lcg(const u64 V[9], unsigned c, u64 X[9]) {
  u64 vh[9], cc[9] = {c, 0, 0, 0, 0, 0, 0, 0, 0};
  shr_bits(vh, 9, V, 9, 336);
  sub_n(X, V, vh, 9);
  add_n(X, X, cc, 9);
  if (cmp_n(X, kM, 9) == 0) memset(X, 0, 9 * sizeof(u64));
}

// S8c-4 (D4), definition: V = floor(2^576 X / m), c = X - V + floor(V / 2^336)
void to_ranlux_def(const u64 X[9], u64 V[9], unsigned* c) {
  u64 num[18] = {0}, q[18], rem[9];
  for (int i = 0; i < 9; i++) num[9 + i] = X[i];
  divmod_m(num, q, rem);
  for (int i = 0; i < 9; i++) V[i] = q[i];  // X < m  =>  quotient < 2^576
  u64 vh[9], t[9];
  shr_bits(vh, 9, V, 9, 336);
  sub_n(t, X, V, 9);
  add_n(t, t, vh, 9);
  *c = (unsigned)t[0];
}

// S8c-4 (D4), shift/add form (what the engine uses; "converts the LCG
// state back to RANLUX numbers"):  Xh = X >> 336, Xl = X mod 2^336, S = Xl + Xh,
//   D = S 2^240 - S - Xh 2^336   (signed)
//   T = Xh - 1 if D < 0;  Xh if 0 <= D < m;  Xh + 1 if D >= m
//   V = X + T,  c = (V >> 336) - T
void to_ranlux(const u64 X[9], u64 V[9], unsigned* c) {
  u64 xh[10], xl[10], s[10], d[10], tmp[10], t[10];
  shr_bits(xh, 10, X, 9, 336);
  for (int i = 0; i < 9; i++) xl[i] = X[i];
  xl[9] = 0;
  mask_bits(xl, 10, 336);
  add_n(s, xl, xh, 10);
  shl_bits(d, 10, s, 10, 240);      // S 2^240 < 2^577: fits 640 bits
  sub_n(d, d, s, 10);
  shl_bits(tmp, 10, xh, 10, 336);
  sub_n(d, d, tmp, 10);             // two's complement, |D| < 2^578
  memcpy(t, xh, sizeof(t));
  u64 one[10] = {1, 0, 0, 0, 0, 0, 0, 0, 0, 0};
  u64 m10[10];
  for (int i = 0; i < 9; i++) m10[i] = kM[i];
  m10[9] = 0;
  if ((int64_t)d[9] < 0) sub_n(t, t, one, 10);            // T = Xh - 1
  else if (cmp_n(d, m10, 10) >= 0) add_n(t, t, one, 10);  // T = Xh + 1
  u64 x10[10], v[10], vh[10], cc[10];
  for (int i = 0; i < 9; i++) x10[i] = X[i];
  x10[9] = 0;
  add_n(v, x10, t, 10);             // T may be -1 (two's complement): wraps correctly
  v[9] = 0;
  shr_bits(vh, 10, v, 9, 336);
  sub_n(cc, vh, t, 10);
  for (int i = 0; i < 9; i++) V[i] = v[i];
  *c = (unsigned)cc[0];
}

// --------------------------------------------------------------- engine ---
// S8c-6/7/8 (D5-D8).  State = (X, pos): X the LCG state, pos in [0, 12] the
// number of draws already consumed from the block to_ranlux(X).
struct Engine {
  u64 A[9];   // a^p mod m
  u64 X[9];   // LCG state
  u64 V[9];   // to_ranlux(X), valid if have_block
  unsigned c;
  int pos;
  bool have_block;
};

void engine_seed(Engine* e, const u64 A[9], const u64 G[9], u64 seed) {
  // D7: X_seed = (A^(2^96))^seed mod m, start state 1; fresh stream pos = 12
  memcpy(e->A, A, sizeof(e->A));
  u64 ex[1] = {seed};
  powmod(G, ex, 1, e->X);
  e->pos = 12;
  e->have_block = false;
}
void compute_G(const u64 A[9], u64 G[9]) {  // G = A^(2^96): 96 squarings
  memcpy(G, A, 9 * sizeof(u64));
  for (int i = 0; i < 96; i++) mulmod(G, G, G);
}
u64 engine_draw48(Engine* e) {  // D8: one draw as a 48-bit integer
  if (e->pos == 12) {
    mulmod(e->A, e->X, e->X);  // D5 advance: X <- A X mod m
    e->pos = 0;
    e->have_block = false;
  }
  if (!e->have_block) {
    to_ranlux(e->X, e->V, &e->c);
    e->have_block = true;
  }
  int bit = 48 * e->pos;  // D6: draw j = bits [48 j, 48 j + 48) of V
  u64 w = e->V[bit / 64] >> (bit % 64);
  if (bit % 64 > 16) w |= e->V[bit / 64 + 1] << (64 - bit % 64);
  e->pos++;
  return w & 0xFFFFFFFFFFFFull;
}
double to_double(u64 k48) {  // S8c-11: k 2^-48, exact
  return std::ldexp((double)k48, -48);
}
void engine_skip(Engine* e, u64 n) {  // D8 skip(n): n draws, full 64-bit range
  if (n == 0) return;
  // k = floor((pos + n - 1) / 12) in 65-bit safe form
  u128 t = (u128)e->pos + n - 1;
  u64 k = (u64)(t / 12);
  int newpos = (int)((u128)e->pos + n - (u128)12 * k);
  u64 Ak[9], ex[1] = {k};
  powmod(e->A, ex, 1, Ak);
  mulmod(Ak, e->X, e->X);
  e->pos = newpos;
  e->have_block = false;
}

template <class F>
void parallel_for(u64 n, int nthreads, F f) {
  if (nthreads <= 1 || n < 2) { f(0, n, 0); return; }
  std::vector<std::thread> th;
  u64 chunk = (n + nthreads - 1) / nthreads;
  for (int t = 0; t < nthreads; t++) {
    u64 lo = (u64)t * chunk, hi = lo + chunk < n ? lo + chunk : n;
    if (lo >= hi) break;
    th.emplace_back(f, lo, hi, t);
  }
  for (auto& x : th) x.join();
}

}  // namespace

// ------------------------------------------------------------- C exports ---
extern "C" {

void orc_modulus(u64 out[9]) { memcpy(out, kM, sizeof(kM)); }
void orc_multiply9x9(const u64* a, const u64* b, u64* out18) { multiply9x9(a, b, out18); }
void orc_mod_m(const u64* z18, u64* out9) { mod_m(z18, out9); }
void orc_mod_m_longdiv(const u64* z18, u64* out9) { divmod_m(z18, nullptr, out9); }
void orc_mulmod(const u64* a, const u64* b, u64* out9) { mulmod(a, b, out9); }
void orc_powmod(const u64* base, const u64* e, int ne, u64* out9) { powmod(base, e, ne, out9); }
void orc_multiplier(uint32_t p, u64* out9) { multiplier_ap(p, out9); }
void orc_swb_steps(u64* V9, unsigned* c, u64 nsteps) { swb_steps(V9, c, nsteps); }
void orc_to_lcg(const u64* V9, unsigned c, u64* X9) { to_lcg(V9, c, X9); }
void orc_to_ranlux(const u64* X9, u64* V9, unsigned* c) { to_ranlux(X9, V9, c); }
void orc_to_ranlux_def(const u64* X9, u64* V9, unsigned* c) { to_ranlux_def(X9, V9, c); }
void orc_seed_state(u64 seed, uint32_t p, u64* X9) {
  u64 A[9], G[9];
  Engine e;
  multiplier_ap(p, A);
  compute_G(A, G);
  engine_seed(&e, A, G, seed);
  memcpy(X9, e.X, sizeof(e.X));
}
// test hook for S8c-7: seed with exponent 2^log2e instead of 2^96
void orc_seed_state_exp(u64 seed, uint32_t p, int log2e, u64* X9) {
  u64 A[9], G[9];
  multiplier_ap(p, A);
  memcpy(G, A, sizeof(G));
  for (int i = 0; i < log2e; i++) mulmod(G, G, G);
  u64 ex[1] = {seed};
  powmod(G, ex, 1, X9);
}

// cfg2 (BASELINE.json configs[1]): each uint64[9] state x in [0, 2^576)
// <- A^reps x mod m, canonical, in place; states is [n][9]
void orc_advance_states(u64* states, u64 n, uint32_t p, uint32_t reps, int nthreads) {
  u64 A[9];
  multiplier_ap(p, A);
  parallel_for(n, nthreads, [&](u64 lo, u64 hi, int) {
    for (u64 i = lo; i < hi; i++) {
      u64* x = states + 9 * i;
      for (uint32_t r = 0; r < reps; r++) mulmod(A, x, x);
      if (reps == 0) {  // still canonicalise
        u64 z[18] = {0};
        memcpy(z, x, 9 * sizeof(u64));
        mod_m(z, x);
      }
    }
  });
}

// General stream generator.  Stream i: seeded with seeds[i] (D7), then
// skip(skips[i]) if skips != null (D8), then n_per_stream draws.
//   out48   (nullable) [n_streams][n_per_stream] 48-bit integers, stream-major
//   outd    (nullable) [n_streams][n_per_stream] doubles, stream-major
//   sum/sumsq (nullable) per-stream S, Q:  S = S + d;  Q = fma(d, d, Q)  in draw order (S8c-14)
//   X_out (nullable) [n][9] final LCG state, V_out (nullable) [n][9] its RANLUX block,
//   c_out (nullable) carry, pos_out (nullable) cursor
void orc_streams(const u64* seeds, const u64* skips, u64 n_streams, uint32_t p, u64 n_per_stream,
                 u64* out48, double* outd, double* sum, double* sumsq, u64* X_out, u64* V_out,
                 unsigned* c_out, unsigned* pos_out, int nthreads) {
  u64 A[9], G[9];
  multiplier_ap(p, A);
  compute_G(A, G);
  parallel_for(n_streams, nthreads, [&](u64 lo, u64 hi, int) {
    for (u64 i = lo; i < hi; i++) {
      Engine e;
      engine_seed(&e, A, G, seeds[i]);
      if (skips) engine_skip(&e, skips[i]);
      double S = 0.0, Q = 0.0;
      for (u64 t = 0; t < n_per_stream; t++) {
        u64 k = engine_draw48(&e);
        double d = to_double(k);
        if (out48) out48[i * n_per_stream + t] = k;
        if (outd) outd[i * n_per_stream + t] = d;
        S = S + d;
        Q = std::fma(d, d, Q);
      }
      if (sum) sum[i] = S;
      if (sumsq) sumsq[i] = Q;
      if (X_out) memcpy(X_out + 9 * i, e.X, 9 * sizeof(u64));
      if (V_out || c_out) {
        u64 V[9];
        unsigned c;
        to_ranlux(e.X, V, &c);
        if (V_out) memcpy(V_out + 9 * i, V, sizeof(V));
        if (c_out) c_out[i] = c;
      }
      if (pos_out) pos_out[i] = (unsigned)e.pos;
    }
  });
}

// Single engine driven call by call from a given (X, pos): used by the skip /
// cursor pins.  ops[k] > 0: draw ops[k] numbers (48-bit ints appended to out48);
// ops[k] < 0 is not used; skip amounts come from skipn[k] when is_skip[k] != 0.
void orc_engine_run(u64* X9, unsigned* pos, uint32_t p, const unsigned char* is_skip, const u64* amount,
                    int nops, u64* out48) {
  Engine e;
  multiplier_ap(p, e.A);
  memcpy(e.X, X9, sizeof(e.X));
  e.pos = (int)*pos;
  e.have_block = false;
  u64 w = 0;
  for (int k = 0; k < nops; k++) {
    if (is_skip[k]) engine_skip(&e, amount[k]);
    else
      for (u64 t = 0; t < amount[k]; t++) out48[w++] = engine_draw48(&e);
  }
  memcpy(X9, e.X, sizeof(e.X));
  *pos = (unsigned)e.pos;
}

// Standard normal deviates from pairs of 48-bit draws (reading N-1; not in the paper, which
// stops at uniform numbers).  The plain Box-Muller definition (Box & Muller 1958) on
// u0 = k[2i] 2^-48, u1 = k[2i+1] 2^-48, both in [0, 1):
//     r = sqrt(-2 ln(1 - u0)),   z[2i] = r cos(2 pi u1),   z[2i+1] = r sin(2 pi u1)
// (1 - u0 is in (0, 1] and exact, so the logarithm is finite).  Evaluated in long double (x87 64-bit
// mantissa) and rounded once to fp64.  cos / sin of 2 pi u1 use the exact identities for a quarter
// turn and its complement -- t = 4 u1 is exact, q = floor(t), f = t - q, angle = (pi / 2) f, and
// cos(pi/2 f) = sin(pi/2 (1 - f)) for f > 1/2 -- so that the exact zeros of the definition
// (u1 = 0, 1/4, 1/2, 3/4) are zeros here too and the relative error is ~2^-63 everywhere, also next to them.
void orc_normals(const u64* k, u64 n_pairs, double* z) {
  const long double half_pi = 1.57079632679489661923132169163975144L;
  for (u64 i = 0; i < n_pairs; i++) {
    const double u0 = (double)k[2 * i] * 0x1p-48, u1 = (double)k[2 * i + 1] * 0x1p-48;
    const long double r = sqrtl(-2.0L * logl(1.0L - (long double)u0));
    const double t = 4.0 * u1;                 // exact
    const int q = (int)t;                      // 0 .. 3
    const double f = t - (double)q;            // exact, in [0, 1)
    const bool upper = f > 0.5;                // cos(pi/2 f) = sin(pi/2 (1 - f)): arguments stay in [0, pi/4]
    const long double ang = half_pi * (long double)(upper ? 1.0 - f : f);
    const long double c = upper ? sinl(ang) : cosl(ang), s = upper ? cosl(ang) : sinl(ang);
    long double cq, sq;                        // cos, sin of ang + q pi / 2
    switch (q) {
      case 0: cq = c; sq = s; break;
      case 1: cq = -s; sq = c; break;
      case 2: cq = -c; sq = -s; break;
      default: cq = s; sq = -c; break;
    }
    z[2 * i] = (double)(r * cq);
    z[2 * i + 1] = (double)(r * sq);
  }
}

int orc_hardware_threads(void) {
  unsigned n = std::thread::hardware_concurrency();
  return n ? (int)n : 1;
}

}  // extern "C"
