// Host-side modular arithmetic of the library (multiplier a^p, seeding / skip tables).
//
// Product code, independent of oracle/: a small variable-length unsigned integer on
// 32-bit words and reduction modulo m = 2^576 - 2^240 + 1 by repeatedly
// replacing the part above bit 576 through 2^576 == 2^240 - 1 (mod m), then subtracting m
// while the value is >= m.  Cold path: a few hundred modular products per handle.
#pragma once
#include <algorithm>
#include <cstdint>
#include <vector>

namespace rlx {
namespace host {

struct Big {
  std::vector<uint32_t> w;  // little-endian, no leading zero words

  Big() {}
  explicit Big(uint64_t v) {
    if (v) w.push_back((uint32_t)v);
    if (v >> 32) w.push_back((uint32_t)(v >> 32));
  }
  void trim() {
    while (!w.empty() && w.back() == 0) w.pop_back();
  }
  bool is_zero() const { return w.empty(); }
  size_t bits() const {
    if (w.empty()) return 0;
    uint32_t t = w.back();
    size_t b = 0;
    while (t) { b++; t >>= 1; }
    return 32 * (w.size() - 1) + b;
  }
  static int cmp(const Big& a, const Big& b) {
    if (a.w.size() != b.w.size()) return a.w.size() < b.w.size() ? -1 : 1;
    for (size_t i = a.w.size(); i-- > 0;)
      if (a.w[i] != b.w[i]) return a.w[i] < b.w[i] ? -1 : 1;
    return 0;
  }
  static Big add(const Big& a, const Big& b) {
    Big r;
    size_t n = std::max(a.w.size(), b.w.size());
    r.w.resize(n + 1);
    uint64_t c = 0;
    for (size_t i = 0; i < n; i++) {
      uint64_t s = c + (i < a.w.size() ? a.w[i] : 0) + (i < b.w.size() ? b.w[i] : 0);
      r.w[i] = (uint32_t)s;
      c = s >> 32;
    }
    r.w[n] = (uint32_t)c;
    r.trim();
    return r;
  }
  static Big sub(const Big& a, const Big& b) {  // requires a >= b
    Big r;
    r.w.resize(a.w.size());
    int64_t c = 0;
    for (size_t i = 0; i < a.w.size(); i++) {
      int64_t s = (int64_t)a.w[i] - (i < b.w.size() ? b.w[i] : 0) + c;
      r.w[i] = (uint32_t)s;
      c = s >> 32;
    }
    r.trim();
    return r;
  }
  static Big mul(const Big& a, const Big& b) {
    Big r;
    if (a.is_zero() || b.is_zero()) return r;
    r.w.assign(a.w.size() + b.w.size(), 0);
    for (size_t i = 0; i < a.w.size(); i++) {
      uint64_t c = 0;
      for (size_t j = 0; j < b.w.size(); j++) {
        uint64_t s = (uint64_t)a.w[i] * b.w[j] + r.w[i + j] + c;
        r.w[i + j] = (uint32_t)s;
        c = s >> 32;
      }
      r.w[i + b.w.size()] = (uint32_t)c;
    }
    r.trim();
    return r;
  }
  static Big shl(const Big& a, size_t s) {
    Big r;
    if (a.is_zero()) return r;
    size_t ws = s / 32, bs = s % 32;
    r.w.assign(a.w.size() + ws + 1, 0);
    for (size_t i = 0; i < a.w.size(); i++) {
      r.w[i + ws] |= bs ? (a.w[i] << bs) : a.w[i];
      if (bs) r.w[i + ws + 1] |= a.w[i] >> (32 - bs);
    }
    r.trim();
    return r;
  }
  static Big shr(const Big& a, size_t s) {
    Big r;
    size_t ws = s / 32, bs = s % 32;
    if (ws >= a.w.size()) return r;
    r.w.assign(a.w.size() - ws, 0);
    for (size_t i = 0; i < r.w.size(); i++) {
      uint32_t lo = a.w[i + ws];
      uint32_t hi = (i + ws + 1 < a.w.size()) ? a.w[i + ws + 1] : 0;
      r.w[i] = bs ? (lo >> bs) | (hi << (32 - bs)) : lo;
    }
    r.trim();
    return r;
  }
  static Big low_bits(const Big& a, size_t nbits) {
    Big r;
    size_t nw = (nbits + 31) / 32;
    r.w.assign(a.w.begin(), a.w.begin() + std::min(nw, a.w.size()));
    if (nbits % 32 && r.w.size() == nw) r.w[nw - 1] &= (1u << (nbits % 32)) - 1;
    r.trim();
    return r;
  }
  void to_u32x18(uint32_t out[18]) const {
    for (int i = 0; i < 18; i++) out[i] = (size_t)i < w.size() ? w[i] : 0;
  }
  void to_u64x9(uint64_t out[9]) const {
    uint32_t t[18];
    to_u32x18(t);
    for (int i = 0; i < 9; i++) out[i] = (uint64_t)t[2 * i] | ((uint64_t)t[2 * i + 1] << 32);
  }
};

inline Big modulus() {  // m = 2^576 - 2^240 + 1
  Big one(1);
  return Big::add(Big::sub(Big::shl(one, 576), Big::shl(one, 240)), one);
}

inline Big reduce(Big x) {
  const Big m = modulus();
  while (x.bits() > 576) {  // x = lo + hi 2^576 == lo + hi 2^240 - hi
    Big hi = Big::shr(x, 576), lo = Big::low_bits(x, 576);
    x = Big::sub(Big::add(lo, Big::shl(hi, 240)), hi);
  }
  while (Big::cmp(x, m) >= 0) x = Big::sub(x, m);
  return x;
}
inline Big mulmod(const Big& a, const Big& b) { return reduce(Big::mul(a, b)); }
inline Big powmod(Big base, uint64_t e) {
  Big r(1);
  while (e) {
    if (e & 1) r = mulmod(r, base);
    base = mulmod(base, base);
    e >>= 1;
  }
  return r;
}
// a = b^-1 mod m = m - (m - 1) / 2^24: one subtract-with-borrow step is X <- a X (D2)
inline Big multiplier_a() {
  const Big m = modulus();
  return Big::sub(m, Big::shr(Big::sub(m, Big(1)), 24));
}
inline Big multiplier_ap(uint32_t p) { return powmod(multiplier_a(), p); }
inline Big pow2k(Big base, int k) {  // base^(2^k)
  for (int i = 0; i < k; i++) base = mulmod(base, base);
  return base;
}

// LCG state -> the 24 RANLUX numbers packed in 576 bits + carry (reading D4, shift/add form):
//   Xh = X >> 336, S = (X mod 2^336) + Xh, D = S 2^240 - S - Xh 2^336, T = Xh - [D < 0], V = X + T,
//   c = (V >> 336) - T.  X must be canonical (< m).
inline void to_ranlux(const Big& X, uint32_t v[18], uint32_t* carry) {
  const Big Xh = Big::shr(X, 336);
  const Big S = Big::add(Big::low_bits(X, 336), Xh);
  const bool neg = Big::cmp(Big::shl(S, 240), Big::add(S, Big::shl(Xh, 336))) < 0;
  const Big T = neg ? Big::sub(Xh, Big(1)) : Xh;  // D < 0 implies Xh >= 1
  const Big V = Big::add(X, T);
  V.to_u32x18(v);
  if (carry) {
    const Big d = Big::sub(Big::shr(V, 336), T);
    *carry = d.is_zero() ? 0u : d.w[0];
  }
}
inline Big from_u64x9(const uint64_t in[9]) {
  Big r;
  r.w.resize(18);
  for (int i = 0; i < 9; i++) {
    r.w[2 * i] = (uint32_t)in[i];
    r.w[2 * i + 1] = (uint32_t)(in[i] >> 32);
  }
  r.trim();
  return r;
}

}  // namespace host
}  // namespace rlx
