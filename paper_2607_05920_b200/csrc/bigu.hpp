// bigu.hpp -- minimal host-side unsigned big integer for context precomputation (tables only; never on the hot path).
// Little-endian uint32 limbs, always normalised (no leading zero limbs; zero = empty vector).
#pragma once
#include <algorithm>
#include <cstdint>
#include <vector>

namespace fhe {

struct BigU {
  std::vector<uint32_t> v;

  BigU() {}
  explicit BigU(uint64_t x) {
    while (x) { v.push_back((uint32_t)x); x >>= 32; }
  }
  static BigU pow2(uint32_t e) {
    BigU r;
    r.v.assign(e / 32 + 1, 0u);
    r.v[e / 32] = 1u << (e % 32);
    return r;
  }
  void trim() { while (!v.empty() && v.back() == 0) v.pop_back(); }
  bool is_zero() const { return v.empty(); }
  uint32_t bits() const {
    if (v.empty()) return 0;
    uint32_t top = v.back(), b = 0;
    while (top) { ++b; top >>= 1; }
    return (uint32_t)(v.size() - 1) * 32 + b;
  }
  bool bit(uint32_t i) const { return i / 32 < v.size() && ((v[i / 32] >> (i % 32)) & 1u); }
  uint32_t limb(size_t i) const { return i < v.size() ? v[i] : 0u; }

  static int cmp(const BigU& a, const BigU& b) {
    if (a.v.size() != b.v.size()) return a.v.size() < b.v.size() ? -1 : 1;
    for (size_t i = a.v.size(); i-- > 0;)
      if (a.v[i] != b.v[i]) return a.v[i] < b.v[i] ? -1 : 1;
    return 0;
  }
  BigU& add(const BigU& b) {
    if (v.size() < b.v.size()) v.resize(b.v.size(), 0u);
    uint64_t c = 0;
    for (size_t i = 0; i < v.size(); ++i) {
      c += (uint64_t)v[i] + b.limb(i);
      v[i] = (uint32_t)c;
      c >>= 32;
    }
    if (c) v.push_back((uint32_t)c);
    return *this;
  }
  BigU& add_small(uint32_t x) { return add(BigU((uint64_t)x)); }
  // requires *this >= b
  BigU& sub(const BigU& b) {
    int64_t c = 0;
    for (size_t i = 0; i < v.size(); ++i) {
      int64_t d = (int64_t)v[i] - (int64_t)b.limb(i) + c;
      v[i] = (uint32_t)d;
      c = d >> 32;  // arithmetic shift: 0 or -1
    }
    trim();
    return *this;
  }
  BigU& mul_small(uint32_t m) {
    uint64_t c = 0;
    for (size_t i = 0; i < v.size(); ++i) {
      c += (uint64_t)v[i] * m;
      v[i] = (uint32_t)c;
      c >>= 32;
    }
    if (c) v.push_back((uint32_t)c);
    trim();
    return *this;
  }
  static BigU mul(const BigU& a, const BigU& b) {
    BigU r;
    if (a.is_zero() || b.is_zero()) return r;
    r.v.assign(a.v.size() + b.v.size(), 0u);
    for (size_t i = 0; i < a.v.size(); ++i) {
      uint64_t c = 0;
      for (size_t j = 0; j < b.v.size(); ++j) {
        c += (uint64_t)a.v[i] * b.v[j] + r.v[i + j];
        r.v[i + j] = (uint32_t)c;
        c >>= 32;
      }
      r.v[i + b.v.size()] = (uint32_t)c;
    }
    r.trim();
    return r;
  }
  // exact or floor division by a word; returns remainder
  uint32_t divmod_small(uint32_t d) {
    uint64_t r = 0;
    for (size_t i = v.size(); i-- > 0;) {
      uint64_t cur = (r << 32) | v[i];
      v[i] = (uint32_t)(cur / d);
      r = cur % d;
    }
    trim();
    return (uint32_t)r;
  }
  uint32_t mod_small(uint32_t d) const {
    uint64_t r = 0;
    for (size_t i = v.size(); i-- > 0;) r = ((r << 32) | v[i]) % d;
    return (uint32_t)r;
  }
  BigU& shl1() {
    uint32_t c = 0;
    for (size_t i = 0; i < v.size(); ++i) {
      uint32_t n = v[i] >> 31;
      v[i] = (v[i] << 1) | c;
      c = n;
    }
    if (c) v.push_back(c);
    return *this;
  }
  BigU low_bits(uint32_t nb) const {
    BigU r;
    size_t nl = (nb + 31) / 32;
    r.v.assign(v.begin(), v.begin() + std::min(nl, v.size()));
    if (nb % 32 && r.v.size() == nl) r.v[nl - 1] &= (1u << (nb % 32)) - 1u;
    r.trim();
    return r;
  }
  // binary long division: quotient and remainder of a / m (m != 0).  Sizes here are a few thousand bits.
  static void divmod(const BigU& a, const BigU& m, BigU& q, BigU& r) {
    q = BigU();
    r = BigU();
    uint32_t nb = a.bits();
    q.v.assign((nb + 31) / 32, 0u);
    for (uint32_t i = nb; i-- > 0;) {
      r.shl1();
      if (a.bit(i)) {
        if (r.v.empty()) r.v.push_back(1u); else r.v[0] |= 1u;
      }
      if (cmp(r, m) >= 0) {
        r.sub(m);
        q.v[i / 32] |= 1u << (i % 32);
      }
    }
    q.trim();
  }
  static BigU mod(const BigU& a, const BigU& m) {
    BigU q, r;
    divmod(a, m, q, r);
    return r;
  }
  // value as fixed-length limb array
  void to_limbs(uint32_t* out, size_t n) const {
    for (size_t i = 0; i < n; ++i) out[i] = limb(i);
  }
};

}  // namespace fhe
