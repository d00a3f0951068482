// ring.cuh -- count rings and the counting-tropical element on the device.
//
// element = (energy int32, count in a ring R).  (.) adds energies and multiplies counts,
// (+) keeps the larger energy and adds counts on ties (zero = (-inf, 0), :55).
// R is Z/2^64 (wrapping uint64: a ring homomorphic image of the exact count) or Z/p for the two
// 31-bit primes of include/bbtn.h (CRT mode).
#pragma once
#include <cstdint>

namespace bbtn {

struct RingU64 {
  using T = uint64_t;
  static constexpr bool kCounts = true;
  static __device__ __forceinline__ T mul(T a, T b) { return a * b; }
  static __device__ __forceinline__ T add(T a, T b) { return a + b; }
  static __device__ __forceinline__ T from_small(uint32_t x) { return x; }
};

template <uint32_t P>
struct RingMod {
  using T = uint32_t;
  static constexpr bool kCounts = true;
  // P = 2^31 - C with a small C (1 and 19 for the two primes), so 2^31 == C (mod P): fold the high part of the
  // 62-bit product down twice instead of dividing.  x = hi*2^31 + lo  ->  hi*C + lo < (C+1)*2^31  ->  < 2^31 + C*(C+1).
  static constexpr uint32_t C = 0x80000000u - P;
  static_assert(C >= 1 && C <= 64, "RingMod expects a prime just below 2^31");
  static __device__ __forceinline__ T mul(T a, T b) {
    const uint64_t x = (uint64_t)a * b;                                   // a, b < P  =>  x < 2^62
    const uint64_t y = (uint64_t)(uint32_t)(x >> 31) * C + ((uint32_t)x & 0x7fffffffu);
    const uint32_t z = (uint32_t)(y >> 31) * C + ((uint32_t)y & 0x7fffffffu);   // < 2^31 + C*(C+1) < 2P
    return z >= P ? z - P : z;
  }
  static __device__ __forceinline__ T add(T a, T b) { uint32_t s = a + b; return s >= P ? s - P : s; }   // a,b < 2^31
  static __device__ __forceinline__ T from_small(uint32_t x) { return x % P; }
};

// Search mode (PAPER.md:55 "the tropical number inf for optimization problems"; :81-91): plain max-plus, no count
// plane at all.  The count type is an empty object; kernels reach counts only through ldc/stc below, which touch no
// memory for this ring, so the planes may be null.
struct NoCount {};
struct RingNone {
  using T = NoCount;
  static constexpr bool kCounts = false;
  static __device__ __forceinline__ T mul(T, T) { return T{}; }
  static __device__ __forceinline__ T add(T, T) { return T{}; }
  static __device__ __forceinline__ T from_small(uint32_t) { return T{}; }
};

using RingP1 = RingMod<2147483647u>;
using RingP2 = RingMod<2147483629u>;

// Both primes at once (CRT mode, streaming and fused kernels): the residue mod P1 in the low word and the residue
// mod P2 in the high word of one 64-bit count, so the two prime passes share one read of the energy planes.
struct RingP12 {
  using T = uint64_t;
  static constexpr bool kCounts = true;
  static __device__ __forceinline__ T pack(uint32_t r1, uint32_t r2) { return (uint64_t)r1 | ((uint64_t)r2 << 32); }
  static __device__ __forceinline__ T mul(T a, T b) {
    return pack(RingP1::mul((uint32_t)a, (uint32_t)b), RingP2::mul((uint32_t)(a >> 32), (uint32_t)(b >> 32)));
  }
  static __device__ __forceinline__ T add(T a, T b) {
    return pack(RingP1::add((uint32_t)a, (uint32_t)b), RingP2::add((uint32_t)(a >> 32), (uint32_t)(b >> 32)));
  }
  static __device__ __forceinline__ T from_small(uint32_t x) { return pack(RingP1::from_small(x), RingP2::from_small(x)); }
};

constexpr int32_t NEG_INF = -(1 << 30);
constexpr int32_t ZERO_BELOW = -(1 << 29);

// count-plane accesses (no-ops for RingNone)
template <class R> __device__ __forceinline__ typename R::T ldc(const typename R::T *p, int64_t i) {
  if constexpr (R::kCounts) return p[i]; else return typename R::T{};
}
template <class R> __device__ __forceinline__ void stc(typename R::T *p, int64_t i, typename R::T v) {
  if constexpr (R::kCounts) p[i] = v;
}
template <class R> __device__ __forceinline__ typename R::T czero() {
  if constexpr (R::kCounts) return (typename R::T)0; else return typename R::T{};
}
template <class R> __device__ __forceinline__ typename R::T shfl_xor_c(typename R::T v, int d) {
  if constexpr (R::kCounts) return __shfl_xor_sync(0xffffffffu, v, d); else return v;
}

// acc (+)= (e, c)
template <class R>
__device__ __forceinline__ void oplus(int32_t &acc_e, typename R::T &acc_c, int32_t e, typename R::T c) {
  if (e > acc_e) { acc_e = e; acc_c = c; }
  else if (e == acc_e) acc_c = R::add(acc_c, c);
}

template <class R>
__device__ __forceinline__ void canonicalise(int32_t &e, typename R::T &c) {
  if (e < ZERO_BELOW) { e = NEG_INF; c = czero<R>(); }
}

}  // namespace bbtn

// dispatch a templated launcher over the ring id.  The two primes only ever run packed (RingP12: CRT mode's second
// pass), so the single-prime rings RingP1 / RingP2 are building blocks, not launch targets.
#define BBTN_RING_DISPATCH(ring, ...)                                   \
  do {                                                                  \
    if ((ring) == 0) { using R = ::bbtn::RingU64; __VA_ARGS__; }        \
    else if ((ring) == 4) { using R = ::bbtn::RingP12; __VA_ARGS__; }   \
    else { using R = ::bbtn::RingNone; __VA_ARGS__; }                   \
  } while (0)
