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
  static __device__ __forceinline__ T mul(T a, T b) { return a * b; }
  static __device__ __forceinline__ T add(T a, T b) { return a + b; }
  static __device__ __forceinline__ T from_small(uint32_t x) { return x; }
};

template <uint32_t P>
struct RingMod {
  using T = uint32_t;
  static __device__ __forceinline__ T mul(T a, T b) { return (T)(((uint64_t)a * b) % P); }
  static __device__ __forceinline__ T add(T a, T b) { uint32_t s = a + b; return s >= P ? s - P : s; }   // a,b < 2^31
  static __device__ __forceinline__ T from_small(uint32_t x) { return x % P; }
};

using RingP1 = RingMod<2147483647u>;
using RingP2 = RingMod<2147483629u>;

constexpr int32_t NEG_INF = -(1 << 30);
constexpr int32_t ZERO_BELOW = -(1 << 29);

// acc (+)= (e, c)
template <class R>
__device__ __forceinline__ void oplus(int32_t &acc_e, typename R::T &acc_c, int32_t e, typename R::T c) {
  if (e > acc_e) { acc_e = e; acc_c = c; }
  else if (e == acc_e) acc_c = R::add(acc_c, c);
}

template <class R>
__device__ __forceinline__ void canonicalise(int32_t &e, typename R::T &c) {
  if (e < ZERO_BELOW) { e = NEG_INF; c = 0; }
}

}  // namespace bbtn

// dispatch a templated launcher over the ring id
#define BBTN_RING_DISPATCH(ring, ...)                                   \
  do {                                                                  \
    if ((ring) == 0) { using R = ::bbtn::RingU64; __VA_ARGS__; }        \
    else if ((ring) == 1) { using R = ::bbtn::RingP1; __VA_ARGS__; }    \
    else { using R = ::bbtn::RingP2; __VA_ARGS__; }                     \
  } while (0)
