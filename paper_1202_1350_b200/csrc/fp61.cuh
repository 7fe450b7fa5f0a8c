// fp61.cuh — F_p arithmetic, p = 2^61 - 1, for sm_100a device code (§6.1; PAPER.md:175:
// "multiplying two field elements requires three machine multiplications of 64-bit data types, and a
// handful of additions and bit shifts").  Header-only; nothing here is shared with oracle/.
//
// Representation: canonical uint64 in [0,p).  A product of two canonical words is < 2^122, so the
// 128-bit product (lo = a*b, hi = __umul64hi(a,b)) folds with 2^61 = 1 (mod p):
//   a*b = (lo & p) + (lo >> 61 | hi << 3)   (mod p),   both terms < 2^61 -> sum < 2^62.
// Lazy accumulation: acc128 collects up to 64 unreduced 122-bit products before one fold.
#pragma once
#include <stdint.h>

namespace fp61 {

constexpr uint64_t P = 0x1FFFFFFFFFFFFFFFULL;

__host__ __device__ __forceinline__ uint64_t reduce62(uint64_t x) {  // x < 2^62 + small -> [0,p)
    x = (x & P) + (x >> 61);
    return x >= P ? x - P : x;
}
__host__ __device__ __forceinline__ uint64_t add(uint64_t a, uint64_t b) {
    uint64_t s = a + b;
    return s >= P ? s - P : s;
}
__host__ __device__ __forceinline__ uint64_t sub(uint64_t a, uint64_t b) {
    return a >= b ? a - b : a + P - b;
}
__host__ __device__ __forceinline__ uint64_t neg(uint64_t a) { return a ? P - a : 0; }
__host__ __device__ __forceinline__ uint64_t dbl(uint64_t a) { return add(a, a); }

#ifdef __CUDA_ARCH__
__device__ __forceinline__ uint64_t mulhi(uint64_t a, uint64_t b) { return __umul64hi(a, b); }
#else
__host__ __forceinline__ uint64_t mulhi(uint64_t a, uint64_t b) {
    return (uint64_t)(((unsigned __int128)a * b) >> 64);
}
#endif

// fold a 128-bit value (hi < 2^61 guaranteed by callers: at most 64 products) to canonical
__host__ __device__ __forceinline__ uint64_t fold128(uint64_t hi, uint64_t lo) {
    // value = hi*2^64 + lo;  2^64 = 8 (mod p)  ->  lo&p + lo>>61 + hi*8 pieces
    uint64_t x = (lo & P) + ((lo >> 61) | ((hi << 3) & P)) + (hi >> 58);
    return reduce62(x);  // x < 2^61 + 2^61 + 64
}
__host__ __device__ __forceinline__ uint64_t mul(uint64_t a, uint64_t b) {
    uint64_t lo = a * b, hi = mulhi(a, b);  // hi < 2^58
    uint64_t x = (lo & P) + ((lo >> 61) | (hi << 3));
    return x >= P ? x - P : x;
}

// 128-bit lazy accumulator of full products
struct acc128 {
    uint64_t lo, hi;
    __host__ __device__ __forceinline__ void clear() { lo = 0; hi = 0; }
    __host__ __device__ __forceinline__ void mac(uint64_t a, uint64_t b) {  // += a*b (unreduced)
        uint64_t pl = a * b, ph = mulhi(a, b);
        lo += pl;
        hi += ph + (lo < pl);
    }
    __host__ __device__ __forceinline__ void addw(uint64_t w) {  // += w
        lo += w;
        hi += (lo < w);
    }
    __host__ __device__ __forceinline__ uint64_t value() const { return fold128(hi, lo); }
};

#ifdef __CUDACC__
// (lo,hi) += a*b, and, if pred, (lo1,hi1) += a*b too: one 64x64->128 product, two carry-chain adds (the second predicated)
__device__ __forceinline__ void mac2(uint64_t &lo, uint64_t &hi, uint64_t &lo1, uint64_t &hi1, uint64_t a, uint64_t b,
                                     uint32_t pred) {
    asm("{\n\t.reg .u64 pl, ph;\n\t.reg .pred p;\n\t"
        "setp.ne.u32 p, %6, 0;\n\t"
        "mul.lo.u64 pl, %4, %5;\n\tmul.hi.u64 ph, %4, %5;\n\t"
        "add.cc.u64 %0, %0, pl;\n\taddc.u64 %1, %1, ph;\n\t"
        "@p add.cc.u64 %2, %2, pl;\n\t@p addc.u64 %3, %3, ph;\n\t}"
        : "+l"(lo), "+l"(hi), "+l"(lo1), "+l"(hi1)
        : "l"(a), "l"(b), "r"(pred));
}
#endif

// chi(b, x) = x if b else 1 - x
__host__ __device__ __forceinline__ uint64_t chi(uint32_t b, uint64_t x) { return b ? x : sub(1, x); }

// counter-based challenge generator (reading c-11): splitmix64 stream, output number k
__host__ __device__ __forceinline__ uint64_t draw(uint64_t seed, uint64_t k) {
    uint64_t x = seed + (k + 1) * 0x9E3779B97F4A7C15ULL;
    x ^= x >> 30; x *= 0xBF58476D1CE4E5B9ULL;
    x ^= x >> 27; x *= 0x94D049BB133111EBULL;
    x ^= x >> 31;
    x &= P;
    return x == P ? 0 : x;
}

}  // namespace fp61
