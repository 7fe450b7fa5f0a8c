// vc_state.cuh — device-resident proof state and launch-shape constants shared by the kernels
// and the host driver of libvc.so.  (Nothing here is shared with oracle/.)
#pragma once
#include <stdint.h>

namespace vc {

constexpr int MAX_LOG = 31;        // layers of up to 2^30 gates / tables of 2^31 would not fit anyway
constexpr int MAX_VARS = 64;
constexpr int RED_BLOCK = 256;     // threads per block of the streaming kernels
constexpr int MAX_PART_BLOCKS = 4096;

// Proof state kept on the device between kernels and between vc_prove_layer calls
// (BASELINE.json north_star (3): challenges come from a seeded PRNG kept on the device).
struct DevState {
    uint64_t seed;
    uint64_t ctr;              // next challenge index k of H(seed,k)
    uint64_t claim;            // current claim  V~_i(z)
    uint64_t r;                // latest round challenge
    uint64_t v1, v2;           // A[0] after phase 1, B[0] after phase 2
    uint64_t z[MAX_VARS];      // current claim point
    uint64_t r1[MAX_VARS];     // phase-1 challenges (bind the bits of in1)
    uint64_t r2[MAX_VARS];     // phase-2 challenges (bind the bits of in2)
    uint64_t G[4];             // last round's message (debug)
    unsigned int ticket;       // last-block-done counter of the streaming kernels
    unsigned int flags;        // bit 0: non-canonical input word seen
    unsigned int bar_count;    // rendezvous counter of k_eval_all (directly behind flags: one memset clears both)
    unsigned int bar_gen;
    uint64_t invfact[MAX_VARS + 1];  // 1/k! mod p, written once at load (Lagrange denominators)
};

// Implicit wiring by bit fields (for regular circuits the in-neighbours of a gate
// are "determined with very little arithmetic and no global memory accesses").  An index is
//     in(g) = ( c + sum_f ((g >> p0_f) & (2^len_f - 1)) << q0_f ) & mask,      at most three fields per index,
// which covers the add trees (in = 2g, 2g+1), the squaring layers (g), the two lanes of the square-and-multiply chain
// (g', g' + n by lane), the matrix-product layer (i m + k, m^2 + k m + j from g = (i m + j) m + k) and the sliding window
// of the pattern matcher ((i + j) mod T, T + j from g = i Q + j).  The gate type is t[bit tbit of g] (two lanes) or t[0].
// Unpacked so that the device evaluates a field in four instructions: m = 2^len - 1, and an unused field has m = 0.
struct WireField { uint32_t p0, m, q0, pad; };
struct alignas(16) WireRule {
    WireField f[2][3];
    uint32_t c[2], mask[2];             // mask[w] = 2^k - 1, the smallest that holds every index of operand w (a cyclic window wraps at it)
    uint32_t t[2], tbit, tm;             // type = t[(g >> tbit) & tm]; tm = 0: one type
};

}  // namespace vc
