// vc_round.cuh — streaming schedule, steps a4-a6: the per-round gate-contribution kernel with its
// block+grid reduction and device-side challenge, and the weight-update / table-fold kernel.
#pragma once
#include "vc_kernels.cuh"

namespace vc {

// One gate's contribution to round j of a phase ("each gate
// contributes to only a single term of this sum"):
//   for t in {0,1,2}:  P[g] * chi(b,t) * f_type(x(t), other)   [phase 1]   /  f_type(other, x(t))  [phase 2]
// with x(t) = lo + t (hi - lo).  chi(b,0) = 1-b, chi(b,1) = b, chi(b,2) = 2 if b else -1, so a gate
// feeds exactly two of the three sums: G[b] with weight P and G[2] with weight 2P or -P.
// For MULT the fixed operand is folded into the weight first (Pf = P*other), so the two terms cost
// one multiply each.
template <int PHASE>
__device__ __forceinline__ void gate_terms(uint32_t t, uint64_t Pg, uint64_t other, uint32_t b, uint64_t lo,
                                           uint64_t hi, acc128 &a0, acc128 &a1, acc128 &a2) {
    const uint64_t xb = b ? hi : lo;
    const uint64_t x2 = fp61::sub(fp61::dbl(hi), lo);
    uint64_t Pf = Pg, fb, f2;
    if (t == 1) {  // MULT
        Pf = fp61::mul(Pg, other); fb = xb; f2 = x2;
    } else if (t == 0) {  // ADD
        fb = fp61::add(xb, other); f2 = fp61::add(x2, other);
    } else if (t == 2) {  // SUB
        if (PHASE == 1) { fb = fp61::sub(xb, other); f2 = fp61::sub(x2, other); }
        else { fb = fp61::sub(other, xb); f2 = fp61::sub(other, x2); }
    } else {  // RELAY: f = L
        if (PHASE == 1) { fb = xb; f2 = x2; }
        else { fb = other; f2 = other; }
    }
    const uint64_t c2 = b ? fp61::dbl(Pf) : fp61::neg(Pf);
    // predicated accumulate into G[b]
    const uint64_t pl = Pf * fb, ph = fp61::mulhi(Pf, fb);
    if (b) { a1.lo += pl; a1.hi += ph + (a1.lo < pl); }
    else   { a0.lo += pl; a0.hi += ph + (a0.lo < pl); }
    a2.mac(c2, f2);
}

// Round j of phase PHASE over all n gates of the layer.
//   tab  : the fold table A_j (phase 1) or B_j (phase 2): 2^{s-j} words
//   Vb   : V_{i+1} (phase 1: the fixed operand V_{i+1}[in2[g]])
// The last block writes (G0,G1,G2) to tr[0..2], draws r = H(seed, ctr++), stores it in st->r and
// st->r1[j] / st->r2[j].
template <int PHASE>
__global__ void __launch_bounds__(RED_BLOCK)
k_round(const uint8_t *__restrict__ type, const uint32_t *__restrict__ in1, const uint32_t *__restrict__ in2,
        const uint64_t *__restrict__ Pw, const uint64_t *__restrict__ tab, const uint64_t *__restrict__ Vb,
        DevState *st, uint32_t j, uint32_t n, uint64_t *part, uint64_t *tr) {
    __shared__ uint64_t red[3 * 32];
    acc128 a0, a1, a2; a0.clear(); a1.clear(); a2.clear();
    uint64_t s0 = 0, s1 = 0, s2 = 0; int it = 0;
    const uint64_t v1 = PHASE == 2 ? st->v1 : 0;
    for (uint32_t g = blockIdx.x * blockDim.x + threadIdx.x; g < n; g += gridDim.x * blockDim.x) {
        const uint32_t t = type[g], i1 = in1[g], i2 = in2[g];
        const uint32_t idx = PHASE == 1 ? i1 : i2;
        const uint32_t b = (idx >> j) & 1u, u = idx >> (j + 1);
        const ulonglong2 pr = *reinterpret_cast<const ulonglong2 *>(tab + 2 * (size_t)u);
        const uint64_t other = PHASE == 1 ? Vb[i2] : v1;
        gate_terms<PHASE>(t, Pw[g], other, b, pr.x, pr.y, a0, a1, a2);
        if (++it == 32) {
            s0 = fp61::add(s0, a0.value()); s1 = fp61::add(s1, a1.value()); s2 = fp61::add(s2, a2.value());
            a0.clear(); a1.clear(); a2.clear(); it = 0;
        }
    }
    uint64_t v[3] = {fp61::add(s0, a0.value()), fp61::add(s1, a1.value()), fp61::add(s2, a2.value())};
    if (grid_sum_last_block<3>(v, part, st, red) && threadIdx.x == 0) {
        tr[0] = v[0]; tr[1] = v[1]; tr[2] = v[2];
        st->G[0] = v[0]; st->G[1] = v[1]; st->G[2] = v[2];
        const uint64_t r = fp61::draw(st->seed, st->ctr);
        st->ctr += 1;
        st->r = r;
        if (PHASE == 1) st->r1[j] = r; else st->r2[j] = r;
    }
}

// a6: P[g] *= chi(bit_j(idx[g]), r);  fold: out[u] = tab[2u] + r (tab[2u+1] - tab[2u]), u < half.
// When half == 1 the single folded value is V~_{i+1}(r1) (resp. r2): stored as v1 (resp. v2).
template <int PHASE>
__global__ void __launch_bounds__(RED_BLOCK)
k_update(const uint32_t *__restrict__ idx, uint64_t *__restrict__ Pw, const uint64_t *__restrict__ tab,
         uint64_t *__restrict__ out, DevState *st, uint32_t j, uint32_t n, uint32_t half) {
    const uint64_t r = st->r, omr = fp61::sub(1, r);
    const uint32_t tid = blockIdx.x * blockDim.x + threadIdx.x, stride = gridDim.x * blockDim.x;
    for (uint32_t g = tid; g < n; g += stride) {
        const uint32_t b = (idx[g] >> j) & 1u;
        Pw[g] = fp61::mul(Pw[g], b ? r : omr);
    }
    for (uint32_t u = tid; u < half; u += stride) {
        const ulonglong2 pr = *reinterpret_cast<const ulonglong2 *>(tab + 2 * (size_t)u);
        const uint64_t f = fp61::add(pr.x, fp61::mul(r, fp61::sub(pr.y, pr.x)));
        out[u] = f;
        if (half == 1) { if (PHASE == 1) st->v1 = f; else st->v2 = f; }
    }
}

}  // namespace vc
