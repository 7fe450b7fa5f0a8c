/* oracle/gkr_oracle.c — O-cmt: plain, slow, single-threaded CPU prover + verifier for the GKR
 * layer sum-check over F_p, p = 2^61 - 1.
 *
 * TEST INFRASTRUCTURE ONLY.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this.  It shares no code, header, table or constant with the
 * CUDA path (paper_1202_1350_b200/csrc); the two agree only through the paper's mathematics.
 *
 * What it follows:
 *   - PAPER.md:93-101 (§3.1): one iteration per circuit layer; V's challenges are random field
 *     elements; P's responses are low-degree polynomials given by their evaluations; iteration i
 *     involves only two adjacent layers.
 *   - PAPER.md:121-123 (§4.1.1): each gate contributes independently to exactly one term of each
 *     message, so one pass over the layer's gates per message, all arithmetic in F_p.
 *   - PAPER.md:197 (§6.1): F_p with p = 2^61 - 1, integers embed naturally, no floating point.
 *   - SURVEY.md §8(c) "Algorithm (O-cmt)" for every convention the paper leaves open (layer
 *     numbering, variable order, message format t = 0,1,2, gate types, the two-claims->one line
 *     reduction, the challenge generator).  Those readings are listed in DESIGN.md.
 *
 * Parity pins (tests/test_oracle_*.py, -m "not gpu"): field ops vs Python big ints; eq tables and
 * MLEs vs the literal product/sum definition; every round message vs the exponential-size sum of
 * oracle/gkr_def.py on tiny random circuits with all four gate types; g(0)+g(1) = claim in every
 * round at every size; A[0] = V~(r1), B[0] = V~(r2); wiring sums; line restriction; circuit outputs
 * vs directly computed F2 / F0 / matmul / pattern counts; verifier accepts honest transcripts and
 * rejects any single-word tamper at the predicted (layer, round).
 * PARITY UNPINNED (conventions of this build, fixed by no printed value in the paper): the challenge
 * stream H(seed,k) beyond its published splitmix64 known-answer, the bit order of the bound
 * variables, the transcript layout and the gate-type codes.
 *
 * Arithmetic: unsigned __int128 products and the C '%' operator; no Mersenne tricks, no blocking,
 * no reordering beyond the per-gate pass the paper states.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef unsigned __int128 u128;

#define ORC_P ((uint64_t)2305843009213693951ULL) /* 2^61 - 1 */

enum { ORC_ADD = 0, ORC_MULT = 1, ORC_SUB = 2, ORC_RELAY = 3, ORC_SUM = 4 };
enum { ORC_OK = 0, ORC_ERR_ARG = 1, ORC_ERR_SHAPE = 2, ORC_ERR_NOMEM = 5 };

typedef struct {
    uint32_t log_size;     /* layer has 2^log_size gates */
    const uint8_t *type;   /* 0 ADD, 1 MULT, 2 SUB, 3 RELAY; 4 SUM only as the single gate of layer 0 (see orc_prove_sum_layer) */
    const uint32_t *in1;   /* indices into the layer below */
    const uint32_t *in2;
} orc_layer;

/* Optional per-layer debug record for the pins. */
typedef struct {
    uint64_t r1[64];
    uint64_t r2[64];
    uint64_t v1, v2;
    uint64_t Wsum[4];      /* sum over gates of type tau of the final weight P[g] */
    uint64_t tau;
} orc_layer_debug;

/* ---------------------------------------------------------------- field */
uint64_t orc_p(void) { return ORC_P; }
uint64_t orc_add(uint64_t a, uint64_t b) { return (uint64_t)(((u128)a + b) % ORC_P); }
uint64_t orc_sub(uint64_t a, uint64_t b) { return (uint64_t)(((u128)a + ORC_P - b) % ORC_P); }
uint64_t orc_mul(uint64_t a, uint64_t b) { return (uint64_t)(((u128)a * b) % ORC_P); }
uint64_t orc_pow(uint64_t a, uint64_t e) {
    uint64_t r = 1;
    while (e) { if (e & 1) r = orc_mul(r, a); a = orc_mul(a, a); e >>= 1; }
    return r;
}
uint64_t orc_inv(uint64_t a) { return orc_pow(a, ORC_P - 2); } /* Fermat */

/* chi(b,x) = x if b = 1 else 1 - x  (SURVEY.md §8 conventions) */
static uint64_t chi(uint32_t b, uint64_t x) { return b ? x : orc_sub(1, x); }

/* gate function by type (reading c-3) */
static uint64_t gate_f(uint8_t t, uint64_t L, uint64_t R) {
    switch (t) {
    case ORC_ADD: return orc_add(L, R);
    case ORC_MULT: return orc_mul(L, R);
    case ORC_SUB: return orc_sub(L, R);
    default: return L; /* RELAY */
    }
}

/* ---------------------------------------------------------------- challenges (reading c-11)
 * H(seed,k) = splitmix64 output number k of the stream seeded with `seed`:
 * state_k = seed + (k+1)*0x9E3779B97F4A7C15, then the splitmix64 finaliser.
 * to_field: keep the low 61 bits; if that equals p use 0. */
uint64_t orc_mix(uint64_t seed, uint64_t k) {
    uint64_t x = seed + (k + 1) * 0x9E3779B97F4A7C15ULL;
    x = (x ^ (x >> 30)) * 0xBF58476D1CE4E5B9ULL;
    x = (x ^ (x >> 27)) * 0x94D049BB133111EBULL;
    return x ^ (x >> 31);
}
uint64_t orc_draw(uint64_t seed, uint64_t k) {
    uint64_t v = orc_mix(seed, k) & ORC_P;
    return v == ORC_P ? 0 : v;
}

/* ---------------------------------------------------------------- eq tables and MLEs
 * T[u] = eq(u,x) = prod_k chi(u_k, x_k), built one variable at a time (variable k = bit k). */
void orc_eq_table(const uint64_t *x, uint32_t s, uint64_t *T) {
    T[0] = 1;
    for (uint32_t k = 0; k < s; k++) {
        uint64_t half = (uint64_t)1 << k;
        for (uint64_t u = 0; u < half; u++) {
            uint64_t e = T[u];
            T[u] = orc_mul(e, chi(0, x[k]));
            T[u + half] = orc_mul(e, chi(1, x[k]));
        }
    }
}

/* V~(x) = sum_u eq(u,x) V[u] */
uint64_t orc_mle(const uint64_t *V, uint32_t s, const uint64_t *x) {
    uint64_t n = (uint64_t)1 << s, acc = 0;
    uint64_t *T = (uint64_t *)malloc(n * sizeof(uint64_t));
    if (!T) return ~(uint64_t)0;
    orc_eq_table(x, s, T);
    for (uint64_t u = 0; u < n; u++) acc = orc_add(acc, orc_mul(T[u], V[u]));
    free(T);
    return acc;
}

/* The sum gate of very large fan-in at the output (reading c-19): layer 0 is ONE gate of type SUM whose
 * in-neighbours are all gates of layer 1 (in1/in2 are not read). */
static int is_sum_layer(const orc_layer *L) { return L->log_size == 0 && L->type[0] == ORC_SUM; }

/* ---------------------------------------------------------------- evaluation (a1)
 * V[d] <- input; for i = d-1..0: V_i[g] = f_type(V_{i+1}[in1[g]], V_{i+1}[in2[g]]).
 * V is an array of d+1 caller-allocated buffers. */
int orc_evaluate(const orc_layer *layers, uint32_t d, uint32_t log_input, const uint64_t *input,
                 uint64_t *const *V) {
    uint64_t n_in = (uint64_t)1 << log_input;
    for (uint64_t u = 0; u < n_in; u++) {
        if (input[u] >= ORC_P) return ORC_ERR_ARG;
        V[d][u] = input[u];
    }
    for (int64_t i = (int64_t)d - 1; i >= 0; i--) {
        const orc_layer *L = &layers[i];
        uint64_t n = (uint64_t)1 << L->log_size;
        uint64_t nb = (uint64_t)1 << ((uint32_t)i + 1 < d ? layers[i + 1].log_size : log_input);
        if (i == 0 && is_sum_layer(L)) {            /* y = sum of every value of layer 1 */
            uint64_t acc = 0;
            for (uint64_t u = 0; u < nb; u++) acc = orc_add(acc, V[1][u]);
            V[0][0] = acc;
            continue;
        }
        for (uint64_t g = 0; g < n; g++) {
            if (L->type[g] > 3 || L->in1[g] >= nb || L->in2[g] >= nb) return ORC_ERR_SHAPE;
            V[i][g] = gate_f(L->type[g], V[i + 1][L->in1[g]], V[i + 1][L->in2[g]]);
        }
    }
    return ORC_OK;
}

/* ---------------------------------------------------------------- start claim (a2)
 * z_0 = s_0 draws; claim = V~_0(z_0). */
int orc_start(const uint64_t *V0, uint32_t s0, uint64_t seed, uint64_t *ctr, uint64_t *z, uint64_t *claim) {
    for (uint32_t k = 0; k < s0; k++) z[k] = orc_draw(seed, (*ctr)++);
    *claim = orc_mle(V0, s0, z);
    return ORC_OK;
}

/* Lagrange interpolation on nodes 0..n-1 evaluated at tau (plain formula with field inverses). */
uint64_t orc_lagrange(const uint64_t *q, uint32_t n, uint64_t tau) {
    uint64_t tot = 0;
    for (uint32_t k = 0; k < n; k++) {
        uint64_t num = 1, den = 1;
        for (uint32_t m = 0; m < n; m++) {
            if (m == k) continue;
            num = orc_mul(num, orc_sub(tau, m));
            den = orc_mul(den, orc_sub(k, m));
        }
        tot = orc_add(tot, orc_mul(q[k], orc_mul(num, orc_inv(den))));
    }
    return tot;
}

/* value at r of the degree-<=2 polynomial through (0,G0),(1,G1),(2,G2) */
uint64_t orc_interp2(const uint64_t *G, uint64_t r) { return orc_lagrange(G, 3, r); }

/* ---------------------------------------------------------------- one layer of the prover (a3-a7)
 * L      : the gates of layer i;  s_i = L->log_size
 * s      : log2 size of layer i+1;  Vb = V_{i+1} (2^s words)
 * z      : in: the claim point (s_i words); out: the next claim point (s words). Buffer >= max(s_i,s).
 * claim  : in: claimed V~_i(z); out: q(tau) = claimed V~_{i+1}(z').  (P does not use the incoming value.)
 * tr     : 7s+1 words: per round (G[0],G[1],G[2]), 2s rounds, then q[0..s].
 * Follows SURVEY.md §8(c) O-cmt line by line. */
int orc_prove_layer(const orc_layer *L, uint32_t s, const uint64_t *Vb, uint64_t seed, uint64_t *ctr,
                    uint64_t *z, uint64_t *claim, uint64_t *tr, orc_layer_debug *dbg) {
    if (s == 0 || s > 63) return ORC_ERR_SHAPE;
    uint64_t n = (uint64_t)1 << L->log_size, nb = (uint64_t)1 << s;
    uint64_t *Pw = (uint64_t *)malloc(n * sizeof(uint64_t));
    uint64_t *A = (uint64_t *)malloc(nb * sizeof(uint64_t));
    uint64_t r1[64], r2[64], q[65], pt[64];
    if (!Pw || !A) { free(Pw); free(A); return ORC_ERR_NOMEM; }
    const uint8_t *type = L->type;
    uint64_t w = 0;

    /* P[g] = eq(g,z) = beta(z,g) for all g (a3) */
    orc_eq_table(z, L->log_size, Pw);

    /* phase 1 binds bit j of in1; phase 2 binds bit j of in2 (a4-a6) */
    uint64_t v1 = 0, v2 = 0;
    for (int phase = 1; phase <= 2; phase++) {
        const uint32_t *idx = phase == 1 ? L->in1 : L->in2;
        uint64_t *rr = phase == 1 ? r1 : r2;
        memcpy(A, Vb, nb * sizeof(uint64_t)); /* A (resp. B) = copy(V_{i+1}) */
        for (uint32_t j = 0; j < s; j++) {
            uint64_t G[3];
            for (uint64_t t = 0; t < 3; t++) {
                uint64_t acc = 0;
                for (uint64_t g = 0; g < n; g++) {
                    uint32_t b = (idx[g] >> j) & 1;
                    uint64_t u = (uint64_t)idx[g] >> (j + 1);
                    uint64_t lo = A[2 * u], hi = A[2 * u + 1];
                    uint64_t x = orc_add(lo, orc_mul(t, orc_sub(hi, lo)));
                    uint64_t f = phase == 1 ? gate_f(type[g], x, Vb[L->in2[g]])
                                            : gate_f(type[g], v1, x);
                    acc = orc_add(acc, orc_mul(orc_mul(Pw[g], chi(b, t)), f));
                }
                G[t] = acc;
            }
            tr[w++] = G[0]; tr[w++] = G[1]; tr[w++] = G[2];
            uint64_t r = orc_draw(seed, (*ctr)++);
            rr[j] = r;
            for (uint64_t g = 0; g < n; g++) Pw[g] = orc_mul(Pw[g], chi((idx[g] >> j) & 1, r));
            uint64_t half = nb >> (j + 1);
            for (uint64_t u = 0; u < half; u++)
                A[u] = orc_add(A[2 * u], orc_mul(r, orc_sub(A[2 * u + 1], A[2 * u])));
        }
        if (phase == 1) v1 = A[0]; else v2 = A[0];
    }

    /* line restriction q(t) = V~_{i+1}(r1 + t (r2 - r1)), t = 0..s (a7; reading c-5) */
    for (uint32_t t = 0; t <= s; t++) {
        for (uint32_t k = 0; k < s; k++) pt[k] = orc_add(r1[k], orc_mul(t, orc_sub(r2[k], r1[k])));
        q[t] = orc_mle(Vb, s, pt);
        tr[w++] = q[t];
    }
    uint64_t tau = orc_draw(seed, (*ctr)++);
    for (uint32_t k = 0; k < s; k++) z[k] = orc_add(r1[k], orc_mul(tau, orc_sub(r2[k], r1[k])));
    *claim = orc_lagrange(q, s + 1, tau);

    if (dbg) {
        memset(dbg, 0, sizeof(*dbg));
        memcpy(dbg->r1, r1, s * sizeof(uint64_t));
        memcpy(dbg->r2, r2, s * sizeof(uint64_t));
        dbg->v1 = v1; dbg->v2 = v2; dbg->tau = tau;
        for (uint64_t g = 0; g < n; g++) dbg->Wsum[type[g]] = orc_add(dbg->Wsum[type[g]], Pw[g]);
    }
    free(Pw); free(A);
    return ORC_OK;
}

/* ---------------------------------------------------------------- the sum gate at the output (reading c-19)
 * "The GKR protocol typically assumes that all gates have fan-in two, but [8] explains how the protocol can be modified
 * to handle a single sum-gate of very large fan-in at the output."  The output is y = sum_{w in {0,1}^s} V_1[w], and V_1[w]
 * = V~_1(w) on Boolean w, so the claim "y" is a sum of the multilinear V~_1 over the cube: a sum-check over its s variables,
 * bit 0 first (reading c-2).  Round j:
 *     g_j(t) = sum over Boolean suffixes b of V~_1(r_0..r_{j-1}, t, b)          (degree 1 in t: sent as g_j(0), g_j(1))
 *     V checks g_j(0) + g_j(1) = claim, draws r_j, claim <- g_j(r_j) = g_j(0) + r_j (g_j(1) - g_j(0)).
 * After s rounds the claim is V~_1(r) at ONE point: z' = r, no line restriction and no tau.
 * A = copy(V_1) is folded by r_j after every round, as in the layer sum-check (a6).  tr: 2 s words; s draws. */
int orc_prove_sum_layer(uint32_t s, const uint64_t *Vb, uint64_t seed, uint64_t *ctr, uint64_t *z, uint64_t *claim,
                        uint64_t *tr) {
    if (s == 0 || s > 63) return ORC_ERR_SHAPE;
    uint64_t nb = (uint64_t)1 << s, w = 0;
    uint64_t *A = (uint64_t *)malloc(nb * sizeof(uint64_t));
    if (!A) return ORC_ERR_NOMEM;
    memcpy(A, Vb, nb * sizeof(uint64_t));
    for (uint32_t j = 0; j < s; j++) {
        uint64_t half = nb >> (j + 1), G0 = 0, G1 = 0;
        for (uint64_t u = 0; u < half; u++) { G0 = orc_add(G0, A[2 * u]); G1 = orc_add(G1, A[2 * u + 1]); }
        tr[w++] = G0; tr[w++] = G1;
        uint64_t r = orc_draw(seed, (*ctr)++);
        z[j] = r;
        for (uint64_t u = 0; u < half; u++)
            A[u] = orc_add(A[2 * u], orc_mul(r, orc_sub(A[2 * u + 1], A[2 * u])));
    }
    *claim = A[0];
    free(A);
    return ORC_OK;
}

/* Entry state of layer i taken in isolation.  The challenges are a function of (seed, counter) alone (reading c-11),
 * the counter advances by s_0 for z_0 and by 2 s_{l+1} + 1 per proved layer l (2s round challenges, then tau), and
 * the claim point of layer i >= 1 is z = l(tau) = r1 + tau (r2 - r1) with r1, r2, tau the draws of layer i-1
 * (reading c-5).  logs[0..i] = log sizes of layers 0..i.  Writes z[0 .. logs[i]) and returns the counter at which
 * layer i's own draws start.  (The claim at z is V~_i(z) by definition: orc_mle.) */
uint64_t orc_layer_entry(const uint32_t *logs, uint32_t i, uint64_t seed, int sum_out, uint64_t *z) {
    if (i == 0) {
        for (uint32_t k = 0; k < logs[0]; k++) z[k] = orc_draw(seed, k);
        return logs[0];
    }
    /* sum_out: layer 0 is the sum gate (s_0 = 0): it takes s_1 draws and hands z = (r_0..r_{s_1 - 1}) to layer 1 */
    uint64_t c0 = logs[0];
    for (uint32_t l = 0; l + 1 < i; l++) c0 += (sum_out && l == 0) ? logs[1] : 2ull * logs[l + 1] + 1;
    const uint32_t s = logs[i];
    if (sum_out && i == 1) {
        for (uint32_t k = 0; k < s; k++) z[k] = orc_draw(seed, c0 + k);
        return c0 + s;
    }
    const uint64_t tau = orc_draw(seed, c0 + 2ull * s);
    for (uint32_t k = 0; k < s; k++) {
        const uint64_t r1 = orc_draw(seed, c0 + k), r2 = orc_draw(seed, c0 + s + k);
        z[k] = orc_add(r1, orc_mul(tau, orc_sub(r2, r1)));
    }
    return c0 + 2ull * s + 1;
}

static uint32_t log_below(const orc_layer *layers, uint32_t d, uint32_t log_input, uint32_t i) {
    return i + 1 < d ? layers[i + 1].log_size : log_input;
}

/* words layer i writes: (G0,G1,G2) x 2s rounds, then q[0..s]; the sum gate: (G0,G1) x s rounds */
static uint64_t layer_words(const orc_layer *layers, uint32_t d, uint32_t log_input, uint32_t i) {
    uint64_t s = log_below(layers, d, log_input, i);
    return (i == 0 && is_sum_layer(&layers[0])) ? 2 * s : 7 * s + 1;
}

uint64_t orc_transcript_words(const orc_layer *layers, uint32_t d, uint32_t log_input) {
    uint64_t w = 0;
    for (uint32_t i = 0; i < d; i++) w += layer_words(layers, d, log_input, i);
    return w;
}

/* ---------------------------------------------------------------- whole prover
 * evaluate, start claim, then every layer 0..d-1.  outputs: 2^{s_0} words; transcript: all layers
 * concatenated, layer 0 first.  final_z (log_input words) and final_claim are optional. */
int orc_prove(const orc_layer *layers, uint32_t d, uint32_t log_input, const uint64_t *input, uint64_t seed,
              uint64_t *outputs, uint64_t *transcript, uint64_t cap_words, uint64_t *final_z, uint64_t *final_claim) {
    if (d == 0) return ORC_ERR_ARG;
    if (cap_words < orc_transcript_words(layers, d, log_input)) return ORC_ERR_ARG;
    uint64_t **V = (uint64_t **)calloc(d + 1, sizeof(uint64_t *));
    if (!V) return ORC_ERR_NOMEM;
    int rc = ORC_OK;
    for (uint32_t i = 0; i <= d; i++) {
        uint32_t ls = i < d ? layers[i].log_size : log_input;
        V[i] = (uint64_t *)malloc(sizeof(uint64_t) << ls);
        if (!V[i]) rc = ORC_ERR_NOMEM;
    }
    uint64_t z[64], claim = 0, ctr = 0, w = 0;
    if (rc == ORC_OK) rc = orc_evaluate(layers, d, log_input, input, V);
    if (rc == ORC_OK) {
        memcpy(outputs, V[0], sizeof(uint64_t) << layers[0].log_size);
        rc = orc_start(V[0], layers[0].log_size, seed, &ctr, z, &claim);
    }
    for (uint32_t i = 0; i < d && rc == ORC_OK; i++) {
        uint32_t s = log_below(layers, d, log_input, i);
        if (i == 0 && is_sum_layer(&layers[0])) rc = orc_prove_sum_layer(s, V[1], seed, &ctr, z, &claim, transcript + w);
        else rc = orc_prove_layer(&layers[i], s, V[i + 1], seed, &ctr, z, &claim, transcript + w, NULL);
        w += layer_words(layers, d, log_input, i);
    }
    if (rc == ORC_OK && final_z) memcpy(final_z, z, log_input * sizeof(uint64_t));
    if (rc == ORC_OK && final_claim) *final_claim = claim;
    for (uint32_t i = 0; i <= d; i++) free(V[i]);
    free(V);
    return rc;
}

/* ---------------------------------------------------------------- verifier
 * Same draw order as the prover.  Start claim from the CLAIMED outputs; each round: G0+G1 == claim,
 * claim <- interp2(G, r); after 2s rounds v1 = q[0], v2 = q[1] and the wiring check
 * claim == sum_tau W_tau f_tau(v1,v2); then z <- l(tau), claim <- q(tau); at the end
 * claim == V~_d(z) of the input.  Rejection is reported through accept/fail_layer/fail_round:
 * fail_round m < 2s: round check m failed; fail_round = 2s: wiring check failed; fail_layer = d:
 * the closing input check failed.  A sum gate at the output (reading c-19) has s round checks and nothing else. */
int orc_verify(const orc_layer *layers, uint32_t d, uint32_t log_input, const uint64_t *input,
               const uint64_t *outputs, uint64_t seed, const uint64_t *transcript, uint64_t n_words,
               int *accept, uint32_t *fail_layer, uint32_t *fail_round) {
    *accept = 0; *fail_layer = 0; *fail_round = 0;
    if (n_words != orc_transcript_words(layers, d, log_input)) return ORC_ERR_ARG;
    uint64_t z[64], ctr = 0, claim, w = 0;
    for (uint32_t k = 0; k < layers[0].log_size; k++) z[k] = orc_draw(seed, ctr++);
    claim = orc_mle(outputs, layers[0].log_size, z);
    for (uint32_t i = 0; i < d; i++) {
        const orc_layer *L = &layers[i];
        uint32_t s = log_below(layers, d, log_input, i);
        uint64_t n = (uint64_t)1 << L->log_size, nb = (uint64_t)1 << s;
        uint64_t r[128];
        if (i == 0 && is_sum_layer(L)) {      /* the sum gate: s linear rounds, then the claim is V~_1(r) at z = r */
            for (uint32_t m = 0; m < s; m++) {
                const uint64_t *G = transcript + w; w += 2;
                if (orc_add(G[0], G[1]) != claim) { *fail_layer = 0; *fail_round = m; return ORC_OK; }
                z[m] = orc_draw(seed, ctr++);
                claim = orc_add(G[0], orc_mul(z[m], orc_sub(G[1], G[0])));
            }
            continue;
        }
        for (uint32_t m = 0; m < 2 * s; m++) {
            const uint64_t *G = transcript + w; w += 3;
            if (orc_add(G[0], G[1]) != claim) { *fail_layer = i; *fail_round = m; return ORC_OK; }
            r[m] = orc_draw(seed, ctr++);
            claim = orc_interp2(G, r[m]);
        }
        const uint64_t *q = transcript + w; w += s + 1;
        uint64_t v1 = q[0], v2 = q[1];
        uint64_t *Tz = (uint64_t *)malloc(n * sizeof(uint64_t));
        uint64_t *T1 = (uint64_t *)malloc(nb * sizeof(uint64_t));
        uint64_t *T2 = (uint64_t *)malloc(nb * sizeof(uint64_t));
        if (!Tz || !T1 || !T2) { free(Tz); free(T1); free(T2); return ORC_ERR_NOMEM; }
        orc_eq_table(z, L->log_size, Tz);
        orc_eq_table(r, s, T1);
        orc_eq_table(r + s, s, T2);
        uint64_t W[4] = {0, 0, 0, 0};
        for (uint64_t g = 0; g < n; g++)
            W[L->type[g]] = orc_add(W[L->type[g]], orc_mul(Tz[g], orc_mul(T1[L->in1[g]], T2[L->in2[g]])));
        free(Tz); free(T1); free(T2);
        uint64_t rhs = 0;
        for (uint8_t t = 0; t < 4; t++) rhs = orc_add(rhs, orc_mul(W[t], gate_f(t, v1, v2)));
        if (rhs != claim) { *fail_layer = i; *fail_round = 2 * s; return ORC_OK; }
        uint64_t tau = orc_draw(seed, ctr++);
        for (uint32_t k = 0; k < s; k++) z[k] = orc_add(r[k], orc_mul(tau, orc_sub(r[s + k], r[k])));
        claim = orc_lagrange(q, s + 1, tau);
    }
    for (uint64_t u = 0; u < ((uint64_t)1 << log_input); u++)
        if (input[u] >= ORC_P) return ORC_ERR_ARG;
    if (orc_mle(input, log_input, z) != claim) { *fail_layer = d; *fail_round = 0; return ORC_OK; }
    *accept = 1;
    return ORC_OK;
}
