/*
 * oracle.c -- plain CPU oracle for the FlexMoE routed-expert FFN hot path.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this.  It shares no code, header, table or
 * helper with the CUDA path under paper_2606_27866_b200/csrc/, and neither imports the other.
 *
 * What it computes is a plainly defined result (the method is exact, not an approximation),
 * written out in the paper's order and notation:
 *   pack   : Eq. 3     W~gate = P W_gate, W~up = P W_up, W~down = W_down P^T
 *   route  : Alg. 2 l.5-6 "Sort(eid)", read as the STABLE sort by
 *            (expert id, flat index t*k+j)  -- DESIGN.md reading R5
 *   ffn    : Eq. 1 / Eq. 4 with the prefix mask m(r) realised by the loop
 *            bound c < r_e, router weight applied after the down projection and summed over
 *            the k slots in slot order (Alg. 1 l.19; Alg. 2 l.19-20)
 *   rho    : Eq. 12   rho = 1 - mean_e r_e / I
 *   width  : k = ceil(r * d_ff) in exact integer arithmetic (reading R2)
 *
 * Arithmetic: bf16 inputs are widened exactly; every product and sum is carried in FXO_REAL
 * (double for the *_f64 entry points -- the default oracle; float for *_f32, the "plain fp32
 * oracle" of BASELINE.json's north_star, kept to show its own error is ~1e-6).  Plain
 * sequential loops in index order, one token at a time; OpenMP only across tokens.  No
 * blocking, no sorting, no alignment, no interleaving: it loops per token as Alg. 1's math does.
 *
 * Pins (tests/test_oracle_pins.py): P1 dense equality vs an independent torch fp64 einsum,
 * P2 slice == mask, P3 permutation invariance, P4 channel additivity / nestedness, P5 linearity
 * in router weights, P6 numpy brute force, P7 Alg.1 == Alg.2 emulation, P8 grouping vs numpy
 * stable argsort/bincount/cumsum, P9 Fig. 6 -> rho = 0.4031, P10 Table 2 linear byte model.
 * Parity unpinned: SiLU at large-magnitude arguments and the summation order inside a dot
 * product (any order is accepted within the stated tolerance).
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#ifndef FXO_REAL
#define FXO_REAL double
#endif
#ifndef FXO_SUF
#define FXO_SUF f64
#endif
#define FXO_CAT_(a, b) a##_##b
#define FXO_CAT(a, b) FXO_CAT_(a, b)
#define FXO_NAME(base) FXO_CAT(base, FXO_SUF)

static inline FXO_REAL bf16_widen(uint16_t b)
{
    uint32_t u = (uint32_t)b << 16;
    float f;
    memcpy(&f, &u, 4);
    return (FXO_REAL)f;
}

/* silu(z) = z / (1 + exp(-z))   (reading R1: phi = SiLU) */
static inline FXO_REAL silu(FXO_REAL z)
{
#if defined(FXO_IS_FLOAT)
    return z / (1.0f + expf(-z));
#else
    return z / (1.0 + exp(-z));
#endif
}

/*
 * Routed-expert FFN with per-expert retained widths (Eq. 4 summed over the token's k experts).
 *   x        [T][d]      bf16 bits
 *   Gt, Ut   [E][I][d]   bf16 bits, channel-RANKED (output of fxo_pack)
 *   Dt       [E][d][I]   bf16 bits, channel-RANKED
 *   r        [E]         retained widths, 0 <= r_e <= I
 *   ids, w   [T][k]      expert ids / router weights
 *   rows     [n_rows]    token indices to evaluate (NULL -> 0..n_rows-1); rows of y are
 *                        independent given the routing, so a subset is an exact check
 *   y        [n_rows][d] output in FXO_REAL (no rounding to bf16)
 */
void FXO_NAME(fxo_moe_ffn)(const uint16_t* x, const uint16_t* Gt, const uint16_t* Ut,
                           const uint16_t* Dt, const int32_t* r, const int32_t* ids,
                           const float* w, int T, int k, int E, int d, int I,
                           const int32_t* rows, int n_rows, FXO_REAL* y)
{
    (void)T; (void)E;
#pragma omp parallel
    {
        FXO_REAL* xt = (FXO_REAL*)malloc(sizeof(FXO_REAL) * (size_t)d);
        FXO_REAL* h = (FXO_REAL*)malloc(sizeof(FXO_REAL) * (size_t)(I > 0 ? I : 1));
#pragma omp for schedule(dynamic, 1)
        for (int q = 0; q < n_rows; ++q) {
            const int t = rows ? rows[q] : q;
            FXO_REAL* yt = y + (size_t)q * d;
            for (int i = 0; i < d; ++i) { xt[i] = bf16_widen(x[(size_t)t * d + i]); yt[i] = 0; }   /* Y <- 0 */
            for (int j = 0; j < k; ++j) {
                const int e = ids[(size_t)t * k + j];
                const int re = r[e];
                const uint16_t* G = Gt + (size_t)e * I * d;
                const uint16_t* U = Ut + (size_t)e * I * d;
                const uint16_t* D = Dt + (size_t)e * d * I;
                for (int c = 0; c < re; ++c) {                 /* prefix mask m(r): c < r_e */
                    FXO_REAL g = 0, u = 0;
                    for (int i = 0; i < d; ++i) {
                        g += bf16_widen(G[(size_t)c * d + i]) * xt[i];
                        u += bf16_widen(U[(size_t)c * d + i]) * xt[i];
                    }
                    h[c] = silu(g) * u;
                }
                const FXO_REAL wj = (FXO_REAL)w[(size_t)t * k + j];
                for (int i = 0; i < d; ++i) {
                    FXO_REAL o = 0;
                    for (int c = 0; c < re; ++c) o += bf16_widen(D[(size_t)i * I + c]) * h[c];
                    yt[i] += wj * o;                           /* weight by router score, add into Y */
                }
            }
        }
        free(xt);
        free(h);
    }
}

#ifdef FXO_COMMON
/* Eq. 3: gather rows of gate/up and columns of down by the ranking permutation.
 * channel_rank[e][p] = ORIGINAL index of the p-th ranked channel (reading R3). */
void fxo_pack(int E, int I, int d, const uint16_t* Wg, const uint16_t* Wu, const uint16_t* Wd,
              const int32_t* channel_rank, uint16_t* Gt, uint16_t* Ut, uint16_t* Dt)
{
    for (int e = 0; e < E; ++e)
        for (int p = 0; p < I; ++p) {
            const int src = channel_rank ? channel_rank[(size_t)e * I + p] : p;
            memcpy(Gt + ((size_t)e * I + p) * d, Wg + ((size_t)e * I + src) * d, sizeof(uint16_t) * (size_t)d);
            memcpy(Ut + ((size_t)e * I + p) * d, Wu + ((size_t)e * I + src) * d, sizeof(uint16_t) * (size_t)d);
            for (int i = 0; i < d; ++i)
                Dt[((size_t)e * d + i) * I + p] = Wd[((size_t)e * d + i) * I + src];
        }
}

/* Grouping: counts, exclusive offsets (offsets[E] = T*k), stable perm and its inverse.
 * Returns 0, or -1 if an id is outside [0,E). */
int fxo_route(const int32_t* ids, int T, int k, int E, int32_t* counts, int32_t* offsets,
              int32_t* perm, int32_t* inv_perm)
{
    const int A = T * k;
    for (int e = 0; e < E; ++e) counts[e] = 0;
    for (int f = 0; f < A; ++f) {
        if (ids[f] < 0 || ids[f] >= E) return -1;
        counts[ids[f]]++;
    }
    offsets[0] = 0;
    for (int e = 0; e < E; ++e) offsets[e + 1] = offsets[e] + counts[e];
    int pos = 0;
    for (int e = 0; e < E; ++e)
        for (int f = 0; f < A; ++f)
            if (ids[f] == e) perm[pos++] = f;
    for (int p = 0; p < A; ++p) inv_perm[perm[p]] = p;
    return 0;
}

/* Eq. 12 for n cells (one layer: n = E): rho = 1 - (1/n) sum r/I */
double fxo_budget_rho(const int32_t* r, int n, int I)
{
    double s = 0;
    for (int i = 0; i < n; ++i) s += (double)r[i] / (double)I;
    return 1.0 - s / (double)n;
}

/* k = ceil(I * num/den) in integers (reading R2) */
int32_t fxo_ratio_to_width(int I, int num, int den)
{
    return (int32_t)(((int64_t)I * num + den - 1) / den);
}
#endif
