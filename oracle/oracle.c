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
 *   saliency : Eq. 2   s_j = mean_b sum_{theta in Theta_j} (theta * g_theta^(b))^2, Theta_j = row j of
 *            W_gate, row j of W_up, column j of W_down
 *   rank   : Eq. 3's pi: channels by DESCENDING s, ties -> lower original index first (reading R4)
 *   router : the frozen router's front end (reading R10; PAPER.md:478, 545 take its output as given): top-k of the
 *            logits (ties -> lower expert id), softmax over the k selected logits (= full softmax renormalised)
 *   actions: Eq. 6 hard action k* = argmax_k softmax((alpha + g) / tau) with the Gumbel noise g passed
 *            in, width = ceil(r_k* I); Eq. 10 cost C = sum_e q_e sum_k p_ek r_k,
 *            p = softmax(alpha)
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
 * stable argsort/bincount/cumsum, P9 Fig. 6 -> rho = 0.4031, P10 Table 2 linear byte model,
 * P11 saliency (closed form for constant gradients, a^2 scaling, channel equivariance, additivity
 * over the three matrices, python brute force), P12 rank (numpy stable argsort, planted order, ties),
 * P13 router front end (the generator's full-softmax route, closed forms, shift invariance, k = E),
 * P14 actions (Fig. 6 histogram via noise-free argmax, temperature invariance of the argmax, Eq. 10
 * closed forms).
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

/*
 * Eq. 2: grouped first-order Taylor saliency of every hidden channel.
 *   Wg, Wu [E][I][d], Wd [E][d][I]                 weights, bf16 bits (ORIGINAL channel order)
 *   Gg, Gu [B][E][I][d], Gd [B][E][d][I]           gradients of the B ranking batches, bf16 bits
 *   s      [E][I]                                   out, double
 * s[e][j] = (1/B) sum_b [ sum_i (Wg[e][j][i] Gg[b][e][j][i])^2 + sum_i (Wu.. Gu..)^2 + sum_i (Wd[e][i][j] Gd[b][e][i][j])^2 ]
 */
void fxo_saliency(const uint16_t* Wg, const uint16_t* Wu, const uint16_t* Wd, const uint16_t* Gg,
                  const uint16_t* Gu, const uint16_t* Gd, int B, int E, int I, int d, double* s)
{
    const size_t per = (size_t)E * I * d;
#pragma omp parallel for collapse(2) schedule(static)
    for (int e = 0; e < E; ++e)
        for (int j = 0; j < I; ++j) {
            double acc = 0;
            for (int b = 0; b < B; ++b) {
                double sb = 0;                                   /* s^(b)_{e,j} */
                for (int i = 0; i < d; ++i) {
                    const size_t row = ((size_t)e * I + j) * d + i;      /* (e, j, i) of gate / up   */
                    const size_t col = ((size_t)e * d + i) * I + j;      /* (e, i, j) of down        */
                    const double tg = (double)bf16_widen(Wg[row]) * (double)bf16_widen(Gg[b * per + row]);
                    const double tu = (double)bf16_widen(Wu[row]) * (double)bf16_widen(Gu[b * per + row]);
                    const double td = (double)bf16_widen(Wd[col]) * (double)bf16_widen(Gd[b * per + col]);
                    sb += tg * tg + tu * tu + td * td;
                }
                acc += sb;
            }
            s[(size_t)e * I + j] = acc / (double)B;
        }
}

/* Eq. 3's permutation: sort s in descending order; equal saliencies keep ascending original index
 * (reading R4).  rank[e][p] = ORIGINAL index of the p-th most important channel (reading R3).  A total order, so the
 * library sort gives exactly one result. */
static const double* fxo_sort_keys;
static int fxo_rank_cmp(const void* a, const void* b)
{
    const int32_t ia = *(const int32_t*)a, ib = *(const int32_t*)b;
    const double sa = fxo_sort_keys[ia], sb = fxo_sort_keys[ib];
    if (sa > sb) return -1;
    if (sa < sb) return 1;
    return ia < ib ? -1 : (ia > ib ? 1 : 0);
}
void fxo_rank(const double* s, int E, int I, int32_t* rank)
{
    for (int e = 0; e < E; ++e) {
        int32_t* r = rank + (size_t)e * I;
        for (int j = 0; j < I; ++j) r[j] = j;
        fxo_sort_keys = s + (size_t)e * I;
        qsort(r, (size_t)I, sizeof(int32_t), fxo_rank_cmp);
    }
}

/* Router front end (reading R10): for every token the k largest logits (fp32 comparison, ties -> lower expert id), in
 * descending order; weights = softmax over those k logits (equal to the softmax over all E renormalised to sum 1),
 * computed in double and rounded once to fp32. */
void fxo_router_topk(const float* logits, int T, int E, int k, int32_t* ids, float* w)
{
    for (int t = 0; t < T; ++t) {
        const float* l = logits + (size_t)t * E;
        int32_t* id = ids + (size_t)t * k;
        for (int j = 0; j < k; ++j) {
            int best = -1;
            for (int e = 0; e < E; ++e) {
                int taken = 0;
                for (int q = 0; q < j; ++q) taken |= (id[q] == e);
                if (taken) continue;
                if (best < 0 || l[e] > l[best]) best = e;        /* strict: the lower id wins a tie */
            }
            id[j] = best;
        }
        double den = 0;
        for (int j = 0; j < k; ++j) den += exp((double)l[id[j]] - (double)l[id[0]]);
        for (int j = 0; j < k; ++j) w[(size_t)t * k + j] = (float)(exp((double)l[id[j]] - (double)l[id[0]]) / den);
    }
}

/* Eq. 6: z_soft = softmax((alpha + g) / tau), hard action = argmax_k z_soft (ties -> lower k), forward
 * value of the straight-through estimator (Eq. 7) = the hard one-hot, so the sampled width is ceil(r_k* I) with the
 * ratio r_k = num[k] / den (exact integers).  alpha, gumbel [E][K] fp32 (the noise is an INPUT).
 * Both sides decide the argmax on the fp32 sum alpha + g (softmax and the division by tau > 0 are monotone). */
void fxo_sample_actions(const float* alpha, const float* gumbel, int E, int K, const int32_t* num, int den, int I,
                        int32_t* action, int32_t* width)
{
    for (int e = 0; e < E; ++e) {
        int best = 0;
        float vbest = alpha[(size_t)e * K] + gumbel[(size_t)e * K];
        for (int k = 1; k < K; ++k) {
            const float v = alpha[(size_t)e * K + k] + gumbel[(size_t)e * K + k];
            if (v > vbest) { vbest = v; best = k; }
        }
        action[e] = best;
        width[e] = fxo_ratio_to_width(I, num[best], den);
    }
}

/* Eq. 10 for one layer: C = sum_e q_e sum_k p_ek r_k, p_e = softmax(alpha_e) (clean, no noise, no tau),
 * q_e = n_e / sum n (the load ratio of expert e in this layer), r_k = num[k] / den. */
double fxo_action_cost(const float* alpha, int E, int K, const int32_t* num, int den, const int32_t* counts)
{
    double total = 0, C = 0;
    for (int e = 0; e < E; ++e) total += (double)counts[e];
    for (int e = 0; e < E; ++e) {
        double mx = alpha[(size_t)e * K], z = 0, er = 0;
        for (int k = 1; k < K; ++k) if (alpha[(size_t)e * K + k] > mx) mx = alpha[(size_t)e * K + k];
        for (int k = 0; k < K; ++k) z += exp((double)alpha[(size_t)e * K + k] - mx);
        for (int k = 0; k < K; ++k) er += exp((double)alpha[(size_t)e * K + k] - mx) / z * ((double)num[k] / (double)den);
        C += (total > 0 ? (double)counts[e] / total : 0.0) * er;
    }
    return C;
}
#endif
