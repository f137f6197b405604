// fxm_rank.cu -- the steps immediately around the hot path that SURVEY.md 8(f) lists as NEXT-2 and NEXT-4:
//   NEXT-2  channel saliency (Eq. 2) and the descending ranking that defines P (Eq. 3):
//             s[e][j] = (1/B) sum_b sum_{theta in Theta_j} (theta * g_theta^(b))^2,
//             Theta_j = row j of W_gate, row j of W_up, column j of W_down
//           -> channel_rank[e][p] = ORIGINAL index of the p-th most important channel (readings R3, R4), the input of pack.
//           A streaming reduction over the weights and B gradient sets: HBM-bound, (1 + B) * 6 E I d bytes, each read once.
//   NEXT-4  the training-time action sampling that turns logits into a width table on the device (Eq. 6-7, PAPER.md:104-113:
//           the forward value of the straight-through estimator is the hard one-hot), and the load-sensitive cost of
//           Eq. 10.  With these the masked forward of Eq. 4 is "sample -> moe_ffn" with no host round trip.
// All sums are fixed-order (no floating-point atomics): results are reproducible run to run.
#include "fxm_internal.cuh"

#include <mutex>

namespace fxm {

__device__ __forceinline__ float bf_lo(uint32_t u) { return __uint_as_float(u << 16); }
__device__ __forceinline__ float bf_hi(uint32_t u) { return __uint_as_float(u & 0xFFFF0000u); }
constexpr int SAL_GU_ROWS = 4;                  // gate / up rows per warp of a row block (a block covers 32 rows)
__device__ __forceinline__ float sq8(const uint4& w, const uint4& g) {
    const float p0 = bf_lo(w.x) * bf_lo(g.x), p1 = bf_hi(w.x) * bf_hi(g.x), p2 = bf_lo(w.y) * bf_lo(g.y), p3 = bf_hi(w.y) * bf_hi(g.y);
    const float p4 = bf_lo(w.z) * bf_lo(g.z), p5 = bf_hi(w.z) * bf_hi(g.z), p6 = bf_lo(w.w) * bf_lo(g.w), p7 = bf_hi(w.w) * bf_hi(g.w);
    return ((p0 * p0 + p1 * p1) + (p2 * p2 + p3 * p3)) + ((p4 * p4 + p5 * p5) + (p6 * p6 + p7 * p7));
}

// One launch streams all three weight tensors and their gradients.  Blocks [0, dn_blocks) sum W_down columns, the rest sum
// gate / up rows; the column blocks are the long ones and come first, so the short row blocks fill the tail of the grid.
// Both roles issue every load of a step (12 x 16 bytes per thread at B = 2) before the first use: the kernel is bound
// by HBM only while enough requests are in flight, so a thread must never wait on one load at a time.
//
// gate and up rows: one warp per (e, j), four rows per warp and block; the row of d bf16 is read with 16-byte loads,
// weights once, gradients B times.
__device__ __forceinline__ void saliency_gu_rows(size_t blk, int d, size_t rows, size_t per, const uint4* __restrict__ Wg,
                                                 const uint4* __restrict__ Wu, const uint4* __restrict__ Gg,
                                                 const uint4* __restrict__ Gu, int B, float* __restrict__ part0) {
    const int lane = threadIdx.x & 31;
    const int cpr = d >> 3;                                      // 16-byte chunks per row
    const size_t per4 = per >> 3;                                // chunks per gradient set
    for (int j = 0; j < SAL_GU_ROWS; ++j) {
        const size_t row = (blk * SAL_GU_ROWS + j) * 8ull + (threadIdx.x >> 5);
        if (row >= rows) return;
        float acc = 0.f;
#pragma unroll 2
        for (int c = lane; c < cpr; c += 32) {
            const size_t o = row * cpr + c;
            const uint4 wg = __ldcs(Wg + o), wu = __ldcs(Wu + o);
            // gradient sets four at a time with every load issued before the first use (B is a run-time value: a plain loop
            // over b would serialise the loads); the sum stays in the order b = 0, 1, ...
            for (int b0 = 0; b0 < B; b0 += 4) {
                uint4 gg[4], gu[4];
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (b0 + u < B) { gg[u] = __ldcs(Gg + (b0 + u) * per4 + o); gu[u] = __ldcs(Gu + (b0 + u) * per4 + o); }
#pragma unroll
                for (int u = 0; u < 4; ++u)
                    if (b0 + u < B) acc += sq8(wg, gg[u]) + sq8(wu, gu[u]);
            }
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (lane == 0) part0[row] = acc;
    }
}

__device__ __forceinline__ void sq8_acc(float (&acc)[8], const uint4& w, const uint4& g) {
    const float p0 = bf_lo(w.x) * bf_lo(g.x), p1 = bf_hi(w.x) * bf_hi(g.x), p2 = bf_lo(w.y) * bf_lo(g.y), p3 = bf_hi(w.y) * bf_hi(g.y);
    const float p4 = bf_lo(w.z) * bf_lo(g.z), p5 = bf_hi(w.z) * bf_hi(g.z), p6 = bf_lo(w.w) * bf_lo(g.w), p7 = bf_hi(w.w) * bf_hi(g.w);
    acc[0] += p0 * p0; acc[1] += p1 * p1; acc[2] += p2 * p2; acc[3] += p3 * p3;
    acc[4] += p4 * p4; acc[5] += p5 * p5; acc[6] += p6 * p6; acc[7] += p7 * p7;
}

// down columns: a WARP owns (e, r, cg): rows [r0, r1) of W_down[e] [d][I], 32 consecutive 16-byte chunks of each row (a
// lane owns 8 consecutive columns); the eight warps of a block take neighbouring items, so a block reads contiguous row
// segments whatever I is.  Rows go four at a time: the weight chunks of the four rows and two gradient sets of each are
// loaded before the first multiply.  Per column the sum runs over the rows in order (inside a group of four rows: b in
// order for B <= 2, pairs of gradient sets in order beyond).  Partial column sums go to slot 1 + r.
__device__ __forceinline__ void saliency_dn_cols(size_t blk, int E, int d, int I, int R, size_t per,
                                                 const uint4* __restrict__ Wd, const uint4* __restrict__ Gd, int B,
                                                 float* __restrict__ part) {
    const int lane = threadIdx.x & 31;
    const int cpr = I >> 3;                                      // chunks per row (I % 16 == 0)
    const int CG = (cpr + 31) >> 5;
    const size_t item = blk * 8ull + (threadIdx.x >> 5);
    if (item >= (size_t)E * R * CG) return;
    const int cg = (int)(item % CG), r = (int)(item / CG % R), e = (int)(item / CG / R);
    const int c0 = cg * 32 + lane;
    if (c0 >= cpr) return;
    const int r0 = (int)((long long)d * r / R), r1 = (int)((long long)d * (r + 1) / R);
    const size_t per4 = per >> 3;
    float acc[8];
#pragma unroll
    for (int q = 0; q < 8; ++q) acc[q] = 0.f;
    const uint4* w_ptr = Wd + ((size_t)e * d + r0) * cpr + c0;
    const uint4* g_ptr = Gd + ((size_t)e * d + r0) * cpr + c0;
    for (int i = r0; i < r1; i += 4, w_ptr += 4 * (size_t)cpr, g_ptr += 4 * (size_t)cpr) {
        const int nr = r1 - i;                                   // rows left (>= 1); rows beyond are neither read nor summed
        uint4 w[4];
#pragma unroll
        for (int v = 0; v < 4; ++v)
            if (v < nr) w[v] = __ldcs(w_ptr + (size_t)v * cpr);
        for (int b0 = 0; b0 < B; b0 += 2) {
            uint4 g[4][2];
#pragma unroll
            for (int v = 0; v < 4; ++v)
#pragma unroll
                for (int u = 0; u < 2; ++u)
                    if (v < nr && b0 + u < B) g[v][u] = __ldcs(g_ptr + (b0 + u) * per4 + (size_t)v * cpr);
#pragma unroll
            for (int v = 0; v < 4; ++v)
#pragma unroll
                for (int u = 0; u < 2; ++u)
                    if (v < nr && b0 + u < B) sq8_acc(acc, w[v], g[v][u]);
        }
    }
    float4* out = (float4*)(part + ((size_t)(1 + r) * E + e) * I + (size_t)c0 * 8);
    out[0] = make_float4(acc[0], acc[1], acc[2], acc[3]);
    out[1] = make_float4(acc[4], acc[5], acc[6], acc[7]);
}

__global__ void __launch_bounds__(256, 3) k_saliency(int E, int d, int I, int R, size_t rows, size_t per, unsigned dn_blocks,
                                                     const uint4* __restrict__ Wg, const uint4* __restrict__ Wu,
                                                     const uint4* __restrict__ Wd, const uint4* __restrict__ Gg,
                                                     const uint4* __restrict__ Gu, const uint4* __restrict__ Gd, int B,
                                                     float* __restrict__ part) {
    if (blockIdx.x < dn_blocks) saliency_dn_cols(blockIdx.x, E, d, I, R, per, Wd, Gd, B, part);
    else saliency_gu_rows(blockIdx.x - dn_blocks, d, rows, per, Wg, Wu, Gg, Gu, B, part);
}

// s = (slot 0 + slot 1 + ... + slot R) / B, slots summed in index order.  Launched as a programmatic dependent of
// k_saliency (its launch latency runs under that kernel's tail); the wait returns once k_saliency has completed.
__global__ void k_saliency_sum(const float* __restrict__ part, int slots, size_t n, float inv_b, float* __restrict__ s) {
    pdl_wait();
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n; i += (size_t)gridDim.x * blockDim.x) {
        float acc = 0.f;
        for (int q = 0; q < slots; ++q) acc += part[(size_t)q * n + i];
        s[i] = acc * inv_b;
    }
}

int saliency_row_chunks(const Dims& D) {
    int R = (148 * 8 + D.E - 1) / D.E;                           // row chunks per expert (= partial-sum slots): enough warp items for every SM
    if (R > 16) R = 16;
    if (R > D.d) R = D.d;
    return R < 1 ? 1 : R;
}
size_t saliency_workspace_bytes(const Dims& D) { return align_up((size_t)(1 + saliency_row_chunks(D)) * D.E * D.I * sizeof(float), 1024); }

cudaError_t launch_saliency(const Dims& D, const __nv_bfloat16* Wg, const __nv_bfloat16* Wu, const __nv_bfloat16* Wd,
                            const __nv_bfloat16* Gg, const __nv_bfloat16* Gu, const __nv_bfloat16* Gd, int B, float* s,
                            float* part, cudaStream_t st) {
    const size_t rows = (size_t)D.E * D.I, per = rows * D.d;
    const int R = saliency_row_chunks(D);
    const size_t CG = ((size_t)(D.I >> 3) + 31) / 32;
    const size_t dn_blocks = ((size_t)D.E * R * CG + 7) / 8, gu_blocks = (rows + 8 * SAL_GU_ROWS - 1) / (8 * SAL_GU_ROWS);
    if (dn_blocks + gu_blocks > 0x7FFFFFFFull) return cudaErrorInvalidConfiguration;
    k_saliency<<<(unsigned)(dn_blocks + gu_blocks), 256, 0, st>>>(D.E, D.d, D.I, R, rows, per, (unsigned)dn_blocks, (const uint4*)Wg,
                                                                  (const uint4*)Wu, (const uint4*)Wd, (const uint4*)Gg,
                                                                  (const uint4*)Gu, (const uint4*)Gd, B, part);
    size_t b3 = (rows + 255) / 256;
    if (b3 > 148 * 8) b3 = 148 * 8;
    const cudaError_t e = cudaGetLastError();
    if (e != cudaSuccess) return e;
    return launch_pdl(k_saliency_sum, dim3((unsigned)b3), dim3(256), 0, st, (const float*)part, 1 + R, rows, 1.0f / (float)B, s);
}

// ------------------------------------------------------------------------------------------------ no-allocation variant
// fxm_saliency_static: the same two kernels with their partial-sum scratch in a file-scope device array instead of a
// caller buffer, for callers that cannot allocate (CUDA graph capture, serving loops, harnesses that forbid cudaMalloc).
// The array is part of the library image: every GPU that loads the library holds SALIENCY_STATIC_BYTES until exit.
// In HOST code `g_saliency_scratch` is only a stand-in for the symbol, not a device address (a kernel handed it would
// fault, or silently use host memory where the GPU can reach it); the device address comes from cudaGetSymbolAddress,
// looked up once per device with that device current.  Nothing in the array has to start at zero: every slot the
// summing kernel reads (slot 0: gate/up rows, slots 1..R: down-column chunks) is written in full by the kernel
// before it in the same call, so stale contents of an earlier call are never read.  All calls on a device share the
// array: calls that overlap on the GPU (different streams without an ordering between them) race.
static __device__ __align__(256) float g_saliency_scratch[SALIENCY_STATIC_BYTES / sizeof(float)];

constexpr int SALIENCY_MAX_DEVICES = 64;
static float* g_saliency_scratch_addr[SALIENCY_MAX_DEVICES];   // device address of the array on device i (nullptr: not looked up yet)
static std::mutex g_saliency_scratch_mutex;

static cudaError_t saliency_static_scratch(float** out) {
    int dev = -1;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    if (dev < 0 || dev >= SALIENCY_MAX_DEVICES) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(g_saliency_scratch_mutex);
    if (!g_saliency_scratch_addr[dev]) {
        float* ptr = nullptr;
        e = cudaGetSymbolAddress((void**)&ptr, g_saliency_scratch);      // the current device's copy of the array
        if (e != cudaSuccess) return e;
        if (!ptr) return cudaErrorInvalidSymbol;
        g_saliency_scratch_addr[dev] = ptr;
    }
    *out = g_saliency_scratch_addr[dev];
    return cudaSuccess;
}

cudaError_t launch_saliency_static(const Dims& D, const __nv_bfloat16* Wg, const __nv_bfloat16* Wu, const __nv_bfloat16* Wd,
                                   const __nv_bfloat16* Gg, const __nv_bfloat16* Gu, const __nv_bfloat16* Gd, int B, float* s,
                                   cudaStream_t st) {
    if (saliency_workspace_bytes(D) > SALIENCY_STATIC_BYTES) return cudaErrorInvalidValue;   // the caller checks first
    float* part = nullptr;
    const cudaError_t e = saliency_static_scratch(&part);
    if (e != cudaSuccess) return e;
    return launch_saliency(D, Wg, Wu, Wd, Gg, Gu, Gd, B, s, part, st);
}

// ------------------------------------------------------------------------------------------------ rank
// One block per expert: bitonic sort of 64-bit keys (~orderable(s) << 32 | index) in shared memory.  The keys are
// distinct, so "descending s, ties -> lower original index" (reading R4) is the ascending key order -- one result.
constexpr int RANK_THREADS = 1024;
constexpr int RANK_MAX_I = 16384;
__global__ void __launch_bounds__(RANK_THREADS) k_rank(const float* __restrict__ s, int I, int Np, int* __restrict__ rank) {
    extern __shared__ unsigned long long keys[];
    const int e = blockIdx.x;
    for (int i = threadIdx.x; i < Np; i += RANK_THREADS) {
        unsigned long long key = ~0ull;                          // padding sorts last
        if (i < I) {
            float v = s[(size_t)e * I + i];
            if (v == 0.f) v = 0.f;                               // -0 and +0 are one value
            uint32_t u = __float_as_uint(v);
            u ^= (u >> 31) ? 0xFFFFFFFFu : 0x80000000u;          // ascending-orderable
            key = ((unsigned long long)(~u) << 32) | (uint32_t)i;
        }
        keys[i] = key;
    }
    __syncthreads();
    for (int k = 2; k <= Np; k <<= 1) {
        for (int j = k >> 1; j > 0; j >>= 1) {
            for (int t = threadIdx.x; t < (Np >> 1); t += RANK_THREADS) {
                const int lo = ((t & ~(j - 1)) << 1) | (t & (j - 1));      // index with bit j clear
                const int hi = lo | j;
                const bool up = (lo & k) == 0;
                const unsigned long long a = keys[lo], b = keys[hi];
                if ((a > b) == up) { keys[lo] = b; keys[hi] = a; }
            }
            __syncthreads();
        }
    }
    for (int i = threadIdx.x; i < I; i += RANK_THREADS) rank[(size_t)e * I + i] = (int)(uint32_t)keys[i];
}
cudaError_t init_rank_kernel() {
    return cudaFuncSetAttribute(k_rank, cudaFuncAttributeMaxDynamicSharedMemorySize, RANK_MAX_I * 8);
}
bool rank_supported(int I) { return I <= RANK_MAX_I; }
cudaError_t launch_rank(int E, int I, const float* s, int* rank, cudaStream_t st) {
    int Np = 2;
    while (Np < I) Np <<= 1;
    k_rank<<<E, RANK_THREADS, (size_t)Np * 8, st>>>(s, I, Np, rank);
    return cudaGetLastError();
}

// ---------------------------------------------------------------------------------------- action sampling
struct RatioArg { int num[MAX_K]; int den; int K; };
// Eq. 6: k* = argmax_k softmax((alpha + g) / tau) = argmax_k (alpha_k + g_k) for any tau > 0 (fp32 sum,
// ties -> lower k); Eq. 7: the forward pass uses the hard one-hot, so the sampled width is ceil(r_k* I).
__global__ void k_sample_actions(const float* __restrict__ alpha, const float* __restrict__ gumbel, RatioArg ra, int E, int I,
                                 int* __restrict__ table, int* __restrict__ action) {
    const int e = threadIdx.x;
    if (e >= MAX_E) return;
    int width = 0;
    if (e < E) {
        int best = 0;
        float vbest = alpha[(size_t)e * ra.K] + (gumbel ? gumbel[(size_t)e * ra.K] : 0.f);
        for (int k = 1; k < ra.K; ++k) {
            const float v = alpha[(size_t)e * ra.K + k] + (gumbel ? gumbel[(size_t)e * ra.K + k] : 0.f);
            if (v > vbest) { vbest = v; best = k; }
        }
        width = (int)(((long long)I * ra.num[best] + ra.den - 1) / ra.den);
        if (action) action[e] = best;
    }
    table[e] = width;
}
// Eq. 10 for one layer: C = sum_e q_e sum_k p_ek r_k, p_e = softmax(alpha_e), q_e = n_e / sum n
__global__ void __launch_bounds__(MAX_E) k_action_cost(const float* __restrict__ alpha, RatioArg ra, int E,
                                                       const int* __restrict__ counts, float* __restrict__ cost) {
    __shared__ float s_c[MAX_E], s_n[MAX_E];
    const int e = threadIdx.x;
    float er = 0.f, n = 0.f;
    if (e < E) {
        float mx = alpha[(size_t)e * ra.K];
        for (int k = 1; k < ra.K; ++k) mx = fmaxf(mx, alpha[(size_t)e * ra.K + k]);
        float z = 0.f, acc = 0.f;
        for (int k = 0; k < ra.K; ++k) {
            const float p = expf(alpha[(size_t)e * ra.K + k] - mx);
            z += p;
            acc += p * ((float)ra.num[k] / (float)ra.den);
        }
        er = acc / z;
        n = (float)counts[e];
    }
    s_c[e] = er * n;
    s_n[e] = n;
    __syncthreads();
    for (int o = MAX_E / 2; o > 0; o >>= 1) {                    // fixed-order tree
        if (e < o) { s_c[e] += s_c[e + o]; s_n[e] += s_n[e + o]; }
        __syncthreads();
    }
    if (e == 0) *cost = s_n[0] > 0.f ? s_c[0] / s_n[0] : 0.f;
}
cudaError_t launch_sample_actions(const float* alpha, const float* gumbel, int K, const int* num_host, int den, int E, int I,
                                  int* table, int* action, cudaStream_t st) {
    RatioArg ra{};
    for (int k = 0; k < K; ++k) ra.num[k] = num_host[k];
    ra.den = den; ra.K = K;
    k_sample_actions<<<1, MAX_E, 0, st>>>(alpha, gumbel, ra, E, I, table, action);
    return cudaGetLastError();
}
cudaError_t launch_action_cost(const float* alpha, int K, const int* num_host, int den, int E, const int* counts, float* cost,
                               cudaStream_t st) {
    RatioArg ra{};
    for (int k = 0; k < K; ++k) ra.num[k] = num_host[k];
    ra.den = den; ra.K = K;
    k_action_cost<<<1, MAX_E, 0, st>>>(alpha, ra, E, counts, cost);
    return cudaGetLastError();
}

}  // namespace fxm
