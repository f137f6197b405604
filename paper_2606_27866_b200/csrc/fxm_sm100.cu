// fxm_sm100.cu -- steps a4/a5/a6 on Blackwell: persistent, warp-specialised grouped GEMMs on tcgen05 tensor
// cores with TMEM accumulators, fed by contiguous cp.async.bulk (TMA unit) copies of pre-swizzled tiles.
//
//   a4  GEMM-1 + SwiGLU (Eq. 4; Alg. 2 l.12-16):
//         D[128 packed rows, N tokens] = Wgu_tile[128, d] . Xs_tile[N, d]^T      ("swap-AB": weights on UMMA M)
//       packed rows interleave gate/up in groups of 16, so gate channel c sits in TMEM lane l and its up twin
//       in lane l+16 of the SAME warp quadrant: SwiGLU is one __shfl_xor(.,16) away.  h = silu(g)*u, channels
//       >= r_e forced to 0 (the paper's pad-zero rule), one rounding to bf16, tile written to
//       the H panel with one bulk store.
//   a5  GEMM-2 + scale + combine (Alg. 2 l.18-20):
//         D[128 out features, N tokens] = Wd_tile[128, r_e] . H_tile[N, r_e]^T
//       K loop bounded by ceil(r_e/64): pruned K steps are never loaded or issued.  The epilogue rounds the
//       accumulator to bf16 and stores it to O[row][feature] (a warp writes 64 contiguous bytes per token);
//       the router-weight scale and the sum over a token's k experts are a gather in k_combine (no atomics,
//       slot order, fp32, one rounding).
//   a6  decode-sized T uses the same kernels: N shrinks to 16 and the kernel becomes a weight streamer
//       (16 KB bulk copies back to back, MMA cost negligible).
//
// Why swap-AB: the per-expert row count n_e is small and ragged in MoE (C2: ~273), and UMMA M is fixed at 128
// while N is any multiple of 16 -- tokens on N waste < 6 % where tokens on M would waste ~40 %.
//
// Warp roles (192 threads): warp 0 = bulk-copy producer, warp 1 = MMA issuer (+TMEM owner), warps 2-5 = epilogue
// (warp w reads TMEM lanes 32*(w%4)..+31).  Pipelines: smem full/empty ring (producer<->MMA), TMEM
// full/empty x2 (MMA<->epilogue, double-buffered accumulator so the epilogue of tile i overlaps the MMAs
// of tile i+1).  Work items are taken with a static stride over the device-side schedule written by the
// route kernel, so the launch shape never depends on routing or budget.
#include "fxm_ptx.cuh"

namespace fxm {

// ------------------------------------------------------------------------------------------------ kernel
struct GemmArgs {
    Dims D;
    const uint8_t* packed;     // gate/up region first, then down region
    const int* r_table;
    const int4* items;         // GEMM-1: explicit work items {e, row0, nvalid, cb}; GEMM-2: token tiles {e,row0,nvalid,.}
    const Sched* sched;
    const uint8_t* Bsrc;       // Xs (GEMM-1) or H (GEMM-2) panels
    uint8_t* H;                // GEMM-1 output panels
    uint8_t* O;                // GEMM-2 output panels
    DevState* state;
    int P;                     // panel row capacity
};

template <int MODE, int TN, int STAGES>
struct SmemPlan {
    static constexpr int STAGE_BYTES = WT_BYTES + TN * ROW_BYTES;
    static constexpr int STAGING_BYTES = MODE == 1 ? TN * ROW_BYTES : 0;   // H tile (GEMM-2 stores from registers)
    static constexpr int BAR_OFF = STAGES * STAGE_BYTES + STAGING_BYTES;
    static constexpr int TOTAL = BAR_OFF + 256 + 1024;              // + barriers + alignment slack
};

template <int MODE, int TN, int STAGES>
__global__ void __launch_bounds__(192, 1) k_gemm_sm100(const GemmArgs a) {
    extern __shared__ uint8_t smem_raw[];
    using Plan = SmemPlan<MODE, TN, STAGES>;
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    const uint32_t bar_base = smem_base + Plan::BAR_OFF;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (STAGES + s); };
    auto tfull_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + s); };
    auto tempty_bar = [&](int s) { return bar_base + 8u * (2 * STAGES + 2 + s); };
    volatile uint32_t* tmem_slot = (volatile uint32_t*)(smem_gen + Plan::BAR_OFF + 8 * (2 * STAGES + 4));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const Dims& D = a.D;

    if (threadIdx.x == 0) {
        for (int s = 0; s < STAGES; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int s = 0; s < 2; ++s) { mbar_init(tfull_bar(s), 1); mbar_init(tempty_bar(s), 128); }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(smem_u32((const void*)tmem_slot), 2 * TN);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int W = MODE == 1 ? a.sched->W1 : a.sched->W2;
    const uint8_t* dn = a.packed + gu_bytes(D);

    if (warp == 0) {
        // ===================================================== producer: one lane issues every bulk copy
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int wi = blockIdx.x; wi < W; wi += gridDim.x) {
                const int4 it = MODE == 1 ? a.items[wi] : a.items[wi / D.nDB];
                const int e = it.x, row0 = it.y;
                const uint32_t nb = (uint32_t)((it.z + 15) & ~15) * ROW_BYTES;
                const uint8_t* asrc;
                size_t astride;
                int nk;
                if (MODE == 1) {
                    asrc = a.packed + gu_tile_index(D, e, it.w, 0) * WT_BYTES;
                    astride = WT_BYTES;
                    nk = D.nKB1;
                } else {
                    asrc = dn + dn_tile_index(D, e, 0, wi % D.nDB) * WT_BYTES;
                    astride = (size_t)D.nDB * WT_BYTES;
                    nk = (a.r_table[e] + KB - 1) / KB;
                }
                const uint8_t* bsrc = a.Bsrc + (size_t)row0 * ROW_BYTES;
                const size_t bstride = (size_t)a.P * ROW_BYTES;
                for (int kb = 0; kb < nk; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u, a.state);
                    const uint32_t sa = smem_base + stage * Plan::STAGE_BYTES;
                    mbar_expect_tx(full_bar(stage), WT_BYTES + nb);
                    bulk_g2s(sa, asrc + kb * astride, WT_BYTES, full_bar(stage));
                    bulk_g2s(sa + WT_BYTES, bsrc + kb * bstride, nb, full_bar(stage));
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================================================== MMA issuer: one lane issues every tcgen05.mma
        if (lane == 0) {
            int stage = 0, as = 0;
            uint32_t phase = 0, aphase = 0;
            for (int wi = blockIdx.x; wi < W; wi += gridDim.x) {
                const int4 it = MODE == 1 ? a.items[wi] : a.items[wi / D.nDB];
                const uint32_t n = (uint32_t)(it.z + 15) & ~15u;
                const int nk = MODE == 1 ? D.nKB1 : (a.r_table[it.x] + KB - 1) / KB;
                const uint32_t idesc = make_idesc(n);
                const uint32_t d_tmem = tmem_base + (uint32_t)as * TN;
                mbar_wait(tempty_bar(as), aphase ^ 1u, a.state);
                tc_fence_after();
                for (int kb = 0; kb < nk; ++kb) {
                    mbar_wait(full_bar(stage), phase, a.state);
                    tc_fence_after();
                    const uint32_t sa = smem_base + stage * Plan::STAGE_BYTES;
                    const uint64_t adesc = make_desc_sw128(sa), bdesc = make_desc_sw128(sa + WT_BYTES);
#pragma unroll
                    for (int kk = 0; kk < KB / 16; ++kk)      // +32 bytes along K inside the swizzle atom = +2 in desc units
                        umma_bf16(d_tmem, adesc + 2u * kk, bdesc + 2u * kk, idesc, (uint32_t)((kb | kk) != 0));
                    umma_commit(empty_bar(stage));             // frees the smem slot when these MMAs retire
                    if (++stage == STAGES) { stage = 0; phase ^= 1u; }
                }
                umma_commit(tfull_bar(as));                    // accumulator complete -> epilogue
                if (++as == 2) { as = 0; aphase ^= 1u; }
            }
        }
    } else {
        // ===================================================== epilogue warps 2..5
        const int q = warp & 3;                                // TMEM lane quadrant this warp may read
        const int et = threadIdx.x - 64;                       // 0..127
        uint8_t* staging = smem_gen + STAGES * Plan::STAGE_BYTES;
        const uint32_t staging_s = smem_base + STAGES * Plan::STAGE_BYTES;
        int as = 0;
        uint32_t aphase = 0;
        for (int wi = blockIdx.x; wi < W; wi += gridDim.x) {
            const int4 it = MODE == 1 ? a.items[wi] : a.items[wi / D.nDB];
            const int e = it.x, row0 = it.y, nvalid = it.z;
            const int n = (nvalid + 15) & ~15;
            const int r = a.r_table[e];
            const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)as * TN;
            mbar_wait(tfull_bar(as), aphase, a.state);
            tc_fence_after();
            if (MODE == 1) {
                const int cb = it.w;
                const int ch = q * 16 + (lane & 15);           // channel within the block handled by this lane pair
                const bool keep = cb * CB + ch < r;            // tail mask of the last retained block
                const int odd = lane >> 4;                     // lanes 0-15 finish even token columns, 16-31 odd ones
                for (int c0 = 0; c0 < n; c0 += 16) {
                    uint32_t v[16];
                    tmem_ld16(taddr + c0, v);
                    tmem_ld_wait();
#pragma unroll
                    for (int m = 0; m < 8; ++m) {
                        const float mine0 = __uint_as_float(v[2 * m]), mine1 = __uint_as_float(v[2 * m + 1]);
                        const float send = odd ? mine0 : mine1;                    // what the twin lane needs
                        const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
                        const float g = odd ? recv : mine0;                        // gate lives in lanes 0-15
                        const float u = odd ? mine1 : recv;                        // up lives in lanes 16-31
                        float h = __fdividef(g, 1.f + __expf(-g)) * u;
                        if (!keep) h = 0.f;
                        const uint32_t t = c0 + 2 * m + odd;
                        *(__nv_bfloat16*)(staging + sw128_off(t, ch)) = __float2bfloat16_rn(h);
                    }
                }
                tc_fence_before();
                mbar_arrive(tempty_bar(as));                   // accumulator drained -> MMA may reuse it
                fence_proxy_async_smem();                      // generic-proxy smem writes -> visible to the bulk engine
                epi_bar_sync();
                if (et == 0) {
                    bulk_s2g(a.H + ((size_t)cb * a.P + row0) * ROW_BYTES, staging_s, (uint32_t)n * ROW_BYTES);
                    bulk_commit();
                    bulk_wait_read0();                         // staging may be overwritten after this
                }
                epi_bar_sync();
            } else {
                // lane = output feature; 16 token columns per load; 32 lanes -> 64 contiguous bytes of one O row
                uint8_t* dst = a.O + o_off(a.P, row0, (wi % D.nDB) * WT_ROWS + q * 32 + lane);
                for (int c0 = 0; c0 < n; c0 += 16) {
                    uint32_t v[16];
                    tmem_ld16(taddr + c0, v);
                    tmem_ld_wait();
#pragma unroll
                    for (int jj = 0; jj < 16; ++jj)
                        *(__nv_bfloat16*)(dst + (size_t)(c0 + jj) * (2 * WT_ROWS)) = __float2bfloat16_rn(__uint_as_float(v[jj]));
                }
                tc_fence_before();
                mbar_arrive(tempty_bar(as));
            }
            if (++as == 2) { as = 0; aphase ^= 1u; }
        }
        if (MODE == 1 && et == 0) bulk_wait0();
    }

    tc_fence_before();
    __syncthreads();
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, 2 * TN);
    }
}

// ---------------------------------------------------------------------------------------------- launchers
template <int MODE, int TN, int STAGES>
static cudaError_t launch_t(const GemmArgs& a, int num_sms, cudaStream_t st) {
    using Plan = SmemPlan<MODE, TN, STAGES>;
    k_gemm_sm100<MODE, TN, STAGES><<<num_sms, 192, Plan::TOTAL, st>>>(a);
    return cudaGetLastError();
}

cudaError_t init_sm100_kernels() {
    cudaError_t e;
#define FXM_SET(MODE, TN, ST)                                                                                     \
    e = cudaFuncSetAttribute(k_gemm_sm100<MODE, TN, ST>, cudaFuncAttributeMaxDynamicSharedMemorySize,             \
                             SmemPlan<MODE, TN, ST>::TOTAL);                                                            \
    if (e != cudaSuccess) return e;
    FXM_SET(1, 128, 5)
    FXM_SET(2, 128, 5)
    FXM_SET(1, 256, 4)
    FXM_SET(2, 256, 4)
#undef FXM_SET
    return cudaSuccess;
}

cudaError_t launch_gemm1_sm100(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                               DevState* state, int tile_n, int num_sms, cudaStream_t st) {
    GemmArgs a{};
    a.D = D; a.packed = packed; a.r_table = r_table; a.items = ws.items1; a.sched = ws.sched; a.Bsrc = ws.Xs;
    a.H = ws.H; a.state = state; a.P = ws.P;
    return tile_n == 256 ? launch_t<1, 256, 4>(a, num_sms, st) : launch_t<1, 128, 5>(a, num_sms, st);
}

cudaError_t launch_gemm2_sm100(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                               DevState* state, int tile_n, int num_sms, cudaStream_t st) {
    GemmArgs a{};
    a.D = D; a.packed = packed; a.r_table = r_table; a.items = ws.tt; a.sched = ws.sched; a.Bsrc = ws.H;
    a.O = ws.O; a.state = state; a.P = ws.P;
    return tile_n == 256 ? launch_t<2, 256, 4>(a, num_sms, st) : launch_t<2, 128, 5>(a, num_sms, st);
}

}  // namespace fxm
