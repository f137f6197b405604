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
//       K loop bounded by ceil(r_e/64): pruned K steps are never loaded or issued.  The epilogue transposes the
//       accumulator through shared memory into rows of 128 output features (bf16) and writes the tile to the
//       O panel with one bulk store; the router-weight scale and the sum over a token's k experts are a gather
//       in k_combine (no atomics, slot order, fp32, one rounding).
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
#include "fxm_internal.cuh"

namespace fxm {

// ------------------------------------------------------------------------------------------ PTX wrappers
__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ uint32_t mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok;
}
// Bounded wait: a pipeline bug must end in a trap + sticky flag, never in a hung GPU.
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity, DevState* state) {
    if (mbar_try_wait(bar, parity)) return;
    const long long t0 = clock64();
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if ((++spins & 0xFFFu) == 0 && clock64() - t0 > 4000000000LL) {
            atomicOr(&state->flags, 2u);
            __threadfence_system();
            __trap();
        }
    }
}
__device__ __forceinline__ void fence_barrier_init() { asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory"); }
__device__ __forceinline__ void fence_proxy_async_smem() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }

// global -> shared bulk copy (contiguous), completion on an mbarrier
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
// shared -> global bulk copy (contiguous), bulk-group completion
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src, uint32_t bytes) {
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait_read0() { asm volatile("cp.async.bulk.wait_group.read 0;" ::: "memory"); }
__device__ __forceinline__ void bulk_wait0() { asm volatile("cp.async.bulk.wait_group 0;" ::: "memory"); }

__device__ __forceinline__ void tmem_alloc(uint32_t dst_smem, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// D[tmem] (+)= A[smem] * B[smem]; bf16 x bf16 -> fp32, M = 128, K = 16 per instruction
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc)
        : "memory");
}
// arrive on an mbarrier when all MMAs issued so far by this thread have completed
__device__ __forceinline__ void umma_commit(uint32_t bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void tmem_ld16(uint32_t taddr, uint32_t (&v)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 {%0,%1,%2,%3,%4,%5,%6,%7,%8,%9,%10,%11,%12,%13,%14,%15}, [%16];"
        : "=r"(v[0]), "=r"(v[1]), "=r"(v[2]), "=r"(v[3]), "=r"(v[4]), "=r"(v[5]), "=r"(v[6]), "=r"(v[7]), "=r"(v[8]),
          "=r"(v[9]), "=r"(v[10]), "=r"(v[11]), "=r"(v[12]), "=r"(v[13]), "=r"(v[14]), "=r"(v[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void epi_bar_sync() { asm volatile("bar.sync 1, 128;" ::: "memory"); }

// K-major, 128-byte-swizzled shared-memory matrix descriptor (sm_100 format): start>>4 | LBO(ignored)=1<<16 |
// SBO = 1024 B (8 rows) >>4 at bit 32 | version 1 at bit 46 | layout SWIZZLE_128B (2) at bit 61.
__device__ __forceinline__ uint64_t make_desc_sw128(uint32_t saddr) {
    return (uint64_t)((saddr & 0x3FFFFu) >> 4) | (1ull << 16) | (64ull << 32) | (1ull << 46) | (2ull << 61);
}
// instruction descriptor, kind::f16: D fp32 (bit 4), A bf16 (bit 7), B bf16 (bit 10), both K-major, N>>3 at 17, M>>4 at 24
__device__ __forceinline__ uint32_t make_idesc(uint32_t n) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((n >> 3) << 17) | ((128u >> 4) << 24);
}

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
    static constexpr int STAGING_BYTES = TN * (MODE == 1 ? ROW_BYTES : O_ROW_BYTES);   // H tile / O tile
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
                const int db = wi % D.nDB;
                uint8_t* mine = staging + (q * 32 + lane) * 2;       // this lane's output feature inside an O row
                for (int c0 = 0; c0 < n; c0 += 16) {
                    uint32_t v[16];
                    tmem_ld16(taddr + c0, v);
                    tmem_ld_wait();
#pragma unroll
                    for (int jj = 0; jj < 16; ++jj)                 // 32 lanes -> 64 contiguous bytes of row c0+jj
                        *(__nv_bfloat16*)(mine + (c0 + jj) * O_ROW_BYTES) = __float2bfloat16_rn(__uint_as_float(v[jj]));
                }
                tc_fence_before();
                mbar_arrive(tempty_bar(as));
                fence_proxy_async_smem();
                epi_bar_sync();
                if (et == 0) {
                    bulk_s2g(a.O + ((size_t)db * a.P + row0) * O_ROW_BYTES, staging_s, (uint32_t)n * O_ROW_BYTES);
                    bulk_commit();
                    bulk_wait_read0();
                }
                epi_bar_sync();
            }
            if (++as == 2) { as = 0; aphase ^= 1u; }
        }
        if (et == 0) bulk_wait0();
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
    FXM_SET(2, 256, 3)
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
    return tile_n == 256 ? launch_t<2, 256, 3>(a, num_sms, st) : launch_t<2, 128, 5>(a, num_sms, st);
}

}  // namespace fxm
