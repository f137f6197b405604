// fxm_pair.cu -- steps a4/a5 as CTA-PAIR kernels (tcgen05.mma.cta_group::2): two SMs of one TPC share a tile.
//
//   a4  GEMM-1 + SwiGLU (Eq. 4; Alg. 2 l.12-16), swap-AB:
//         D[256 packed weight rows, N tokens] = Wgu[256, d] . Xs[N, d]^T,   UMMA M = 256 over the pair:
//         CTA r of the pair owns channel block cb = 2*cbp + r (64 gate + 64 up rows, lanes 0..127 of ITS TMEM).
//   a5  GEMM-2 (Alg. 2 l.18):
//         D[256 out features, N tokens] = Wd[256, r_e] . H[N, r_e]^T,  CTA r owns feature block db = 2*dbp + r;
//         K loop bounded by ceil(r_e/64): pruned K steps are never loaded or issued.
//
// Token tiles are up to 512 rows: a tile is one or two SUB-TILES of <= 256 tokens (UMMA N <= 256) that share the
// weight operand -- each weight byte is pulled from HBM/L2 into shared memory once per (expert, token tile), so a
// ragged expert (e.g. 273 tokens = 256 + 32 padded) does not re-read its weights for the tail.  Sub-tile s lives
// in TMEM columns [256 s, 256 s + N_s); sub-tiles are handed to the epilogue round-robin over the two halves, so
// tiles of <= 256 tokens are double-buffered (the epilogue of one overlaps the MMAs of the next).
//
// Per CTA and pipeline stage: A = one 16 KB weight tile, B0/B1 = this CTA's HALF of each sub-tile's token rows
// (the pair MMA reads N/2 rows from each CTA's shared memory).  Everything is moved by contiguous cp.async.bulk
// copies of pre-swizzled SW128 K-major data; no tensor map is needed.
//
// Warp roles (192 threads per CTA):  warp 0 = bulk-copy producer (both CTAs), warp 1 = MMA issuer in the leader
// CTA / RELAY in the peer CTA (forwards "my operands have landed" to the leader's barrier, since a plain bulk copy
// can only signal a barrier of its own CTA), warps 2-5 = epilogue (each CTA drains its own TMEM lanes).
// Barriers: full[s] (local, tx bytes), pfull[s] (leader, 1 remote arrive), empty[s] (both CTAs, multicast commit),
// tfull[h] (both CTAs, multicast commit), tempty[h] (leader, one arrive per CTA).
#include "fxm_ptx.cuh"

namespace fxm {

constexpr int PAIR_NSUB = 256;                  // tokens per sub-tile (UMMA N max)
constexpr int PAIR_BHALF = PAIR_NSUB / 2 * ROW_BYTES;   // 16 KB: one CTA's half of a sub-tile's B operand
constexpr int PAIR_STAGE = WT_BYTES + 2 * PAIR_BHALF;   // 48 KB
constexpr int PAIR_STAGES = 4;

struct PairArgs {
    Dims D;
    const uint8_t* packed;
    const int* r_table;
    const int4* items;         // GEMM-1: pair items {e, row0, valid rows, cbp}; GEMM-2: token tiles {e, row0, valid rows, .}
    const Sched* sched;
    const uint8_t* Bsrc;       // Xs (GEMM-1) or H (GEMM-2) panels
    uint8_t* H;                // GEMM-1 output panels
    uint8_t* O;                // GEMM-2 output rows [P][dpad] bf16
    DevState* state;
    int P;
};

template <int MODE>
struct PairSmem {
    static constexpr int STAGING = MODE == 1 ? PAIR_NSUB * ROW_BYTES : 0;     // H sub-tile (GEMM-2 stores straight from registers)
    static constexpr int BAR_OFF = PAIR_STAGES * PAIR_STAGE + STAGING;
    static constexpr int TOTAL = BAR_OFF + 256 + 1024;
};

// ------------------------------------------------------------------------------------------ cluster PTX
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_id_x() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%clusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ uint32_t cluster_count_x() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%nclusterid.x;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// arrive on the mbarrier at the same shared-memory offset in CTA `rank` of the cluster.  Default semantics
// (release at CTA scope): the signals forwarded this way order asynchronous-proxy traffic (bulk copies into shared
// memory, tcgen05 reads of shared / tensor memory) whose completion the arriving thread has already observed on a
// barrier; a cluster-scope release would put a GPU-wide MEMBAR on the critical path of every pipeline stage.
__device__ __forceinline__ void mbar_arrive_remote(uint32_t bar, uint32_t rank) {
    asm volatile(
        "{\n\t.reg .b32 ra;\n\t"
        "mapa.shared::cluster.u32 ra, %0, %1;\n\t"
        "mbarrier.arrive.shared::cluster.b64 _, [ra];\n\t}"
        ::"r"(bar), "r"(rank)
        : "memory");
}
__device__ __forceinline__ void tmem_alloc2(uint32_t dst_smem, uint32_t ncols) {
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(dst_smem), "r"(ncols) : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
__device__ __forceinline__ void tmem_dealloc2(uint32_t taddr, uint32_t ncols) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "r"(ncols) : "memory");
}
// D[tmem, both CTAs] (+)= A[smem, 128 rows per CTA] * B[smem, N/2 rows per CTA]; bf16 -> fp32, M = 256, K = 16
__device__ __forceinline__ void umma2_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc, uint32_t acc) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], %1, %2, %3, p;\n\t}"
        ::"r"(d_tmem), "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(acc)
        : "memory");
}
// when all MMAs issued so far have completed, arrive on the mbarrier at this offset in BOTH CTAs of the pair
__device__ __forceinline__ void umma2_commit_mc(uint32_t bar) {
    const uint16_t mask = 3;
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;"
                 ::"r"(bar), "h"(mask)
                 : "memory");
}
__device__ __forceinline__ uint32_t make_idesc2(uint32_t n) {     // M = 256 (pair), N = n
    return (1u << 4) | (1u << 7) | (1u << 10) | ((n >> 3) << 17) | ((256u >> 4) << 24);
}

// ------------------------------------------------------------------------------------------------ kernel
struct PairItem {
    int e, row0, n0, n1, blk, nk, r;
    bool valid;               // false: this CTA's weight block lies beyond the retained width (odd block count)
};

template <int MODE>
__device__ __forceinline__ PairItem pair_item(const PairArgs& a, int wi, uint32_t rank) {
    const Dims& D = a.D;
    PairItem it;
    int4 q;
    int pairblk;
    if (MODE == 1) {
        q = a.items[wi];
        pairblk = q.w;
    } else {
        const int nDBp = (D.nDB + 1) >> 1;
        q = a.items[wi / nDBp];
        pairblk = wi % nDBp;
    }
    it.e = q.x;
    it.row0 = q.y;
    const int n = (q.z + 15) & ~15;
    it.n0 = n < PAIR_NSUB ? n : PAIR_NSUB;
    it.n1 = n - it.n0;
    it.r = a.r_table[it.e];
    const int nb = (it.r + CB - 1) / CB;
    const int blk = 2 * pairblk + (int)rank;
    const int limit = MODE == 1 ? nb : D.nDB;
    it.valid = blk < limit;
    it.blk = it.valid ? blk : 2 * pairblk;      // a pruned / non-existent twin block: load the leader's block again, discard
    it.nk = MODE == 1 ? D.nKB1 : nb;
    return it;
}

template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(192, 1) k_gemm_pair(const PairArgs a) {
    extern __shared__ uint8_t smem_raw[];
    using Plan = PairSmem<MODE>;
    constexpr int ST = PAIR_STAGES;
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    const uint32_t bar_base = smem_base + Plan::BAR_OFF;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto pfull_bar = [&](int s) { return bar_base + 8u * (ST + s); };
    auto empty_bar = [&](int s) { return bar_base + 8u * (2 * ST + s); };
    auto tfull_bar = [&](int h) { return bar_base + 8u * (3 * ST + h); };
    auto tempty_bar = [&](int h) { return bar_base + 8u * (3 * ST + 2 + h); };
    volatile uint32_t* tmem_slot = (volatile uint32_t*)(smem_gen + Plan::BAR_OFF + 8 * (3 * ST + 4));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const Dims& D = a.D;

    if (threadIdx.x == 0) {
        for (int s = 0; s < ST; ++s) { mbar_init(full_bar(s), 1); mbar_init(pfull_bar(s), 1); mbar_init(empty_bar(s), 1); }
        for (int h = 0; h < 2; ++h) { mbar_init(tfull_bar(h), 1); mbar_init(tempty_bar(h), 2); }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc2(smem_u32((const void*)tmem_slot), 512);
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                                       // barriers of both CTAs are initialised before any remote use
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;

    const int W = MODE == 1 ? a.sched->W1 : a.sched->W2;
    const int wi0 = (int)cluster_id_x(), wstep = (int)cluster_count_x();
    const uint8_t* dn = a.packed + gu_bytes(D);

    if (warp == 0) {
        // ===================================================== producer (both CTAs): this CTA's A tile and B halves
        if (lane == 0) {
            int stage = 0;
            uint32_t phase = 0;
            for (int wi = wi0; wi < W; wi += wstep) {
                const PairItem it = pair_item<MODE>(a, wi, rank);
                const uint8_t* asrc;
                size_t astride;
                if (MODE == 1) {
                    asrc = a.packed + gu_tile_index(D, it.e, it.blk, 0) * WT_BYTES;
                    astride = WT_BYTES;
                } else {
                    asrc = dn + dn_tile_index(D, it.e, 0, it.blk) * WT_BYTES;
                    astride = (size_t)D.nDB * WT_BYTES;
                }
                const uint32_t h0 = (uint32_t)it.n0 >> 1, h1 = (uint32_t)it.n1 >> 1;      // rows of each sub-tile this CTA holds
                const uint8_t* b0 = a.Bsrc + (size_t)(it.row0 + rank * h0) * ROW_BYTES;
                const uint8_t* b1 = a.Bsrc + (size_t)(it.row0 + PAIR_NSUB + rank * h1) * ROW_BYTES;
                const size_t bstride = (size_t)a.P * ROW_BYTES;
                const uint32_t tx = WT_BYTES + (h0 + h1) * ROW_BYTES;
                for (int kb = 0; kb < it.nk; ++kb) {
                    mbar_wait(empty_bar(stage), phase ^ 1u, a.state);
                    const uint32_t sa = smem_base + stage * PAIR_STAGE;
                    mbar_expect_tx(full_bar(stage), tx);
                    bulk_g2s(sa, asrc + kb * astride, WT_BYTES, full_bar(stage));
                    bulk_g2s(sa + WT_BYTES, b0 + kb * bstride, h0 * ROW_BYTES, full_bar(stage));
                    if (h1) bulk_g2s(sa + WT_BYTES + PAIR_BHALF, b1 + kb * bstride, h1 * ROW_BYTES, full_bar(stage));
                    if (++stage == ST) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0 && rank == 0) {
            // ================================================= MMA issuer (leader CTA): one thread issues for the pair
            int stage = 0;
            uint32_t phase = 0, sc = 0;
            for (int wi = wi0; wi < W; wi += wstep) {
                const PairItem it = pair_item<MODE>(a, wi, rank);
                const uint32_t hA = sc & 1u, hB = (sc + 1u) & 1u;
                mbar_wait(tempty_bar(hA), ((sc >> 1) & 1u) ^ 1u, a.state);
                if (it.n1) mbar_wait(tempty_bar(hB), (((sc + 1u) >> 1) & 1u) ^ 1u, a.state);
                tc_fence_after();
                const uint32_t d0 = tmem_base + hA * PAIR_NSUB, d1 = tmem_base + hB * PAIR_NSUB;
                const uint32_t id0 = make_idesc2((uint32_t)it.n0), id1 = make_idesc2((uint32_t)(it.n1 ? it.n1 : 16));
                for (int kb = 0; kb < it.nk; ++kb) {
                    mbar_wait(full_bar(stage), phase, a.state);
                    mbar_wait(pfull_bar(stage), phase, a.state);
                    tc_fence_after();
                    const uint32_t sa = smem_base + stage * PAIR_STAGE;
                    const uint64_t adesc = make_desc_sw128(sa);
                    const uint64_t bd0 = make_desc_sw128(sa + WT_BYTES), bd1 = make_desc_sw128(sa + WT_BYTES + PAIR_BHALF);
#pragma unroll
                    for (int kk = 0; kk < KB / 16; ++kk)
                        umma2_bf16(d0, adesc + 2u * kk, bd0 + 2u * kk, id0, (uint32_t)((kb | kk) != 0));
                    if (it.n1) {
#pragma unroll
                        for (int kk = 0; kk < KB / 16; ++kk)
                            umma2_bf16(d1, adesc + 2u * kk, bd1 + 2u * kk, id1, (uint32_t)((kb | kk) != 0));
                    }
                    umma2_commit_mc(empty_bar(stage));          // frees this stage in BOTH CTAs when the MMAs retire
                    if (++stage == ST) { stage = 0; phase ^= 1u; }
                }
                umma2_commit_mc(tfull_bar(hA));
                if (it.n1) umma2_commit_mc(tfull_bar(hB));
                sc += it.n1 ? 2u : 1u;
            }
        } else if (lane == 0) {
            // ================================================= relay (peer CTA): my operands of stage s have landed
            int stage = 0;
            uint32_t phase = 0;
            for (int wi = wi0; wi < W; wi += wstep) {
                const PairItem it = pair_item<MODE>(a, wi, rank);
                for (int kb = 0; kb < it.nk; ++kb) {
                    mbar_wait(full_bar(stage), phase, a.state);
                    mbar_arrive_remote(pfull_bar(stage), 0);
                    if (++stage == ST) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else {
        // ===================================================== epilogue warps 2..5 (both CTAs, own TMEM lanes)
        const int q = warp & 3;
        const int et = threadIdx.x - 64;
        uint8_t* staging = smem_gen + ST * PAIR_STAGE;
        const uint32_t staging_s = smem_base + ST * PAIR_STAGE;
        const int dpad = D.nDB * WT_ROWS;
        uint32_t sc = 0;
        for (int wi = wi0; wi < W; wi += wstep) {
            const PairItem it = pair_item<MODE>(a, wi, rank);
            const int nsub = it.n1 ? 2 : 1;
            for (int s = 0; s < nsub; ++s, ++sc) {
                const uint32_t h = sc & 1u;
                const int n = s ? it.n1 : it.n0;
                const int rowS = it.row0 + s * PAIR_NSUB;
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + h * PAIR_NSUB;
                mbar_wait(tfull_bar(h), (sc >> 1) & 1u, a.state);
                tc_fence_after();
                if (MODE == 1) {
                    if (it.valid) {
                        const int ch = q * 16 + (lane & 15);
                        const bool keep = it.blk * CB + ch < it.r;       // tail mask of the last retained block (pad-zero rule)
                        const int odd = lane >> 4;
                        for (int c0 = 0; c0 < n; c0 += 16) {
                            uint32_t v[16];
                            tmem_ld16(taddr + c0, v);
                            tmem_ld_wait();
#pragma unroll
                            for (int m = 0; m < 8; ++m) {
                                const float mine0 = __uint_as_float(v[2 * m]), mine1 = __uint_as_float(v[2 * m + 1]);
                                const float send = odd ? mine0 : mine1;
                                const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
                                const float g = odd ? recv : mine0;
                                const float u = odd ? mine1 : recv;
                                float hv = __fdividef(g, 1.f + __expf(-g)) * u;
                                if (!keep) hv = 0.f;
                                const uint32_t t = c0 + 2 * m + odd;
                                *(__nv_bfloat16*)(staging + sw128_off(t, ch)) = __float2bfloat16_rn(hv);
                            }
                        }
                    }
                    tc_fence_before();
                    fence_proxy_async_smem();
                    epi_bar_sync();
                    if (et == 0) {
                        if (rank == 0) mbar_arrive(tempty_bar(h)); else mbar_arrive_remote(tempty_bar(h), 0);
                        if (it.valid) {
                            bulk_s2g(a.H + ((size_t)it.blk * a.P + rowS) * ROW_BYTES, staging_s, (uint32_t)n * ROW_BYTES);
                            bulk_commit();
                            bulk_wait_read0();
                        }
                    }
                    epi_bar_sync();
                } else {
                    if (it.valid) {
                        // lane = output feature; 16 token columns per load; 32 lanes -> 64 contiguous bytes of one O row
                        uint8_t* dst = a.O + ((size_t)rowS * dpad + it.blk * WT_ROWS + q * 32 + lane) * 2;
                        for (int c0 = 0; c0 < n; c0 += 16) {
                            uint32_t v[16];
                            tmem_ld16(taddr + c0, v);
                            tmem_ld_wait();
#pragma unroll
                            for (int jj = 0; jj < 16; ++jj)
                                *(__nv_bfloat16*)(dst + (size_t)(c0 + jj) * dpad * 2) = __float2bfloat16_rn(__uint_as_float(v[jj]));
                        }
                    }
                    tc_fence_before();
                    epi_bar_sync();
                    if (et == 0) {
                        if (rank == 0) mbar_arrive(tempty_bar(h)); else mbar_arrive_remote(tempty_bar(h), 0);
                    }
                }
            }
        }
        if (MODE == 1 && et == 0) bulk_wait0();
    }

    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                                       // the peer may still be reading my shared memory / arriving on my barriers
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc2(tmem_base, 512);
    }
}

// ---------------------------------------------------------------------------------------------- launchers
template <int MODE>
static cudaError_t launch_pair_t(const PairArgs& a, int num_sms, cudaStream_t st) {
    k_gemm_pair<MODE><<<num_sms / 2 * 2, 192, PairSmem<MODE>::TOTAL, st>>>(a);   // cluster dims are compiled in
    return cudaGetLastError();
}

cudaError_t init_pair_kernels() {
    cudaError_t e = cudaFuncSetAttribute(k_gemm_pair<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, PairSmem<1>::TOTAL);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_gemm_pair<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, PairSmem<2>::TOTAL);
}

cudaError_t launch_gemm1_pair(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                              DevState* state, int num_sms, cudaStream_t st) {
    PairArgs a{};
    a.D = D; a.packed = packed; a.r_table = r_table; a.items = ws.items1; a.sched = ws.sched; a.Bsrc = ws.Xs;
    a.H = ws.H; a.state = state; a.P = ws.P;
    return launch_pair_t<1>(a, num_sms, st);
}

cudaError_t launch_gemm2_pair(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                              DevState* state, int num_sms, cudaStream_t st) {
    PairArgs a{};
    a.D = D; a.packed = packed; a.r_table = r_table; a.items = ws.tt; a.sched = ws.sched; a.Bsrc = ws.H;
    a.O = ws.O; a.state = state; a.P = ws.P;
    return launch_pair_t<2>(a, num_sms, st);
}

}  // namespace fxm
