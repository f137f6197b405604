// fxm_pair.cu -- steps a4/a5 as CTA-PAIR kernels (tcgen05.mma.cta_group::2): two SMs of one TPC share a tile.
//
//   a4  GEMM-1 + SwiGLU (Eq. 4; Alg. 2 l.12-16), swap-AB:
//         D[256 packed weight rows, N tokens] = Wgu[256, d] . Xs[N, d]^T,   UMMA M = 256 over the pair:
//         CTA r of the pair owns channel block cb = 2*cbp + r (64 gate + 64 up rows, lanes 0..127 of ITS TMEM).
//         Epilogue: h = silu(g) * u (gate lane l, up lane l+16: one shuffle), channels >= r_e forced to 0 (the
//         paper's pad-zero rule), one rounding to bf16, stored straight into the swizzled H panel.
//   a5  GEMM-2 (Alg. 2 l.18):
//         D[256 out features, N tokens] = Wd[256, r_e] . H[N, r_e]^T,  CTA r owns feature block db = 2*dbp + r;
//         K loop bounded by ceil(r_e/64): pruned K steps are never loaded or issued.  Epilogue: one rounding to
//         bf16, O[row][feature]; the router-weight scale and the sum over k experts are the gather in k_combine.
//
// Token tiles are up to 512 rows: a tile is one or two SUB-TILES of <= 256 tokens (UMMA N <= 256) that share the
// weight operand -- each weight byte is pulled from HBM into shared memory once per (expert, token tile), so a
// ragged expert (e.g. 273 tokens = 256 + 32 padded) does not re-read its weights for the tail.  Sub-tile s lives
// in TMEM columns [256 s, 256 s + N_s); sub-tiles are handed to the epilogue round-robin over the two halves, so
// tiles of <= 256 tokens are double-buffered (the epilogue of one overlaps the MMAs of the next).
//
// Two operand rings per CTA, because the operands have different latencies: the WEIGHT ring is deep (8 x 16 KB:
// weights have no reuse inside a token tile and come from HBM, ~2-3 us away under load), the TOKEN ring is
// shallow (3 x 32 KB: this CTA's half of each sub-tile's rows, re-read by every weight block, so they come from
// L2).  Everything is moved by contiguous cp.async.bulk copies of pre-swizzled SW128 K-major data.
//
// Warp roles (384 threads per CTA): warp 0 = weight producer, warp 2 = token producer, warp 1 = MMA issuer in the
// leader CTA / RELAY in the peer CTA (forwards "my operands of this k-block have landed" to the leader's barrier,
// since a plain bulk copy can only signal a barrier of its own CTA), warps 4-11 = epilogue (each CTA drains its
// own TMEM lanes; two warps per lane quadrant, each taking half of the columns).
// Barriers: fullA/fullB (local, tx bytes), pfull (leader, 1 remote arrive per k-block), emptyA/emptyB (both CTAs,
// multicast commit), tfull[h] (both CTAs, multicast commit), tempty[h] (leader, one arrive per CTA).
#include "fxm_ptx.cuh"

namespace fxm {

constexpr int PAIR_NSUB = 256;                  // tokens per sub-tile (UMMA N max)
constexpr int PAIR_BHALF = PAIR_NSUB / 2 * ROW_BYTES;   // 16 KB: one CTA's half of a sub-tile's B operand
constexpr int PAIR_BSLOT = 2 * PAIR_BHALF;      // 32 KB
constexpr int PAIR_NA = 8;                      // weight ring depth
constexpr int PAIR_NB = 3;                      // token ring depth
constexpr int PAIR_THREADS = 384;

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

constexpr int PAIR_A_OFF = 0;
constexpr int PAIR_B_OFF = PAIR_NA * WT_BYTES;
constexpr int PAIR_BAR_OFF = PAIR_B_OFF + PAIR_NB * PAIR_BSLOT;
constexpr int PAIR_SMEM = PAIR_BAR_OFF + 512 + 1024;      // + barriers + alignment slack

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

__device__ __forceinline__ void epi_bar_sync256() { asm volatile("bar.sync 1, 256;" ::: "memory"); }

template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PAIR_THREADS, 1) k_gemm_pair(const PairArgs a) {
    extern __shared__ uint8_t smem_raw[];
    constexpr int NA = PAIR_NA, NB = PAIR_NB;
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    const uint32_t bar_base = smem_base + PAIR_BAR_OFF;
    auto fullA = [&](int s) { return bar_base + 8u * s; };
    auto emptyA = [&](int s) { return bar_base + 8u * (NA + s); };
    auto pfull = [&](int s) { return bar_base + 8u * (2 * NA + s); };
    auto fullB = [&](int s) { return bar_base + 8u * (3 * NA + s); };
    auto emptyB = [&](int s) { return bar_base + 8u * (3 * NA + NB + s); };
    auto tfull_bar = [&](int h) { return bar_base + 8u * (3 * NA + 2 * NB + h); };
    auto tempty_bar = [&](int h) { return bar_base + 8u * (3 * NA + 2 * NB + 2 + h); };
    volatile uint32_t* tmem_slot = (volatile uint32_t*)(smem_gen + PAIR_BAR_OFF + 8 * (3 * NA + 2 * NB + 4));

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const Dims& D = a.D;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NA; ++s) { mbar_init(fullA(s), 1); mbar_init(emptyA(s), 1); mbar_init(pfull(s), 1); }
        for (int s = 0; s < NB; ++s) { mbar_init(fullB(s), 1); mbar_init(emptyB(s), 1); }
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
        // ===================================================== weight producer (both CTAs): this CTA's 16 KB A tiles
        if (lane == 0) {
            int sa = 0;
            uint32_t pa = 0;
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
                for (int kb = 0; kb < it.nk; ++kb) {
                    mbar_wait(emptyA(sa), pa ^ 1u, a.state);
                    mbar_expect_tx(fullA(sa), WT_BYTES);
                    bulk_g2s(smem_base + PAIR_A_OFF + sa * WT_BYTES, asrc + kb * astride, WT_BYTES, fullA(sa));
                    if (++sa == NA) { sa = 0; pa ^= 1u; }
                }
            }
        }
    } else if (warp == 2) {
        // ===================================================== token producer (both CTAs): this CTA's half of each sub-tile
        if (lane == 0) {
            int sb = 0;
            uint32_t pb = 0;
            const size_t bstride = (size_t)a.P * ROW_BYTES;
            for (int wi = wi0; wi < W; wi += wstep) {
                const PairItem it = pair_item<MODE>(a, wi, rank);
                const uint32_t h0 = (uint32_t)it.n0 >> 1, h1 = (uint32_t)it.n1 >> 1;      // rows of each sub-tile this CTA holds
                const uint8_t* b0 = a.Bsrc + (size_t)(it.row0 + rank * h0) * ROW_BYTES;
                const uint8_t* b1 = a.Bsrc + (size_t)(it.row0 + PAIR_NSUB + rank * h1) * ROW_BYTES;
                for (int kb = 0; kb < it.nk; ++kb) {
                    mbar_wait(emptyB(sb), pb ^ 1u, a.state);
                    const uint32_t sbase = smem_base + PAIR_B_OFF + sb * PAIR_BSLOT;
                    mbar_expect_tx(fullB(sb), (h0 + h1) * ROW_BYTES);
                    bulk_g2s(sbase, b0 + kb * bstride, h0 * ROW_BYTES, fullB(sb));
                    if (h1) bulk_g2s(sbase + PAIR_BHALF, b1 + kb * bstride, h1 * ROW_BYTES, fullB(sb));
                    if (++sb == NB) { sb = 0; pb ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        if (lane == 0 && rank == 0) {
            // ================================================= MMA issuer (leader CTA): one thread issues for the pair
            int sa = 0, sb = 0;
            uint32_t pa = 0, pb = 0, sc = 0;
            for (int wi = wi0; wi < W; wi += wstep) {
                const PairItem it = pair_item<MODE>(a, wi, rank);
                const uint32_t hA = sc & 1u, hB = (sc + 1u) & 1u;
                mbar_wait(tempty_bar(hA), ((sc >> 1) & 1u) ^ 1u, a.state);
                if (it.n1) mbar_wait(tempty_bar(hB), (((sc + 1u) >> 1) & 1u) ^ 1u, a.state);
                tc_fence_after();
                const uint32_t d0 = tmem_base + hA * PAIR_NSUB, d1 = tmem_base + hB * PAIR_NSUB;
                const uint32_t id0 = make_idesc2((uint32_t)it.n0), id1 = make_idesc2((uint32_t)(it.n1 ? it.n1 : 16));
                for (int kb = 0; kb < it.nk; ++kb) {
                    mbar_wait(fullA(sa), pa, a.state);
                    mbar_wait(fullB(sb), pb, a.state);
                    mbar_wait(pfull(sa), pa, a.state);          // the peer CTA's halves of this k-block
                    tc_fence_after();
                    const uint32_t sB = smem_base + PAIR_B_OFF + sb * PAIR_BSLOT;
                    const uint64_t adesc = make_desc_sw128(smem_base + PAIR_A_OFF + sa * WT_BYTES);
                    const uint64_t bd0 = make_desc_sw128(sB), bd1 = make_desc_sw128(sB + PAIR_BHALF);
#pragma unroll
                    for (int kk = 0; kk < KB / 16; ++kk)
                        umma2_bf16(d0, adesc + 2u * kk, bd0 + 2u * kk, id0, (uint32_t)((kb | kk) != 0));
                    if (it.n1) {
#pragma unroll
                        for (int kk = 0; kk < KB / 16; ++kk)
                            umma2_bf16(d1, adesc + 2u * kk, bd1 + 2u * kk, id1, (uint32_t)((kb | kk) != 0));
                    }
                    umma2_commit_mc(emptyA(sa));                // frees the slots in BOTH CTAs when these MMAs retire
                    umma2_commit_mc(emptyB(sb));
                    if (++sa == NA) { sa = 0; pa ^= 1u; }
                    if (++sb == NB) { sb = 0; pb ^= 1u; }
                }
                umma2_commit_mc(tfull_bar(hA));
                if (it.n1) umma2_commit_mc(tfull_bar(hB));
                sc += it.n1 ? 2u : 1u;
            }
        } else if (lane == 0) {
            // ================================================= relay (peer CTA): my operands of this k-block have landed
            int sa = 0, sb = 0;
            uint32_t pa = 0, pb = 0;
            for (int wi = wi0; wi < W; wi += wstep) {
                const PairItem it = pair_item<MODE>(a, wi, rank);
                for (int kb = 0; kb < it.nk; ++kb) {
                    mbar_wait(fullA(sa), pa, a.state);
                    mbar_wait(fullB(sb), pb, a.state);
                    mbar_arrive_remote(pfull(sa), 0);
                    if (++sa == NA) { sa = 0; pa ^= 1u; }
                    if (++sb == NB) { sb = 0; pb ^= 1u; }
                }
            }
        }
    } else if (warp >= 4) {
        // ===================================================== epilogue warps 4..11 (both CTAs, own TMEM lanes)
        const int q = warp & 3;                                // TMEM lane quadrant this warp may read
        const int grp = (warp - 4) >> 2;                       // which half of the columns
        const int et = threadIdx.x - 128;
        const int dpad = D.nDB * WT_ROWS;
        uint32_t sc = 0;
        for (int wi = wi0; wi < W; wi += wstep) {
            const PairItem it = pair_item<MODE>(a, wi, rank);
            const int nsub = it.n1 ? 2 : 1;
            for (int s = 0; s < nsub; ++s, ++sc) {
                const uint32_t h = sc & 1u;
                const int n = s ? it.n1 : it.n0;
                const int split = ((n >> 4) + 1) / 2 * 16;    // columns [0, split) -> group 0, [split, n) -> group 1
                const int cbeg = grp ? split : 0, cend = grp ? n : split;
                const int rowS = it.row0 + s * PAIR_NSUB;
                const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + h * PAIR_NSUB;
                mbar_wait(tfull_bar(h), (sc >> 1) & 1u, a.state);
                tc_fence_after();
                if (it.valid && cbeg < cend) {
                    // two register buffers: the TMEM load of the next 16 columns is in flight while these are processed
                    uint32_t va[16], vb[16];
                    if (MODE == 1) {
                        const int ch = q * 16 + (lane & 15);
                        const bool keep = it.blk * CB + ch < it.r;       // tail mask of the last retained block (pad-zero rule)
                        const int odd = lane >> 4;
                        uint8_t* hrow = a.H + ((size_t)it.blk * a.P + rowS) * ROW_BYTES;
                        auto swiglu16 = [&](const uint32_t (&v)[16], int c0) {
#pragma unroll
                            for (int m = 0; m < 8; ++m) {
                                const float mine0 = __uint_as_float(v[2 * m]), mine1 = __uint_as_float(v[2 * m + 1]);
                                const float send = odd ? mine0 : mine1;                    // what the twin lane needs
                                const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
                                const float g = odd ? recv : mine0;                        // gate lives in lanes 0-15
                                const float u = odd ? mine1 : recv;                        // up lives in lanes 16-31
                                float hv = __fdividef(g, 1.f + __expf(-g)) * u;
                                if (!keep) hv = 0.f;
                                const uint32_t t = c0 + 2 * m + odd;                       // 16 lanes -> one full 32-byte sector
                                *(__nv_bfloat16*)(hrow + sw128_off(t, ch)) = __float2bfloat16_rn(hv);
                            }
                        };
                        tmem_ld16(taddr + cbeg, va);
                        for (int c0 = cbeg; c0 < cend; c0 += 32) {
                            tmem_ld_wait();
                            if (c0 + 16 < cend) tmem_ld16(taddr + c0 + 16, vb);
                            swiglu16(va, c0);
                            tmem_ld_wait();
                            if (c0 + 32 < cend) tmem_ld16(taddr + c0 + 32, va);
                            if (c0 + 16 < cend) swiglu16(vb, c0 + 16);
                        }
                    } else {
                        // lane = output feature; 16 token columns per load; 32 lanes -> 64 contiguous bytes of one O row
                        uint8_t* dst = a.O + ((size_t)rowS * dpad + it.blk * WT_ROWS + q * 32 + lane) * 2;
                        auto store16 = [&](const uint32_t (&v)[16], int c0) {
#pragma unroll
                            for (int jj = 0; jj < 16; ++jj)
                                *(__nv_bfloat16*)(dst + (size_t)(c0 + jj) * dpad * 2) = __float2bfloat16_rn(__uint_as_float(v[jj]));
                        };
                        tmem_ld16(taddr + cbeg, va);
                        for (int c0 = cbeg; c0 < cend; c0 += 32) {
                            tmem_ld_wait();
                            if (c0 + 16 < cend) tmem_ld16(taddr + c0 + 16, vb);
                            store16(va, c0);
                            tmem_ld_wait();
                            if (c0 + 32 < cend) tmem_ld16(taddr + c0 + 32, va);
                            if (c0 + 16 < cend) store16(vb, c0 + 16);
                        }
                    }
                }
                tc_fence_before();
                epi_bar_sync256();                             // all 8 warps have drained this half of TMEM
                if (et == 0) {
                    if (rank == 0) mbar_arrive(tempty_bar(h)); else mbar_arrive_remote(tempty_bar(h), 0);
                }
            }
        }
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
    k_gemm_pair<MODE><<<num_sms / 2 * 2, PAIR_THREADS, PAIR_SMEM, st>>>(a);   // cluster dims are compiled in
    return cudaGetLastError();
}

cudaError_t init_pair_kernels() {
    cudaError_t e = cudaFuncSetAttribute(k_gemm_pair<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, PAIR_SMEM);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_gemm_pair<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, PAIR_SMEM);
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
