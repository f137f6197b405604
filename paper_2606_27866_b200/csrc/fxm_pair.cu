// fxm_pair.cu -- steps a4/a5 as CTA-PAIR kernels (tcgen05.mma.cta_group::2): two SMs of one TPC share a tile.
//
//   a4  GEMM-1 + SwiGLU (Eq. 4; Alg. 2 l.12-16), swap-AB:
//         D[256 packed weight rows, N tokens] = Wgu[256, d] . X[pi][N, d]^T,   UMMA M = 256 over the pair:
//         CTA r of the pair owns channel block cb = 2*cbp + r (64 gate + 64 up rows, lanes 0..127 of ITS TMEM).
//         Epilogue: h = silu(g) * u (gate lane l, up lane l+16: one shuffle), channels >= r_e forced to 0 (the
//         paper's pad-zero rule), one rounding to bf16 -> the swizzled H panel.
//   a5  GEMM-2 + router-weight scale + scatter-add combine (Alg. 2 l.18-20):
//         D[256 out features, N tokens] = Wd[256, r_e] . H[N, r_e]^T,  CTA r owns feature block db = 2*dbp + r;
//         K loop bounded by ceil(r_e/64): pruned K steps are never loaded or issued.  Epilogue: every epilogue warp
//         pulls its share of the accumulator into registers (tcgen05.ld), hands the TMEM columns back to the MMA
//         warp at once, then scales each token column by its router weight in fp32 and adds it into the fp32
//         accumulator yacc[token][feature] with red.global.add.f32 -- a warp covers 32 consecutive features of one
//         token = one 128-byte line per instruction (measured on B200: 5.7 TB/s of fp32 adds, the speed of plain
//         stores; cp.reduce.async.bulk is 3x slower).  No O panels, no combine kernel, no third rounding.
//
// Token tiles are up to 512 rows: a tile is one or two SUB-TILES of <= 256 tokens (UMMA N <= 256, balanced split)
// that share the weight operand -- each weight byte is pulled into shared memory once per (expert, token tile).
//
// Pipeline (what the in-kernel timeline of the previous version showed: the MMA thread was ISSUE-bound -- three
// barrier waits, two commits and a register->uniform-register "waterfall" per instruction, because it ran in a
// divergent `lane == 0` branch -- and the epilogue was serialised with the main loop):
//   * every role runs WARP-UNIFORM: all 32 lanes walk the loops and poll the barriers, one elected lane issues the
//     asynchronous instruction, so descriptors and addresses live in uniform registers;
//   * ONE ring of stages, each stage = this CTA's 16 KB weight tile + its half of the token rows of one k-block;
//     the stage size follows the largest token tile of the call (Sched::max_n), so small tiles get a deep ring;
//   * ONE wait per k-block for the MMA warp: the leader's full barrier counts its own producer's arrive(+tx) AND the
//     peer CTA's relay ("my half has landed"); ONE multicast commit frees the stage in both CTAs;
//   * TMEM is a circular column allocator: a sub-tile takes N contiguous columns, so the MMAs of the next item start
//     as soon as the columns they need are drained (tiles of <= 256 tokens are fully double-buffered);
//   * the GEMM-1 epilogue stages its output in shared memory in the final layout and writes it with bulk stores (the H
//     panels make a CTA's output of a sub-tile one contiguous range); the GEMM-2 epilogue has no staging at all;
//   * GEMM-1 takes its token rows straight from x (X[pi], Alg. 2 l.7): TMA tile::gather4 through a tensor map over
//     x [T][d], four rows per instruction, landing in the swizzled K-major operand layout -- no gathered copy of x;
//   * an optional L2 prefetch cursor over the weight tiles exists (FXM_PAIR_PF) but is off: every distance > 0 was slower.
//
// Warp roles: warp 0 = weight producer, warp 1 = MMA issuer (leader CTA) / relay (peer CTA), GEMM-1 only: warps 2-7 =
// gather warps (a gather4 costs one warp ~60 cycles of issue, six of them keep up with the MMAs), then 16 epilogue
// warps (each CTA drains its own TMEM lanes; four warps per lane quadrant).  768 threads (GEMM-1) / 640 (GEMM-2).
// GEMM-1's epilogue warps also zero yacc (the scatter-add target of GEMM-2) before their first tile: they are idle
// while the first tiles are multiplied, so the fp32 accumulator costs no launch and no time of its own.
#include "fxm_ptx.cuh"

#include <cuda.h>          // CUtensorMap and the cuTensorMapEncodeTiled prototype (resolved at run time, no libcuda link)

namespace fxm {

constexpr int PAIR_NSUB = 256;                  // most tokens per sub-tile (UMMA N max)
constexpr int PAIR_EPI_WARPS = 16;              // epilogue warps: 4 per TMEM lane quadrant (the SwiGLU epilogue is issue-bound)
#ifndef FXM_PAIR_GW
#define FXM_PAIR_GW 6
#endif
constexpr int PAIR_GW = FXM_PAIR_GW;                      // gather warps of GEMM-1 (TMA gather4 issue costs ~60 cycles per 4 rows and warp)
// warps: 0 producer, 1 MMA / relay, [GEMM-1: 2..7 gather], then the epilogue warps (first one a multiple of 4)
template <int MODE> struct PairCfg {
    static constexpr int EPI0 = MODE == 1 ? (2 + PAIR_GW + 3) / 4 * 4 : 4;
    static constexpr int THREADS = 32 * (EPI0 + PAIR_EPI_WARPS);
};
constexpr int PAIR_MAX_STAGES = 8;
constexpr int PAIR_SMEM = 232448;               // 227 KB: everything a CTA can have
constexpr int PAIR_AUX = 2048;                  // barriers (264 B) and, at +512, the gather warps' token indices
// after the ring: GEMM-1 two 16 KB epilogue staging buffers; GEMM-2 two sets of 512 {token, router weight} pairs
template <int MODE> struct PairSmem {
    static constexpr int EXTRA = MODE == 1 ? 2 * 16384 : 2 * 512 * 8;
    static constexpr int RING = PAIR_SMEM - 1024 /*alignment slack*/ - EXTRA - PAIR_AUX;   // GEMM-1: 4 x 48 KB
};
constexpr int PAIR_GMAX = (PAIR_NSUB / 4 + PAIR_GW - 1) / PAIR_GW;     // most 4-row groups one gather warp issues per k-block
constexpr int PAIR_TQ = 8;                      // TMEM sub-tile barrier ring
#ifndef FXM_PAIR_PF
#define FXM_PAIR_PF 0
#endif
constexpr int PAIR_PF = FXM_PAIR_PF;                     // weight tiles the L2 prefetch cursor runs ahead (measured: 0 is fastest, 12 costs 2-5 %)

struct PairArgs {
    Dims D;
    LayerView V;
    const int* r_table;
    const int4* items;         // token tiles {e, row0, valid rows, GEMM-1 work prefix}; [ntt] = sentinel
    const Sched* sched;
    const uint8_t* Bsrc;       // GEMM-2: the H panels
    const int* tok;            // GEMM-1: token index of every padded row (the gather4 row coordinates)
    uint8_t* H;                // GEMM-1 output panels
    const int2* row_tw;        // GEMM-2: {token or -1, router weight bits} of every padded row
    float* yacc;               // GEMM-2: fp32 scatter-add target [T][d]; GEMM-1 zeroes it
    DevState* state;
    int P;
    int T;
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
// one lane of a converged warp
__device__ __forceinline__ bool elect_one() {
    uint32_t p;
    asm volatile(
        "{\n\t.reg .pred q;\n\t"
        "elect.sync _|q, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, q;\n\t}"
        : "=r"(p));
    return p != 0;
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
// TMA gather4: four rows (row coordinates r0..r3) x 64 bf16 columns starting at `col` of the 2-D tensor behind `map`
// land as four consecutive 128-byte rows at `dst`, 128-byte swizzled by shared-memory address -- the K-major SW128
// operand layout tcgen05.mma reads.  512 bytes complete on `bar`.
__device__ __forceinline__ void tma_gather4(uint32_t dst, const void* map, int col, int4 r, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cta.global.tile::gather4.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5, %6}], [%7];"
        ::"r"(dst), "l"(map), "r"(col), "r"(r.x), "r"(r.y), "r"(r.z), "r"(r.w), "r"(bar)
        : "memory");
}
__device__ __forceinline__ uint32_t make_idesc2(uint32_t n) {     // M = 256 (pair), N = n
    return (1u << 4) | (1u << 7) | (1u << 10) | ((n >> 3) << 17) | ((256u >> 4) << 24);
}
__device__ __forceinline__ void epi_bar_sync_all() { asm volatile("bar.sync 1, %0;" ::"n"(32 * PAIR_EPI_WARPS) : "memory"); }
__device__ __forceinline__ int shfl0(int v) { return __shfl_sync(0xffffffffu, v, 0); }   // also tells the compiler: warp-uniform

// ------------------------------------------------------------------------------------------------ timeline
// -DFXM_TRACE: the leader CTA of every cluster records clock64() stamps of its first 16 items (tuning aid; the
// product build has none of this).  Fields: 0 item start (MMA warp), 1 accumulator columns free, 2 main loop done,
// 3 cycles spent waiting for full stages, 4 epilogue sees the first sub-tile, 5 epilogue done, 6 producer cycles
// spent waiting for empty stages, 7 tokens, 8 k-blocks.
#ifdef FXM_TRACE
__device__ long long g_trace[2][74][16][10];
#define FXM_TR(mode, j, f, v) do { if ((j) < 16 && cluster_id_x() < 74u) g_trace[(mode) - 1][cluster_id_x()][(j)][(f)] = (long long)(v); } while (0)
#define FXM_CLK() clock64()
#else
#define FXM_TR(mode, j, f, v) do { } while (0)
#define FXM_CLK() 0ll
#endif

// ------------------------------------------------------------------------------------------------ items
struct PairItem {
    int e, row0, n0, n1, blk, nk, r;
    uint32_t eblk;            // first channel block of the expert in the weight regions
    bool valid;               // false: this CTA's weight block lies beyond the retained width (odd block count)
};

// `cur` = this role's cursor over the token tiles (GEMM-1: item wi belongs to the tile j with tt[j].w <= wi < tt[j+1].w;
// a role's items ascend, so the cursor only moves forward -- a few L1 hits per item)
template <int MODE>
__device__ __forceinline__ PairItem pair_item(const PairArgs& a, int wi, uint32_t rank, int& cur) {
    const Dims& D = a.D;
    PairItem it;
    int4 q;
    int pairblk;
    // Items of one expert are walked BLOCK-major: (block pair, token tile) instead of (token tile, block pair).  The tiles of
    // an expert read the same weight tiles; with a static stride over the item list they now run on neighbouring clusters in
    // the same round, so the second reader finds the tile in L2 (or merges with the miss in flight) instead of fetching it
    // from HBM again 40 us later.  The tile list stays tile-major (tt[j].w = work prefix of tile j); .z carries the number
    // of tiles of the expert (nt) and the tile's index among them (t0).
    if (MODE == 1) {
        while (__ldg(&a.items[cur + 1].w) <= wi) ++cur;
        q = __ldg(a.items + cur);
        const int nt = (q.z >> 16) & 0xFF, t0 = (q.z >> 24) & 0xFF;
        const int nbp = __ldg(&a.items[cur + 1].w) - q.w;          // block pairs per tile (the same for every tile of the expert)
        const int L = wi - (q.w - t0 * nbp);                        // position inside the expert's nt * nbp items
        pairblk = L / nt;
        const int t = L - pairblk * nt;
        if (t != t0) q = __ldg(a.items + (cur - t0 + t));
    } else {
        const int nDBp = (D.nDB + 1) >> 1;
        const int jt = wi / nDBp;
        q = a.items[jt];
        const int nt = (q.z >> 16) & 0xFF, t0 = (q.z >> 24) & 0xFF;
        const int L = wi - (jt - t0) * nDBp;
        pairblk = L / nt;
        const int t = L - pairblk * nt;
        if (t != t0) q = a.items[jt - t0 + t];
    }
    it.e = q.x;
    it.row0 = q.y;
    const int n = ((q.z & 0xFFFF) + 15) & ~15;
    // one sub-tile up to 256 tokens, else two balanced ones (both multiples of 16)
    it.n0 = n <= PAIR_NSUB ? n : (((n >> 4) + 1) >> 1) << 4;
    it.n1 = n - it.n0;
    it.r = a.r_table[it.e];
    it.eblk = a.V.eblk[it.e];
    const int nb = (it.r + CB - 1) / CB;
    const int blk = 2 * pairblk + (int)rank;
    const int limit = MODE == 1 ? nb : D.nDB;
    it.valid = blk < limit;
    it.blk = it.valid ? blk : 2 * pairblk;      // a pruned / non-existent twin block: load the leader's block again, discard
    it.nk = MODE == 1 ? D.nKB1 : nb;
    return it;
}

// Circular TMEM column allocator, replayed identically by the MMA warp and by every epilogue thread: sub-tile
// number q (in issue order) takes w contiguous columns at the returned offset.  `need` = how many sub-tiles must
// have been drained before the MMAs of q may write (sub-tiles are drained in order): the newest earlier sub-tile
// whose columns overlap, and q - PAIR_TQ because the barrier ring has PAIR_TQ entries.
// (lo / hi are indexed with run-time values and therefore live in local memory; a register-only shift-register form
// was tried and backed out -- no measured gain.)
struct TmemRing {
    uint32_t head, seq;
    uint32_t lo[PAIR_TQ], hi[PAIR_TQ];
    __device__ __forceinline__ void init() { head = 0; seq = 0; }
    __device__ __forceinline__ uint32_t record(uint32_t c, uint32_t w) {      // -> sub-tiles that must be drained first
        uint32_t nd = seq >= (uint32_t)PAIR_TQ ? seq - PAIR_TQ + 1 : 0;
#pragma unroll
        for (uint32_t i = 1; i < (uint32_t)PAIR_TQ; ++i) {
            if (i <= seq) {
                const uint32_t s = seq - i;
                if (lo[s % PAIR_TQ] < c + w && hi[s % PAIR_TQ] > c && s + 1 > nd) nd = s + 1;
            }
        }
        lo[seq % PAIR_TQ] = c;
        hi[seq % PAIR_TQ] = c + w;
        ++seq;
        return nd;
    }
    // the one or two sub-tiles of an item (n0 + n1 <= 512); they never overlap each other
    __device__ __forceinline__ void alloc_item(uint32_t n0, uint32_t n1, uint32_t& c0, uint32_t& c1, uint32_t& need) {
        if (head + n0 > 512u) head = 0;
        c0 = head;
        c1 = 0;
        if (n1) {
            if (c0 + n0 + n1 <= 512u) c1 = c0 + n0;
            else if (n1 <= c0) c1 = 0;
            else { c0 = 0; c1 = n0; }
        }
        head = n1 ? c1 + n1 : c0 + n0;
        need = record(c0, n0);
        if (n1) need = max(need, record(c1, n1));              // disjoint from [c0, c0 + n0) by construction
    }
};

// ------------------------------------------------------------------------------------------------ kernel
template <int MODE>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(PairCfg<MODE>::THREADS, 1)
k_gemm_pair(const PairArgs a, const __grid_constant__ CUtensorMap xmap) {
    constexpr int EPI0 = PairCfg<MODE>::EPI0;
    extern __shared__ uint8_t smem_raw[];
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    constexpr int PAIR_RING_BYTES = PairSmem<MODE>::RING;
    constexpr int PAIR_EXTRA = PairSmem<MODE>::EXTRA;
    [[maybe_unused]] const uint32_t stg_base = smem_base + PAIR_RING_BYTES;   // GEMM-1: epilogue staging, 2 x 16 KB
    [[maybe_unused]] uint8_t* stg_gen = smem_gen + PAIR_RING_BYTES;            // GEMM-2: row info, 2 x 512 x {token, weight}
    const uint32_t bar_base = smem_base + PAIR_RING_BYTES + PAIR_EXTRA;
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (PAIR_MAX_STAGES + s); };
    auto tfull_bar = [&](uint32_t q) { return bar_base + 8u * (2 * PAIR_MAX_STAGES + (q % PAIR_TQ)); };
    auto tempty_bar = [&](uint32_t q) { return bar_base + 8u * (2 * PAIR_MAX_STAGES + PAIR_TQ + (q % PAIR_TQ)); };
    volatile uint32_t* tmem_slot = (volatile uint32_t*)(smem_gen + PAIR_RING_BYTES + PAIR_EXTRA + 8 * (2 * PAIR_MAX_STAGES + 2 * PAIR_TQ));
    [[maybe_unused]] int4* gidx = (int4*)(smem_gen + PAIR_RING_BYTES + PAIR_EXTRA + 512);   // [PAIR_GW][PAIR_GMAX] token indices

    const int warp = shfl0(threadIdx.x >> 5), lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    pdl_launch_dependents();
    const Dims& D = a.D;

    if (threadIdx.x == 0) {
        for (int s = 0; s < PAIR_MAX_STAGES; ++s) {
            // leader: own producer + the peer's relay; GEMM-1: + one arrival per gather warp
            mbar_init(full_bar(s), (rank == 0 ? 2 : 1) + (MODE == 1 ? PAIR_GW : 0));
            mbar_init(empty_bar(s), 1);
        }
        // "columns drained": one arrival per epilogue warp of both CTAs (a warp arrives as soon as its share is in registers)
        for (int q = 0; q < PAIR_TQ; ++q) { mbar_init(tfull_bar(q), 1); mbar_init(tempty_bar(q), 2 * PAIR_EPI_WARPS); }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc2(smem_u32((const void*)tmem_slot), 512);
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                                       // barriers of both CTAs are initialised before any remote use
    tc_fence_after();
    const uint32_t tmem_base = *tmem_slot;
    pdl_wait();                                               // everything above overlapped the previous kernel's tail

    // ring geometry of this call: a stage holds one 16 KB weight tile and this CTA's half of the widest token tile
    const int max_n = a.sched->max_n;
    const uint32_t stage_bytes = WT_BYTES + (((uint32_t)max_n * (ROW_BYTES / 2) + 1023u) & ~1023u);
    const int NS = min(PAIR_MAX_STAGES, (int)(PAIR_RING_BYTES / stage_bytes));


    constexpr bool gather = MODE == 1;                        // GEMM-1 token rows come straight from x via TMA gather4
    const int W = MODE == 1 ? a.sched->W1 : a.sched->W2;
    const int wi0 = (int)cluster_id_x(), wstep = (int)cluster_count_x();
    int cur = 0;                                              // every role walks the same item sequence with its own tile cursor
    [[maybe_unused]] int pf_cur = 0;
    auto a_src = [&](const PairItem& it, size_t& stride) -> const uint8_t* {
        if (MODE == 1) { stride = WT_BYTES; return a.V.gu + gu_tile_off(D, it.eblk, it.blk, 0); }
        stride = (size_t)D.nDB * WT_BYTES;
        return a.V.dn + dn_tile_off(D, it.eblk, 0, it.blk);
    };

    // Register budget (GEMM-1, 768 threads): the epilogue warps hold a 64-value share of the accumulator, the producer /
    // MMA / gather warps need few registers.  The pool is the CTA's OWN launch allocation (768 threads x 80 registers = 61440;
    // the SM's remaining registers are not part of it -- an inc beyond it waits forever): 8 x 32 x 48 + 16 x 32 x 96 = 61440.  Every role adjusts its own budget at
    // the top of its branch (that is where ptxas picks it up).  setmaxnreg is WARPGROUP-aligned: all four warps of a warpgroup must
    // execute the same instruction, so one dec dominates every non-epilogue role (warps 0-7 = two whole warpgroups).
#define FXM_REG_DEC() do { if constexpr (MODE == 1) asm volatile("setmaxnreg.dec.sync.aligned.u32 48;" ::: "memory"); } while (0)
#define FXM_REG_INC() do { if constexpr (MODE == 1) asm volatile("setmaxnreg.inc.sync.aligned.u32 96;" ::: "memory"); } while (0)
    if (warp < EPI0) {
    FXM_REG_DEC();
    if (warp == 0) {
        // ===================================================== producer (both CTAs): weight tile + token half per k-block
        const bool leader_lane = elect_one();
        const uint64_t pol_stream = l2_policy_evict_first();     // weight tiles: read once
        int s = 0;
        uint32_t ph = 0;
        const size_t bstride = (size_t)a.P * ROW_BYTES;
        // L2 prefetch cursor over the same weight-tile sequence, PAIR_PF tiles ahead (prefetching the token halves as
        // well was measured and did not help: they are shared by the clusters of an expert and mostly hit L2)
        int pf_wi = wi0, pf_kb = 0, pf_nk = 0;
        const uint8_t* pf_src = nullptr;
        size_t pf_stride = 0;
        auto pf_load_item = [&]() {
            if (pf_wi < W) {
                const PairItem pit = pair_item<MODE>(a, pf_wi, rank, pf_cur);
                pf_src = a_src(pit, pf_stride);
                pf_nk = pit.nk;
            }
        };
        auto pf_step = [&]() {
            if (pf_wi >= W) return;
            if (leader_lane) bulk_prefetch_l2(pf_src + pf_kb * pf_stride, WT_BYTES);
            if (++pf_kb == pf_nk) { pf_kb = 0; pf_wi += wstep; pf_load_item(); }
        };
        pf_load_item();
        for (int i = 0; i < PAIR_PF; ++i) pf_step();
        int tj = 0;
        for (int wi = wi0; wi < W; wi += wstep, ++tj) {
            const PairItem it = pair_item<MODE>(a, wi, rank, cur);
            long long tw = 0;
            size_t astride;
            const uint8_t* asrc = a_src(it, astride);
            const uint32_t h0 = (uint32_t)it.n0 >> 1, h1 = (uint32_t)it.n1 >> 1;      // rows of each sub-tile this CTA holds
            const uint8_t* b0 = a.Bsrc + (size_t)(it.row0 + rank * h0) * ROW_BYTES;
            const uint8_t* b1 = a.Bsrc + (size_t)(it.row0 + it.n0 + rank * h1) * ROW_BYTES;
            const uint32_t tx = WT_BYTES + (h0 + h1) * ROW_BYTES;
            for (int kb = 0; kb < it.nk; ++kb) {
                const long long tw0 = FXM_CLK();
                mbar_wait(empty_bar(s), ph ^ 1u, a.state);
                tw += FXM_CLK() - tw0;
                if (leader_lane) {
                    const uint32_t sb = smem_base + s * stage_bytes;
                    mbar_expect_tx(full_bar(s), tx);
                    bulk_g2s_hint(sb, asrc + kb * astride, WT_BYTES, full_bar(s), pol_stream);
                    if (!gather) {                                     // else: the gather warps bring the same bytes
                        bulk_g2s(sb + WT_BYTES, b0 + kb * bstride, h0 * ROW_BYTES, full_bar(s));
                        if (h1) bulk_g2s(sb + WT_BYTES + h0 * ROW_BYTES, b1 + kb * bstride, h1 * ROW_BYTES, full_bar(s));
                    }
                }
                pf_step();
                if (++s == NS) { s = 0; ph ^= 1u; }
            }
            if (rank == 0 && leader_lane) FXM_TR(MODE, tj, 6, tw);
        }
    } else if (MODE == 1 && gather && warp >= 2 && warp < 2 + PAIR_GW) {
        // ===================================================== gather warps (both CTAs; GEMM-1 with the gather fused)
        // X[pi] (Alg. 2 l.7) without a copy of x in global memory: this CTA's half of the token rows of a
        // k-block comes straight from x, four rows per TMA gather4 (group g = rows 4g..4g+3 of the half, sub-tile 0
        // first).  Warp gw issues groups gw, gw + PAIR_GW, ...; their token indices sit in this warp's slice of gidx.
        const int gw = warp - 2;
        const bool leader_lane = elect_one();
        int4* myidx = gidx + gw * PAIR_GMAX;
        int s = 0;
        uint32_t ph = 0;
        for (int wi = wi0; wi < W; wi += wstep) {
            const PairItem it = pair_item<MODE>(a, wi, rank, cur);
            const int h0 = it.n0 >> 1, h1 = it.n1 >> 1;
            const int ng0 = h0 >> 2, ng = (h0 + h1) >> 2;
            const int cnt = ng > gw ? (ng - gw + PAIR_GW - 1) / PAIR_GW : 0;
            __syncwarp();                                             // the previous item's gather4s have read their indices
            if (lane < cnt) {
                const int g = gw + PAIR_GW * lane;
                const int p = g < ng0 ? it.row0 + (int)rank * h0 + 4 * g : it.row0 + it.n0 + (int)rank * h1 + 4 * (g - ng0);
                myidx[lane] = __ldg((const int4*)(a.tok + p));
            }
            __syncwarp();
            for (int kb = 0; kb < it.nk; ++kb) {
                mbar_wait(empty_bar(s), ph ^ 1u, a.state);
                if (leader_lane) {
                    const uint32_t dst = smem_base + s * stage_bytes + WT_BYTES + (uint32_t)gw * (4u * ROW_BYTES);
                    for (int j = 0; j < cnt; ++j)
                        tma_gather4(dst + (uint32_t)j * (PAIR_GW * 4u * ROW_BYTES), &xmap, kb * KB, myidx[j], full_bar(s));
                    // Every gather warp ARRIVES on the stage's full barrier, also when it had no group to bring (a token tile of
                    // 16-32 rows has fewer 4-row groups than gather warps).  A warp that only polls the empty barriers takes part
                    // in no handshake: the pipeline can lap it, and two phases behind a parity wait can no longer tell "not yet"
                    // from "long ago" -- found as an intermittent time-out at decode-sized T (about one call in 100, always
                    // warps gw >= 2 on an empty barrier).  Skipping the waits instead lets the warp run AHEAD, which aliases
                    // the same way once it has rows to bring again.  With the arrival it can do neither.
                    mbar_arrive(full_bar(s));
                }
                __syncwarp();
                if (++s == NS) { s = 0; ph ^= 1u; }
            }
        }
    } else if (warp == 1 && rank != 0) {
        // ===================================================== relay (peer CTA): "my half of this k-block has landed"
        const bool leader_lane = elect_one();
        int s = 0;
        uint32_t ph = 0;
        for (int wi = wi0; wi < W; wi += wstep) {
            const PairItem it = pair_item<MODE>(a, wi, rank, cur);
            for (int kb = 0; kb < it.nk; ++kb) {
                mbar_wait(full_bar(s), ph, a.state);
                if (leader_lane) mbar_arrive_remote(full_bar(s), 0);
                if (++s == NS) { s = 0; ph ^= 1u; }
            }
        }
    } else if (warp == 1) {
        // ===================================================== MMA issuer (leader CTA): one elected lane issues for the pair
        const bool leader_lane = elect_one();
        TmemRing ring;
        ring.init();
        int s = 0;
        uint32_t ph = 0, drained = 0;
        int tj = 0;
        for (int wi = wi0; wi < W; wi += wstep, ++tj) {
            const PairItem it = pair_item<MODE>(a, wi, rank, cur);
            [[maybe_unused]] const long long t_start = FXM_CLK();
            long long tw = 0;
            uint32_t c0, c1, need;
            const uint32_t q0 = ring.seq;
            ring.alloc_item((uint32_t)it.n0, (uint32_t)it.n1, c0, c1, need);
            for (; drained < need; ++drained) mbar_wait(tempty_bar(drained), (drained / PAIR_TQ) & 1u, a.state);
            tc_fence_after();
            [[maybe_unused]] const long long t_acc = FXM_CLK();
            const uint32_t d0 = tmem_base + c0, d1 = tmem_base + c1;
            const uint32_t id0 = make_idesc2((uint32_t)it.n0), id1 = make_idesc2((uint32_t)(it.n1 ? it.n1 : 16));
            const uint32_t boff1 = WT_BYTES + ((uint32_t)it.n0 >> 1) * ROW_BYTES;
            for (int kb = 0; kb < it.nk; ++kb) {
                const long long tw0 = FXM_CLK();
                mbar_wait(full_bar(s), ph, a.state);                 // both halves of this k-block (own producer + relay)
                tw += FXM_CLK() - tw0;
                tc_fence_after();
                if (leader_lane) {
                    const uint32_t sb = smem_base + s * stage_bytes;
                    const uint64_t adesc = make_desc_sw128(sb);
                    const uint64_t bd0 = make_desc_sw128(sb + WT_BYTES), bd1 = make_desc_sw128(sb + boff1);
#pragma unroll
                    for (int kk = 0; kk < KB / 16; ++kk)
                        umma2_bf16(d0, adesc + 2u * kk, bd0 + 2u * kk, id0, (uint32_t)((kb | kk) != 0));
                    if (it.n1) {
#pragma unroll
                        for (int kk = 0; kk < KB / 16; ++kk)
                            umma2_bf16(d1, adesc + 2u * kk, bd1 + 2u * kk, id1, (uint32_t)((kb | kk) != 0));
                    }
                    umma2_commit_mc(empty_bar(s));                    // frees the stage in BOTH CTAs when these MMAs retire
                }
                __syncwarp();
                if (++s == NS) { s = 0; ph ^= 1u; }
            }
            if (leader_lane) {
                umma2_commit_mc(tfull_bar(q0));
                if (it.n1) umma2_commit_mc(tfull_bar(q0 + 1));
                FXM_TR(MODE, tj, 0, t_start); FXM_TR(MODE, tj, 1, t_acc); FXM_TR(MODE, tj, 2, FXM_CLK()); FXM_TR(MODE, tj, 3, tw);
                FXM_TR(MODE, tj, 7, it.n0 + it.n1); FXM_TR(MODE, tj, 8, it.nk);
            }
            __syncwarp();
        }
    }
    } else {
        FXM_REG_INC();
        // ===================================================== epilogue warps (both CTAs, own TMEM lanes)
        const int q = warp & 3;                                // TMEM lane quadrant this warp may read
        constexpr int NWQ = PAIR_EPI_WARPS / 4;                // warps per lane quadrant
        const int wq = (warp - EPI0) >> 2;                        // which share of the 16-column groups
        const int et = threadIdx.x - 32 * EPI0;
        TmemRing ring;
        ring.init();
        int tj = 0;
        if constexpr (MODE == 1) {
            // Y <- 0 (Alg. 2 l.1): zero the fp32 scatter-add target of GEMM-2.  These warps have nothing
            // to do until the first tile has been multiplied; the stores drain while the tensor pipe works.
            if (a.yacc) {
                uint4* z = (uint4*)a.yacc;
                const size_t n4 = (size_t)a.T * D.d / 4;
                const size_t nthr = (size_t)gridDim.x * (32 * PAIR_EPI_WARPS);
                for (size_t i = (size_t)blockIdx.x * (32 * PAIR_EPI_WARPS) + et; i < n4; i += nthr) z[i] = make_uint4(0, 0, 0, 0);
            }
            // A warp owns up to four 16-token groups of a sub-tile (its lane quadrant = 16 gate + 16 up channels): it pulls
            // them into 64 registers and hands the TMEM columns back to the MMA warp AT ONCE -- the next tile's MMAs run
            // while SwiGLU is computed from registers.  The bf16 results go to a 32 KB staging buffer in the FINAL global
            // layout (swizzled H panel rows of this CTA's channel block), one bulk store per sub-tile.
            const uint64_t pol_keep = l2_policy_evict_last();         // H panels: read back by GEMM-2
            const int chn = q * 16 + (lane & 15);
            const int odd = lane >> 4;
            uint32_t soff[8];                                         // staging offset of token row 2m + odd (rows repeat every 8)
#pragma unroll
            for (int m = 0; m < 8; ++m) soff[m] = sw128_off((uint32_t)(2 * m + odd), (uint32_t)chn);
            bool store_pending = false;
            for (int wi = wi0; wi < W; wi += wstep, ++tj) {
                const PairItem it = pair_item<MODE>(a, wi, rank, cur);
                const int nsub = it.n1 ? 2 : 1;
                uint32_t cc0, cc1, need_unused;
                const uint32_t sq0 = ring.seq;
                ring.alloc_item((uint32_t)it.n0, (uint32_t)it.n1, cc0, cc1, need_unused);
                const bool keep = it.blk * CB + chn < it.r;           // tail mask of the last retained block (pad-zero rule)
                for (int sidx = 0; sidx < nsub; ++sidx) {
                    const int n = sidx ? it.n1 : it.n0;
                    const uint32_t col0 = sidx ? cc1 : cc0;
                    const uint32_t sq = sq0 + sidx;
                    const int rowS = it.row0 + (sidx ? it.n0 : 0);
                    const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + col0;
                    const int ngrp = n >> 4;                           // <= 16 groups in a sub-tile of <= 256 tokens
                    const int gbeg = ngrp * wq / NWQ, gend = ngrp * (wq + 1) / NWQ;     // <= 4 of them are this warp's
                    mbar_wait(tfull_bar(sq), (sq / PAIR_TQ) & 1u, a.state);
                    if (et == 0 && rank == 0 && sidx == 0) FXM_TR(MODE, tj, 4, FXM_CLK());
                    tc_fence_after();
                    uint32_t v[4][16];
                    if (it.valid) {
#pragma unroll
                        for (int u = 0; u < 4; ++u)
                            if (gbeg + u < gend) tmem_ld16(taddr + (uint32_t)(gbeg + u) * 16u, v[u]);
                        tmem_ld_wait();
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) {                                   // this warp no longer needs the columns
                        if (rank == 0) mbar_arrive(tempty_bar(sq)); else mbar_arrive_remote(tempty_bar(sq), 0);
                    }
                    if (store_pending) {                               // the previous sub-tile's bulk store has read the staging buffer
                        if (et == 0) bulk_wait_read0();
                        epi_bar_sync_all();
                        store_pending = false;
                    }
                    if (it.valid) {
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            if (gbeg + u < gend) {
                                uint8_t* sg = stg_gen + (uint32_t)(gbeg + u) * (16u * ROW_BYTES);
#pragma unroll
                                for (int m = 0; m < 8; ++m) {
                                    const float mine0 = __uint_as_float(v[u][2 * m]), mine1 = __uint_as_float(v[u][2 * m + 1]);
                                    const float send = odd ? mine0 : mine1;                    // what the twin lane needs
                                    const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
                                    const float g = odd ? recv : mine0;                        // gate lives in lanes 0-15
                                    const float up = odd ? mine1 : recv;                       // up lives in lanes 16-31
                                    float hv = __fdividef(g, 1.f + __expf(-g)) * up;
                                    if (!keep) hv = 0.f;
                                    *(__nv_bfloat16*)(sg + soff[m]) = __float2bfloat16_rn(hv);
                                }
                            }
                        }
                    }
                    fence_proxy_async_smem();                          // staging writes -> visible to the bulk-copy engine
                    epi_bar_sync_all();
                    if (et == 0 && it.valid) {
                        bulk_s2g_hint(a.H + ((size_t)it.blk * a.P + rowS) * ROW_BYTES, stg_base, (uint32_t)n * ROW_BYTES, pol_keep);
                        bulk_commit();
                    }
                    store_pending = it.valid;                          // warp-uniform across the CTA
                    if (et == 0 && rank == 0 && sidx == nsub - 1) FXM_TR(MODE, tj, 5, FXM_CLK());
                }
            }
            if (et == 0) bulk_wait0();
        } else {
            // GEMM-2: "Z <- Z (.) alpha;  Y <- ScatterAdd(Y, pi, Z)" (Alg. 2 l.19-20) straight from the
            // accumulator.  A warp owns up to four 16-column groups of a sub-tile (its lane quadrant = 32 output features):
            // it loads them into 64 registers, tells the MMA warp that it is done with the columns, and only then scales and
            // adds: lane = feature, so each red.global.add.f32 of the warp is one 128-byte line of yacc[token].
            int2* rinfo = (int2*)stg_gen;                              // [2][512] {token or -1, router weight bits}
            const int feat0 = q * 32 + lane;
            for (int wi = wi0; wi < W; wi += wstep, ++tj) {
                const PairItem it = pair_item<MODE>(a, wi, rank, cur);
                const int nsub = it.n1 ? 2 : 1;
                int2* ri = rinfo + (tj & 1) * 512;
                if (et < it.n0 + it.n1) ri[et] = __ldg(a.row_tw + it.row0 + et);
                epi_bar_sync_all();                                    // row info of this item is in place (and the buffer of item tj-2 is free)
                uint32_t cc0, cc1, need_unused;
                const uint32_t sq0 = ring.seq;
                ring.alloc_item((uint32_t)it.n0, (uint32_t)it.n1, cc0, cc1, need_unused);
                const int feat = it.blk * WT_ROWS + feat0;
                const bool fok = it.valid && feat < D.d;               // padded rows of the last feature block (d % 128 == 64)
                float* ycol = a.yacc + feat;
                for (int sidx = 0; sidx < nsub; ++sidx) {
                    const int n = sidx ? it.n1 : it.n0;
                    const uint32_t col0 = sidx ? cc1 : cc0;
                    const uint32_t sq = sq0 + sidx;
                    const int2* rr = ri + (sidx ? it.n0 : 0);
                    const uint32_t taddr = tmem_base + ((uint32_t)(q * 32) << 16) + col0;
                    const int ngrp = n >> 4;                               // <= 16 groups in a sub-tile of <= 256 tokens
                    const int gbeg = ngrp * wq / NWQ, gend = ngrp * (wq + 1) / NWQ;     // <= 4 of them are this warp's
                    mbar_wait(tfull_bar(sq), (sq / PAIR_TQ) & 1u, a.state);
                    if (et == 0 && rank == 0 && sidx == 0) FXM_TR(MODE, tj, 4, FXM_CLK());
                    tc_fence_after();
                    uint32_t v[4][16];
                    if (it.valid) {
#pragma unroll
                        for (int u = 0; u < 4; ++u)
                            if (gbeg + u < gend) tmem_ld16(taddr + (uint32_t)(gbeg + u) * 16u, v[u]);
                        tmem_ld_wait();
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) {                                   // this warp no longer needs the columns
                        if (rank == 0) mbar_arrive(tempty_bar(sq)); else mbar_arrive_remote(tempty_bar(sq), 0);
                    }
                    if (fok) {
#pragma unroll
                        for (int u = 0; u < 4; ++u) {
                            if (gbeg + u < gend) {
                                const int2* r16 = rr + (gbeg + u) * 16;
#pragma unroll
                                for (int jj = 0; jj < 16; ++jj) {
                                    const int2 tw = r16[jj];           // same address in every lane: a broadcast
                                    if (tw.x >= 0)
                                        asm volatile("red.relaxed.gpu.global.add.f32 [%0], %1;" ::"l"(ycol + (size_t)tw.x * D.d),
                                                     "f"(__int_as_float(tw.y) * __uint_as_float(v[u][jj])) : "memory");
                                }
                            }
                        }
                    }
                    if (et == 0 && rank == 0 && sidx == nsub - 1) FXM_TR(MODE, tj, 5, FXM_CLK());
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
static cudaError_t launch_pair_t(const PairArgs& a, const CUtensorMap& xmap, int num_sms, cudaStream_t st) {
    return launch_pdl(k_gemm_pair<MODE>, dim3(num_sms / 2 * 2), dim3(PairCfg<MODE>::THREADS), PAIR_SMEM, st, a, xmap);
}

// x [T][d] bf16 as a 2-D tensor {d, T} with box {64 columns, 1 row} and 128-byte swizzle: the shape tile::gather4 wants
cudaError_t encode_x_map(const void* x, int T, int d, void* map_out) {
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult qres;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &qres);
        if (e != cudaSuccess) return e;
        if (qres != cudaDriverEntryPointSuccess || !p) return cudaErrorNotSupported;
        fn = (EncodeFn)p;
    }
    const cuuint64_t gdim[2] = {(cuuint64_t)d, (cuuint64_t)T};
    const cuuint64_t gstride[1] = {(cuuint64_t)d * 2};
    const cuuint32_t box[2] = {(cuuint32_t)KB, 1};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = fn((CUtensorMap*)map_out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(x), gdim, gstride, box,
                          estr, CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                          CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t init_pair_kernels() {
    cudaError_t e = cudaFuncSetAttribute(k_gemm_pair<1>, cudaFuncAttributeMaxDynamicSharedMemorySize, PAIR_SMEM);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_gemm_pair<2>, cudaFuncAttributeMaxDynamicSharedMemorySize, PAIR_SMEM);
}

cudaError_t launch_gemm1_pair(const Dims& D, const LayerView& V, const int* r_table, const Workspace& ws, int T,
                              DevState* state, int num_sms, const void* x_map, cudaStream_t st) {
    PairArgs a{};
    a.D = D; a.V = V; a.r_table = r_table; a.items = ws.tt; a.sched = ws.sched; a.tok = ws.row_tok;
    a.H = ws.H; a.yacc = ws.yacc; a.T = T; a.state = state; a.P = ws.P;
    return launch_pair_t<1>(a, *(const CUtensorMap*)x_map, num_sms, st);
}

cudaError_t launch_gemm2_pair(const Dims& D, const LayerView& V, const int* r_table, const Workspace& ws,
                              DevState* state, int num_sms, cudaStream_t st) {
    PairArgs a{};
    a.D = D; a.V = V; a.r_table = r_table; a.items = ws.tt; a.sched = ws.sched; a.Bsrc = ws.H;
    a.row_tw = ws.row_tw; a.yacc = ws.yacc; a.state = state; a.P = ws.P;
    return launch_pair_t<2>(a, CUtensorMap{}, num_sms, st);
}

}  // namespace fxm

#ifdef FXM_TRACE
extern "C" int fxm_trace_read(void* dst) { return (int)cudaMemcpyFromSymbol(dst, fxm::g_trace, sizeof(fxm::g_trace)); }
#endif
