// fxm_decode.cu -- step a6: the decode-shaped routed-expert FFN (a2..a5 of SURVEY.md 8(a)) as ONE launch.
//
//   y[t] = sum_j topk_w[t][j] * W~down_e[:, :r_e] ( silu(W~gate_e[:r_e] x[t]) (.) W~up_e[:r_e] x[t] ),  e = topk_ids[t][j]
//   (Eq. 4; Alg. 2.)  With a handful of tokens per expert the call is a stream of
//   the retained weight prefix of every ACTIVE expert, read exactly once: HBM-bound.
//
// One SM pulls only ~40 GB/s through its bulk-copy ring, so the HBM roofline needs ALL 148 SMs streaming the same
// number of bytes -- also when the call has fewer 64-channel work items than SMs (T = 1 at 75 % pruned: 80 items).  The
// kernel therefore cuts the weight stream at TILE granularity, in two phases separated by a grid barrier:
//   phase 1  gate/up.  The tiles of all items (item = run (expert e, <= 16 tokens) x retained channel block cb), in the
//            order (item, k-block), form one list of W * d/64 tiles; CTA c owns the contiguous range [c T1/G, (c+1) T1/G).
//            A range is a few PIECES (parts of one item): D1[128 packed rows, 16 tokens] += Wgu_tile . Xe^T over the
//            piece's k-blocks, then the fp32 partial goes to scratch slot (item + c) -- unique per (item, CTA).
//   phase 2  down.  Tiles in the order (item, feature block): W * ceil(d/128) tiles, again one contiguous range per CTA.
//            For every piece (item, feature blocks db0..db1) the epilogue warps sum the item's partials (the slots of the
//            CTAs that touched it), apply SwiGLU (gate lane l, up lane l+16: one shuffle) and the pad-zero rule for
//            channels >= r_e, round once to bf16 -> Hs; Y[db] += Wd_tile(e, cb, db) . Hs^T accumulates in
//            TMEM over the consecutive pieces of a run; at the end of the run segment the touched feature blocks are
//            scaled by the router weight (Alg. 2 l.19) and added to yacc[t][:] with fp32 reductions (l.20 ScatterAdd).
//   Both phases are balanced to +-1 tile whatever the routing and the budget.  With no more runs than CTAs (a handful of
//   tokens) the CTAs are first dealt out to the runs, so that no range crosses a run boundary (struct Split).
// Roles (320 threads): warp 0 weight producer (16 KB cp.async.bulk per tile through a shared-memory ring; it starts
// fetching phase-2 tiles while the grid barrier is still closing), warp 1 MMA issuer, warps 2-5 epilogue, warps 6-9
// stage the <= 16 token rows x[t] of a run into swizzled K-major panels Xe (X[pi], Alg. 2 l.7).
// Synchronisation between CTAs (all resident: grid = #SMs, one CTA per SM; nothing a CTA waits for depends on a later
// kernel, so none of this can deadlock):
//   * phase 1 -> phase 2 is NOT a grid barrier: a phase-2 piece waits for the per-item counter of ITS item (the two or
//     three CTAs that hold phase-1 pieces of it each add 1 after their partial is in global memory);
//   * "yacc is zeroed" is a split barrier: every CTA arrives in its prologue and checks before its first reduction;
//   * one grid barrier before yacc -> y (one rounding to bf16), a single ever-growing counter (see cnt_arrive).
// The launch is an ordinary one with the programmatic-dependent-launch attribute.
// TMEM columns: [0,32) two phase-1 accumulators, [32, 32 + 16 nDB) the Y partial.  Needs nDB <= 30 (d <= 3840).
#include "fxm_ptx.cuh"

namespace fxm {

constexpr int DEC_THREADS = 320;
constexpr int DEC_N = 16;                         // tokens per run = UMMA N
constexpr int DEC_XE_KB_BYTES = DEC_N * ROW_BYTES;   // 2 KB of Xe per k-block
constexpr int DEC_MAX_SLOTS = 12;
constexpr int DEC_SMEM_MAX = 232448;              // 227 KB
constexpr int DEC_PART = WT_ROWS * DEC_N;         // floats of one phase-1 partial: 128 packed rows x 16 tokens (8 KB)
constexpr int DEC_ALIGN_MIN_CTAS = 12;            // the run-aligned split is used when every run gets at least this many CTAs
constexpr int DEC_MAX_CTAS = 160;                 // the partial-slot capacity is sized for at most this many CTAs

struct DecArgs {
    Dims D;
    LayerView V;
    const int* r_table;
    const uint4* x;            // [T][d] bf16
    const int* ids;            // [T][k]
    const float* topk_w;       // [T][k]
    float* yacc;               // [T][d] fp32 scratch (workspace)
    float* part;               // phase-1 partials: [(items + #CTAs)][128][16] fp32 (workspace)
    const uint2* y_add;        // [T][d] bf16 or null: shared-expert output added in fp32 before the rounding of y
    __nv_bfloat16* y;          // [T][d]
    DevState* state;
    uint32_t* icnt;            // [items] phase-1 pieces written per item (blob tail; zero on entry, zeroed again on exit)
    int T, k, A;
    int slots;                 // ring depth
    int pf;                    // L2 prefetch distance in 16 KB tiles (0 = none)
};

// persistent auxiliary shared memory (after ring, Xe, Hs)
struct DecAux {
    int run_en[DEC_MAX_RUNS];      // expert | tokens << 16
    int run_pos[DEC_MAX_RUNS];     // first sorted position of the run
    int run_ib[DEC_MAX_RUNS + 1];  // first item of the run; [n_runs] = W
    int16_t perm[DEC_MAX_A];       // sorted position -> flat assignment index
    float wts[DEC_MAX_A];          // topk_w by flat assignment index (read once in the prologue)
    int r[MAX_E];
    uint32_t eb[MAX_E];            // first channel block of each expert in the weight regions (LayerView::eblk)
    uint64_t bars[2 * DEC_MAX_SLOTS + 16];
    uint32_t tmem_slot;
    int n_runs, W;
    int aligned;                   // 1: the CTAs are dealt out to the runs first (crun), no CTA's range crosses a run boundary
    int16_t crun[DEC_MAX_CTAS + 2];    // aligned: first CTA of run r (r <= n_runs <= G); crun[n_runs] = G
    unsigned long long ztarget;    // value of DevState::dec_zcnt at which every CTA of THIS launch has zeroed its slice of yacc
};
// prologue-only scratch, aliased on the weight ring (>= 4 slots = 64 KB)
struct DecTmp {
    int16_t ids[DEC_MAX_A];
    int cnt[MAX_E], off[MAX_E + 1], ibase[MAX_E + 1], gbase[MAX_E + 1];
    int wh[DEC_THREADS / 32][MAX_E];   // per-warp expert histogram, then the warp's running base
};

__host__ __device__ inline int dec_fixed_smem(const Dims& D) {
    return 1024 + D.nKB1 * DEC_XE_KB_BYTES + 2 * DEC_XE_KB_BYTES + (int)((sizeof(DecAux) + 1023) / 1024 * 1024);
}

// one lane of a converged warp.  The asynchronous instructions (bulk copies, tcgen05.mma / commit) take their operands
// from uniform registers: they are issued by ONE elected lane inside loops that all 32 lanes walk, so the compiler keeps
// addresses and descriptors uniform (a `lane == 0` branch costs a register->uniform waterfall per instruction).
__device__ __forceinline__ bool dec_elect_one() {
    uint32_t p;
    asm volatile(
        "{\n\t.reg .pred q;\n\t"
        "elect.sync _|q, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, q;\n\t}"
        : "=r"(p));
    return p != 0;
}
__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ unsigned long long ld_acquire_u64(const unsigned long long* p) {
    unsigned long long v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
// Grid-wide synchronisation without a reset and without a chain of dependent round trips (all CTAs are resident, see the
// header).  A counter only grows; every launch on a layer has the same grid size G and adds exactly G, so the value a
// CTA's own arrival returns names the target of ITS launch, (old / G + 1) * G.  The arrival is a release (it publishes
// what the CTA wrote before the preceding block-level barrier), the poll is an acquire.  After the last arrival a
// poller needs one L2 round trip -- the two-level counter + generation word this replaces needed four.
__device__ __forceinline__ unsigned long long cnt_arrive(unsigned long long* c) {
    unsigned long long old;
    asm volatile("atom.acq_rel.gpu.global.add.u64 %0, [%1], 1;" : "=l"(old) : "l"(c) : "memory");
    return old;
}
__device__ __forceinline__ unsigned long long cnt_target(unsigned long long old, uint32_t G) { return (old / G + 1ull) * G; }
__device__ __forceinline__ void wait_timeout(DevState* st) {
    atomicOr(&st->flags, 2u);
    if (st->hflag) *(volatile uint32_t*)st->hflag = 2u;
    __threadfence_system();
    __trap();
}
__device__ __forceinline__ void cnt_wait(const unsigned long long* c, unsigned long long target, DevState* st) {
    if (ld_acquire_u64(c) >= target) return;
    const long long t0 = clock64();
    uint32_t spins = 0;
    while (ld_acquire_u64(c) < target) {
        __nanosleep(64);
        if ((++spins & 0x3FFu) == 0 && clock64() - t0 > 4000000000LL) wait_timeout(st);
    }
}
// item readiness: the phase-1 pieces of an item are written by a few CTAs; each adds 1 (release) after its partial is in
// global memory, the phase-2 reader polls (acquire) until all of them have
__device__ __forceinline__ void item_signal(uint32_t* c) {
    asm volatile("red.release.gpu.global.add.u32 [%0], 1;" ::"l"(c) : "memory");
}
__device__ __forceinline__ void item_wait(const uint32_t* c, uint32_t need, DevState* st) {
    if (ld_acquire_u32(c) >= need) return;
    const long long t0 = clock64();
    uint32_t spins = 0;
    while (ld_acquire_u32(c) < need) {
        __nanosleep(32);
        if ((++spins & 0x3FFu) == 0 && clock64() - t0 > 4000000000LL) wait_timeout(st);
    }
}
__device__ __forceinline__ void red_add_f32(float* p, float v) {
    asm volatile("red.relaxed.gpu.global.add.f32 [%0], %1;" ::"l"(p), "f"(v) : "memory");
}

__device__ __forceinline__ void tmem_ld2(uint32_t taddr, uint32_t& v0, uint32_t& v1) {
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x2.b32 {%0, %1}, [%2];" : "=r"(v0), "=r"(v1) : "r"(taddr) : "memory");
}

// ---- the two tile lists.  Phase p has tiles_per_item = nKB1 (p = 1) or nDB (p = 2); tile t belongs to item t / tpi.
// A PIECE is the part of one item inside a CTA's range: item, local tile range [a, b).
struct Piece { int item, a, b; };
struct PieceIter {
    long long t, hi;
    int tpi;
    __device__ __forceinline__ void init(long long lo_, long long hi_, int tpi_) { t = lo_; hi = hi_; tpi = tpi_; }
    __device__ __forceinline__ bool next(Piece& p) {
        if (t >= hi) return false;
        p.item = (int)(t / tpi);
        p.a = (int)(t - (long long)p.item * tpi);
        const long long room = hi - t;
        p.b = room < (long long)(tpi - p.a) ? p.a + (int)room : tpi;
        t += p.b - p.a;
        return true;
    }
};
// run cursor: items ascend, so the run of an item is found by walking forward
__device__ __forceinline__ int run_of(const DecAux* ax, int item, int& cur) {
    while (ax->run_ib[cur + 1] <= item) ++cur;
    return cur;
}
// CTA that owns tile t of a list of Tn tiles split over G CTAs as [c Tn / G, (c + 1) Tn / G)
__device__ __forceinline__ int cta_of_tile(long long t, long long Tn, int G) { return (int)(((t + 1) * G - 1) / Tn); }

// How the tile list of a phase (tpi tiles per item) is cut into one contiguous range per CTA.
//   flat:    CTA c owns [c Tn / G, (c + 1) Tn / G) of the whole list (balanced to +-1 tile; ranges cross run boundaries).
//   aligned: when the call has no more runs than CTAs (a handful of tokens), the CTAs are dealt out to the runs in
//            proportion to their items (run r gets the CTAs [crun[r], crun[r+1])) and each run's tiles are cut evenly
//            among ITS CTAs.  No range crosses a run boundary, so no CTA restages x in phase 1 or drains and refills its
//            Y partial in phase 2 -- measured at C4 T=1: the four CTAs with a run boundary finished phase 2 ~3 us after
//            the rest and the whole grid waited for them.  Costs an imbalance of one part in (CTAs per run), so it is used
//            only when every run gets >= DEC_ALIGN_MIN_CTAS CTAs (with 2-3 CTAs per run -- T=64 and a heterogeneous table --
//            it cost 35 %).
struct Split {
    // 32-bit arithmetic: tiles of a phase <= 320 runs * 256 blocks * 60 tiles = 4.9 M, times G <= 160 stays below 2^32
    const DecAux* ax;
    uint32_t W;
    int G, aligned;
    __device__ __forceinline__ void range(int c, int tpi, long long& lo, long long& hi) const {
        if (!aligned) { const uint32_t Tn = W * (uint32_t)tpi; lo = Tn * (uint32_t)c / (uint32_t)G; hi = Tn * (uint32_t)(c + 1) / (uint32_t)G; return; }
        int r = 0;
        while ((int)ax->crun[r + 1] <= c) ++r;
        const uint32_t c0 = ax->crun[r], nc = ax->crun[r + 1] - c0;
        const uint32_t tb = (uint32_t)ax->run_ib[r] * tpi, n = (uint32_t)(ax->run_ib[r + 1] - ax->run_ib[r]) * tpi;
        lo = tb + n * ((uint32_t)c - c0) / nc;
        hi = tb + n * ((uint32_t)c - c0 + 1) / nc;
    }
    // owner of tile t, which belongs to run `run`
    __device__ __forceinline__ int owner(long long t, int run, int tpi) const {
        if (!aligned) return (int)((((uint32_t)t + 1u) * (uint32_t)G - 1u) / (W * (uint32_t)tpi));
        const uint32_t c0 = ax->crun[run], nc = ax->crun[run + 1] - c0;
        const uint32_t tb = (uint32_t)ax->run_ib[run] * tpi, n = (uint32_t)(ax->run_ib[run + 1] - ax->run_ib[run]) * tpi;
        return (int)(c0 + (((uint32_t)t - tb + 1u) * nc - 1u) / n);
    }
    // does CTA c (a CTA of run `run` when aligned) own any tile of the phase?
    __device__ __forceinline__ bool holds(int c, int run, int tpi) const {
        if (!aligned) { const uint32_t Tn = W * (uint32_t)tpi; return Tn * (uint32_t)c / (uint32_t)G != Tn * (uint32_t)(c + 1) / (uint32_t)G; }
        const uint32_t c0 = ax->crun[run], nc = ax->crun[run + 1] - c0;
        const uint32_t n = (uint32_t)(ax->run_ib[run + 1] - ax->run_ib[run]) * tpi;
        return n * ((uint32_t)c - c0) / nc != n * ((uint32_t)c - c0 + 1) / nc;
    }
};

#ifdef FXM_TRACE
__device__ unsigned long long g_dtrace[148][16];
__device__ __forceinline__ unsigned long long dec_now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define DEC_TR(f) do { if (threadIdx.x == 0 && blockIdx.x < 148) g_dtrace[blockIdx.x][f] = dec_now(); } while (0)
#define DEC_TRE(f) do { if (threadIdx.x == 64 && blockIdx.x < 148) g_dtrace[blockIdx.x][f] = dec_now(); } while (0)
#define DEC_TRM(f) do { if (threadIdx.x == 32 && blockIdx.x < 148) g_dtrace[blockIdx.x][f] = dec_now(); } while (0)
#else
#define DEC_TRM(f) do { } while (0)
#define DEC_TR(f) do { } while (0)
#define DEC_TRE(f) do { } while (0)
#endif

__global__ void __launch_bounds__(DEC_THREADS, 1) k_decode(const DecArgs a) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const Dims& D = a.D;
    const uint32_t smem_base = (smem_u32(smem_raw) + 1023u) & ~1023u;
    uint8_t* smem_gen = smem_raw + (smem_base - smem_u32(smem_raw));
    const int NS = a.slots;
    const uint32_t ring_s = smem_base;
    const uint32_t xe_off = (uint32_t)NS * WT_BYTES;
    const uint32_t hs_off = xe_off + (uint32_t)D.nKB1 * DEC_XE_KB_BYTES;
    const uint32_t aux_off = hs_off + 2u * DEC_XE_KB_BYTES;
    uint8_t* xe_gen = smem_gen + xe_off;
    uint8_t* hs_gen = smem_gen + hs_off;
    DecAux* ax = (DecAux*)(smem_gen + aux_off);
    DecTmp* tp = (DecTmp*)smem_gen;                       // prologue-only: the ring is idle until the roles start
    const uint32_t bar_base = smem_base + aux_off + (uint32_t)offsetof(DecAux, bars);
    auto full_bar = [&](int s) { return bar_base + 8u * s; };
    auto empty_bar = [&](int s) { return bar_base + 8u * (DEC_MAX_SLOTS + s); };
    const uint32_t bx = bar_base + 8u * (2 * DEC_MAX_SLOTS);
    const uint32_t xfull = bx, xempty = bx + 8, yfull = bx + 16, yempty = bx + 24;
    auto a1full = [&](int b) { return bx + 32u + 8u * b; };
    auto a1empty = [&](int b) { return bx + 48u + 8u * b; };
    auto hfull = [&](int b) { return bx + 64u + 8u * b; };
    auto hempty = [&](int b) { return bx + 80u + 8u * b; };

    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int E = D.E, A = a.A, k = a.k;
    DEC_TR(0);
    const uint32_t G = gridDim.x;
    pdl_launch_dependents();

    // ------------------------------------------------------------------------------------------ prologue
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        mbar_init(xfull, 128); mbar_init(xempty, 1); mbar_init(yfull, 1); mbar_init(yempty, 128);
        for (int b = 0; b < 2; ++b) {
            mbar_init(a1full(b), 1); mbar_init(a1empty(b), 128); mbar_init(hfull(b), 128); mbar_init(hempty(b), 1);
        }
        fence_barrier_init();
    }
    if (warp == 1) tmem_alloc(smem_u32(&ax->tmem_slot), 512);
    pdl_wait();                                              // the previous kernel may still use the workspace / write x, ids
    // Every global load of the prologue is issued at once (ids, router weights, the width table, the block index: one
    // DRAM round trip when the lines are cold), the zeroing below runs while they are in flight, then they are consumed.
    constexpr int PER = (DEC_MAX_A + DEC_THREADS - 1) / DEC_THREADS;
    static_assert(MAX_E <= DEC_THREADS, "one width per thread");
    int idv[PER];
    float wv[PER];
#pragma unroll
    for (int u = 0; u < PER; ++u) {
        const int f = tid + u * DEC_THREADS;
        idv[u] = f < A ? __ldg(a.ids + f) : 0;
        wv[u] = f < A ? __ldg(a.topk_w + f) : 0.f;
    }
    const int rv = tid < E ? __ldg(a.r_table + tid) : 0;
    const uint32_t ebv = tid < E ? __ldg(a.V.eblk + tid) : 0u;
    // a handful of tokens: pull x into L2 now, the stagers ask for their rows only after the grouping
    if (tid == 0 && (size_t)a.T * D.d * 2 <= 65536) bulk_prefetch_l2(a.x, (uint32_t)((size_t)a.T * D.d * 2));
    // zero this CTA's slice of the fp32 accumulator; the arrival below (after the next block barrier) publishes it, and every
    // CTA checks that ALL slices are published before its first reduction (a split barrier: arrive here, wait ~20 us later)
    {
        float4* z = (float4*)a.yacc;
        const size_t n4 = (size_t)a.T * D.d / 4;
        for (size_t i = (size_t)blockIdx.x * DEC_THREADS + tid; i < n4; i += (size_t)G * DEC_THREADS)
            z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    // counts (Alg. 2 l.4-6, stable counting sort as in fxm_route.cu): warp w owns the contiguous chunk [w*chunk, (w+1)*chunk)
    // of the flat assignments; per 32-wide step the lowest lane of every group of equal ids adds the group size to
    // the warp's histogram row
    constexpr int NW = DEC_THREADS / 32;
    const int chunk = ((A + NW - 1) / NW + 31) & ~31;
    const int wlo = min(A, warp * chunk), whi = min(A, wlo + chunk);
    for (int i = tid; i < NW * MAX_E; i += DEC_THREADS) (&tp->wh[0][0])[i] = 0;
    // Xe / Hs start as zeros (rows beyond a run's token count are never staged)
    for (int i = tid; i < (int)((aux_off - xe_off) / 16); i += DEC_THREADS) ((uint4*)xe_gen)[i] = make_uint4(0, 0, 0, 0);
    {
        bool bad = false;
#pragma unroll
        for (int u = 0; u < PER; ++u) {
            const int f = tid + u * DEC_THREADS;
            if (f < A) {
                int id = idv[u];
                if (id < 0 || id >= E) { bad = true; id = -1; }
                tp->ids[f] = (int16_t)id;
                ax->wts[f] = wv[u];
            }
        }
        if (bad) atomicOr(&a.state->flags, 1u);
        if (tid < MAX_E) { ax->r[tid] = rv; ax->eb[tid] = ebv; }
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = ax->tmem_slot;
    unsigned long long zold = 0;
    if (tid == DEC_THREADS - 1) zold = cnt_arrive(&a.state->dec_zcnt);     // the result is not needed before the end of the prologue
    for (int base = wlo; base < whi; base += 32) {
        const int f = base + lane;
        const int id = f < whi ? (int)tp->ids[f] : -1;
        const unsigned m = __match_any_sync(0xffffffffu, id);
        if (id >= 0 && lane == __ffs(m) - 1) tp->wh[warp][id] += __popc(m);
        __syncwarp();
    }
    __syncthreads();
    if (tid < E) {                                                  // exclusive scan over the warps, per expert
        int run = 0;
#pragma unroll
        for (int w = 0; w < NW; ++w) {
            const int c = tp->wh[w][tid];
            tp->wh[w][tid] = run;
            run += c;
        }
        tp->cnt[tid] = run;
    }
    __syncthreads();
    // warp 0: exclusive scans over experts: sorted offsets, item base, run base
    if (warp == 0) {
        int c_off = 0, c_items = 0, c_runs = 0;
        for (int base = 0; base < E; base += 32) {
            const int e = base + lane;
            const int n = e < E ? tp->cnt[e] : 0;
            const int r = e < E ? ax->r[e] : 0;
            const int ng = (n > 0 && r > 0) ? (n + DEC_N - 1) / DEC_N : 0;     // idle / width-0 experts: no work
            const int ni = ng * ((r + CB - 1) / CB);
            int s_n = n, s_i = ni, s_g = ng;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int t1 = __shfl_up_sync(0xffffffffu, s_n, o), t2 = __shfl_up_sync(0xffffffffu, s_i, o);
                const int t3 = __shfl_up_sync(0xffffffffu, s_g, o);
                if (lane >= o) { s_n += t1; s_i += t2; s_g += t3; }
            }
            if (e < E) {
                tp->off[e] = c_off + s_n - n;
                tp->ibase[e] = c_items + s_i - ni;
                tp->gbase[e] = c_runs + s_g - ng;
            }
            c_off += __shfl_sync(0xffffffffu, s_n, 31);
            c_items += __shfl_sync(0xffffffffu, s_i, 31);
            c_runs += __shfl_sync(0xffffffffu, s_g, 31);
        }
        if (lane == 0) {
            tp->off[E] = c_off; tp->ibase[E] = c_items; tp->gbase[E] = c_runs;
            ax->W = c_items;
            ax->n_runs = c_runs;
            ax->run_ib[c_runs] = c_items;
        }
    }
    __syncthreads();
    // stable positions (ascending flat index inside an expert, reading R5): expert offset + earlier warps + earlier
    // steps of this warp + lower lanes of this step
    for (int base = wlo; base < whi; base += 32) {
        const int f = base + lane;
        const int id = f < whi ? (int)tp->ids[f] : -1;
        const unsigned m = __match_any_sync(0xffffffffu, id);
        if (id >= 0) ax->perm[tp->off[id] + tp->wh[warp][id] + __popc(m & ((1u << lane) - 1u))] = (int16_t)f;
        __syncwarp();
        if (id >= 0 && lane == __ffs(m) - 1) tp->wh[warp][id] += __popc(m);
        __syncwarp();
    }
    // the run table of the WHOLE call: run (e, g) = tokens [16 g, 16 g + 16) of expert e's segment, items = its retained blocks
    if (tid < E) {
        const int n = tp->cnt[tid], r = ax->r[tid];
        const int nb = (r + CB - 1) / CB;
        const int ng = tp->gbase[tid + 1] - tp->gbase[tid];
        for (int g = 0; g < ng; ++g) {
            const int slot = tp->gbase[tid] + g;
            ax->run_en[slot] = tid | (min(DEC_N, n - g * DEC_N) << 16);
            ax->run_pos[slot] = tp->off[tid] + g * DEC_N;
            ax->run_ib[slot] = tp->ibase[tid] + g * nb;
        }
    }
    if (tid == DEC_THREADS - 1) ax->ztarget = cnt_target(zold, G);
    fence_proxy_async_smem();                                // the zeros of Xe / Hs -> visible to the tensor core's reads
    __syncthreads();
    const int W = ax->W;
    // deal the CTAs out to the runs (see Split) when every run gets enough of them
    if (warp == 0) {
        const int nr = ax->n_runs;
        bool ok = nr >= 1 && nr <= (int)G && W > 0;
        if (ok) {
            for (int r = lane; r <= nr; r += 32) ax->crun[r] = (int16_t)((uint32_t)G * (uint32_t)ax->run_ib[r] / (uint32_t)W);
            __syncwarp();
            for (int r = lane; r < nr; r += 32) ok = ok && ax->crun[r + 1] - ax->crun[r] >= DEC_ALIGN_MIN_CTAS;
        }
        ok = __all_sync(0xffffffffu, ok);
        if (lane == 0) ax->aligned = ok ? 1 : 0;
    }
    __syncthreads();
    Split sp;
    sp.ax = ax; sp.W = (uint32_t)W; sp.G = (int)G; sp.aligned = ax->aligned;
    long long lo1, hi1, lo2, hi2;
    sp.range((int)blockIdx.x, D.nKB1, lo1, hi1);
    sp.range((int)blockIdx.x, D.nDB, lo2, hi2);
    DEC_TR(1);

    if (warp == 0) {
        // ===================================================== weight producer: phase-1 range, then the phase-2 range
        // every weight byte is read exactly once: evict_first keeps the stream from displacing anything -- measured
        // -7 % at C4 T=1 and -10 % at C2 T=16, but +3.5 % when the call streams multi-GB at full HBM rate (C4 T=32/64 at
        // 0 %), so the hint is used below ~1.2 GB per call.
        // One SM's ring (6 slots at C4) keeps only ~96 KB in flight: at DRAM latency that is ~40 GB/s per SM, and a CTA
        // whose whole range is a few dozen tiles never reaches even that.  So an L2 prefetch cursor runs `pf` tiles ahead
        // of the ring over the same tile sequence (both phases): for small calls pf covers the CTA's entire range -- every
        // DRAM request of the call is in flight within microseconds of the prologue and the ring then hits L2.
        const bool el = dec_elect_one();
        const uint64_t pol_stream = l2_policy_evict_first();
        const bool hint = a.pf == 0 && (size_t)W * (size_t)(D.nKB1 + D.nDB) * WT_BYTES < ((size_t)1200 << 20);
        int stage = 0;
        uint32_t phase = 0;
        // the tile sequence of this CTA as contiguous segments; two cursors walk it: the ring loads and the L2 prefetch
        struct Seq {
            PieceIter it;
            int cur, ph;
            const uint8_t* base;
            int count, j;
        };
        auto seq_init = [&](Seq& q) { q.it.init(lo1, hi1, D.nKB1); q.cur = 0; q.ph = 1; q.count = 0; q.j = 0; q.base = nullptr; };
        auto seq_next_tile = [&](Seq& q, const uint8_t*& tile) -> bool {
            while (q.j == q.count) {
                Piece p;
                if (!q.it.next(p)) {
                    if (q.ph == 2) return false;
                    q.ph = 2; q.cur = 0;
                    q.it.init(lo2, hi2, D.nDB);
                    continue;
                }
                const int run = run_of(ax, p.item, q.cur);
                const int e = ax->run_en[run] & 0xFFFF, cb = p.item - ax->run_ib[run];
                q.base = q.ph == 1 ? a.V.gu + gu_tile_off(D, ax->eb[e], cb, p.a) : a.V.dn + dn_tile_off(D, ax->eb[e], cb, p.a);
                q.count = p.b - p.a;
                q.j = 0;
            }
            tile = q.base + (size_t)q.j * WT_BYTES;
            ++q.j;
            return true;
        };
        Seq ld, pf;
        seq_init(ld);
        seq_init(pf);
        const uint8_t* t;
        bool pf_live = a.pf > 0;
        for (int i = 0; i < a.pf && pf_live; ++i) {
            pf_live = seq_next_tile(pf, t);
            if (pf_live && el) bulk_prefetch_l2(t, WT_BYTES);
        }
        while (seq_next_tile(ld, t)) {                        // phase-2 tiles run ahead of grid barrier A: weights do not depend on phase 1
            if (pf_live) {
                const uint8_t* tp2;
                pf_live = seq_next_tile(pf, tp2);
                if (pf_live && el) bulk_prefetch_l2(tp2, WT_BYTES);
            }
            mbar_wait(empty_bar(stage), phase ^ 1u, a.state);
            if (el) {
                mbar_expect_tx(full_bar(stage), WT_BYTES);
                if (hint) bulk_g2s_hint(ring_s + stage * WT_BYTES, t, WT_BYTES, full_bar(stage), pol_stream);
                else bulk_g2s(ring_s + stage * WT_BYTES, t, WT_BYTES, full_bar(stage));
            }
            if (++stage == NS) { stage = 0; phase ^= 1u; }
        }
    } else if (warp == 1) {
        // ===================================================== MMA issuer
        const bool el = dec_elect_one();
        const uint32_t idesc = make_idesc(DEC_N);
        int stage = 0;
        uint32_t phase = 0;
        PieceIter it;
        Piece p;
        int cur = 0, prev_run = -1, nrun = 0, i = 0;
        // ---- phase 1: D1[b] = sum over the piece's k-blocks of Wgu(e, cb, kb) . Xe[kb]^T
        it.init(lo1, hi1, D.nKB1);
        bool more = it.next(p);
        while (more) {
            const int run = run_of(ax, p.item, cur);
            if (run != prev_run) { mbar_wait(xfull, (uint32_t)(nrun & 1), a.state); if (nrun == 0) DEC_TRM(11); ++nrun; prev_run = run; }
            const int b = i & 1, u = i >> 1;
            mbar_wait(a1empty(b), (uint32_t)((u & 1) ^ 1), a.state);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + (uint32_t)b * DEC_N;
            for (int kb = p.a; kb < p.b; ++kb) {
                mbar_wait(full_bar(stage), phase, a.state);
                if (i == 0 && kb == p.a) DEC_TRM(4);
                tc_fence_after();
                if (el) {
                    const uint64_t adesc = make_desc_sw128(ring_s + stage * WT_BYTES);
                    const uint64_t bdesc = make_desc_sw128(smem_base + xe_off + (uint32_t)kb * DEC_XE_KB_BYTES);
#pragma unroll
                    for (int kk = 0; kk < KB / 16; ++kk)
                        umma_bf16(d_tmem, adesc + 2u * kk, bdesc + 2u * kk, idesc, (uint32_t)((kb != p.a) | (kk != 0)));
                    umma_commit(empty_bar(stage));
                }
                __syncwarp();
                if (++stage == NS) { stage = 0; phase ^= 1u; }
            }
            Piece nx;
            more = it.next(nx);
            int cur2 = cur;
            const bool run_ends = !more || run_of(ax, nx.item, cur2) != run;
            if (el) {
                umma_commit(a1full(b));
                if (run_ends) umma_commit(xempty);              // Xe may be restaged once these MMAs retire
            }
            __syncwarp();
            p = nx;
            ++i;
        }
        DEC_TRM(8);
        // ---- phase 2: Y[db] += Wd(e, cb, db) . Hs[b]^T, accumulated in TMEM over the consecutive pieces of a run
        cur = 0; prev_run = -1; i = 0;
        int nseg = 0;
        uint32_t touched = 0;
        it.init(lo2, hi2, D.nDB);
        more = it.next(p);
        while (more) {
            const int run = run_of(ax, p.item, cur);
            if (run != prev_run) {                                // a new run segment: the previous Y partial must be drained
                mbar_wait(yempty, (uint32_t)((nseg & 1) ^ 1), a.state);
                touched = 0;
                prev_run = run;
            }
            const int b = i & 1, u = i >> 1;
            mbar_wait(hfull(b), (uint32_t)(u & 1), a.state);
            if (i == 0) DEC_TRM(9);
            tc_fence_after();
            const uint64_t bdesc = make_desc_sw128(smem_base + hs_off + (uint32_t)b * DEC_XE_KB_BYTES);
            for (int db = p.a; db < p.b; ++db) {
                mbar_wait(full_bar(stage), phase, a.state);
                tc_fence_after();
                const uint32_t acc = (touched >> db) & 1u;
                if (el) {
                    const uint64_t adesc = make_desc_sw128(ring_s + stage * WT_BYTES);
                    const uint32_t d_tmem = tmem_base + 2u * DEC_N + (uint32_t)db * DEC_N;
#pragma unroll
                    for (int kk = 0; kk < KB / 16; ++kk)
                        umma_bf16(d_tmem, adesc + 2u * kk, bdesc + 2u * kk, idesc, (uint32_t)(acc | (kk != 0)));
                    umma_commit(empty_bar(stage));
                }
                __syncwarp();
                touched |= 1u << db;
                if (++stage == NS) { stage = 0; phase ^= 1u; }
            }
            Piece nx;
            more = it.next(nx);
            int cur2 = cur;
            const bool run_ends = !more || run_of(ax, nx.item, cur2) != run;
            if (el) {
                umma_commit(hempty(b));
                if (run_ends) umma_commit(yfull);
            }
            __syncwarp();
            if (run_ends) ++nseg;
            p = nx;
            ++i;
        }
        DEC_TRM(10);
    } else if (warp < 6) {
        // ===================================================== epilogue warps 2..5 (TMEM lane quadrant q = warp & 3)
        const int q = warp & 3;
        const uint32_t lane_base = (uint32_t)(q * 32) << 16;
        const int row = q * 32 + lane;                              // packed gate/up row (phase 1), output feature in a block (phase 2)
        PieceIter it;
        Piece p;
        int i = 0;
        // ---- phase 1: the piece's fp32 partial -> scratch slot (item + CTA): 64 contiguous bytes per thread
        it.init(lo1, hi1, D.nKB1);
        while (it.next(p)) {
            const int b = i & 1, u = i >> 1;
            uint32_t v[16];
            mbar_wait(a1full(b), (uint32_t)(u & 1), a.state);
            tc_fence_after();
            tmem_ld16(tmem_base + lane_base + (uint32_t)b * DEC_N, v);
            tmem_ld_wait();
            tc_fence_before();
            mbar_arrive(a1empty(b));
            float4* dst = (float4*)(a.part + ((size_t)(p.item + (int)blockIdx.x) * WT_ROWS + row) * DEC_N);
#pragma unroll
            for (int m = 0; m < 4; ++m)
                dst[m] = make_float4(__uint_as_float(v[4 * m]), __uint_as_float(v[4 * m + 1]), __uint_as_float(v[4 * m + 2]),
                                     __uint_as_float(v[4 * m + 3]));
            // the piece is written: tell the readers of this item (no grid barrier between the phases -- a phase-2 piece
            // waits only for the few CTAs that hold pieces of ITS item)
            asm volatile("bar.sync 2, 128;" ::: "memory");
            if (tid == 64) item_signal(a.icnt + p.item);
            ++i;
        }
        DEC_TRE(2);
        // ---- phase 2
        int cur = 0, prev_run = -1, nseg = 0;
        uint32_t touched = 0;
        i = 0;
        it.init(lo2, hi2, D.nDB);
        // the CTAs c0 .. c1 hold the phase-1 pieces of an item (except those whose own range is empty)
        auto item_ctas = [&](int item, int run, int& c0, int& c1) {
            const long long t0 = (long long)item * D.nKB1;
            c0 = sp.owner(t0, run, D.nKB1);
            c1 = sp.owner(t0 + D.nKB1 - 1, run, D.nKB1);
        };
        auto item_need = [&](int item, int run) -> uint32_t {
            int c0, c1;
            item_ctas(item, run, c0, c1);
            uint32_t need = 0;
            for (int c = c0; c <= c1; ++c) need += sp.holds(c, run, D.nKB1) ? 1u : 0u;
            return need;
        };
        auto load_partials = [&](int item, int run, float (&out)[16]) {
            int c0, c1;
            item_ctas(item, run, c0, c1);
#pragma unroll
            for (int m = 0; m < 16; ++m) out[m] = 0.f;
            for (int c = c0; c <= c1; c += 2) {          // two pieces per step: eight independent 16-byte loads in flight per thread
                const bool h0 = sp.holds(c, run, D.nKB1), h1 = c + 1 <= c1 && sp.holds(c + 1, run, D.nKB1);
                const float4* s0 = (const float4*)(a.part + ((size_t)(item + c) * WT_ROWS + row) * DEC_N);
                const float4* s1 = s0 + (size_t)WT_ROWS * DEC_N / 4;
                float4 f0[4], f1[4];
#pragma unroll
                for (int m = 0; m < 4; ++m) {
                    f0[m] = h0 ? __ldcg(s0 + m) : make_float4(0.f, 0.f, 0.f, 0.f);
                    f1[m] = h1 ? __ldcg(s1 + m) : make_float4(0.f, 0.f, 0.f, 0.f);
                }
#pragma unroll
                for (int m = 0; m < 4; ++m) {
                    out[4 * m] += f0[m].x + f1[m].x; out[4 * m + 1] += f0[m].y + f1[m].y;
                    out[4 * m + 2] += f0[m].z + f1[m].z; out[4 * m + 3] += f0[m].w + f1[m].w;
                }
            }
        };
        bool more = it.next(p);
        while (more) {
            const int run = run_of(ax, p.item, cur);
            if (run != prev_run) { touched = 0; prev_run = run; }
            const int en = ax->run_en[run];
            const int e = en & 0xFFFF, nt = en >> 16;
            const int cb = p.item - ax->run_ib[run];
            const int b = i & 1, u = i >> 1;
            // h of item (run, cb): sum of the partials of the CTAs that touched the item in phase 1
            float acc[16];
            if (lane == 0) item_wait(a.icnt + p.item, item_need(p.item, run), a.state);
            __syncwarp();
            if (i == 0) DEC_TRE(3);
            load_partials(p.item, run, acc);
            Piece nx;
            more = it.next(nx);
            int cur2 = cur;
            const int run_nx = more ? run_of(ax, nx.item, cur2) : -1;
            const int ch = q * 16 + (lane & 15);
            const bool keep = cb * CB + ch < ax->r[e];              // tail of the last retained block (pad-zero rule)
            const int odd = lane >> 4;
            mbar_wait(hempty(b), (uint32_t)((u & 1) ^ 1), a.state);
            uint8_t* hs = hs_gen + b * DEC_XE_KB_BYTES;
#pragma unroll
            for (int m = 0; m < 8; ++m) {
                const float mine0 = acc[2 * m], mine1 = acc[2 * m + 1];
                const float send = odd ? mine0 : mine1;
                const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
                const float gte = odd ? recv : mine0;               // gate lives in lanes 0-15
                const float up = odd ? mine1 : recv;                // up lives in lanes 16-31
                float h = __fdividef(gte, 1.f + __expf(-gte)) * up;
                if (!keep) h = 0.f;
                const uint32_t t = 2 * m + odd;
                *(__nv_bfloat16*)(hs + sw128_off(t, ch)) = __float2bfloat16_rn(h);
            }
            fence_proxy_async_smem();
            mbar_arrive(hfull(b));
            if (i == 0) {
                // every CTA's slice of yacc is zeroed (they arrived in their prologues, ~20 us ago): checked here, while the
                // tensor core works on the first piece, and not in front of the first reduction
                if (lane == 0) cnt_wait(&a.state->dec_zcnt, ax->ztarget, a.state);
                __syncwarp();
            }
            touched |= ((p.b >= 32 ? 0xFFFFFFFFu : ((1u << p.b) - 1u)) & ~((1u << p.a) - 1u));
            const bool run_ends = !more || run_nx != run;
            if (run_ends) {
                // ---- end of the run segment: touched feature blocks of Y -> yacc (router-weight scale + ScatterAdd, Alg. 2 l.19-20)
                int tok = 0;
                float wt = 0.f;
                if (lane < nt) {
                    const int f = ax->perm[ax->run_pos[run] + lane];
                    tok = f / k;
                    wt = ax->wts[f];
                }
                mbar_wait(yfull, (uint32_t)(nseg & 1), a.state);
                tc_fence_after();
                if (nt <= 2) {
                    // one or two tokens (single-token decode): two columns per feature block, eight blocks per TMEM wait
                    const int t0 = __shfl_sync(0xffffffffu, tok, 0), t1 = __shfl_sync(0xffffffffu, tok, 1);
                    const float w0 = __shfl_sync(0xffffffffu, wt, 0), w1 = __shfl_sync(0xffffffffu, wt, 1);
                    for (int db0 = 0; db0 < D.nDB; db0 += 8) {
                        uint32_t v0[8], v1[8];
#pragma unroll
                        for (int u = 0; u < 8; ++u)
                            if (db0 + u < D.nDB && ((touched >> (db0 + u)) & 1u))
                                tmem_ld2(tmem_base + lane_base + 2u * DEC_N + (uint32_t)(db0 + u) * DEC_N, v0[u], v1[u]);
                        tmem_ld_wait();
#pragma unroll
                        for (int u = 0; u < 8; ++u) {
                            const int feat = (db0 + u) * WT_ROWS + row;
                            if (db0 + u < D.nDB && ((touched >> (db0 + u)) & 1u) && feat < D.d) {
                                red_add_f32(a.yacc + (size_t)t0 * D.d + feat, w0 * __uint_as_float(v0[u]));
                                if (nt == 2) red_add_f32(a.yacc + (size_t)t1 * D.d + feat, w1 * __uint_as_float(v1[u]));
                            }
                        }
                    }
                } else
                for (int db = 0; db < D.nDB; ++db) {
                    if (!((touched >> db) & 1u)) continue;
                    uint32_t v[16];
                    tmem_ld16(tmem_base + lane_base + 2u * DEC_N + (uint32_t)db * DEC_N, v);
                    tmem_ld_wait();
                    const int feat = db * WT_ROWS + row;
#pragma unroll
                    for (int tk = 0; tk < DEC_N; ++tk) {
                        const int t = __shfl_sync(0xffffffffu, tok, tk);
                        const float w = __shfl_sync(0xffffffffu, wt, tk);
                        if (tk < nt && feat < D.d) red_add_f32(a.yacc + (size_t)t * D.d + feat, w * __uint_as_float(v[tk]));
                    }
                }
                tc_fence_before();
                mbar_arrive(yempty);
                DEC_TRE(12);
                ++nseg;
            }
            p = nx;
            ++i;
        }
    } else {
        // ===================================================== stagers, warps 6..9: x rows of a run -> Xe (phase 1 only)
        const int st = tid - 192;                                   // 0..127
        const int cpr = D.d >> 3;                                   // 16-byte chunks per x row
        PieceIter it;
        Piece p;
        int cur = 0, prev_run = -1, nrun = 0, staged = 0;           // staged = rows of Xe that may hold a previous run's tokens
        it.init(lo1, hi1, D.nKB1);
        while (it.next(p)) {
            const int run = run_of(ax, p.item, cur);
            if (run == prev_run) continue;
            prev_run = run;
            const int nt = ax->run_en[run] >> 16, pos = ax->run_pos[run];
            // row-outer / chunk-inner: no divisions; 2 rows x up to 4 column steps = 8 loads in flight per thread.  The
            // loads of the first batch are issued BEFORE the wait for the panel (only the stores need it free), so a run
            // of one or two tokens is already in registers when the previous run's last MMA retires.
            bool waited = false;
            for (int pr0 = 0; pr0 < nt; pr0 += 2) {
                const uint4* s0 = a.x + (size_t)((int)ax->perm[pos + pr0] / k) * cpr;
                const uint4* s1 = pr0 + 1 < nt ? a.x + (size_t)((int)ax->perm[pos + pr0 + 1] / k) * cpr : nullptr;
                for (int c0 = st; c0 < cpr; c0 += 512) {
                    uint4 v0[4], v1[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int c = c0 + 128 * u;
                        v0[u] = c < cpr ? __ldg(s0 + c) : make_uint4(0, 0, 0, 0);
                        v1[u] = (s1 && c < cpr) ? __ldg(s1 + c) : make_uint4(0, 0, 0, 0);
                    }
                    if (!waited) {
                        mbar_wait(xempty, (uint32_t)((nrun & 1) ^ 1), a.state);
                        ++nrun;
                        waited = true;
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int c = c0 + 128 * u;
                        if (c < cpr) {
                            uint8_t* dst = xe_gen + (size_t)(c >> 3) * DEC_XE_KB_BYTES;
                            *(uint4*)(dst + sw128_chunk((uint32_t)pr0, (uint32_t)(c & 7))) = v0[u];
                            if (s1) *(uint4*)(dst + sw128_chunk((uint32_t)(pr0 + 1), (uint32_t)(c & 7))) = v1[u];
                        }
                    }
                }
            }
            if (!waited) {                                          // threads beyond the row width (d < 1024) issued nothing
                mbar_wait(xempty, (uint32_t)((nrun & 1) ^ 1), a.state);
                ++nrun;
            }
            // rows of a previous, larger run must not leak into this one: clear rows nt .. staged-1
            for (int pr = nt; pr < staged; ++pr)
                for (int c = st; c < cpr; c += 128)
                    *(uint4*)(xe_gen + (size_t)(c >> 3) * DEC_XE_KB_BYTES + sw128_chunk((uint32_t)pr, (uint32_t)(c & 7))) = make_uint4(0, 0, 0, 0);
            staged = nt;
            fence_proxy_async_smem();
            mbar_arrive(xfull);
        }
    }

    // ------------------------------------------------------------------------------------------ yacc -> y
    // final grid barrier: every reduction into yacc is performed before anybody rounds it.  The arrival of thread 0 is a
    // release that follows the block barrier, so it covers the reductions of all 320 threads.
    tc_fence_before();
    __syncthreads();
    DEC_TR(4);
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, 512);
    }
    if (tid == 0) {
#ifdef FXM_TRACE
        asm volatile("fence.acq_rel.gpu;" ::: "memory");
        DEC_TR(13);
#endif
        // both counters grow by exactly G per launch, so the target of this launch's final barrier is the number the
        // prologue arrival already returned: the arrival here needs no return value (no round trip before the poll)
        asm volatile("red.release.gpu.global.add.u64 [%0], 1;" ::"l"(&a.state->dec_bcnt) : "memory");
        DEC_TR(7);
        cnt_wait(&a.state->dec_bcnt, ax->ztarget, a.state);
    }
    __syncthreads();
    DEC_TR(5);
    // the item counters go back to zero for the next call (nobody reads them after the barrier above)
    for (int i = (int)((long long)W * blockIdx.x / G) + tid; i < (int)((long long)W * (blockIdx.x + 1) / G); i += DEC_THREADS) a.icnt[i] = 0u;
    {
        const size_t n4 = (size_t)a.T * D.d / 4;
        const float4* src = (const float4*)a.yacc;
        uint2* dst = (uint2*)a.y;
        for (size_t i = (size_t)blockIdx.x * DEC_THREADS + tid; i < n4; i += (size_t)G * DEC_THREADS) {
            float4 f = __ldcg(src + i);
            if (a.y_add) {
                const uint2 sa = __ldg(a.y_add + i);
                f.x += __uint_as_float(sa.x << 16); f.y += __uint_as_float(sa.x & 0xFFFF0000u);
                f.z += __uint_as_float(sa.y << 16); f.w += __uint_as_float(sa.y & 0xFFFF0000u);
            }
            const __nv_bfloat162 b0 = __floats2bfloat162_rn(f.x, f.y), b1 = __floats2bfloat162_rn(f.z, f.w);
            uint2 o;
            o.x = *(const uint32_t*)&b0;
            o.y = *(const uint32_t*)&b1;
            dst[i] = o;
        }
    }
    DEC_TR(6);
}

// ---------------------------------------------------------------------------------------------- host side
int decode_slots(const Dims& D) {
    const int avail = DEC_SMEM_MAX - dec_fixed_smem(D);
    int s = avail / WT_BYTES;
    if (s > DEC_MAX_SLOTS) s = DEC_MAX_SLOTS;
    return s;
}

// nCB <= 1024 keeps the tile arithmetic of struct Split inside 32 bits (320 runs x 1024 blocks x 60 tiles x 160 CTAs < 2^32)
bool decode_supported(const Dims& D) { return D.nDB * DEC_N + 2 * DEC_N <= 512 && decode_slots(D) >= 4 && D.nCB <= 1024; }

// most phase-1 partial slots a call with T*k = A assignments can need: (items + CTAs); monotonic in A
size_t decode_part_bytes(const Dims& D, long long A) {
    const long long a = A < DEC_MAX_A ? A : DEC_MAX_A;
    long long runs = a / DEC_N + D.E;
    if (runs > a) runs = a;                                   // a run holds at least one assignment
    return (size_t)(runs * D.nCB + DEC_MAX_CTAS + 1) * DEC_PART * sizeof(float);
}

cudaError_t init_decode_kernel() {
    return cudaFuncSetAttribute(k_decode, cudaFuncAttributeMaxDynamicSharedMemorySize, DEC_SMEM_MAX);
}

cudaError_t launch_decode(const Dims& D, const LayerView& V, const int* r_table, const __nv_bfloat16* x,
                          const int* ids, const float* topk_w, int T, int k, float* yacc, float* part,
                          const __nv_bfloat16* y_add, __nv_bfloat16* y, DevState* state, uint32_t* item_cnt, int num_sms, int pf,
                          cudaStream_t st) {
    DecArgs a{};
    a.D = D; a.V = V; a.r_table = r_table; a.x = (const uint4*)x; a.ids = ids; a.topk_w = topk_w;
    a.yacc = yacc; a.part = part; a.y_add = (const uint2*)y_add; a.y = y; a.state = state; a.icnt = item_cnt; a.T = T; a.k = k; a.A = T * k;
    a.slots = decode_slots(D);
    a.pf = pf;
    const int smem = dec_fixed_smem(D) + a.slots * WT_BYTES;
    const int grid = num_sms < DEC_MAX_CTAS ? num_sms : DEC_MAX_CTAS;
    return launch_pdl(k_decode, dim3(grid), dim3(DEC_THREADS), (size_t)smem, st, a);
}

}  // namespace fxm

#ifdef FXM_TRACE
extern "C" int fxm_dtrace_read(void* dst) { return (int)cudaMemcpyFromSymbol(dst, fxm::g_dtrace, sizeof(fxm::g_dtrace)); }
#endif
