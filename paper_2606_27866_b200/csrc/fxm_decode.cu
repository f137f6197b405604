// fxm_decode.cu -- step a6: the decode-shaped routed-expert FFN (a2..a5 of SURVEY.md 8(a)) as ONE launch.
//
//   y[t] = sum_j topk_w[t][j] * W~down_e[:, :r_e] ( silu(W~gate_e[:r_e] x[t]) (.) W~up_e[:r_e] x[t] ),  e = topk_ids[t][j]
//   (Eq. 4; Alg. 2.)  With a handful of tokens per expert the call is a stream of
//   the retained weight prefix of every ACTIVE expert, read exactly once: HBM-bound.
//
// Design (one persistent CTA per SM, cooperative launch, 320 threads):
//   prologue   every CTA re-derives the grouping from topk_ids in shared memory (stable counting sort, the same
//              definition as fxm_route.cu, Alg. 2 l.4-6) and the flat work list for the CURRENT width table:
//              items (expert e, token group g of <= 16 rows, retained channel block cb), ordered (e, g, cb); pruned
//              blocks, idle experts and width-0 experts have no items.  CTA c owns the contiguous item range
//              [c W / G, (c+1) W / G) and cuts it into RUNS of equal (e, g).
//   warp 0     weight producer: per item the d/64 gate/up tiles (one contiguous range) then the d/128 down tiles (one
//              contiguous range), 16 KB cp.async.bulk each, through a shared-memory ring; an L2 prefetch cursor
//              runs `pf` tiles ahead so the ring is refilled at L2 latency and HBM sees a deep queue.
//   warp 1     MMA issuer.  GEMM-1 (swap-AB): D1[128 packed gate/up rows, 16 tokens] += Wgu_tile . Xe^T over d;
//              GEMM-2: Y[db][128 out features, 16 tokens] += Wd_tile(e, cb, db) . Hs^T with K = 64 channels, for every
//              feature block db.  Y stays in TMEM and accumulates over the consecutive channel blocks of a run.
//              Issue order is software-pipelined: G(0), G(1), D(0), G(2), D(1), ... so the SwiGLU epilogue of
//              item i overlaps the weight stream of item i+1.
//   warps 2-5  epilogue: SwiGLU (gate lane l, up lane l+16: one shuffle), pad-zero rule for channels >= r_e
//              (PAPER.md:579), one rounding to bf16 -> Hs (the B operand of GEMM-2); at the end of a run the
//              fp32 partial Y is scaled by the router weight (Alg. 2 l.19) and added to yacc[t][:] with fp32
//              reductions (Alg. 2 l.20 ScatterAdd).
//   warps 6-9  stage the <= 16 token rows x[t] of the current run into swizzled K-major panels Xe (X[pi], Alg. 2 l.7).
//   grid barriers (sense-reversing counters in DevState; all CTAs are co-resident by the cooperative launch):
//              #0 yacc zeroed by everyone before anyone adds to it, #1 every partial added before yacc -> y (one
//              rounding to bf16).
// TMEM columns: [0,32) two GEMM-1 accumulators, [32, 32 + 16 nDB) the Y partial.  Needs nDB <= 30 (d <= 3840).
#include "fxm_ptx.cuh"

namespace fxm {

constexpr int DEC_THREADS = 320;
constexpr int DEC_N = 16;                         // tokens per group = UMMA N
constexpr int DEC_MAX_RUNS = 320;                 // >= DEC_MAX_A / 16 + MAX_E (total number of runs of a call)
constexpr int DEC_XE_KB_BYTES = DEC_N * ROW_BYTES;   // 2 KB of Xe per k-block
constexpr int DEC_MAX_SLOTS = 12;
constexpr int DEC_SMEM_MAX = 232448;              // 227 KB

struct DecArgs {
    Dims D;
    LayerView V;
    const int* r_table;
    const uint4* x;            // [T][d] bf16
    const int* ids;            // [T][k]
    const float* topk_w;       // [T][k]
    float* yacc;               // [T][d] fp32 scratch (workspace)
    const uint2* y_add;        // [T][d] bf16 or null: shared-expert output added in fp32 before the rounding of y
    __nv_bfloat16* y;          // [T][d]
    DevState* state;
    int T, k, A;
    int slots;                 // ring depth
    int pf;                    // L2 prefetch distance in tiles
};

// persistent auxiliary shared memory (after ring, Xe, Hs)
struct DecAux {
    int4 runs[DEC_MAX_RUNS];   // {e | n << 16, first sorted position, cb_lo, cb_hi}
    int16_t perm[DEC_MAX_A];   // sorted position -> flat assignment index
    int r[MAX_E];
    uint32_t eb[MAX_E];        // first channel block of each expert in the weight regions (LayerView::eblk)
    uint64_t bars[2 * DEC_MAX_SLOTS + 16];
    uint32_t tmem_slot;
    int n_runs, n_items, W;
    uint32_t gen0[2];
};
// prologue-only scratch, aliased on the weight ring (>= 4 slots = 64 KB)
struct DecTmp {
    int16_t ids[DEC_MAX_A];
    int cnt[MAX_E], off[MAX_E + 1], ibase[MAX_E + 1], gbase[MAX_E + 1];
    int wh[DEC_THREADS / 32][MAX_E];   // per-warp expert histogram, then the warp's running base
    int first_run;
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
// Grid barrier, one thread per CTA (all CTAs are co-resident: cooperative launch).  Two levels, because 148 atomics on ONE
// address serialise in L2 (measured: 10-20 us per barrier): CTA b arrives on sub-counter b % 8, the last arriver of a
// sub-counter arrives on the top counter, the last of those bumps the generation word that everyone polls (it lives in
// another 128-byte line than the counters).  Every counter is reset by its last arriver before the generation moves.
__device__ __forceinline__ void grid_arrive(DevState* st, int i, uint32_t G) {
    __threadfence();
    const uint32_t grp = blockIdx.x & 7u;
    const uint32_t gsize = (G - grp + 7u) >> 3;                       // CTAs with this residue
    if (atomicAdd(&st->bar_sub[i][grp], 1u) == gsize - 1u) {
        st->bar_sub[i][grp] = 0u;
        __threadfence();
        const uint32_t ngrp = G < 8u ? G : 8u;
        if (atomicAdd(&st->bar_count[i], 1u) == ngrp - 1u) {
            st->bar_count[i] = 0u;
            __threadfence();
            atomicAdd(&st->bar_gen[i], 1u);
        }
    }
}
__device__ __forceinline__ void grid_wait(DevState* st, int i, uint32_t gen0) {
    const long long t0 = clock64();
    uint32_t spins = 0;
    while (ld_acquire_u32(&st->bar_gen[i]) == gen0) {
        __nanosleep(1000);                                         // 148 pollers: keep the L2 slice of the barrier words quiet
        if ((++spins & 0x3FFu) == 0 && clock64() - t0 > 4000000000LL) {
            atomicOr(&st->flags, 2u);
            if (st->hflag) *(volatile uint32_t*)st->hflag = 2u;
            __threadfence_system();
            __trap();
        }
    }
}

// walks the items of this CTA in (run, channel block) order
struct ItemCur {
    int R, cb;
    __device__ __forceinline__ void init(const DecAux* ax) { R = 0; cb = ax->n_runs > 0 ? ax->runs[0].z : 0; }
    __device__ __forceinline__ bool first(const DecAux* ax) const { return cb == ax->runs[R].z; }
    __device__ __forceinline__ bool last(const DecAux* ax) const { return cb + 1 == ax->runs[R].w; }
    __device__ __forceinline__ int e(const DecAux* ax) const { return ax->runs[R].x & 0xFFFF; }
    __device__ __forceinline__ uint32_t eb(const DecAux* ax) const { return ax->eb[ax->runs[R].x & 0xFFFF]; }
    __device__ __forceinline__ void next(const DecAux* ax) {
        if (++cb == ax->runs[R].w) {
            ++R;
            cb = R < ax->n_runs ? ax->runs[R].z : 0;
        }
    }
};

// the weight stream in issue order, one PART at a time: G(0), G(1), D(0), G(2), D(1), ..., G(n-1), D(n-2), D(n-1).
// A part is a contiguous range of 16 KB tiles: G(i) = the d/64 gate/up tiles of item i, D(i) = its ceil(d/128) down tiles.
struct PartStream {
    const DecAux* ax;
    const uint8_t* gu;
    const uint8_t* dn;
    Dims D;
    ItemCur g, d;
    int i;            // step: the G part of item i, then the D part of item i-1
    int sub;          // 0 = G(i) comes next, 1 = D(i-1) comes next
    __device__ __forceinline__ void init(const DecAux* a, const DecArgs& args) {
        ax = a; D = args.D; gu = args.V.gu; dn = args.V.dn;
        g.init(a); d.init(a);
        i = 0; sub = 0;
    }
    __device__ __forceinline__ bool next(const uint8_t*& base, int& count) {
        const int n = ax->n_items;
        while (n > 0 && i <= n) {
            if (sub == 0) {
                sub = 1;
                if (i < n) {
                    base = gu + gu_tile_off(D, g.eb(ax), g.cb, 0);
                    count = D.nKB1;
                    g.next(ax);
                    return true;
                }
            }
            sub = 0;
            const int ii = i++;
            if (ii >= 1) {
                base = dn + dn_tile_off(D, d.eb(ax), d.cb, 0);
                count = D.nDB;
                d.next(ax);
                return true;
            }
        }
        return false;
    }
};

// -DFXM_TRACE: per-CTA globaltimer stamps (ns): 0 entry, 1 prologue done, 2 roles done (this CTA's last reduction issued),
// 3 grid barrier #1 passed, 4 exit.  Tuning aid only.
#ifdef FXM_TRACE
__device__ unsigned long long g_dtrace[148][8];
__device__ __forceinline__ unsigned long long dec_now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define DEC_TR(f) do { if (threadIdx.x == 0 && blockIdx.x < 148) g_dtrace[blockIdx.x][f] = dec_now(); } while (0)
#else
#define DEC_TR(f) do { } while (0)
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

    // ------------------------------------------------------------------------------------------ prologue
    if (tid == 0) {
        for (int s = 0; s < NS; ++s) { mbar_init(full_bar(s), 1); mbar_init(empty_bar(s), 1); }
        mbar_init(xfull, 128); mbar_init(xempty, 1); mbar_init(yfull, 1); mbar_init(yempty, 128);
        for (int b = 0; b < 2; ++b) {
            mbar_init(a1full(b), 1); mbar_init(a1empty(b), 128); mbar_init(hfull(b), 128); mbar_init(hempty(b), 1);
        }
        fence_barrier_init();
        ax->gen0[0] = ld_acquire_u32(&a.state->bar_gen[0]);      // read before this CTA arrives anywhere
        ax->gen0[1] = ld_acquire_u32(&a.state->bar_gen[1]);
    }
    if (warp == 1) tmem_alloc(smem_u32(&ax->tmem_slot), 512);
    bool bad = false;
    for (int f = tid; f < A; f += DEC_THREADS) {
        int id = a.ids[f];
        if (id < 0 || id >= E) { bad = true; id = -1; }
        tp->ids[f] = (int16_t)id;
    }
    if (bad) atomicOr(&a.state->flags, 1u);
    for (int e = tid; e < MAX_E; e += DEC_THREADS) { ax->r[e] = e < E ? a.r_table[e] : 0; ax->eb[e] = e < E ? a.V.eblk[e] : 0u; }
    // zero this CTA's slice of the fp32 accumulator (grid barrier #0 orders it before every reduction)
    {
        float4* z = (float4*)a.yacc;
        const size_t n4 = (size_t)a.T * D.d / 4;
        for (size_t i = (size_t)blockIdx.x * DEC_THREADS + tid; i < n4; i += (size_t)G * DEC_THREADS)
            z[i] = make_float4(0.f, 0.f, 0.f, 0.f);
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    if (tid == 0) grid_arrive(a.state, 0, G);
    const uint32_t tmem_base = ax->tmem_slot;

    // counts (Alg. 2 l.4-6, stable counting sort as in fxm_route.cu): warp w owns the contiguous chunk [w*chunk, (w+1)*chunk)
    // of the flat assignments; per 32-wide step the lowest lane of every group of equal ids adds the group size to
    // the warp's histogram row
    constexpr int NW = DEC_THREADS / 32;
    const int chunk = ((A + NW - 1) / NW + 31) & ~31;
    const int wlo = min(A, warp * chunk), whi = min(A, wlo + chunk);
    for (int i = tid; i < NW * MAX_E; i += DEC_THREADS) (&tp->wh[0][0])[i] = 0;
    __syncthreads();
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
        }
    }
    __syncthreads();
    const int W = ax->W;
    const int lo = (int)((long long)blockIdx.x * W / (long long)G), hi = (int)((long long)(blockIdx.x + 1) * W / (long long)G);
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
    if (tid < E) {
        // the run that contains item `lo`
        const int r = ax->r[tid];
        const int nb = (r + CB - 1) / CB;
        if (lo < hi && tp->ibase[tid] <= lo && lo < tp->ibase[tid + 1]) tp->first_run = tp->gbase[tid] + (lo - tp->ibase[tid]) / nb;
    }
    if (tid == 0) { ax->n_runs = 0; ax->n_items = hi - lo; }
    __syncthreads();
    if (tid < E && lo < hi) {
        const int n = tp->cnt[tid], r = ax->r[tid];
        const int nb = (r + CB - 1) / CB;
        const int ng = tp->gbase[tid + 1] - tp->gbase[tid];
        for (int g = 0; g < ng; ++g) {
            const int i0 = tp->ibase[tid] + g * nb;             // items [i0, i0 + nb) = channel blocks 0..nb-1 of (e, g)
            const int s = max(i0, lo), t = min(i0 + nb, hi);
            if (s < t) {
                const int slot = tp->gbase[tid] + g - tp->first_run;
                const int nt = min(DEC_N, n - g * DEC_N);
                ax->runs[slot] = make_int4(tid | (nt << 16), tp->off[tid] + g * DEC_N, s - i0, t - i0);
                atomicMax(&ax->n_runs, slot + 1);
            }
        }
    }
    __syncthreads();
    // Xe / Hs start as zeros (rows beyond a run's token count are never staged)
    for (int i = tid; i < (int)((aux_off - xe_off) / 16); i += DEC_THREADS) ((uint4*)xe_gen)[i] = make_uint4(0, 0, 0, 0);
    fence_proxy_async_smem();
    __syncthreads();
    const int n_items = ax->n_items, n_runs = ax->n_runs;
    DEC_TR(1);

    if (warp == 0) {
        // ===================================================== weight producer + L2 prefetch cursor
        // per tile: wait for the slot, arm the barrier, one 16 KB bulk copy; optionally one 16 KB L2 prefetch `pf` tiles
        // further down the same stream (a second cursor).  Measured on B200: the prefetch competes with the ring's own
        // loads for the SM's outstanding requests and every distance > 0 is slower (C4 T=64 0 %: 558 us at 0, 580 at 8,
        // 978 at 64), so the default distance is 0.
        if (n_items > 0) {
            const bool el = dec_elect_one();
            // every weight byte is read exactly once: evict_first keeps the stream from displacing anything -- measured
            // -7 % at C4 T=1 and -10 % at C2 T=16, but +3.5 % when the call streams multi-GB at full HBM rate (C4 T=32/64 at
            // 0 %), so the hint is used below ~1.2 GB per call
            const uint64_t pol_stream = l2_policy_evict_first();
            const bool hint = (size_t)W * (size_t)(D.nKB1 + D.nDB) * WT_BYTES < ((size_t)1200 << 20);
            PartStream ld, pf;
            ld.init(ax, a);
            pf.init(ax, a);
            const uint8_t* pb = nullptr;
            int pc = 0, pj = 0;
            bool pf_live = pf.next(pb, pc);
            auto pf_step = [&]() {
                if (!pf_live) return;
                if (el) bulk_prefetch_l2(pb + (size_t)pj * WT_BYTES, WT_BYTES);
                if (++pj == pc) { pj = 0; pf_live = pf.next(pb, pc); }
            };
            for (int p = 0; p < a.pf; ++p) pf_step();
            int stage = 0;
            uint32_t phase = 0;
            const uint8_t* base = nullptr;
            int count = 0;
            while (ld.next(base, count)) {
                for (int j = 0; j < count; ++j) {
                    if (a.pf > 0) pf_step();
                    mbar_wait(empty_bar(stage), phase ^ 1u, a.state);
                    if (el) {
                        mbar_expect_tx(full_bar(stage), WT_BYTES);
                        if (hint) bulk_g2s_hint(ring_s + stage * WT_BYTES, base + (size_t)j * WT_BYTES, WT_BYTES, full_bar(stage), pol_stream);
                        else bulk_g2s(ring_s + stage * WT_BYTES, base + (size_t)j * WT_BYTES, WT_BYTES, full_bar(stage));
                    }
                    if (++stage == NS) { stage = 0; phase ^= 1u; }
                }
            }
        }
    } else if (warp == 1) {
        // ===================================================== MMA issuer
        if (n_items > 0) {
            const bool el = dec_elect_one();
            ItemCur g, d;
            g.init(ax); d.init(ax);
            int stage = 0;
            uint32_t phase = 0;
            const uint32_t idesc = make_idesc(DEC_N);
            for (int i = 0; i <= n_items; ++i) {
                if (i < n_items) {                                  // ---- G(i): D1[b] = Wgu(e, cb) . Xe^T
                    const int b = i & 1, u = i >> 1;
                    if (g.first(ax)) mbar_wait(xfull, (uint32_t)(g.R & 1), a.state);
                    mbar_wait(a1empty(b), (uint32_t)((u & 1) ^ 1), a.state);
                    tc_fence_after();
                    const uint32_t d_tmem = tmem_base + (uint32_t)b * DEC_N;
                    for (int kb = 0; kb < D.nKB1; ++kb) {
                        mbar_wait(full_bar(stage), phase, a.state);
                        tc_fence_after();
                        if (el) {
                            const uint64_t adesc = make_desc_sw128(ring_s + stage * WT_BYTES);
                            const uint64_t bdesc = make_desc_sw128(smem_base + xe_off + (uint32_t)kb * DEC_XE_KB_BYTES);
#pragma unroll
                            for (int kk = 0; kk < KB / 16; ++kk)
                                umma_bf16(d_tmem, adesc + 2u * kk, bdesc + 2u * kk, idesc, (uint32_t)((kb | kk) != 0));
                            umma_commit(empty_bar(stage));
                        }
                        __syncwarp();
                        if (++stage == NS) { stage = 0; phase ^= 1u; }
                    }
                    if (el) {
                        umma_commit(a1full(b));
                        if (g.last(ax)) umma_commit(xempty);        // Xe may be restaged once these MMAs retire
                    }
                    __syncwarp();
                    g.next(ax);
                }
                if (i >= 1) {                                       // ---- D(i-1): Y[db] += Wd(e, cb, db) . Hs[b]^T
                    const int b = (i - 1) & 1, u = (i - 1) >> 1;
                    const bool first = d.first(ax);
                    if (first) mbar_wait(yempty, (uint32_t)((d.R & 1) ^ 1), a.state);
                    mbar_wait(hfull(b), (uint32_t)(u & 1), a.state);
                    tc_fence_after();
                    const uint64_t bdesc = make_desc_sw128(smem_base + hs_off + (uint32_t)b * DEC_XE_KB_BYTES);
                    for (int db = 0; db < D.nDB; ++db) {
                        mbar_wait(full_bar(stage), phase, a.state);
                        tc_fence_after();
                        if (el) {
                            const uint64_t adesc = make_desc_sw128(ring_s + stage * WT_BYTES);
                            const uint32_t d_tmem = tmem_base + 2u * DEC_N + (uint32_t)db * DEC_N;
#pragma unroll
                            for (int kk = 0; kk < KB / 16; ++kk)
                                umma_bf16(d_tmem, adesc + 2u * kk, bdesc + 2u * kk, idesc, (uint32_t)(!first || kk != 0));
                            umma_commit(empty_bar(stage));
                        }
                        __syncwarp();
                        if (++stage == NS) { stage = 0; phase ^= 1u; }
                    }
                    if (el) {
                        umma_commit(hempty(b));
                        if (d.last(ax)) umma_commit(yfull);
                    }
                    __syncwarp();
                    d.next(ax);
                }
            }
        }
    } else if (warp < 6) {
        // ===================================================== epilogue warps 2..5
        const int q = warp & 3;                                     // TMEM lane quadrant this warp may read
        const uint32_t lane_base = (uint32_t)(q * 32) << 16;
        bool zero_seen = false;
        int i = 0;
        for (int R = 0; R < n_runs; ++R) {
            const int4 run = ax->runs[R];
            const int e = run.x & 0xFFFF, nt = run.x >> 16;
            const int r = ax->r[e];
            for (int cb = run.z; cb < run.w; ++cb, ++i) {
                const int b = i & 1, u = i >> 1;
                uint32_t v[16];
                mbar_wait(a1full(b), (uint32_t)(u & 1), a.state);
                tc_fence_after();
                tmem_ld16(tmem_base + lane_base + (uint32_t)b * DEC_N, v);
                tmem_ld_wait();
                tc_fence_before();
                mbar_arrive(a1empty(b));
                const int ch = q * 16 + (lane & 15);
                const bool keep = cb * CB + ch < r;                 // tail of the last retained block (pad-zero rule)
                const int odd = lane >> 4;
                mbar_wait(hempty(b), (uint32_t)((u & 1) ^ 1), a.state);
                uint8_t* hs = hs_gen + b * DEC_XE_KB_BYTES;
#pragma unroll
                for (int m = 0; m < 8; ++m) {
                    const float mine0 = __uint_as_float(v[2 * m]), mine1 = __uint_as_float(v[2 * m + 1]);
                    const float send = odd ? mine0 : mine1;
                    const float recv = __shfl_xor_sync(0xffffffffu, send, 16);
                    const float gte = odd ? recv : mine0;           // gate lives in lanes 0-15
                    const float up = odd ? mine1 : recv;            // up lives in lanes 16-31
                    float h = __fdividef(gte, 1.f + __expf(-gte)) * up;
                    if (!keep) h = 0.f;
                    const uint32_t t = 2 * m + odd;
                    *(__nv_bfloat16*)(hs + sw128_off(t, ch)) = __float2bfloat16_rn(h);
                }
                fence_proxy_async_smem();
                mbar_arrive(hfull(b));
            }
            // ---- end of run: Y partial -> yacc (router-weight scale + ScatterAdd, Alg. 2 l.19-20)
            int tok = 0;
            float wt = 0.f;
            if (lane < nt) {
                const int f = ax->perm[run.y + lane];
                tok = f / k;
                wt = a.topk_w[f];
            }
            mbar_wait(yfull, (uint32_t)(R & 1), a.state);
            tc_fence_after();
            if (!zero_seen) {
                if (lane == 0) grid_wait(a.state, 0, ax->gen0[0]);
                __syncwarp();
                zero_seen = true;
            }
            for (int db = 0; db < D.nDB; ++db) {
                uint32_t v[16];
                tmem_ld16(tmem_base + lane_base + 2u * DEC_N + (uint32_t)db * DEC_N, v);
                tmem_ld_wait();
                const int feat = db * WT_ROWS + q * 32 + lane;
#pragma unroll
                for (int tk = 0; tk < DEC_N; ++tk) {
                    const int t = __shfl_sync(0xffffffffu, tok, tk);
                    const float w = __shfl_sync(0xffffffffu, wt, tk);
                    if (tk < nt && feat < D.d) atomicAdd(a.yacc + (size_t)t * D.d + feat, w * __uint_as_float(v[tk]));
                }
            }
            tc_fence_before();
            mbar_arrive(yempty);
        }
    } else {
        // ===================================================== stagers, warps 6..9: x rows of the run -> Xe
        const int st = tid - 192;                                   // 0..127
        const int cpr = D.d >> 3;                                   // 16-byte chunks per x row
        for (int R = 0; R < n_runs; ++R) {
            const int4 run = ax->runs[R];
            const int nt = run.x >> 16;
            mbar_wait(xempty, (uint32_t)((R & 1) ^ 1), a.state);
            const int total = nt * cpr;
            for (int i0 = st; i0 < total; i0 += 128 * 8) {
                uint4 v[8];
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int idx = i0 + u * 128;
                    if (idx < total) {
                        const int p = idx / cpr, c = idx - p * cpr;
                        const int f = ax->perm[run.y + p];
                        v[u] = __ldg(a.x + (size_t)(f / k) * cpr + c);
                    }
                }
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int idx = i0 + u * 128;
                    if (idx < total) {
                        const int p = idx / cpr, c = idx - p * cpr;
                        *(uint4*)(xe_gen + (size_t)(c >> 3) * DEC_XE_KB_BYTES + sw128_chunk((uint32_t)p, (uint32_t)(c & 7))) = v[u];
                    }
                }
            }
            fence_proxy_async_smem();
            mbar_arrive(xfull);
        }
    }

    // ------------------------------------------------------------------------------------------ yacc -> y
    __threadfence();                                               // this thread's reductions are performed
    tc_fence_before();
    __syncthreads();
    DEC_TR(2);
    if (warp == 1) {
        tc_fence_after();
        tmem_dealloc(tmem_base, 512);
    }
    if (tid == 0) {
        DEC_TR(5);
        grid_arrive(a.state, 1, G);
        DEC_TR(6);
        grid_wait(a.state, 1, ax->gen0[1]);
        DEC_TR(7);
    }
    __syncthreads();
    DEC_TR(3);
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
    DEC_TR(4);
}

// ---------------------------------------------------------------------------------------------- host side
int decode_slots(const Dims& D) {
    const int avail = DEC_SMEM_MAX - dec_fixed_smem(D);
    int s = avail / WT_BYTES;
    if (s > DEC_MAX_SLOTS) s = DEC_MAX_SLOTS;
    return s;
}

bool decode_supported(const Dims& D) { return D.nDB * DEC_N + 2 * DEC_N <= 512 && decode_slots(D) >= 4; }

cudaError_t init_decode_kernel() {
    return cudaFuncSetAttribute(k_decode, cudaFuncAttributeMaxDynamicSharedMemorySize, DEC_SMEM_MAX);
}

cudaError_t launch_decode(const Dims& D, const LayerView& V, const int* r_table, const __nv_bfloat16* x,
                          const int* ids, const float* topk_w, int T, int k, float* yacc, const __nv_bfloat16* y_add,
                          __nv_bfloat16* y, DevState* state, int num_sms, int pf, cudaStream_t st) {
    DecArgs a{};
    a.D = D; a.V = V; a.r_table = r_table; a.x = (const uint4*)x; a.ids = ids; a.topk_w = topk_w;
    a.yacc = yacc; a.y_add = (const uint2*)y_add; a.y = y; a.state = state; a.T = T; a.k = k; a.A = T * k;
    a.slots = decode_slots(D);
    a.pf = pf;
    const int smem = dec_fixed_smem(D) + a.slots * WT_BYTES;
    void* args[] = {(void*)&a};
    return cudaLaunchCooperativeKernel((const void*)k_decode, dim3(num_sms), dim3(DEC_THREADS), args, (size_t)smem, st);
}

}  // namespace fxm

#ifdef FXM_TRACE
extern "C" int fxm_dtrace_read(void* dst) { return (int)cudaMemcpyFromSymbol(dst, fxm::g_dtrace, sizeof(fxm::g_dtrace)); }
#endif
