// fxm_route.cu -- steps a2 + a3 in ONE launch: router-output grouping (stable per-expert counting sort, bit-exact
// indices) and the device-side tile schedule that skips pruned work.
//   Alg. 2 l.4-6: "(pi, eid) <- Sort(eid)", read as the STABLE sort by (expert id, flat
//   index f = t*k+j) so that exactly one permutation is correct (reading R5).
//   Alg. 2 l.2-3, 8-11: BucketByRetI / AlignUp / view lists are replaced by a tile list
//   computed here from counts[] and the CURRENT width table r[]: only tiles with channel index < r_e and
//   token row < n_e exist.
//
// k_route, grid = RB <= 128 scatter blocks + 1 planner block of 256 threads, no atomics decide any position
// (deterministic and stable):
//   1  block b histograms its flat assignments [b*chunk, (b+1)*chunk) per expert, one histogram row per warp
//      (warp w owns a contiguous sub-range, so "earlier block, earlier warp, earlier 32-wide step, lower lane" is
//      "lower flat index"), and publishes the block row to bhist[b][.];
//   2  grid-wide publish barrier: a ticket counter; the last block to arrive bumps a generation word that the
//      others poll (all RB <= 128 blocks are co-resident: they are small and a B200 has 148 SMs);
//   3  EVERY block sums the published rows itself: all rows -> counts, rows of earlier blocks -> its own base.
//      These are independent loads (no serial scan by a "last block"), a few per thread;
//   4  every block scans counts over the experts (offsets, padded offsets) in shared memory and scatters its own
//      assignments -- the per-warp histograms of step 1 are still in shared memory, nothing is recomputed;
//   5  the PLANNER block (the extra, last block: it has no assignments of its own, so the schedule is written while the
//      others scatter) writes counts / offsets and the schedule for the current width table: the token tiles
//      {expert, first padded row, valid rows, GEMM-1 work prefix}, experts ordered by descending work per tile (rows x
//      retained width) so that a static stride over the work list hands out the heavy tiles first and the light
//      ones in the last, partly filled round.  GEMM-1's work items (tile, pair of retained channel blocks) are not
//      materialised: item wi belongs to the tile j with tt[j].w <= wi < tt[j+1].w (tt[ntt] is a sentinel).
#include "fxm_internal.cuh"

#include <math_constants.h>

namespace fxm {

constexpr int RT_WARPS = RT_THREADS / 32;

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    return v;
}
__device__ __forceinline__ uint32_t ld_acquire_gpu(const uint32_t* p) {
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

// balanced split of np padded rows into nt tiles: rows per tile, a multiple of 16
__device__ __forceinline__ int per_rows(int np, int nt) { return ((np + nt - 1) / nt + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN; }

// -DFXM_TRACE: per-block globaltimer stamps (ns) of the phases (tuning aid; the product build has none of this)
#ifdef FXM_TRACE
__device__ unsigned long long g_rtrace[RT_MAX_BLOCKS][8];
__device__ __forceinline__ unsigned long long rt_now() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t));
    return t;
}
#define RT_TR(f) do { if (threadIdx.x == 0) g_rtrace[blockIdx.x][f] = rt_now(); } while (0)
#else
#define RT_TR(f) do { } while (0)
#endif

// NEXT-3, the router front end (reading R10; the paper takes the router's OUTPUT as given): for one
// token, the k largest of its E logits in descending order (fp32 comparison, ties -> lower expert id) and the softmax
// over those k logits (= the softmax over all E renormalised to sum 1).  One warp per token; lane l holds the logits
// l, l + 32, ...  Each round: every lane offers its best unused logit, a butterfly keeps (larger value, then lower id).
__device__ __forceinline__ void warp_router_topk(const float* __restrict__ lg, int E, int k, int lane,
                                                 int* __restrict__ ids_out, float* __restrict__ w_out) {
    float v[MAX_E / 32];
#pragma unroll
    for (int u = 0; u < MAX_E / 32; ++u) v[u] = (lane + 32 * u) < E ? lg[lane + 32 * u] : -CUDART_INF_F;
    unsigned used = 0;
    float top = 0.f, mine = 0.f, den = 0.f;
    int my_id = 0;
    for (int j = 0; j < k; ++j) {
        float bv = -CUDART_INF_F;
        int bi = 0x7fffffff;
#pragma unroll
        for (int u = 0; u < MAX_E / 32; ++u) {
            const int id = lane + 32 * u;
            if (id < E && !((used >> u) & 1u) && (v[u] > bv || (v[u] == bv && id < bi))) { bv = v[u]; bi = id; }
        }
#pragma unroll
        for (int o = 16; o; o >>= 1) {
            const float ov = __shfl_xor_sync(0xffffffffu, bv, o);
            const int oi = __shfl_xor_sync(0xffffffffu, bi, o);
            if (ov > bv || (ov == bv && oi < bi)) { bv = ov; bi = oi; }
        }
        if ((bi & 31) == lane && bi < E) used |= 1u << (bi >> 5);
        if (j == 0) top = bv;
        const float ex = expf(bv - top);
        den += ex;
        if (lane == j) { mine = ex; my_id = bi; }
    }
    if (lane < k) {
        ids_out[lane] = my_id;
        w_out[lane] = mine / den;
    }
}

struct RouteWs {             // the device pointers of the workspace the kernel writes
    int* poff;
    Sched* sched;
    int* row_flat;
    int* row_tok;
    int2* row_tw;
    int* bhist;
    int4* tt;
    int chunk;
};

__global__ void __launch_bounds__(RT_THREADS)
k_route(const RouteArgs a, const RouteWs w, DevState* __restrict__ state) {
    __shared__ int whist[RT_WARPS][MAX_E];      // per-warp histogram, later the warp's running base
    __shared__ int s_cnt[MAX_E], s_off[MAX_E + 1], s_poff[MAX_E + 1], s_bbase[MAX_E];
    __shared__ int s_key[MAX_E], s_order[MAX_E];
    __shared__ uint32_t s_gen0;
    const Dims& D = a.D;
    const int E = D.E, k = a.k, A = a.T * a.k;
    const int tid = threadIdx.x, lane = tid & 31, wp = tid >> 5;
    const int RB = gridDim.x - 1, b = blockIdx.x;              // block RB is the planner
    const bool planner = b == RB;
    const int* ids = a.logits ? a.ids_out : a.ids;
    RT_TR(0);
    pdl_launch_dependents();
    for (int i = tid; i < RT_WARPS * MAX_E; i += RT_THREADS) (&whist[0][0])[i] = 0;
    pdl_wait();                                                  // the previous call's kernels may still read the workspace
    RT_TR(1);
    if (tid == 0) s_gen0 = ld_acquire_gpu(&state->route_gen);    // before this block arrives anywhere
    if (a.logits && !planner) {
        // ---- 0: the router front end for this block's own tokens (a block owns whole tokens): ids / weights go to the
        //         workspace, the grouping below reads them back (same block: visible after the barrier)
        const int t_lo = min(a.T, b * (w.chunk / k)), t_hi = min(a.T, t_lo + w.chunk / k);
        for (int t = t_lo + wp; t < t_hi; t += RT_WARPS)
            warp_router_topk(a.logits + (size_t)t * E, E, k, lane, a.ids_out + (size_t)t * k, a.w_out + (size_t)t * k);
    }
    __syncthreads();

    // ---- 1: per-warp histogram of this block's chunk
    const int lo = min(A, b * w.chunk), hi = min(A, lo + w.chunk);
    const int sub = w.chunk / RT_WARPS;
    const int wlo = min(hi, lo + wp * sub), whi = min(hi, wlo + sub);
    {
        bool bad = false;
        int* wh = whist[wp];
        for (int base = wlo; base < whi; base += 32) {
            const int f = base + lane;
            int id = f < whi ? ids[f] : -1;
            if (f < whi && (id < 0 || id >= E)) { bad = true; id = -1; }
            const unsigned m = __match_any_sync(0xffffffffu, id);
            if (id >= 0 && lane == __ffs(m) - 1) wh[id] += __popc(m);
            __syncwarp();
        }
        if (bad) atomicOr(&state->flags, 1u);
    }
    __syncthreads();
    if (!planner)
        for (int e = tid; e < E; e += RT_THREADS) {
            int c = 0;
#pragma unroll
            for (int ww = 0; ww < RT_WARPS; ++ww) c += whist[ww][e];
            w.bhist[(size_t)b * E + e] = c;
        }

    // ---- 2: publish barrier over the grid
    __threadfence();
    __syncthreads();
    RT_TR(2);
    if (tid == 0) {
        if (atomicAdd(&state->ticket, 1u) == gridDim.x - 1u) {
            state->ticket = 0;                                   // ready for the next call on this layer
            __threadfence();
            atomicAdd(&state->route_gen, 1u);
        } else {
            const long long t0 = clock64();
            uint32_t spins = 0;
            while (ld_acquire_gpu(&state->route_gen) == s_gen0) {
                if ((++spins & 0x3FFu) == 0 && clock64() - t0 > 4000000000LL) {
                    atomicOr(&state->flags, 2u);
                    if (state->hflag) *(volatile uint32_t*)state->hflag = 2u;
                    __threadfence_system();
                    __trap();
                }
            }
        }
    }
    __syncthreads();

    RT_TR(3);
    // ---- 3: every block sums the published rows: thread (e0, s0) takes rows s0, s0 + S, ... of column e0
    {
        const int S = RT_THREADS / E > 0 ? RT_THREADS / E : 1;   // E <= 256 = RT_THREADS
        const int e0 = tid % E, s0 = tid / E;
        int tot = 0, base = 0;
        if (s0 < S) {
            int bb = s0;
            for (; bb + 15 * S < RB; bb += 16 * S) {             // 16 independent loads in flight per thread
                int c[16];
#pragma unroll
                for (int u = 0; u < 16; ++u) c[u] = __ldcg(w.bhist + (size_t)(bb + u * S) * E + e0);
#pragma unroll
                for (int u = 0; u < 16; ++u) { tot += c[u]; if (bb + u * S < b) base += c[u]; }
            }
            for (; bb < RB; bb += S) {
                const int c = __ldcg(w.bhist + (size_t)bb * E + e0);
                tot += c;
                if (bb < b) base += c;
            }
        }
        // reduce the S partials of a column through shared memory (s_cnt / s_bbase as accumulators)
        for (int e = tid; e < E; e += RT_THREADS) { s_cnt[e] = 0; s_bbase[e] = 0; }
        __syncthreads();
        if (s0 < S) { atomicAdd(&s_cnt[e0], tot); atomicAdd(&s_bbase[e0], base); }   // integer sums: order-independent
        __syncthreads();
    }

    RT_TR(4);
    // ---- 4a: warp 0 scans over the experts -> offsets and padded offsets (expert order); block 0 also orders the
    //          experts by descending work per tile and lays out the token tiles and work prefixes in that order
    if (wp == 0) {
        int c_off = 0, c_poff = 0;
        for (int base = 0; base < E; base += 32) {
            const int e = base + lane;
            const int n = e < E ? s_cnt[e] : 0;
            const int np = (n + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN;
            const int i_off = warp_incl_scan(n, lane), i_poff = warp_incl_scan(np, lane);
            if (e < E) { s_off[e] = c_off + i_off - n; s_poff[e] = c_poff + i_poff - np; }
            c_off += __shfl_sync(0xffffffffu, i_off, 31);
            c_poff += __shfl_sync(0xffffffffu, i_poff, 31);
        }
        if (lane == 0) { s_off[E] = c_off; s_poff[E] = c_poff; }
    }
    __syncthreads();
    if (planner) {
        // work key of an expert: rows of its widest tile x retained width (what one GEMM-2 item of it costs)
        for (int e = tid; e < E; e += RT_THREADS) {
            const int n = s_cnt[e];
            const int r = a.r_table ? a.r_table[e] : D.I;           // no table yet (fxm_route only): full width
            const int np = (n + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN;
            const int nt = (n > 0 && r > 0) ? (np + a.tile_n - 1) / a.tile_n : 0;
            s_key[e] = nt > 0 ? min(per_rows(np, nt), np) * r : 0;
        }
        __syncthreads();
        for (int e = tid; e < E; e += RT_THREADS) {               // rank by (key descending, id ascending)
            const int ke = s_key[e];
            int rk = 0;
            for (int o = 0; o < E; ++o) {
                const int ko = s_key[o];
                rk += (ko > ke) || (ko == ke && o < e);
            }
            s_order[rk] = e;
        }
        __syncthreads();
        if (wp == 0) {
            int c_tiles = 0, c_work = 0, c_max = ROW_ALIGN;
            for (int base = 0; base < E; base += 32) {
                const int pos = base + lane;
                const int e = pos < E ? s_order[pos] : 0;
                const int n = pos < E ? s_cnt[e] : 0;
                const int r = pos < E ? (a.r_table ? a.r_table[e] : D.I) : 0;
                const int np = (n + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN;
                const int nt = (n > 0 && r > 0) ? (np + a.tile_n - 1) / a.tile_n : 0;   // pruned-away / idle experts: no tiles
                const int nb = ((r + CB - 1) / CB + 1) / 2;                          // GEMM-1 pair items per token tile
                const int i_tiles = warp_incl_scan(nt, lane), i_work = warp_incl_scan(nt * nb, lane);
                if (pos < E && nt > 0) {
                    int j = c_tiles + i_tiles - nt, wk = c_work + i_work - nt * nb;
                    const int p0 = s_poff[e];
                    // balanced split of the padded segment into nt tiles of <= tile_n rows, each a multiple of 16 rows
                    const int per = per_rows(np, nt);
                    // .z = valid rows of the tile (>= 1) | tiles of this expert << 16 | index of the tile among them << 24: the
                    // GEMM kernels walk an expert's items block-major ((block, tile) order), so that the tiles of one expert,
                    // which read the same weight tiles, run on neighbouring clusters at the same time (fxm_pair.cu pair_item)
                    const int ntz = nt <= 15 ? nt : 1;
                    int ti = 0;
                    for (int row = 0; row < np; row += per, ++j, wk += nb, ++ti)
                        w.tt[j] = make_int4(e, p0 + row, min(per, n - row) | (ntz << 16) | ((nt <= 15 ? ti : 0) << 24), wk);
                }
                {
                    int mx = nt > 0 ? min(per_rows(np, nt), np) : 0;               // rows of this expert's widest tile
#pragma unroll
                    for (int o = 16; o; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                    c_max = max(c_max, mx);
                }
                c_tiles += __shfl_sync(0xffffffffu, i_tiles, 31);
                c_work += __shfl_sync(0xffffffffu, i_work, 31);
            }
            if (lane == 0) {
                w.tt[c_tiles] = make_int4(0, 0, 0, c_work);          // sentinel: the work prefix of "the tile after the last"
                w.sched->ntt = c_tiles;
                w.sched->W1 = c_work;
                w.sched->W2 = c_tiles * ((D.nDB + 1) / 2);
                w.sched->P_used = s_poff[E];
                w.sched->A = A;
                w.sched->max_n = c_max;
                w.sched->claim1 = 0;
                w.sched->claim2 = 0;
            }
        }
        for (int e = tid; e <= E; e += RT_THREADS) {
            a.offsets[e] = s_off[e];
            w.poff[e] = s_poff[e];
            if (e < E) a.counts[e] = s_cnt[e];
        }
        // padding rows of the expert segments carry no assignment
        for (int e = tid; e < E; e += RT_THREADS)
            for (int p = s_poff[e] + s_cnt[e]; p < s_poff[e + 1]; ++p) {
                w.row_flat[p] = -1;
                w.row_tok[p] = 0;
                w.row_tw[p] = make_int2(-1, 0);
            }
        return;
    }

    RT_TR(5);
    // ---- 4b: exclusive scan over the warps of this block, on top of the block base -> the warp's running base
    for (int e = tid; e < E; e += RT_THREADS) {
        int run = s_bbase[e];
#pragma unroll
        for (int ww = 0; ww < RT_WARPS; ++ww) {
            const int c = whist[ww][e];
            whist[ww][e] = run;
            run += c;
        }
    }
    __syncthreads();

    // ---- stable scatter of this block's assignments
    for (int base = wlo; base < whi; base += 32) {
        const int f = base + lane;
        int id = f < whi ? ids[f] : -1;
        if (id < 0 || id >= E) id = -1;
        const unsigned m = __match_any_sync(0xffffffffu, id);
        if (id >= 0) {
            const int rank = whist[wp][id] + __popc(m & ((1u << lane) - 1u));
            const int pos = s_off[id] + rank;
            const int pr = s_poff[id] + rank;
            const int t = f / k;
            a.perm[pos] = f;
            a.inv_perm[f] = pos;
            w.row_flat[pr] = f;
            w.row_tok[pr] = t;
            const float* tw = a.logits ? a.w_out : a.topk_w;
            w.row_tw[pr] = make_int2(t, tw ? __float_as_int(tw[f]) : 0);
        } else if (f < whi) {
            a.inv_perm[f] = -1;                              // dropped (precondition violation, flagged above)
        }
        __syncwarp();
        if (id >= 0 && lane == __ffs(m) - 1) whist[wp][id] += __popc(m);
        __syncwarp();
    }

    RT_TR(6);
}

// the same front end as a kernel of its own: feeds the fused decode kernel (which re-derives the grouping in every CTA
// and should not redo the top-k there)
__global__ void __launch_bounds__(RT_THREADS) k_router_topk(const float* __restrict__ logits, int T, int E, int k,
                                                            int* __restrict__ ids_out, float* __restrict__ w_out) {
    pdl_launch_dependents();
    pdl_wait();
    const int lane = threadIdx.x & 31;
    for (int t = blockIdx.x * RT_WARPS + (threadIdx.x >> 5); t < T; t += gridDim.x * RT_WARPS)
        warp_router_topk(logits + (size_t)t * E, E, k, lane, ids_out + (size_t)t * k, w_out + (size_t)t * k);
}
cudaError_t launch_router_topk(const float* logits, int T, int E, int k, int* ids_out, float* w_out, cudaStream_t st) {
    int blocks = (T + RT_WARPS - 1) / RT_WARPS;
    if (blocks > 148 * 4) blocks = 148 * 4;
    if (blocks < 1) blocks = 1;
    return launch_pdl(k_router_topk, dim3(blocks), dim3(RT_THREADS), 0, st, logits, T, E, k, ids_out, w_out);
}

cudaError_t launch_route(const RouteArgs& a, const Workspace& ws, DevState* state, cudaStream_t st) {
    RouteWs w{};
    w.poff = ws.poff; w.sched = ws.sched; w.row_flat = ws.row_flat; w.row_tok = ws.row_tok; w.row_tw = ws.row_tw;
    w.bhist = ws.bhist; w.tt = ws.tt; w.chunk = ws.chunk;
    return launch_pdl(k_route, dim3(ws.RB + 1), dim3(RT_THREADS), 0, st, a, w, state);
}

}  // namespace fxm

#ifdef FXM_TRACE
extern "C" int fxm_rtrace_read(void* dst) { return (int)cudaMemcpyFromSymbol(dst, fxm::g_rtrace, sizeof(fxm::g_rtrace)); }
#endif
