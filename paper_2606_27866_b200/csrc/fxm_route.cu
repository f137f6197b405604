// fxm_route.cu -- step a2/a3: router-output grouping (stable per-expert counting sort, bit-exact indices),
// the device-side tile schedule that skips pruned work, and the gather of token rows into sorted panels.
//   Alg. 2 l.4-6: "(pi, eid) <- Sort(eid)", read as the STABLE sort by (expert id, flat
//   index f = t*k+j) so that exactly one permutation is correct (reading R5).
//   Alg. 2 l.2-3, 8-11: BucketByRetI / AlignUp / view lists are replaced by a tile list
//   computed here from counts[] and the CURRENT width table r[]: only tiles with channel index < r_e and
//   token row < n_e exist.
//   Alg. 2 l.7: X[pi] -- the gather of routed token rows into sorted panels.
//
// Three launches, no atomics decide any position (hence deterministic and stable):
//   k_route_plan     grid = RB blocks.  Block b histograms the flat assignments [b*chunk, (b+1)*chunk) per
//                    expert.  The LAST block to publish (ticket counter) turns the RB x E histogram into
//                    exclusive bases over blocks and writes counts, offsets, padded offsets, the token tiles
//                    and the GEMM-1 work items for the current width table.
//   k_scatter        grid = RB blocks.  Block b ranks its assignments: base over blocks + base over the
//                    warps of the block + __match_any_sync rank inside a 32-wide step ("earlier block, earlier
//                    warp, earlier step, lower lane" == "lower flat index"), writes perm / inv_perm / row_flat
//                    / prow.
//   k_gather         full grid, one warp per padded row: x rows -> swizzled K-major panels Xs.
#include "fxm_internal.cuh"

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

// balanced split of np padded rows into nt tiles: rows per tile, a multiple of 16
__device__ __forceinline__ int per_rows(int np, int nt) { return ((np + nt - 1) / nt + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN; }

// per-warp histogram of the block's chunk; warp w owns the contiguous sub-range [wlo, whi)
__device__ __forceinline__ bool block_histogram(const int* __restrict__ ids, int E, int wlo, int whi, int lane,
                                                int* __restrict__ wh /* this warp's [MAX_E] row */) {
    bool bad = false;
    for (int base = wlo; base < whi; base += 32) {
        const int f = base + lane;
        int id = f < whi ? ids[f] : -1;
        if (f < whi && (id < 0 || id >= E)) { bad = true; id = -1; }
        const unsigned m = __match_any_sync(0xffffffffu, id);
        if (id >= 0 && lane == __ffs(m) - 1) wh[id] += __popc(m);
        __syncwarp();
    }
    return bad;
}

__global__ void __launch_bounds__(RT_THREADS)
k_route_plan(Dims D, const int* __restrict__ ids, int A, int chunk, const int* __restrict__ r_table, int tile_n, int grp,
             int* __restrict__ counts, int* __restrict__ offsets, int* __restrict__ bhist, int* __restrict__ poff,
             int4* __restrict__ tt, int4* __restrict__ items1, Sched* __restrict__ sched,
             DevState* __restrict__ state) {
    __shared__ int whist[RT_WARPS][MAX_E];
    __shared__ int s_cnt[MAX_E], s_off[MAX_E + 1], s_poff[MAX_E + 1];
    __shared__ int s_ntt, s_last;
    const int E = D.E;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    pdl_launch_dependents();
    for (int i = tid; i < RT_WARPS * MAX_E; i += RT_THREADS) (&whist[0][0])[i] = 0;
    __syncthreads();
    pdl_wait();                                                  // the previous call's kernels may still read the workspace
    const int lo = min(A, blockIdx.x * chunk), hi = min(A, lo + chunk);
    const int sub = chunk / RT_WARPS;
    const int wlo = min(hi, lo + w * sub), whi = min(hi, wlo + sub);
    if (block_histogram(ids, E, wlo, whi, lane, whist[w])) atomicOr(&state->flags, 1u);
    __syncthreads();
    for (int e = tid; e < E; e += RT_THREADS) {
        int c = 0;
#pragma unroll
        for (int ww = 0; ww < RT_WARPS; ++ww) c += whist[ww][e];
        bhist[(size_t)blockIdx.x * E + e] = c;
    }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = (atomicAdd(&state->ticket, 1u) == gridDim.x - 1);
    __syncthreads();
    if (!s_last) return;
    __threadfence();

    // ---- last block: exclusive scan over blocks, per expert.  Thread (e, s) owns rows [s*L, (s+1)*L) of column e:
    //      pass 1 sums them, the S segment sums are scanned through shared memory, pass 2 writes the prefixes.
    const int RB = gridDim.x;
    const int S = RT_THREADS / E > 0 ? RT_THREADS / E : 1;     // E <= 256 = RT_THREADS
    const int L = (RB + S - 1) / S;
    int* seg = &whist[0][0];                                     // [S][E] <= 256 ints, histogram rows are dead now
    const int e0 = tid % E, s0 = tid / E;
    const int b_lo = min(RB, s0 * L), b_hi = s0 < S ? min(RB, b_lo + L) : b_lo;
    {
        int sum = 0;
        int b = b_lo;
        for (; b + 8 <= b_hi; b += 8) {
            int c[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) c[u] = __ldcg(bhist + (size_t)(b + u) * E + e0);
#pragma unroll
            for (int u = 0; u < 8; ++u) sum += c[u];
        }
        for (; b < b_hi; ++b) sum += __ldcg(bhist + (size_t)b * E + e0);
        __syncthreads();                                         // everyone is done reading whist
        if (s0 < S) seg[s0 * E + e0] = sum;
    }
    __syncthreads();
    {
        int run = 0;
        for (int ss = 0; ss < s0 && ss < S; ++ss) run += seg[ss * E + e0];
        if (s0 == S - 1) {                                       // the last segment also knows the column total
            const int tot = run + seg[s0 * E + e0];
            s_cnt[e0] = tot;
            counts[e0] = tot;
        }
        int b = b_lo;
        for (; b + 8 <= b_hi; b += 8) {
            int c[8];
#pragma unroll
            for (int u = 0; u < 8; ++u) c[u] = __ldcg(bhist + (size_t)(b + u) * E + e0);
#pragma unroll
            for (int u = 0; u < 8; ++u) { bhist[(size_t)(b + u) * E + e0] = run; run += c[u]; }
        }
        for (; b < b_hi; ++b) {
            const int c = __ldcg(bhist + (size_t)b * E + e0);
            bhist[(size_t)b * E + e0] = run;
            run += c;
        }
    }
    __syncthreads();

    // ---- warp 0: scans over experts -> offsets, padded offsets, token tiles, work prefixes
    if (w == 0) {
        int c_off = 0, c_poff = 0, c_tiles = 0, c_work = 0, c_max = ROW_ALIGN;
        for (int base = 0; base < E; base += 32) {
            const int e = base + lane;
            const int n = e < E ? s_cnt[e] : 0;
            const int r = e < E ? (r_table ? r_table[e] : D.I) : 0;   // no table yet (fxm_route only): full width
            const int np = (n + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN;
            const int nt = (n > 0 && r > 0) ? (np + tile_n - 1) / tile_n : 0;   // pruned-away / idle experts: no tiles
            const int nb = ((r + CB - 1) / CB + grp - 1) / grp;                 // GEMM-1 items per token tile
            const int i_off = warp_incl_scan(n, lane), i_poff = warp_incl_scan(np, lane);
            const int i_tiles = warp_incl_scan(nt, lane), i_work = warp_incl_scan(nt * nb, lane);
            if (e < E) {
                s_off[e] = c_off + i_off - n;
                s_poff[e] = c_poff + i_poff - np;
                int j = c_tiles + i_tiles - nt, wk = c_work + i_work - nt * nb;
                const int p0 = c_poff + i_poff - np;
                // balanced split of the padded segment into nt tiles of <= tile_n rows, each a multiple of 16 rows
                const int per = nt > 0 ? per_rows(np, nt) : 0;
                for (int row = 0; row < np && nt > 0; row += per, ++j, wk += nb)
                    tt[j] = make_int4(e, p0 + row, min(per, n - row), wk);      // .z = valid rows of the tile (>= 1)
            }
            {
                int mx = nt > 0 ? min(per_rows(np, nt), np) : 0;          // rows of this expert's widest tile
#pragma unroll
                for (int o = 16; o; o >>= 1) mx = max(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                c_max = max(c_max, mx);
            }
            c_off += __shfl_sync(0xffffffffu, i_off, 31);
            c_poff += __shfl_sync(0xffffffffu, i_poff, 31);
            c_tiles += __shfl_sync(0xffffffffu, i_tiles, 31);
            c_work += __shfl_sync(0xffffffffu, i_work, 31);
        }
        if (lane == 0) {
            s_off[E] = c_off;
            s_poff[E] = c_poff;
            s_ntt = c_tiles;
            sched->ntt = c_tiles;
            sched->W1 = c_work;
            sched->W2 = c_tiles * ((D.nDB + grp - 1) / grp);
            sched->P_used = c_poff;
            sched->A = A;
            sched->max_n = c_max;
            state->ticket = 0;                               // ready for the next call on this layer
        }
    }
    __syncthreads();
    for (int e = tid; e <= E; e += RT_THREADS) { offsets[e] = s_off[e]; poff[e] = s_poff[e]; }
    // GEMM-1 work items: one per (token tile, RETAINED channel block) -- pruned blocks are never listed
    for (int j = tid; j < s_ntt; j += RT_THREADS) {
        const int4 t = tt[j];
        const int nb = (((r_table ? r_table[t.x] : D.I) + CB - 1) / CB + grp - 1) / grp;
        for (int cb = 0; cb < nb; ++cb) items1[t.w + cb] = make_int4(t.x, t.y, t.z, cb);
    }
}

// copy one x row (d bf16) into the swizzled panels Xs[kb][p][.]; src == nullptr writes zeros
__device__ __forceinline__ void put_row(const uint4* __restrict__ src, uint8_t* __restrict__ Xs, int P, int p,
                                        int chunks_per_row, int lane) {
    for (int c0 = lane; c0 < chunks_per_row; c0 += 128) {
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int c = c0 + 32 * u;
            v[u] = (src && c < chunks_per_row) ? __ldg(src + c) : make_uint4(0, 0, 0, 0);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int c = c0 + 32 * u;
            if (c < chunks_per_row)
                *(uint4*)(Xs + ((size_t)(c >> 3) * P + p) * ROW_BYTES + ((((c & 7) ^ p) & 7) << 4)) = v[u];
        }
    }
}

__global__ void __launch_bounds__(RT_THREADS)
k_scatter(Dims D, const int* __restrict__ ids, int A, int chunk, const int* __restrict__ r_table,
          const int* __restrict__ counts, const int* __restrict__ offsets, const int* __restrict__ poff,
          const int* __restrict__ bbase, int* __restrict__ perm, int* __restrict__ inv_perm,
          int* __restrict__ row_flat, int* __restrict__ prow, int* __restrict__ row_tok, int k) {
    __shared__ int whist[RT_WARPS][MAX_E];      // per-warp histogram, then per-warp running base
    const int E = D.E;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    pdl_launch_dependents();
    for (int i = tid; i < RT_WARPS * MAX_E; i += RT_THREADS) (&whist[0][0])[i] = 0;
    __syncthreads();
    pdl_wait();
    const int lo = min(A, blockIdx.x * chunk), hi = min(A, lo + chunk);
    const int sub = chunk / RT_WARPS;
    const int wlo = min(hi, lo + w * sub), whi = min(hi, wlo + sub);
    block_histogram(ids, E, wlo, whi, lane, whist[w]);
    __syncthreads();
    for (int e = tid; e < E; e += RT_THREADS) {      // exclusive scan over the warps of this block, on top of the block base
        int run = bbase[(size_t)blockIdx.x * E + e];
#pragma unroll
        for (int ww = 0; ww < RT_WARPS; ++ww) {
            const int c = whist[ww][e];
            whist[ww][e] = run;
            run += c;
        }
    }
    __syncthreads();

    // ---- stable scatter
    for (int base = wlo; base < whi; base += 32) {
        const int f = base + lane;
        int id = f < whi ? ids[f] : -1;
        if (id < 0 || id >= E) id = -1;
        const unsigned m = __match_any_sync(0xffffffffu, id);
        if (id >= 0) {
            const int rank = whist[w][id] + __popc(m & ((1u << lane) - 1u));
            const int pos = offsets[id] + rank;
            const int pr = poff[id] + rank;
            perm[pos] = f;
            inv_perm[f] = pos;
            row_flat[pr] = f;
            row_tok[pr] = f / k;
            prow[f] = (!r_table || r_table[id] > 0) ? pr : -1;   // width-0 experts get no tiles: nothing to read back
        } else if (f < whi) {
            inv_perm[f] = -1;                                // dropped (precondition violation, flagged by the plan kernel)
            prow[f] = -1;
        }
        __syncwarp();
        if (id >= 0 && lane == __ffs(m) - 1) whist[w][id] += __popc(m);
        __syncwarp();
    }

    // ---- padding rows of the expert segments carry no assignment
    for (int e = blockIdx.x * RT_THREADS + tid; e < E; e += gridDim.x * RT_THREADS)
        for (int p = poff[e] + counts[e]; p < poff[e + 1]; ++p) { row_flat[p] = -1; row_tok[p] = 0; }
}

// Alg. 2 l.7, X[pi]: one warp per padded row p copies x[token(p)] into the swizzled panels; padding
// rows become zeros so no garbage ever reaches a tensor core.
__global__ void __launch_bounds__(256)
k_gather(Dims D, const uint4* __restrict__ x, int k, const int* __restrict__ row_flat, const Sched* __restrict__ sched,
         uint8_t* __restrict__ Xs, int P) {
    const int lane = threadIdx.x & 31;
    const int gw = blockIdx.x * 8 + (threadIdx.x >> 5), nw = gridDim.x * 8;
    pdl_launch_dependents();
    pdl_wait();
    const int P_used = sched->P_used;
    const int chunks_per_row = D.d >> 3;
    for (int p = gw; p < P_used; p += nw) {
        const int f = row_flat[p];
        put_row(f >= 0 ? x + (size_t)(f / k) * chunks_per_row : nullptr, Xs, P, p, chunks_per_row, lane);
    }
}

cudaError_t launch_route_plan(const Dims& D, const int* ids, int T, int k, const int* r_table, int tile_n, int grp,
                              int* counts, int* offsets, const Workspace& ws, DevState* state, cudaStream_t st) {
    return launch_pdl(k_route_plan, dim3(ws.RB), dim3(RT_THREADS), 0, st, D, ids, T * k, ws.chunk, r_table, tile_n, grp, counts,
                      offsets, ws.bhist, ws.poff, ws.tt, ws.items1, ws.sched, state);
}

cudaError_t launch_scatter(const Dims& D, const int* ids, int T, int k, const int* r_table, const int* counts,
                           const int* offsets, int* perm, int* inv_perm, const Workspace& ws, cudaStream_t st) {
    return launch_pdl(k_scatter, dim3(ws.RB), dim3(RT_THREADS), 0, st, D, ids, T * k, ws.chunk, r_table, counts, offsets,
                      (const int*)ws.poff, (const int*)ws.bhist, perm, inv_perm, ws.row_flat, ws.prow, ws.row_tok, k);
}

cudaError_t launch_gather(const Dims& D, const __nv_bfloat16* x, int T, int k, const Workspace& ws, cudaStream_t st) {
    const long long rows = (long long)T * k + (long long)D.E * (ROW_ALIGN - 1);
    long long blocks = (rows + 7) / 8;
    if (blocks > 148 * 8) blocks = 148 * 8;
    if (blocks < 1) blocks = 1;
    return launch_pdl(k_gather, dim3((unsigned)blocks), dim3(256), 0, st, D, (const uint4*)x, k, (const int*)ws.row_flat,
                      (const Sched*)ws.sched, ws.Xs, ws.P);
}

}  // namespace fxm
