// fxm_route.cu -- step a2/a3: router-output grouping (stable per-expert counting sort, bit-exact indices)
// and the device-side tile schedule that skips pruned work.
//   Alg. 2 l.4-6: "(pi, eid) <- Sort(eid)", read as the STABLE sort by (expert id, flat
//   index f = t*k+j) so that exactly one permutation is correct (reading R5).
//   Alg. 2 l.2-3, 8-11: BucketByRetI / AlignUp / view lists are replaced by a tile list
//   computed here from counts[] and the CURRENT width table r[]: only tiles with channel index < r_e and
//   token row < n_e exist.
//
// One CTA of 32 warps.  Warp w owns the contiguous slice [w*chunk, (w+1)*chunk) of the flat assignment
// array, so "earlier warp, earlier step, lower lane" is exactly "lower flat index": ranks are assigned with
// __match_any_sync inside a step, a running per-warp counter across steps, and an exclusive scan over warps
// -- no atomics, hence a deterministic, stable result.
#include "fxm_internal.cuh"

namespace fxm {

constexpr int RT_WARPS = 32;
constexpr int RT_BATCH = 8;       // independent id loads in flight per lane

__device__ __forceinline__ int warp_incl_scan(int v, int lane) {
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, v, o);
        if (lane >= o) v += t;
    }
    return v;
}

__global__ void __launch_bounds__(RT_WARPS * 32, 1)
k_route(Dims D, const int* __restrict__ ids, int A, const int* __restrict__ r_table, int tile_n,
        int* __restrict__ counts, int* __restrict__ offsets, int* __restrict__ perm, int* __restrict__ inv_perm,
        int* __restrict__ poff, int* __restrict__ row_flat, int4* __restrict__ tt, int4* __restrict__ items1,
        Sched* __restrict__ sched, DevState* __restrict__ state) {
    __shared__ int whist[RT_WARPS][MAX_E];      // per-warp histogram, then per-warp running base
    __shared__ int s_cnt[MAX_E], s_off[MAX_E + 1], s_poff[MAX_E + 1];
    __shared__ int s_ntt;
    const int E = D.E;
    const int tid = threadIdx.x, lane = tid & 31, w = tid >> 5;
    for (int i = tid; i < RT_WARPS * MAX_E; i += blockDim.x) (&whist[0][0])[i] = 0;
    __syncthreads();

    int chunk = (A + RT_WARPS - 1) / RT_WARPS;
    chunk = (chunk + 31) & ~31;
    const int lo = min(A, w * chunk), hi = min(A, lo + chunk);
    bool bad = false;

    // ---- pass 1: per-warp histogram
    for (int base = lo; base < hi; base += 32 * RT_BATCH) {
        int idv[RT_BATCH];
#pragma unroll
        for (int b = 0; b < RT_BATCH; ++b) {
            const int f = base + b * 32 + lane;
            idv[b] = f < hi ? ids[f] : -1;
        }
#pragma unroll
        for (int b = 0; b < RT_BATCH; ++b) {
            if (base + b * 32 >= hi) break;                 // warp-uniform
            int id = idv[b];
            const bool in_range = base + b * 32 + lane < hi;
            if (in_range && (id < 0 || id >= E)) { bad = true; id = -1; }
            const unsigned m = __match_any_sync(0xffffffffu, id);
            if (id >= 0 && lane == __ffs(m) - 1) whist[w][id] += __popc(m);
            __syncwarp();
        }
    }
    if (bad) atomicOr(&state->flags, 1u);
    __syncthreads();

    // ---- exclusive scan over warps (per expert)
    if (tid < E) {
        int run = 0;
#pragma unroll 4
        for (int ww = 0; ww < RT_WARPS; ++ww) {
            const int c = whist[ww][tid];
            whist[ww][tid] = run;
            run += c;
        }
        s_cnt[tid] = run;
        counts[tid] = run;
    }
    __syncthreads();

    // ---- warp 0: scans over experts -> offsets, padded offsets, token tiles, work prefixes
    if (w == 0) {
        int c_off = 0, c_poff = 0, c_tiles = 0, c_work = 0;
        for (int base = 0; base < E; base += 32) {
            const int e = base + lane;
            const int n = e < E ? s_cnt[e] : 0;
            const int r = e < E ? (r_table ? r_table[e] : D.I) : 0;   // no table yet (fxm_route only): full width
            const int np = (n + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN;
            const int nt = (n > 0 && r > 0) ? (n + tile_n - 1) / tile_n : 0;   // pruned-away / idle experts: no tiles
            const int nb = (r + CB - 1) / CB;
            const int i_off = warp_incl_scan(n, lane), i_poff = warp_incl_scan(np, lane);
            const int i_tiles = warp_incl_scan(nt, lane), i_work = warp_incl_scan(nt * nb, lane);
            if (e < E) {
                s_off[e] = c_off + i_off - n;
                s_poff[e] = c_poff + i_poff - np;
                int j = c_tiles + i_tiles - nt, wk = c_work + i_work - nt * nb;
                const int p0 = c_poff + i_poff - np;
                for (int row = 0; row < n && nt > 0; row += tile_n, ++j, wk += nb)
                    tt[j] = make_int4(e, p0 + row, min(tile_n, n - row), wk);
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
            sched->W2 = c_tiles * D.nDB;
            sched->P_used = c_poff;
            sched->A = A;
        }
    }
    __syncthreads();
    if (tid <= E) { offsets[tid] = s_off[tid]; poff[tid] = s_poff[tid]; }
    if (tid < E)                                              // padding rows of each segment
        for (int p = s_poff[tid] + s_cnt[tid]; p < s_poff[tid + 1]; ++p) row_flat[p] = -1;
    // GEMM-1 work items: one per (token tile, RETAINED channel block) -- pruned blocks are never listed
    for (int j = tid; j < s_ntt; j += blockDim.x) {
        const int4 t = tt[j];
        const int nb = ((r_table ? r_table[t.x] : D.I) + CB - 1) / CB;
        for (int cb = 0; cb < nb; ++cb) items1[t.w + cb] = make_int4(t.x, t.y, t.z, cb);
    }

    // ---- pass 2: stable scatter
    for (int base = lo; base < hi; base += 32 * RT_BATCH) {
        int idv[RT_BATCH];
#pragma unroll
        for (int b = 0; b < RT_BATCH; ++b) {
            const int f = base + b * 32 + lane;
            idv[b] = f < hi ? ids[f] : -1;
        }
#pragma unroll
        for (int b = 0; b < RT_BATCH; ++b) {
            if (base + b * 32 >= hi) break;
            const int f = base + b * 32 + lane;
            int id = idv[b];
            if (id < 0 || id >= E) id = -1;
            const unsigned m = __match_any_sync(0xffffffffu, id);
            if (id >= 0) {
                const int rank = whist[w][id] + __popc(m & ((1u << lane) - 1u));
                const int pos = s_off[id] + rank;
                perm[pos] = f;
                inv_perm[f] = pos;
                row_flat[s_poff[id] + rank] = f;
            } else if (f < hi) {
                inv_perm[f] = -1;                            // dropped (precondition violation)
            }
            __syncwarp();
            if (id >= 0 && lane == __ffs(m) - 1) whist[w][id] += __popc(m);
            __syncwarp();
        }
    }
}

cudaError_t launch_route(const Dims& D, const int* ids, int T, int k, const int* r_table, int tile_n, int* counts,
                         int* offsets, int* perm, int* inv_perm, const Workspace& ws, DevState* state,
                         cudaStream_t st) {
    k_route<<<1, RT_WARPS * 32, 0, st>>>(D, ids, T * k, r_table, tile_n, counts, offsets, perm, inv_perm, ws.poff,
                                         ws.row_flat, ws.tt, ws.items1, ws.sched, state);
    return cudaGetLastError();
}

}  // namespace fxm
