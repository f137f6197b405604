// fxm_aux.cu -- the bandwidth-only kernels around the two grouped GEMMs:
//   pack / unpack_prefix (Eq. 3), set_table (Eq. 11), prep (gather x rows into
//   the sorted, padded, swizzled panels + zero the combine accumulator; Alg. 2 l.4-7),
//   finalize (one rounding of y to bf16), read_h (debug).
#include "fxm_internal.cuh"

namespace fxm {

// ---------------------------------------------------------------------------------------------- pack
// one thread per 16-byte chunk of the packed gate/up region
__global__ void k_pack_gu(Dims D, const uint4* __restrict__ Wg, const uint4* __restrict__ Wu,
                          const int* __restrict__ rank, uint4* __restrict__ out, size_t n_chunks) {
    for (size_t g = blockIdx.x * (size_t)blockDim.x + threadIdx.x; g < n_chunks; g += (size_t)gridDim.x * blockDim.x) {
        const uint32_t ch = g & 7, pr = (g >> 3) & 127;
        const size_t tile = g >> 10;
        const int kb = (int)(tile % D.nKB1);
        const int cb = (int)((tile / D.nKB1) % D.nCB);
        const int e = (int)(tile / ((size_t)D.nKB1 * D.nCB));
        const int p = cb * CB + (pr >> 5) * 16 + (pr & 15);     // ranked channel position
        const bool is_up = (pr & 31) >= 16;
        uint4 v = make_uint4(0, 0, 0, 0);
        if (p < D.I) {
            const int c = rank ? rank[(size_t)e * D.I + p] : p;  // ORIGINAL channel index (gather semantics)
            const size_t src = (((size_t)e * D.I + c) * D.d + (size_t)kb * KB + ch * 8) >> 3;
            v = is_up ? Wu[src] : Wg[src];
        }
        out[(tile * WT_BYTES + sw128_chunk(pr, ch)) >> 4] = v;
    }
}

// one thread per 16-byte chunk of the packed down region (8 gathered channels of one output feature)
__global__ void k_pack_dn(Dims D, const uint16_t* __restrict__ Wd, const int* __restrict__ rank,
                          uint4* __restrict__ out, size_t n_chunks) {
    for (size_t g = blockIdx.x * (size_t)blockDim.x + threadIdx.x; g < n_chunks; g += (size_t)gridDim.x * blockDim.x) {
        const uint32_t ch = g & 7, pr = (g >> 3) & 127;
        const size_t tile = g >> 10;
        const int db = (int)(tile % D.nDB);
        const int kb2 = (int)((tile / D.nDB) % D.nCB);
        const int e = (int)(tile / ((size_t)D.nDB * D.nCB));
        const int i = db * WT_ROWS + pr;                         // output feature
        uint16_t h[8];
#pragma unroll
        for (int j = 0; j < 8; ++j) {
            const int p = kb2 * KB + ch * 8 + j;                 // ranked channel position
            uint16_t v = 0;
            if (i < D.d && p < D.I) {
                const int c = rank ? rank[(size_t)e * D.I + p] : p;
                v = Wd[((size_t)e * D.d + i) * D.I + c];
            }
            h[j] = v;
        }
        uint4 v4;
        v4.x = h[0] | ((uint32_t)h[1] << 16);
        v4.y = h[2] | ((uint32_t)h[3] << 16);
        v4.z = h[4] | ((uint32_t)h[5] << 16);
        v4.w = h[6] | ((uint32_t)h[7] << 16);
        out[(tile * WT_BYTES + sw128_chunk(pr, ch)) >> 4] = v4;
    }
}

cudaError_t launch_pack(const Dims& D, const __nv_bfloat16* Wg, const __nv_bfloat16* Wu, const __nv_bfloat16* Wd,
                        const int* rank_dev, uint8_t* packed, cudaStream_t st) {
    const size_t n_gu = gu_bytes(D) >> 4, n_dn = dn_bytes(D) >> 4;
    const int threads = 256;
    const int b_gu = (int)((n_gu + threads - 1) / threads < 148 * 64 ? (n_gu + threads - 1) / threads : 148 * 64);
    const int b_dn = (int)((n_dn + threads - 1) / threads < 148 * 64 ? (n_dn + threads - 1) / threads : 148 * 64);
    k_pack_gu<<<b_gu, threads, 0, st>>>(D, (const uint4*)Wg, (const uint4*)Wu, rank_dev, (uint4*)packed, n_gu);
    k_pack_dn<<<b_dn, threads, 0, st>>>(D, (const uint16_t*)Wd, rank_dev, (uint4*)(packed + gu_bytes(D)), n_dn);
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------- unpack_prefix
__global__ void k_unpack_prefix(Dims D, const uint8_t* __restrict__ packed, int e, int r,
                                uint16_t* __restrict__ Wg, uint16_t* __restrict__ Wu, uint16_t* __restrict__ Wd) {
    const size_t n = (size_t)r * D.d;
    const uint8_t* dn = packed + gu_bytes(D);
    for (size_t g = blockIdx.x * (size_t)blockDim.x + threadIdx.x; g < n; g += (size_t)gridDim.x * blockDim.x) {
        {   // gate / up element (p, i)
            const int p = (int)(g / D.d), i = (int)(g % D.d);
            const int cb = p / CB, w = p % CB;
            const uint32_t pr_g = (w / 16) * 32 + (w % 16);
            const uint8_t* t = packed + gu_tile_index(D, e, cb, i / KB) * WT_BYTES;
            Wg[g] = *(const uint16_t*)(t + sw128_off(pr_g, i % KB));
            Wu[g] = *(const uint16_t*)(t + sw128_off(pr_g + 16, i % KB));
        }
        {   // down element (i, p), output row-major [d][r]
            const int i = (int)(g / r), p = (int)(g % r);
            const uint8_t* t = dn + dn_tile_index(D, e, p / KB, i / WT_ROWS) * WT_BYTES;
            Wd[g] = *(const uint16_t*)(t + sw128_off(i % WT_ROWS, p % KB));
        }
    }
}

cudaError_t launch_unpack_prefix(const Dims& D, const uint8_t* packed, int e, int r, __nv_bfloat16* Wg,
                                 __nv_bfloat16* Wu, __nv_bfloat16* Wd, cudaStream_t st) {
    if (r == 0) return cudaSuccess;
    const size_t n = (size_t)r * D.d;
    const int blocks = (int)((n + 255) / 256 < 148 * 32 ? (n + 255) / 256 : 148 * 32);
    k_unpack_prefix<<<blocks, 256, 0, st>>>(D, packed, e, r, (uint16_t*)Wg, (uint16_t*)Wu, (uint16_t*)Wd);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------ set_table
struct TableArg { int r[MAX_E]; };
__global__ void k_set_table(int* __restrict__ dst, TableArg t, int E) {
    const int e = threadIdx.x;
    if (e < MAX_E) dst[e] = e < E ? t.r[e] : 0;
}
cudaError_t launch_set_table(int* table_dev, const int* r_host, int E, cudaStream_t st) {
    TableArg t;
    for (int e = 0; e < MAX_E; ++e) t.r[e] = e < E ? r_host[e] : 0;
    k_set_table<<<1, MAX_E, 0, st>>>(table_dev, t, E);
    return cudaGetLastError();
}

// ----------------------------------------------------------------------------------------------- prep
// One warp per padded row p: copy x[token(p)] (d bf16) into the swizzled panels Xs[kb][p][.]; padding rows
// become zeros so no garbage ever reaches a tensor core.  The same grid zeroes the fp32 accumulator.
__global__ void k_prep(Dims D, const uint4* __restrict__ x, int T, int k, const int* __restrict__ row_flat,
                       const Sched* __restrict__ sched, uint8_t* __restrict__ Xs, int P, float4* __restrict__ yacc) {
    const int lane = threadIdx.x & 31;
    const int warps_per_block = blockDim.x >> 5;
    const int gw = blockIdx.x * warps_per_block + (threadIdx.x >> 5);
    const int nw = gridDim.x * warps_per_block;
    const int P_used = sched->P_used;
    const int chunks_per_row = D.d >> 3;                       // 16-byte chunks in an x row
    for (int p = gw; p < P_used; p += nw) {
        const int f = row_flat[p];
        const uint4* src = f >= 0 ? x + (size_t)(f / k) * chunks_per_row : nullptr;
        for (int c = lane; c < chunks_per_row; c += 32) {
            const uint4 v = src ? src[c] : make_uint4(0, 0, 0, 0);
            const int kb = c >> 3, ch = c & 7;
            *(uint4*)(Xs + ((size_t)kb * P + p) * ROW_BYTES + (((ch ^ p) & 7) << 4)) = v;
        }
    }
    const size_t n4 = (size_t)T * D.d / 4;
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x)
        yacc[i] = make_float4(0.f, 0.f, 0.f, 0.f);
}

cudaError_t launch_prep(const Dims& D, const __nv_bfloat16* x, int T, int k, const Workspace& ws, cudaStream_t st) {
    const int threads = 256;
    size_t want = ((size_t)T * k + 7) / 8;
    const size_t zero_blocks = ((size_t)T * D.d / 4 + threads * 4 - 1) / (threads * 4);
    if (zero_blocks > want) want = zero_blocks;
    int blocks = (int)(want < 148 * 8 ? want : 148 * 8);
    if (blocks < 1) blocks = 1;
    k_prep<<<blocks, threads, 0, st>>>(D, (const uint4*)x, T, k, ws.row_flat, ws.sched, ws.Xs, ws.P, (float4*)ws.yacc);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------- finalize
__global__ void k_finalize(const float4* __restrict__ yacc, uint2* __restrict__ y, size_t n4) {
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n4; i += (size_t)gridDim.x * blockDim.x) {
        const float4 v = yacc[i];
        __nv_bfloat162 a = __floats2bfloat162_rn(v.x, v.y), b = __floats2bfloat162_rn(v.z, v.w);
        uint2 o;
        o.x = *(uint32_t*)&a;
        o.y = *(uint32_t*)&b;
        y[i] = o;
    }
}
cudaError_t launch_finalize(const Dims& D, int T, const Workspace& ws, __nv_bfloat16* y, cudaStream_t st) {
    const size_t n4 = (size_t)T * D.d / 4;
    if (n4 == 0) return cudaSuccess;
    const int blocks = (int)((n4 + 255) / 256 < 148 * 16 ? (n4 + 255) / 256 : 148 * 16);
    k_finalize<<<blocks, 256, 0, st>>>((const float4*)ws.yacc, (uint2*)y, n4);
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------------- read_h
// H_out[s][c] for sorted position s (perm order) and channel c < I, from the swizzled panels.
__global__ void k_read_h(Dims D, int k, const int* __restrict__ ids, const int* __restrict__ r_table,
                         const int* __restrict__ inv_perm, const int* __restrict__ row_flat,
                         const Sched* __restrict__ sched, const uint8_t* __restrict__ H, int P,
                         uint16_t* __restrict__ out) {
    const int P_used = sched->P_used;
    const size_t n = (size_t)P_used * D.I;
    for (size_t g = blockIdx.x * (size_t)blockDim.x + threadIdx.x; g < n; g += (size_t)gridDim.x * blockDim.x) {
        const int p = (int)(g / D.I), c = (int)(g % D.I);
        const int f = row_flat[p];
        if (f < 0) continue;
        const int s = inv_perm[f];
        const uint8_t* row = H + ((size_t)(c / CB) * P + p) * ROW_BYTES;
        const uint16_t v = *(const uint16_t*)(row + ((((c % CB) >> 3) ^ p) & 7) * 16 + ((c & 7) << 1));
        out[(size_t)s * D.I + c] = c < r_table[ids[f]] ? v : (uint16_t)0;   // pruned tiles are never written
    }
    (void)k;
}
cudaError_t launch_read_h(const Dims& D, int T, int k, const int* ids, const int* r_table, const Workspace& ws,
                          __nv_bfloat16* H_out, cudaStream_t st) {
    (void)T;
    k_read_h<<<148 * 8, 256, 0, st>>>(D, k, ids, r_table, ws.inv_perm, ws.row_flat, ws.sched, ws.H, ws.P,
                                      (uint16_t*)H_out);
    return cudaGetLastError();
}

}  // namespace fxm
