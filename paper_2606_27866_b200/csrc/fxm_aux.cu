// fxm_aux.cu -- the bandwidth-only kernels around the two grouped GEMMs:
//   pack / unpack_prefix (Eq. 3), set_table (Eq. 11), combine (router-weighted sum of
//   each token's k expert outputs, one rounding of y to bf16; Alg. 2 l.19-20), read_h (debug).
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

// -------------------------------------------------------------------------------------------- combine
// Alg. 2 l.19-20: Y[token] += alpha * Z_down, done as a GATHER so that no atomics are needed and
// the sum runs in slot order j = 0..k-1 in fp32 with exactly one rounding of y (readings R8, R11):
//   y[t][i] = sum_j topk_w[t][j] * O[prow[t*k+j]][i]
// One block per token; a thread owns 8 consecutive output features (16 bytes of each O row).
__global__ void __launch_bounds__(128) k_combine(Dims D, int k, const int* __restrict__ prow,
                                                 const float* __restrict__ topk_w, const uint8_t* __restrict__ O,
                                                 int P, uint4* __restrict__ y) {
    __shared__ int s_p[MAX_K];
    __shared__ float s_w[MAX_K];
    const int t = blockIdx.x;
    pdl_launch_dependents();
    pdl_wait();
    if (threadIdx.x < k) {
        s_p[threadIdx.x] = prow[(size_t)t * k + threadIdx.x];
        s_w[threadIdx.x] = topk_w[(size_t)t * k + threadIdx.x];
    }
    __syncthreads();
    const int chunks = D.d >> 3;
    const size_t orow = 2 * WT_ROWS;                              // bytes per row of an O panel
    for (int c = threadIdx.x; c < chunks; c += blockDim.x) {
        const uint8_t* col = O + (size_t)(c >> 4) * P * orow + ((size_t)(c & 15) << 4);   // panel c/16, 16-byte chunk c%16
        float acc[8];
#pragma unroll
        for (int q = 0; q < 8; ++q) acc[q] = 0.f;
        for (int j0 = 0; j0 < k; j0 += 4) {
            uint4 v[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                const int p = j0 + u < k ? s_p[j0 + u] : -1;
                v[u] = p >= 0 ? __ldg((const uint4*)(col + (size_t)p * orow)) : make_uint4(0, 0, 0, 0);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                if (j0 + u >= k) break;
                const float wj = s_w[j0 + u];
                const uint32_t h[4] = {v[u].x, v[u].y, v[u].z, v[u].w};
#pragma unroll
                for (int q = 0; q < 4; ++q) {
                    acc[2 * q] += wj * __uint_as_float(h[q] << 16);
                    acc[2 * q + 1] += wj * __uint_as_float(h[q] & 0xFFFF0000u);
                }
            }
        }
        uint4 o;
        __nv_bfloat162 b0 = __floats2bfloat162_rn(acc[0], acc[1]), b1 = __floats2bfloat162_rn(acc[2], acc[3]);
        __nv_bfloat162 b2 = __floats2bfloat162_rn(acc[4], acc[5]), b3 = __floats2bfloat162_rn(acc[6], acc[7]);
        o.x = *(uint32_t*)&b0; o.y = *(uint32_t*)&b1; o.z = *(uint32_t*)&b2; o.w = *(uint32_t*)&b3;
        y[(size_t)t * chunks + c] = o;
    }
}
cudaError_t launch_combine(const Dims& D, int T, int k, const float* topk_w, const Workspace& ws, __nv_bfloat16* y,
                           cudaStream_t st) {
    if (T == 0) return cudaSuccess;
    return launch_pdl(k_combine, dim3(T), dim3(128), 0, st, D, k, (const int*)ws.prow, topk_w, (const uint8_t*)ws.O, ws.P, (uint4*)y);
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
