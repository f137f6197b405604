// fxm_aux.cu -- the bandwidth-only kernels around the two grouped GEMMs:
//   pack / unpack_prefix (Eq. 3), export_clipped (offline clipping), set_table (Eq. 11,
//   PAPER.md:129), finalize (the single rounding of y: fp32 accumulator -> bf16, optional shared-expert add), read_h (debug).
#include "fxm_internal.cuh"

namespace fxm {

// ---------------------------------------------------------------------------------------------- pack
// one thread per 16-byte chunk of the packed gate/up region (full layer: expert e starts at channel block e * nCB), four
// chunks per step: rank entry -> weight chunk is a dependent chain, so the four chains are issued side by side
__global__ void k_pack_gu(Dims D, const uint4* __restrict__ Wg, const uint4* __restrict__ Wu,
                          const int* __restrict__ rank, uint4* __restrict__ out, size_t n_chunks) {
    const size_t stride = (size_t)gridDim.x * blockDim.x;
    for (size_t g0 = blockIdx.x * (size_t)blockDim.x + threadIdx.x; g0 < n_chunks; g0 += 4 * stride) {
        const uint4* src[4];
        size_t dst[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const size_t g = g0 + u * stride;
            src[u] = nullptr;
            dst[u] = 0;
            if (g >= n_chunks) continue;
            const uint32_t ch = g & 7, pr = (g >> 3) & 127;
            const size_t tile = g >> 10;
            const int kb = (int)(tile % D.nKB1);
            const int cb = (int)((tile / D.nKB1) % D.nCB);
            const int e = (int)(tile / ((size_t)D.nKB1 * D.nCB));
            const int p = cb * CB + (pr >> 5) * 16 + (pr & 15);     // ranked channel position
            const bool is_up = (pr & 31) >= 16;
            dst[u] = (tile * WT_BYTES + sw128_chunk(pr, ch)) >> 4;
            if (p < D.I) {
                const int c = rank ? __ldg(rank + (size_t)e * D.I + p) : p;  // ORIGINAL channel index (gather semantics)
                src[u] = (is_up ? Wu : Wg) + ((((size_t)e * D.I + c) * D.d + (size_t)kb * KB + ch * 8) >> 3);
            }
        }
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) v[u] = src[u] ? __ldcs(src[u]) : make_uint4(0, 0, 0, 0);
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (g0 + u * stride < n_chunks) __stcs(out + dst[u], v[u]);
    }
}

// Fallback of k_pack_dn_rows (W_down not 16-byte aligned, or one row larger than the shared-memory budget):
// one thread per 16-byte chunk of the packed down region (8 gathered channels of one output feature), 2-byte global gathers
__global__ void k_pack_dn_gather(Dims D, const uint16_t* __restrict__ Wd, const int* __restrict__ rank,
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

// The packed down region the fast way.  W~down = W_down P^T permutes COLUMNS, so gathering from global memory pulls a
// 32-byte sector per 2-byte element.  Instead block (e, group of `rpb` output features) stages its rows of W_down[e] in
// shared memory with coalesced 16-byte loads (each byte of W_down is read from HBM exactly once), gathers the ranked
// columns from there, and writes its 128-byte rows of every k-block tile: consecutive threads write consecutive 16-byte
// chunks (the SW128 permutation stays inside a 128-byte row), rpb x 128 contiguous bytes per tile.  rpb divides the
// 128-row tile; rows >= d (padded feature block) and channels >= I (padded channel block) are zeros, as in the gather version.
constexpr int PACK_DN_SMEM = 160 * 1024;
__global__ void __launch_bounds__(256) k_pack_dn_rows(Dims D, const uint16_t* __restrict__ Wd, const int* __restrict__ rank,
                                                      uint4* __restrict__ out, int rpb) {
    extern __shared__ __align__(16) uint8_t pack_smem[];
    uint16_t* srow = (uint16_t*)pack_smem;                        // [rpb][I]
    const int groups = D.nDB * WT_ROWS / rpb;
    const int e = blockIdx.x / groups, i0 = (blockIdx.x % groups) * rpb;   // first (padded) output feature of the block
    const int cpr = D.I >> 3;                                    // 16-byte chunks per row (I % 16 == 0)
    const int n_stage = rpb * cpr;
    for (int q0 = threadIdx.x; q0 < n_stage; q0 += 256 * 4) {    // four loads in flight per thread
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const int q = q0 + u * 256, i = i0 + q / cpr;
            v[u] = make_uint4(0, 0, 0, 0);
            if (q < n_stage && i < D.d) v[u] = __ldcs((const uint4*)(Wd + ((size_t)e * D.d + i) * D.I) + q % cpr);
        }
#pragma unroll
        for (int u = 0; u < 4; ++u)
            if (q0 + u * 256 < n_stage) ((uint4*)srow)[q0 + u * 256] = v[u];
    }
    __syncthreads();
    const int db = i0 / WT_ROWS, pr0 = i0 % WT_ROWS;
    const int per_kb = rpb * 8;                                  // chunks of one k-block tile that belong to this block
    const int* rk = rank ? rank + (size_t)e * D.I : nullptr;
    for (int q = threadIdx.x; q < D.nCB * per_kb; q += 256) {
        const int kb2 = q / per_kb, rl = (q % per_kb) >> 3, ch = q & 7;
        const int p0 = kb2 * KB + ch * 8;                        // first ranked channel position of the chunk
        uint4 v4 = make_uint4(0, 0, 0, 0);
        if (p0 < D.I) {                                          // I % 16 == 0: the chunk is inside or outside as a whole
            int c[8];
            if (rk) {
                const int4 a = __ldg((const int4*)(rk + p0)), b = __ldg((const int4*)(rk + p0) + 1);
                c[0] = a.x; c[1] = a.y; c[2] = a.z; c[3] = a.w; c[4] = b.x; c[5] = b.y; c[6] = b.z; c[7] = b.w;
            } else {
#pragma unroll
                for (int j = 0; j < 8; ++j) c[j] = p0 + j;
            }
            const uint16_t* row = srow + (size_t)rl * D.I;
            v4.x = row[c[0]] | ((uint32_t)row[c[1]] << 16);
            v4.y = row[c[2]] | ((uint32_t)row[c[3]] << 16);
            v4.z = row[c[4]] | ((uint32_t)row[c[5]] << 16);
            v4.w = row[c[6]] | ((uint32_t)row[c[7]] << 16);
        }
        const size_t tile = ((size_t)e * D.nCB + kb2) * D.nDB + db;
        __stcs(out + ((tile * WT_BYTES + sw128_chunk(pr0 + rl, ch)) >> 4), v4);
    }
}

__global__ void k_eblk_full(uint32_t* __restrict__ eblk, int E, int nCB) {
    const int e = blockIdx.x * blockDim.x + threadIdx.x;
    if (e < E) eblk[e] = (uint32_t)e * (uint32_t)nCB;
}

cudaError_t launch_pack(const Dims& D, const __nv_bfloat16* Wg, const __nv_bfloat16* Wu, const __nv_bfloat16* Wd,
                        const int* rank_dev, uint8_t* packed, uint32_t* eblk_dev, cudaStream_t st) {
    const size_t n_gu = gu_bytes(D) >> 4, n_dn = dn_bytes(D) >> 4;
    const int threads = 256;
    const int b_gu = (int)((n_gu + threads - 1) / threads < 148 * 64 ? (n_gu + threads - 1) / threads : 148 * 64);
    const int b_dn = (int)((n_dn + threads - 1) / threads < 148 * 64 ? (n_dn + threads - 1) / threads : 148 * 64);
    k_pack_gu<<<b_gu, threads, 0, st>>>(D, (const uint4*)Wg, (const uint4*)Wu, rank_dev, (uint4*)packed, n_gu);
    // output features per block of k_pack_dn_rows (divides 128): 16 while that leaves five blocks per SM (<= 40 KB of rows),
    // 8 if that does; fewer only when a row is so long that 8 of them exceed the shared-memory budget
    int rpb = 16;
    if ((size_t)rpb * D.I * 2 > 40 * 1024) rpb = 8;
    while (rpb && (size_t)rpb * D.I * 2 > (size_t)PACK_DN_SMEM) rpb >>= 1;
    if (rpb && ((uintptr_t)Wd & 15u) == 0) {
        const size_t smem = (size_t)rpb * D.I * 2;
        cudaError_t e = cudaFuncSetAttribute(k_pack_dn_rows, cudaFuncAttributeMaxDynamicSharedMemorySize, PACK_DN_SMEM);
        if (e != cudaSuccess) return e;
        k_pack_dn_rows<<<D.E * (D.nDB * WT_ROWS / rpb), threads, smem, st>>>(D, (const uint16_t*)Wd, rank_dev,
                                                                           (uint4*)(packed + gu_bytes(D)), rpb);
    } else {
        k_pack_dn_gather<<<b_dn, threads, 0, st>>>(D, (const uint16_t*)Wd, rank_dev, (uint4*)(packed + gu_bytes(D)), n_dn);
    }
    k_eblk_full<<<1, MAX_E, 0, st>>>(eblk_dev, D.E, D.nCB);
    return cudaGetLastError();
}

// --------------------------------------------------------------------------------------- unpack_prefix
__global__ void k_unpack_prefix(Dims D, LayerView V, int e, int r,
                                uint16_t* __restrict__ Wg, uint16_t* __restrict__ Wu, uint16_t* __restrict__ Wd) {
    const size_t n = (size_t)r * D.d;
    const uint32_t eb = V.eblk[e];
    for (size_t g = blockIdx.x * (size_t)blockDim.x + threadIdx.x; g < n; g += (size_t)gridDim.x * blockDim.x) {
        {   // gate / up element (p, i)
            const int p = (int)(g / D.d), i = (int)(g % D.d);
            const int cb = p / CB, w = p % CB;
            const uint32_t pr_g = (w / 16) * 32 + (w % 16);
            const uint8_t* t = V.gu + gu_tile_off(D, eb, cb, i / KB);
            Wg[g] = *(const uint16_t*)(t + sw128_off(pr_g, i % KB));
            Wu[g] = *(const uint16_t*)(t + sw128_off(pr_g + 16, i % KB));
        }
        {   // down element (i, p), output row-major [d][r]
            const int i = (int)(g / r), p = (int)(g % r);
            const uint8_t* t = V.dn + dn_tile_off(D, eb, p / KB, i / WT_ROWS);
            Wd[g] = *(const uint16_t*)(t + sw128_off(i % WT_ROWS, p % KB));
        }
    }
}

cudaError_t launch_unpack_prefix(const Dims& D, const LayerView& V, int e, int r, __nv_bfloat16* Wg,
                                 __nv_bfloat16* Wu, __nv_bfloat16* Wd, cudaStream_t st) {
    if (r == 0) return cudaSuccess;
    const size_t n = (size_t)r * D.d;
    const int blocks = (int)((n + 255) / 256 < 148 * 32 ? (n + 255) / 256 : 148 * 32);
    k_unpack_prefix<<<blocks, 256, 0, st>>>(D, V, e, r, (uint16_t*)Wg, (uint16_t*)Wu, (uint16_t*)Wd);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------- export_clipped
// Offline clipping (Table 2): the retained prefix ceil(r_e / 64) channel blocks of every
// expert, copied back to back.  A channel block is nKB1 (gate/up) resp. nDB (down) consecutive 16 KB tiles in both the
// source and the destination, so the export is a segmented copy: HBM-bound, bytes = 2 x the clipped blob.
// Block (e, part) streams its expert's share with 16-byte loads/stores; eblk_dst is the exclusive scan of the block counts.
__global__ void __launch_bounds__(256) k_export_clipped(Dims D, LayerView src, const int* __restrict__ r,
                                                        uint8_t* __restrict__ gu_dst, uint8_t* __restrict__ dn_dst,
                                                        uint32_t* __restrict__ eblk_dst, int parts) {
    __shared__ uint32_t s_base;
    const int e = blockIdx.x / parts, part = blockIdx.x % parts;
    if (threadIdx.x < 32) {                                      // exclusive scan of ceil(r / 64) over experts < e
        uint32_t acc = 0;
        for (int o = threadIdx.x; o < e; o += 32) acc += (uint32_t)((r[o] + CB - 1) / CB);
#pragma unroll
        for (int o = 16; o; o >>= 1) acc += __shfl_xor_sync(0xffffffffu, acc, o);
        if (threadIdx.x == 0) {
            s_base = acc;
            if (part == 0) eblk_dst[e] = acc;
        }
    }
    __syncthreads();
    const uint32_t dbase = s_base, sbase = src.eblk[e];
    const int nb = (r[e] + CB - 1) / CB;
    const size_t gu_n = (size_t)nb * D.nKB1 * (WT_BYTES / 16), dn_n = (size_t)nb * D.nDB * (WT_BYTES / 16);   // uint4 counts
    const uint4* gs = (const uint4*)(src.gu + gu_tile_off(D, sbase, 0, 0));
    const uint4* ds = (const uint4*)(src.dn + dn_tile_off(D, sbase, 0, 0));
    uint4* gd = (uint4*)(gu_dst + gu_tile_off(D, dbase, 0, 0));
    uint4* dd = (uint4*)(dn_dst + dn_tile_off(D, dbase, 0, 0));
    const size_t stride = (size_t)parts * 256;
    for (size_t i = (size_t)part * 256 + threadIdx.x; i < gu_n + dn_n; i += 4 * stride) {
        uint4 v[4];
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const size_t j = i + u * stride;
            if (j < gu_n + dn_n) v[u] = j < gu_n ? __ldcs(gs + j) : __ldcs(ds + (j - gu_n));
        }
#pragma unroll
        for (int u = 0; u < 4; ++u) {
            const size_t j = i + u * stride;
            if (j < gu_n + dn_n) {
                if (j < gu_n) __stcs(gd + j, v[u]); else __stcs(dd + (j - gu_n), v[u]);
            }
        }
    }
}

cudaError_t launch_export_clipped(const Dims& D, const LayerView& src, const int* r_dev, uint8_t* gu_dst, uint8_t* dn_dst,
                                  uint32_t* eblk_dst, cudaStream_t st) {
    int parts = (148 * 8 + D.E - 1) / D.E;                        // ~8 blocks per SM in total
    if (parts < 1) parts = 1;
    k_export_clipped<<<D.E * parts, 256, 0, st>>>(D, src, r_dev, gu_dst, dn_dst, eblk_dst, parts);
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

// ------------------------------------------------------------------------------------------- finalize
// The end of Alg. 2 l.19-20: the fp32 scatter-add target becomes y.  This is the ONE rounding of y
// (reading R11); y_add, if given, is the shared-expert output added in fp32 before it.
// 8 elements per thread: 32 B of yacc in, 16 B of y out.
__global__ void __launch_bounds__(256) k_finalize(const float4* __restrict__ yacc, const uint4* __restrict__ y_add,
                                                  uint4* __restrict__ y, size_t n8) {
    pdl_launch_dependents();
    pdl_wait();
    for (size_t i = blockIdx.x * (size_t)blockDim.x + threadIdx.x; i < n8; i += (size_t)gridDim.x * blockDim.x) {
        float4 a = __ldcs(yacc + 2 * i), b = __ldcs(yacc + 2 * i + 1);
        if (y_add) {
            const uint4 s = __ldg(y_add + i);
            a.x += __uint_as_float(s.x << 16); a.y += __uint_as_float(s.x & 0xFFFF0000u);
            a.z += __uint_as_float(s.y << 16); a.w += __uint_as_float(s.y & 0xFFFF0000u);
            b.x += __uint_as_float(s.z << 16); b.y += __uint_as_float(s.z & 0xFFFF0000u);
            b.z += __uint_as_float(s.w << 16); b.w += __uint_as_float(s.w & 0xFFFF0000u);
        }
        const __nv_bfloat162 p0 = __floats2bfloat162_rn(a.x, a.y), p1 = __floats2bfloat162_rn(a.z, a.w);
        const __nv_bfloat162 p2 = __floats2bfloat162_rn(b.x, b.y), p3 = __floats2bfloat162_rn(b.z, b.w);
        uint4 o;
        o.x = *(const uint32_t*)&p0; o.y = *(const uint32_t*)&p1; o.z = *(const uint32_t*)&p2; o.w = *(const uint32_t*)&p3;
        y[i] = o;
    }
}
cudaError_t launch_finalize(const Dims& D, int T, const float* yacc, const __nv_bfloat16* y_add, __nv_bfloat16* y,
                            cudaStream_t st) {
    if (T == 0) return cudaSuccess;
    const size_t n8 = (size_t)T * D.d / 8;                        // d % 64 == 0
    size_t blocks = (n8 + 255) / 256;
    if (blocks > 148 * 8) blocks = 148 * 8;
    return launch_pdl(k_finalize, dim3((unsigned)blocks), dim3(256), 0, st, (const float4*)yacc, (const uint4*)y_add, (uint4*)y, n8);
}

// --------------------------------------------------------------------------------------------- read_h
// H_out[s][c] for sorted position s (perm order) and channel c < I, from the swizzled panels.  raw = 0: columns of
// blocks that were never issued (c >= ceil64(r_e)) and, by definition, every column >= r_e read as 0; raw = 1: columns
// below ceil64(r_e) are returned exactly as the GEMM-1 epilogue wrote them (the test of the kernel's pad-zero rule),
// columns of never-issued blocks are 0.
__global__ void k_read_h(Dims D, int k, const int* __restrict__ ids, const int* __restrict__ r_table,
                         const int* __restrict__ inv_perm, const int* __restrict__ row_flat,
                         const Sched* __restrict__ sched, const uint8_t* __restrict__ H, int P,
                         uint16_t* __restrict__ out, int raw) {
    const int P_used = sched->P_used;
    const size_t n = (size_t)P_used * D.I;
    for (size_t g = blockIdx.x * (size_t)blockDim.x + threadIdx.x; g < n; g += (size_t)gridDim.x * blockDim.x) {
        const int p = (int)(g / D.I), c = (int)(g % D.I);
        const int f = row_flat[p];
        if (f < 0) continue;
        const int s = inv_perm[f];
        const uint8_t* row = H + ((size_t)(c / CB) * P + p) * ROW_BYTES;
        const uint16_t v = *(const uint16_t*)(row + ((((c % CB) >> 3) ^ p) & 7) * 16 + ((c & 7) << 1));
        const int r = r_table[ids[f]];
        const int lim = raw ? (r + CB - 1) / CB * CB : r;            // pruned blocks are never written
        out[(size_t)s * D.I + c] = c < lim ? v : (uint16_t)0;
    }
    (void)k;
}
cudaError_t launch_read_h(const Dims& D, int T, int k, const int* ids, const int* r_table, const Workspace& ws,
                          __nv_bfloat16* H_out, int raw, cudaStream_t st) {
    (void)T;
    k_read_h<<<148 * 8, 256, 0, st>>>(D, k, ids, r_table, ws.inv_perm, ws.row_flat, ws.sched, ws.H, ws.P,
                                      (uint16_t*)H_out, raw);
    return cudaGetLastError();
}

}  // namespace fxm
