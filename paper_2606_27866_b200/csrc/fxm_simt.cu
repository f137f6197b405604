// fxm_simt.cu -- the slow, structurally simple DEBUG path for steps a4/a5 (FXM_IMPL_SIMT_DEBUG).
// It runs on the SAME packed weights, schedule, H panels and fp32 accumulator as the tcgen05 kernels, one
// CTA per work item, plain loads and fp32 FMAs -- no tensor cores, no async copies, no mbarriers -- so a
// disagreement between the two paths isolates the fast kernels.  It is a CUDA path (not a CPU fallback) and
// is never selected unless the caller asks for it with fxm_set_impl().
//   a4: G = X_e W~gate[0:r_e]^T, U = X_e W~up[0:r_e]^T, H = silu(G) (.) U, channels >= r_e forced to 0
//       (Eq. 4; Alg. 2 l.12-16)
//   a5: yacc[token(row)] += topk_w(row) * H_e[row, 0:r_e] W~down[:, 0:r_e]^T (Alg. 2 l.18-20)
#include "fxm_internal.cuh"

namespace fxm {

__device__ __forceinline__ float bf16_bits_to_float(uint16_t b) { return __uint_as_float((uint32_t)b << 16); }

constexpr int SIMT_TOK = 8;   // tokens per register block

// block = 128 threads = the 128 packed rows of one gate/up tile; grid.x = work item (token tile j, channel block cb)
__global__ void __launch_bounds__(128) k_gemm1_simt(Dims D, LayerView V,
                                                    const int* __restrict__ r_table, const int4* __restrict__ tt,
                                                    const Sched* __restrict__ sched, const uint16_t* __restrict__ x,
                                                    const int* __restrict__ row_tok, uint8_t* __restrict__ H, int P) {
    __shared__ float s_acc[128][SIMT_TOK + 1];
    // work item = (token tile j, channel block cb < ceil(r_e / 64)); the schedule's own GEMM-1 items are CTA-PAIR
    // items (two channel blocks each), so this path enumerates single blocks itself: tile j, block cb = 0 .. nCB - 1
    const int ntt = sched->ntt;
    for (int wi = blockIdx.x; wi < ntt * D.nCB; wi += gridDim.x) {
        const int4 t = tt[wi / D.nCB];
        const int e = t.x, row0 = t.y, nvalid = t.z & 0xFFFF, cb = wi % D.nCB;
        const int r = r_table[e];
        if (cb * CB >= r) continue;                                   // pruned block: never issued
        const uint32_t eb = V.eblk[e];
        const int pr = threadIdx.x;
        const int npad = (nvalid + ROW_ALIGN - 1) / ROW_ALIGN * ROW_ALIGN;
        for (int t0 = 0; t0 < npad; t0 += SIMT_TOK) {
            float acc[SIMT_TOK];
#pragma unroll
            for (int q = 0; q < SIMT_TOK; ++q) acc[q] = 0.f;
            for (int kb = 0; kb < D.nKB1; ++kb) {
                const uint8_t* wt = V.gu + gu_tile_off(D, eb, cb, kb);
                for (int c = 0; c < KB; ++c) {
                    const float wv = bf16_bits_to_float(*(const uint16_t*)(wt + sw128_off(pr, c)));
#pragma unroll
                    for (int q = 0; q < SIMT_TOK; ++q) {
                        const int p = row0 + t0 + q;                   // padding rows read token 0 (X[pi], Alg. 2 l.7)
                        acc[q] += wv * bf16_bits_to_float(x[(size_t)row_tok[p] * D.d + kb * KB + c]);
                    }
                }
            }
            __syncthreads();
#pragma unroll
            for (int q = 0; q < SIMT_TOK; ++q) s_acc[pr][q] = acc[q];
            __syncthreads();
            // 64 channels x SIMT_TOK tokens of SwiGLU; thread -> (channel, token) pairs
            for (int i = threadIdx.x; i < CB * SIMT_TOK; i += blockDim.x) {
                const int ch = i % CB, q = i / CB;
                const int prg = (ch / 16) * 32 + (ch % 16);
                const float g = s_acc[prg][q], u = s_acc[prg + 16][q];
                float h = g / (1.f + __expf(-g)) * u;
                if (cb * CB + ch >= r) h = 0.f;                      // tail mask of the last retained block
                const int p = row0 + t0 + q;
                const __nv_bfloat16 hb = __float2bfloat16_rn(h);
                *(__nv_bfloat16*)(H + ((size_t)cb * P + p) * ROW_BYTES + ((((ch >> 3) ^ p) & 7) << 4) + ((ch & 7) << 1)) = hb;
            }
        }
    }
}

// block = 128 threads = 128 output features of one down tile row-block; grid.x = work item (token tile j, db)
__global__ void __launch_bounds__(128) k_gemm2_simt(Dims D, LayerView V,
                                                    const int* __restrict__ r_table, const int4* __restrict__ tt,
                                                    const Sched* __restrict__ sched, const uint8_t* __restrict__ H,
                                                    const int2* __restrict__ row_tw, float* __restrict__ yacc, int P) {
    const int ntt = sched->ntt;
    for (int wi = blockIdx.x; wi < ntt * D.nDB; wi += gridDim.x) {
        const int j = wi / D.nDB, db = wi % D.nDB;
        const int4 t = tt[j];
        const int e = t.x, row0 = t.y, nvalid = t.z & 0xFFFF;
        const int r = r_table[e];
        const uint32_t eb = V.eblk[e];
        const int nkb = (r + KB - 1) / KB;
        const int pr = threadIdx.x, i = db * WT_ROWS + pr;
        for (int t0 = 0; t0 < nvalid; t0 += SIMT_TOK) {
            float acc[SIMT_TOK];
#pragma unroll
            for (int q = 0; q < SIMT_TOK; ++q) acc[q] = 0.f;
            for (int kb2 = 0; kb2 < nkb; ++kb2) {
                const uint8_t* wt = V.dn + dn_tile_off(D, eb, kb2, db);
                for (int c = 0; c < KB; ++c) {
                    const float wv = bf16_bits_to_float(*(const uint16_t*)(wt + sw128_off(pr, c)));
#pragma unroll
                    for (int q = 0; q < SIMT_TOK; ++q) {
                        const int p = row0 + t0 + q;
                        const uint8_t* hp = H + ((size_t)kb2 * P + p) * ROW_BYTES + ((((c >> 3) ^ p) & 7) << 4) + ((c & 7) << 1);
                        acc[q] += wv * bf16_bits_to_float(*(const uint16_t*)hp);
                    }
                }
            }
#pragma unroll
            for (int q = 0; q < SIMT_TOK; ++q) {
                if (t0 + q < nvalid && i < D.d) {
                    const int2 tw = row_tw[row0 + t0 + q];             // {token, router weight}: scale + scatter-add
                    if (tw.x >= 0) atomicAdd(yacc + (size_t)tw.x * D.d + i, __int_as_float(tw.y) * acc[q]);
                }
            }
        }
    }
}

cudaError_t launch_gemm1_simt(const Dims& D, const LayerView& V, const int* r_table, const __nv_bfloat16* x,
                              const Workspace& ws, cudaStream_t st) {
    k_gemm1_simt<<<148 * 16, 128, 0, st>>>(D, V, r_table, ws.tt, ws.sched, (const uint16_t*)x, ws.row_tok, ws.H, ws.P);
    return cudaGetLastError();
}
cudaError_t launch_gemm2_simt(const Dims& D, const LayerView& V, const int* r_table, const Workspace& ws,
                              cudaStream_t st) {
    k_gemm2_simt<<<148 * 16, 128, 0, st>>>(D, V, r_table, ws.tt, ws.sched, ws.H, ws.row_tw, ws.yacc, ws.P);
    return cudaGetLastError();
}

}  // namespace fxm
