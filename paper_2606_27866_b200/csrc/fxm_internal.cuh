// fxm_internal.cuh -- shared declarations of the CUDA path (layout math, workspace map, launchers).
// Nothing here is shared with oracle/ (the CPU oracle has its own plain row-major view of the problem).
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <stdint.h>
#include <stddef.h>

namespace fxm {

// ------------------------------------------------------------------------------------------------
// Tile geometry.  Every operand of both grouped GEMMs is stored as "SW128 K-major" tiles:
// rows of 64 bf16 (128 bytes), the 16-byte chunk index of a row XOR-ed with (row & 7) -- exactly what
// tcgen05.mma expects in shared memory for LayoutType SWIZZLE_128B, so a tile is moved with ONE
// contiguous cp.async.bulk and never re-arranged on chip.
// ------------------------------------------------------------------------------------------------
constexpr int KB = 64;                 // K elements per tile row (128 bytes)
constexpr int ROW_BYTES = 128;
constexpr int WT_ROWS = 128;           // weight tile rows = UMMA M
constexpr int WT_BYTES = WT_ROWS * ROW_BYTES;   // 16 KB
constexpr int CB = 64;                 // channels per gate/up tile (64 gate rows + 64 up rows)
constexpr int ROW_ALIGN = 16;          // padded-row alignment of an expert segment (UMMA N granularity)
constexpr int MAX_E = 256;
constexpr int MAX_K = 16;
constexpr int TABLE_STRIDE = 256;      // int32 per resident budget table
constexpr int MAX_TABLES = 16;         // FXM_MAX_BUDGETS registered + 1 "set_budget" slot
constexpr int DEC_MAX_A = 1024;        // most assignments T*k the fused decode kernel takes (int16 indices, smem routing)

// byte offset of element (row, col) inside a swizzled tile whose rows are 128 B; row is the row index
// relative to a base that is a multiple of 8 rows.
__host__ __device__ inline uint32_t sw128_off(uint32_t row, uint32_t col) {
    return row * ROW_BYTES + ((((col >> 3) ^ row) & 7u) << 4) + ((col & 7u) << 1);
}
// byte offset of 16-byte chunk `ch` (0..7) of `row`
__host__ __device__ inline uint32_t sw128_chunk(uint32_t row, uint32_t ch) {
    return row * ROW_BYTES + (((ch ^ row) & 7u) << 4);
}

// byte offset of output feature i of padded row p in the O panels
__host__ __device__ inline size_t o_off(int P, int p, int i) {
    return ((size_t)(i >> 7) * P + p) * (2 * WT_ROWS) + (size_t)(i & 127) * 2;
}

struct Dims {
    int E, d, I;
    int Ip;      // ceil64(I)
    int nCB;     // Ip / 64  channel blocks
    int nKB1;    // d / 64   K blocks of GEMM-1
    int nDB;     // ceil(d / 128) row blocks of the down projection
};

// packed blob: [gate/up tiles][down tiles][tables][state]
//   gate/up tile (e, cb, kb):  rows pr=0..127: g16 = pr/32, w = pr%32; w<16 -> gate channel cb*64+g16*16+w,
//                              else up channel cb*64+g16*16+(w-16); cols = x features kb*64 .. +63
//   down tile (e, kb2, db):    rows = output features db*128 .. +127, cols = channels kb2*64 .. +63
__host__ __device__ inline size_t gu_tile_index(const Dims& D, int e, int cb, int kb) {
    return ((size_t)e * D.nCB + cb) * D.nKB1 + kb;
}
__host__ __device__ inline size_t dn_tile_index(const Dims& D, int e, int kb2, int db) {
    return ((size_t)e * D.nCB + kb2) * D.nDB + db;
}
__host__ __device__ inline size_t gu_bytes(const Dims& D) { return (size_t)D.E * D.nCB * D.nKB1 * WT_BYTES; }
__host__ __device__ inline size_t dn_bytes(const Dims& D) { return (size_t)D.E * D.nCB * D.nDB * WT_BYTES; }

struct DevState {           // lives at the tail of the packed blob (zeroed by pack)
    uint32_t flags;         // bit0: expert id out of range; bit1: pipeline wait timed out
    uint32_t ticket;        // route: blocks that have published their histogram (reset by the last one)
    uint32_t bar_count[2];  // decode kernel: top-level arrivals at grid barrier 0 / 1 (reset by the last arriver)
    uint32_t bar_sub[2][8]; // decode kernel: first-level arrivals, CTA b uses counter b % 8 (reset by their last arrivers)
    uint32_t pad0[12];      // -> 128 bytes: the polled words below live in their own line
    uint32_t bar_gen[2];    // decode kernel: generation of grid barrier 0 / 1 (sense reversal; never reset)
    uint32_t pad1[30];
};

// ------------------------------------------------------------------------------------------------
// Workspace map (all offsets 1024-byte aligned).  P = padded-row capacity for this call.
// ------------------------------------------------------------------------------------------------
struct Sched {              // written by the route kernel, read by everything after it
    int ntt;                // number of token tiles (experts with n_e == 0 or r_e == 0 get none: pruned work is never issued)
    int W1;                 // GEMM-1 work items  = sum_j ceil(r_e(j) / 64)
    int W2;                 // GEMM-2 work items  = ntt * nDB
    int P_used;             // padded rows in use
    int A;                  // T * k
    int max_n;              // rows of the widest token tile (multiple of 16; 16 if there is none)
    int pad[10];
};

struct Workspace {
    int* counts;            // [E]
    int* offsets;           // [E+1]
    int* poff;              // [E+1] padded-row offset of each expert segment (multiple of 16)
    Sched* sched;
    int* perm;              // [A]
    int* inv_perm;          // [A]
    int* row_flat;          // [P]  flat assignment index f = t*k+j of each padded row, -1 for padding
    int* prow;              // [A]  padded row of each flat assignment; -1 = dropped or expert of width 0
    int* row_tok;           // [P]  token index t = f / k of each padded row (0 for padding rows): the gather4 row coordinates
    int* bhist;             // [RB][E] per-route-block expert histogram, then exclusive base over blocks
    int4* tt;               // [NT] token tiles: {expert, first padded row, valid rows, GEMM-1 work prefix}
    int4* items1;           // [NT*nCB] GEMM-1 work items {expert, first padded row, valid rows, channel block}
    uint8_t* Xs;            // [nKB1][P][128 B]  gathered activations, swizzled panels
    uint8_t* H;             // [nCB][P][128 B]   SwiGLU activations, swizzled panels
    uint8_t* O;             // [nDB][P][256 B]  expert outputs, bf16: panel db holds features db*128..+127 of every padded row
    float* yacc;            // [T][d] fp32 accumulator of the fused decode kernel (only when T*k <= DEC_MAX_A)
    int RB;                 // route blocks
    int chunk;              // flat assignments per route block
    int P;                  // padded-row capacity (multiple of 16)
    int NT;                 // token-tile capacity
    size_t bytes;           // total
};

constexpr int TILE_N_MAX = 256;   // largest token tile any kernel uses (schedule capacity is sized for the smallest)
constexpr int TILE_N_MIN = 128;

__host__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

constexpr int RT_THREADS = 256;   // route kernels: 8 warps per block
// flat assignments per route block: a multiple of 256 that keeps the grid at <= 128 blocks
__host__ inline int route_chunk(long long A) {
    const long long per = (A + 127) / 128;
    return (int)((per + 255) / 256 * 256 > 0 ? (per + 255) / 256 * 256 : 256);
}

__host__ inline Workspace map_workspace(const Dims& D, int T, int k, void* base) {
    Workspace w{};
    const size_t A = (size_t)T * k;
    const int P = (int)align_up(A + (size_t)(ROW_ALIGN - 1) * D.E, ROW_ALIGN) + ROW_ALIGN;
    const int NT = (int)(A / TILE_N_MIN) + D.E + 1;
    const int chunk = route_chunk((long long)A);
    const int RB = (int)((A + chunk - 1) / chunk) > 0 ? (int)((A + chunk - 1) / chunk) : 1;
    size_t o = 0;
    auto take = [&](size_t n) { size_t r = o; o = align_up(o + n, 1024); return r; };
    uint8_t* b = (uint8_t*)base;
    w.counts = (int*)(b + take(sizeof(int) * MAX_E));
    w.offsets = (int*)(b + take(sizeof(int) * (MAX_E + 1)));
    w.poff = (int*)(b + take(sizeof(int) * (MAX_E + 1)));
    w.sched = (Sched*)(b + take(sizeof(Sched)));
    w.perm = (int*)(b + take(sizeof(int) * (A + 1)));
    w.inv_perm = (int*)(b + take(sizeof(int) * (A + 1)));
    w.row_flat = (int*)(b + take(sizeof(int) * (size_t)P));
    w.prow = (int*)(b + take(sizeof(int) * (A + 1)));
    w.row_tok = (int*)(b + take(sizeof(int) * (size_t)P));
    w.bhist = (int*)(b + take(sizeof(int) * (size_t)RB * D.E));
    w.tt = (int4*)(b + take(sizeof(int4) * (size_t)NT));
    w.items1 = (int4*)(b + take(sizeof(int4) * (size_t)NT * D.nCB));
    w.Xs = b + take((size_t)D.nKB1 * P * ROW_BYTES);
    w.H = b + take((size_t)D.nCB * P * ROW_BYTES);
    w.O = b + take((size_t)P * D.nDB * WT_ROWS * 2);
    w.yacc = (float*)(b + take(A <= (size_t)DEC_MAX_A ? (size_t)T * D.d * sizeof(float) : 0));
    w.RB = RB;
    w.chunk = chunk;
    w.P = P;
    w.NT = NT;
    w.bytes = o;
    return w;
}

// ------------------------------------------------------------------------------------------------
// Programmatic dependent launch: the kernels of one fxm_moe_ffn are launched with the programmatic-stream-serialization
// attribute, call pdl_launch_dependents() first thing (the next kernel may be scheduled onto free SMs and run its
// prologue) and pdl_wait() before their first access to global memory that an earlier kernel of the stream may still
// be writing or reading (it returns once the preceding kernel has completed and flushed).  Every kernel of the chain
// waits, so completion is transitive.  This hides the launch latency and the prologue of each of the six kernels.
// ------------------------------------------------------------------------------------------------
#ifdef __CUDACC__
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
#endif
template <typename... KArgs, typename... Args>
inline cudaError_t launch_pdl(void (*kernel)(KArgs...), dim3 grid, dim3 block, size_t smem, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg{};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = st;
    cudaLaunchAttribute at[1];
    at[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    at[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = at;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kernel, KArgs(args)...);
}

// ------------------------------------------------------------------------------------------------
// Launchers (each enqueues on `st` and returns cudaGetLastError()).
// ------------------------------------------------------------------------------------------------
cudaError_t launch_pack(const Dims& D, const __nv_bfloat16* Wg, const __nv_bfloat16* Wu, const __nv_bfloat16* Wd,
                        const int* rank_dev /*[E][I] or null*/, uint8_t* packed, cudaStream_t st);
cudaError_t launch_unpack_prefix(const Dims& D, const uint8_t* packed, int e, int r, __nv_bfloat16* Wg,
                                 __nv_bfloat16* Wu, __nv_bfloat16* Wd, cudaStream_t st);
cudaError_t launch_set_table(int* table_dev, const int* r_host, int E, cudaStream_t st);
// a2/a3 part 1: per-block histograms; the last block to finish scans them and writes counts/offsets/poff/tt/items1/sched
// tile_n = max rows of a token tile; grp = weight blocks per work item (1: single-CTA kernels, 2: CTA-pair kernels)
cudaError_t launch_route_plan(const Dims& D, const int* ids, int T, int k, const int* r_table, int tile_n, int grp,
                              int* counts, int* offsets, const Workspace& ws, DevState* state, cudaStream_t st);
// a2 part 2: stable scatter (perm / inv_perm / row_flat / prow)
cudaError_t launch_scatter(const Dims& D, const int* ids, int T, int k, const int* r_table, const int* counts,
                           const int* offsets, int* perm, int* inv_perm, const Workspace& ws, cudaStream_t st);
// gather of the x rows into the sorted, padded, swizzled panels ws.Xs
cudaError_t launch_gather(const Dims& D, const __nv_bfloat16* x, int T, int k, const Workspace& ws, cudaStream_t st);
// y[t] = sum_j topk_w[t][j] * O[row of (t,j)]   (fp32 sum in slot order, one rounding)
cudaError_t launch_combine(const Dims& D, int T, int k, const float* topk_w, const Workspace& ws, __nv_bfloat16* y,
                           cudaStream_t st);
cudaError_t launch_read_h(const Dims& D, int T, int k, const int* ids, const int* r_table, const Workspace& ws,
                          __nv_bfloat16* H_out, cudaStream_t st);

// SIMT debug path (same layouts, no tensor cores, no async copies)
cudaError_t launch_gemm1_simt(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                              cudaStream_t st);
cudaError_t launch_gemm2_simt(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                              cudaStream_t st);

// tcgen05 / TMEM / bulk-copy path
cudaError_t launch_gemm1_sm100(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                               DevState* state, int tile_n, int num_sms, cudaStream_t st);
cudaError_t launch_gemm2_sm100(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                               DevState* state, int tile_n, int num_sms, cudaStream_t st);
cudaError_t init_sm100_kernels();   // cudaFuncSetAttribute for the dynamic shared memory sizes

// CTA-pair path (cta_group::2, token tiles up to 512 rows); the schedule must have been planned with grp = 2
constexpr int PAIR_TILE_N = 512;
// x_map: a CUtensorMap (128 bytes, passed by value to the kernel) over x [T][d] bf16 with box {64, 1} and 128-byte
// swizzle: GEMM-1 gathers its token rows straight from x with TMA gather4 (no Xs copy).  nullptr = read the Xs panels.
cudaError_t launch_gemm1_pair(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                              DevState* state, int num_sms, const void* x_map, cudaStream_t st);
// encodes the tensor map above through the driver entry point cuTensorMapEncodeTiled (no libcuda link dependency)
cudaError_t encode_x_map(const void* x, int T, int d, void* map_out /* 128 bytes, 64-byte aligned */);
cudaError_t launch_gemm2_pair(const Dims& D, const uint8_t* packed, const int* r_table, const Workspace& ws,
                              DevState* state, int num_sms, cudaStream_t st);
cudaError_t init_pair_kernels();

// fused single-launch decode kernel (fxm_decode.cu): T*k <= DEC_MAX_A, d <= 3840
bool decode_supported(const Dims& D);
cudaError_t init_decode_kernel();
cudaError_t launch_decode(const Dims& D, const uint8_t* packed, const int* r_table, const __nv_bfloat16* x,
                          const int* ids, const float* topk_w, int T, int k, float* yacc, __nv_bfloat16* y,
                          DevState* state, int num_sms, int pf, cudaStream_t st);

}  // namespace fxm
