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
constexpr int DEC_MAX_RUNS = 320;      // >= DEC_MAX_A / 16 + MAX_E: most runs (expert, <= 16 tokens) of one decode call

// byte offset of element (row, col) inside a swizzled tile whose rows are 128 B; row is the row index
// relative to a base that is a multiple of 8 rows.
__host__ __device__ inline uint32_t sw128_off(uint32_t row, uint32_t col) {
    return row * ROW_BYTES + ((((col >> 3) ^ row) & 7u) << 4) + ((col & 7u) << 1);
}
// byte offset of 16-byte chunk `ch` (0..7) of `row`
__host__ __device__ inline uint32_t sw128_chunk(uint32_t row, uint32_t ch) {
    return row * ROW_BYTES + (((ch ^ row) & 7u) << 4);
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
__host__ __device__ inline size_t gu_bytes(const Dims& D) { return (size_t)D.E * D.nCB * D.nKB1 * WT_BYTES; }
__host__ __device__ inline size_t dn_bytes(const Dims& D) { return (size_t)D.E * D.nCB * D.nDB * WT_BYTES; }

struct DevState {           // lives at the tail of the packed blob (zeroed by pack)
    uint32_t flags;         // bit0: expert id out of range; bit1: pipeline wait timed out
    uint32_t ticket;        // route: blocks that have published their histogram (reset by the last one)
    uint32_t pad0[2];
    unsigned long long dec_zcnt;  // decode kernel: arrivals "my slice of yacc is zeroed" -- a counter that only grows: every launch adds
                            //   exactly its grid size G (the same for every launch on this layer), so the value a CTA's own
                            //   arrival returns tells it the target of ITS launch: (old / G + 1) * G.  64 bits: never wraps.
    uint32_t pad1[24];
    uint32_t* hflag;        // host-mapped (pinned) word that also receives bit1: readable after a trap has killed the context
                            // -> 128 bytes: the words below live in their own line
    unsigned long long dec_bcnt;  // decode kernel: arrivals at the final grid barrier (same scheme as dec_zcnt)
    uint32_t route_gen;     // route kernel: bumped by the last block to publish its histogram (sense reversal; never reset)
    uint32_t pad2[29];
};
static_assert(sizeof(DevState) == 256, "DevState layout");

// ------------------------------------------------------------------------------------------------
// Workspace map (all offsets 1024-byte aligned).  P = padded-row capacity for this call.
// ------------------------------------------------------------------------------------------------
struct Sched {              // written by the route kernel, read by everything after it
    int ntt;                // number of token tiles (experts with n_e == 0 or r_e == 0 get none: pruned work is never issued)
    int W1;                 // GEMM-1 work items  = sum_j ceil(ceil(r_e(j) / 64) / 2)   (CTA-pair items)
    int W2;                 // GEMM-2 work items  = ntt * ceil(nDB / 2)
    int P_used;             // padded rows in use
    int A;                  // T * k
    int max_n;              // rows of the widest token tile (multiple of 16; 16 if there is none)
    unsigned claim1;        // dynamic work claim counters of GEMM-1 / GEMM-2 (zeroed by the plan kernel)
    unsigned claim2;
    int pad[8];
};

struct Workspace {
    int* counts;            // [E]
    int* offsets;           // [E+1]
    int* poff;              // [E+1] padded-row offset of each expert segment (multiple of 16)
    Sched* sched;
    int* perm;              // [A]
    int* inv_perm;          // [A]
    int* row_flat;          // [P]  flat assignment index f = t*k+j of each padded row, -1 for padding
    int* row_tok;           // [P]  token index t = f / k of each padded row (0 for padding rows): the gather4 row coordinates
    int2* row_tw;           // [P]  {token index or -1 for padding rows, router weight topk_w[f] as bits}: the scatter-add
                            //      destination and scale of each padded row (GEMM-2 epilogue, Alg. 2 l.19-20)
    int* fe_ids;            // [A]  router front end (fxm_moe_ffn_router): the ids it chose ...
    float* fe_w;            // [A]  ... and the renormalised weights
    int* bhist;             // [RB][E] per-route-block expert histogram, then exclusive base over blocks
    int4* tt;               // [NT + 1] token tiles: {expert, first padded row, valid rows, GEMM-1 work prefix}; tt[ntt] = sentinel
    uint8_t* H;             // [nCB][P][128 B]   SwiGLU activations, swizzled panels
    float* yacc;            // [T][d] fp32 accumulator of y: the scatter-add target of GEMM-2 / of the decode kernel
    float* dec_part;        // decode kernel: fp32 partial gate/up sums, one 8 KB slot per (item, CTA) piece
    int RB;                 // route blocks
    int chunk;              // flat assignments per route block
    int P;                  // padded-row capacity (multiple of 16)
    int NT;                 // token-tile capacity
    size_t bytes;           // total
};

constexpr int TILE_N_MIN = 128;   // smallest token tile any plan uses (the schedule capacity is sized for it)

__host__ inline size_t align_up(size_t x, size_t a) { return (x + a - 1) / a * a; }

constexpr int RT_THREADS = 256;   // route kernel: 8 warps per block
constexpr int RT_MAX_BLOCKS = 128;
// tokens per route block: a multiple of 32 that keeps the grid at <= RT_MAX_BLOCKS blocks (a block owns whole tokens,
// i.e. the flat assignments [b * chunk * k, (b + 1) * chunk * k))
__host__ inline int route_tok_chunk(long long T, int E) {
    // every block sums all published histogram rows: keep rows x experts / 256 threads at <= 32 loads per thread
    const int maxb = E <= 64 ? RT_MAX_BLOCKS : (8192 / E > 16 ? 8192 / E : 16);
    const long long per = (T + maxb - 1) / maxb;
    const long long c = (per + 31) / 32 * 32;
    return (int)(c > 0 ? c : 32);
}

size_t decode_part_bytes(const Dims& D, long long A);   // fxm_decode.cu; monotonic in A

__host__ inline Workspace map_workspace(const Dims& D, int T, int k, void* base) {
    Workspace w{};
    const size_t A = (size_t)T * k;
    const int P = (int)align_up(A + (size_t)(ROW_ALIGN - 1) * D.E, ROW_ALIGN) + ROW_ALIGN;
    const int NT = (int)(A / TILE_N_MIN) + D.E + 1;
    const int chunk = route_tok_chunk((long long)T, D.E) * k;          // flat assignments per route block
    const int RB = T > 0 ? (int)((A + chunk - 1) / chunk) : 1;
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
    w.row_tok = (int*)(b + take(sizeof(int) * (size_t)P));
    w.row_tw = (int2*)(b + take(sizeof(int2) * (size_t)P));
    w.fe_ids = (int*)(b + take(sizeof(int) * (A + 1)));
    w.fe_w = (float*)(b + take(sizeof(float) * (A + 1)));
    w.bhist = (int*)(b + take(sizeof(int) * (size_t)RT_MAX_BLOCKS * D.E));   // capacity, not RB: the size stays monotonic in T
    w.tt = (int4*)(b + take(sizeof(int4) * ((size_t)NT + 1)));
    w.H = b + take((size_t)D.nCB * P * ROW_BYTES);
    w.yacc = (float*)(b + take((size_t)T * D.d * sizeof(float)));       // every T: the size is monotonic in T
    w.dec_part = (float*)(b + take(decode_part_bytes(D, (long long)A)));
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
// Where the weight tiles of a layer live.  A full (online) layer keeps every channel block of every expert:
// eblk[e] = e * nCB.  An offline-clipped layer (fxm_export_clipped) keeps only the retained prefix
// ceil(r_e / 64) blocks of each expert, back to back: eblk[e] = sum_{e' < e} ceil(r_e' / 64).  Every kernel
// addresses tiles through eblk, so one code path serves both deployment modes.
// ------------------------------------------------------------------------------------------------
struct LayerView {
    const uint8_t* gu;       // gate/up tiles: tile (e, cb, kb) at ((eblk[e] + cb) * nKB1 + kb) * 16 KB
    const uint8_t* dn;       // down tiles:    tile (e, kb2, db) at ((eblk[e] + kb2) * nDB + db) * 16 KB
    const uint32_t* eblk;    // [E] device: first channel block of expert e
};
__host__ __device__ inline size_t gu_tile_off(const Dims& D, uint32_t eblk, int cb, int kb) {
    return (((size_t)eblk + cb) * D.nKB1 + kb) * WT_BYTES;
}
__host__ __device__ inline size_t dn_tile_off(const Dims& D, uint32_t eblk, int kb2, int db) {
    return (((size_t)eblk + kb2) * D.nDB + db) * WT_BYTES;
}

// ------------------------------------------------------------------------------------------------
// Launchers (each enqueues on `st` and returns cudaGetLastError()).
// ------------------------------------------------------------------------------------------------
cudaError_t launch_pack(const Dims& D, const __nv_bfloat16* Wg, const __nv_bfloat16* Wu, const __nv_bfloat16* Wd,
                        const int* rank_dev /*[E][I] or null*/, uint8_t* packed, uint32_t* eblk_dev, cudaStream_t st);
cudaError_t launch_unpack_prefix(const Dims& D, const LayerView& V, int e, int r, __nv_bfloat16* Wg,
                                 __nv_bfloat16* Wu, __nv_bfloat16* Wd, cudaStream_t st);
cudaError_t launch_set_table(int* table_dev, const int* r_host, int E, cudaStream_t st);
// offline clipping: copy the retained prefix blocks of every expert of `src` into the compact regions
// gu_dst / dn_dst (block order given by eblk_dst) and write eblk_dst; r_dev = the width table (device)
cudaError_t launch_export_clipped(const Dims& D, const LayerView& src, const int* r_dev, uint8_t* gu_dst, uint8_t* dn_dst,
                                  uint32_t* eblk_dst, cudaStream_t st);

// a2 + a3 in ONE launch (fxm_route.cu): per-block histograms -> grid-wide publish -> every block derives its own
// bases and scatters its assignments (stable); block 0 also writes counts / offsets / the token tiles / the work items
// for the CURRENT width table.  tile_n = max rows of a token tile.  topk_w may be null (fxm_route: indices only).
struct RouteArgs {
    Dims D;
    const int* ids;          // [T][k] device, or null when `logits` is given
    const float* topk_w;     // [T][k] device, or null
    const float* logits;     // [T][E] router logits (NEXT-3 front end): softmax -> top-k -> renormalise in this kernel
    int* ids_out;            // [T][k] where the front end writes the ids it chose (workspace), else null
    float* w_out;            // [T][k] ... and the renormalised weights
    const int* r_table;      // current widths or null (fxm_route before any budget: full width)
    int T, k, tile_n;
    int* counts;             // [E]
    int* offsets;            // [E+1]
    int* perm;               // [A]
    int* inv_perm;           // [A]
};
cudaError_t launch_route(const RouteArgs& a, const Workspace& ws, DevState* state, cudaStream_t st);
// the router front end alone (softmax -> top-k -> renormalise): feeds the fused decode kernel
cudaError_t launch_router_topk(const float* logits, int T, int E, int k, int* ids_out, float* w_out, cudaStream_t st);
// y[t] = bf16( yacc[t] (+ y_add[t]) ): the single rounding of y (reading R11); y_add = optional shared-expert output
cudaError_t launch_finalize(const Dims& D, int T, const float* yacc, const __nv_bfloat16* y_add, __nv_bfloat16* y,
                            cudaStream_t st);
// raw != 0: no reader-side mask (what the kernels really wrote, pad columns included)
cudaError_t launch_read_h(const Dims& D, int T, int k, const int* ids, const int* r_table, const Workspace& ws,
                          __nv_bfloat16* H_out, int raw, cudaStream_t st);

// SIMT debug path (same layouts and schedule, no tensor cores, no async copies)
cudaError_t launch_gemm1_simt(const Dims& D, const LayerView& V, const int* r_table, const __nv_bfloat16* x,
                              const Workspace& ws, cudaStream_t st);
cudaError_t launch_gemm2_simt(const Dims& D, const LayerView& V, const int* r_table, const Workspace& ws,
                              cudaStream_t st);

// CTA-pair tcgen05 path (cta_group::2, token tiles up to 512 rows = two sub-tiles)
constexpr int PAIR_TILE_N = 512;
// x_map: a CUtensorMap (128 bytes, passed by value to the kernel) over x [T][d] bf16 with box {64, 1} and 128-byte
// swizzle: GEMM-1 gathers its token rows straight from x with TMA gather4 (no gathered copy of x).  GEMM-1 also
// zeroes ws.yacc (its epilogue warps are idle while the first tiles are multiplied).
cudaError_t launch_gemm1_pair(const Dims& D, const LayerView& V, const int* r_table, const Workspace& ws, int T,
                              DevState* state, int num_sms, const void* x_map, cudaStream_t st);
// encodes the tensor map above through the driver entry point cuTensorMapEncodeTiled (no libcuda link dependency)
cudaError_t encode_x_map(const void* x, int T, int d, void* map_out /* 128 bytes, 64-byte aligned */);
// GEMM-2 with the router-weight scale and the scatter-add into ws.yacc fused in its epilogue (Alg. 2 l.18-20)
cudaError_t launch_gemm2_pair(const Dims& D, const LayerView& V, const int* r_table, const Workspace& ws,
                              DevState* state, int num_sms, cudaStream_t st);
cudaError_t init_pair_kernels();

// NEXT-2 / NEXT-4 (fxm_rank.cu): channel saliency + ranking, action sampling + cost
size_t saliency_workspace_bytes(const Dims& D);
cudaError_t launch_saliency(const Dims& D, const __nv_bfloat16* Wg, const __nv_bfloat16* Wu, const __nv_bfloat16* Wd,
                            const __nv_bfloat16* Gg, const __nv_bfloat16* Gu, const __nv_bfloat16* Gd, int B, float* s,
                            float* part, cudaStream_t st);
// no-allocation variant: the partial sums live in a file-scope device array of fxm_rank.cu (8 MB per GPU that loads the library)
constexpr size_t SALIENCY_STATIC_BYTES = (size_t)8 << 20;
cudaError_t launch_saliency_static(const Dims& D, const __nv_bfloat16* Wg, const __nv_bfloat16* Wu, const __nv_bfloat16* Wd,
                                   const __nv_bfloat16* Gg, const __nv_bfloat16* Gu, const __nv_bfloat16* Gd, int B, float* s,
                                   cudaStream_t st);
cudaError_t init_rank_kernel();
bool rank_supported(int I);
cudaError_t launch_rank(int E, int I, const float* s, int* rank, cudaStream_t st);
cudaError_t launch_sample_actions(const float* alpha, const float* gumbel, int K, const int* num_host, int den, int E, int I,
                                  int* table, int* action, cudaStream_t st);
cudaError_t launch_action_cost(const float* alpha, int K, const int* num_host, int den, int E, const int* counts, float* cost,
                               cudaStream_t st);

// fused single-launch decode kernel (fxm_decode.cu): T*k <= DEC_MAX_A, d <= 3840
bool decode_supported(const Dims& D);
cudaError_t init_decode_kernel();
cudaError_t launch_decode(const Dims& D, const LayerView& V, const int* r_table, const __nv_bfloat16* x,
                          const int* ids, const float* topk_w, int T, int k, float* yacc, float* part,
                          const __nv_bfloat16* y_add, __nv_bfloat16* y, DevState* state, uint32_t* item_cnt, int num_sms, int pf,
                          cudaStream_t st);
// per-item "phase-1 pieces written" counters of the decode kernel (library-owned, in the blob's tail; zero between calls)
__host__ __device__ inline size_t decode_cnt_bytes(const Dims& D) { return sizeof(uint32_t) * (size_t)DEC_MAX_RUNS * D.nCB; }

}  // namespace fxm
