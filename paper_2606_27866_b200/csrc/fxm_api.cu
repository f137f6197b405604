// fxm_api.cu -- the C ABI of include/flexmoe.h: argument validation, host metadata, launch sequencing.
// No arithmetic of the method lives here; every step of the path runs in the kernels of this directory.
#include "../../include/flexmoe.h"
#include <cstdio>
#include "fxm_internal.cuh"

#include <algorithm>
#include <cstring>
#include <new>
#include <vector>

using namespace fxm;

struct fxm_layer {
    Dims D;
    LayerView V;             // where the weight tiles live (inside the caller's packed / clipped blob)
    uint8_t* blob;           // caller's buffer
    int* tables;             // [MAX_TABLES][TABLE_STRIDE] int32
    DevState* state;
    uint32_t* dec_cnt;       // decode kernel: per-item piece counters (blob tail, zero between calls)
    int* rank_dev;           // device copy of channel_rank (full layers packed with a ranking), else null
    int clipped;             // 1: offline-clipped layer: widths are bounded by r_clip
    std::vector<int> r_clip; // [E] exported widths of a clipped layer
    int n_registered;
    int current;             // index of the table the next moe_ffn reads; -1 = none installed
    int impl;
    int num_sms;
    int tile_n_override;     // 0 = PAIR_TILE_N
    int dec_max_A;           // the fused decode kernel takes calls with T*k <= dec_max_A (0 = never)
    int dec_pf;              // its L2 prefetch distance in 16 KB tiles
    int last_launches;       // kernels enqueued by the last fxm_moe_ffn
    uint32_t* host_flags;    // pinned, device-mapped word: bit1 (pipeline timeout) survives a trapped context
    alignas(64) unsigned char x_map[128];   // CUtensorMap over the x of the last general-path call (gather4 source)
    const void* x_map_ptr;   // the x it was encoded for
    int x_map_T;
    std::vector<int> host_tables;   // mirror of the resident tables (validation / introspection only)
    // fxm_moe_ffn_host: inputs travel on a side stream into one of two staging sets so that the host->device copy of
    // call i+1 overlaps the kernels and the device->host copy of call i
    cudaStream_t h2d_stream;
    cudaEvent_t ev_in[2];    // inputs of set b have landed (recorded on h2d_stream)
    cudaEvent_t ev_done[2];  // the kernels that read set b have finished (recorded on the caller's stream)
    cudaEvent_t ev_tail;     // the whole previous host call (kernels + y copy) has finished
    cudaStream_t d2h_stream; // fxm_moe_ffn_host_pipelined: y travels back here, under the kernels of the next call
    cudaEvent_t ev_y[2];     // the y copy that reads device buffer b has finished (recorded on d2h_stream)
    unsigned y_pending;      // bit b: ev_y[b] has not been waited for by the caller's stream yet
    unsigned host_calls;
    const void* host_ws;     // layout key of the previous host call: (workspace, bytes, T, k)
    size_t host_ws_bytes;
    int host_T, host_k;
    std::vector<cudaEvent_t> prof_events;   // fxm_profile_begin: (FXM_N_KERNELS + 1) events per recorded call
    int prof_capacity;       // calls that can still be recorded
    int prof_calls;          // calls recorded so far
};

static size_t host_stage_bytes(const Dims& D, int T, int k) {
    // device staging of the host-buffer entry point: two input sets {x bf16 [T][d], ids int32 [T][k], w fp32 [T][k]}
    // and two y bf16 [T][d] (the pipelined entry point copies y of call i back while call i+1 writes the other one)
    return 4 * align_up((size_t)T * D.d * 2, 1024) + 4 * align_up((size_t)T * k * 4, 1024);
}

static bool make_dims(int E, int d, int I, Dims* D) {
    if (E < 1 || E > MAX_E || d < 64 || d % 64 != 0 || I < 16 || I % 16 != 0) return false;
    D->E = E; D->d = d; D->I = I;
    D->Ip = (I + CB - 1) / CB * CB;
    D->nCB = D->Ip / CB;
    D->nKB1 = d / KB;
    D->nDB = (d + WT_ROWS - 1) / WT_ROWS;
    return true;
}

// tail of a blob, after `wbytes` of weight tiles: [16 budget tables][state][eblk][decode item counters][channel_rank copy
// (full layers only)]
struct Tail { size_t tables, state, eblk, dcnt, rank, total; };
static Tail tail_map(const Dims& D, size_t wbytes, bool with_rank) {
    Tail t;
    t.tables = align_up(wbytes, 1024);
    t.state = t.tables + sizeof(int) * MAX_TABLES * TABLE_STRIDE;
    t.eblk = align_up(t.state + sizeof(DevState), 1024);
    t.dcnt = align_up(t.eblk + sizeof(uint32_t) * MAX_E, 1024);
    t.rank = align_up(t.dcnt + decode_cnt_bytes(D), 1024);
    t.total = with_rank ? align_up(t.rank + sizeof(int) * (size_t)D.E * D.I, 1024) : t.rank;
    return t;
}
static size_t packed_total(const Dims& D) { return tail_map(D, gu_bytes(D) + dn_bytes(D), true).total; }

// ---- clipped blob (offline clipping): [header 2 KB][gate/up tiles of the retained blocks][down tiles][tail]
constexpr uint32_t CLIP_MAGIC = 0x4D584643u;    // "CFXM"
constexpr size_t CLIP_HEADER_BYTES = 2048;
struct ClipHeader { uint32_t magic, version; int32_t E, d, I, reserved[3]; int32_t r[MAX_E]; };
static_assert(sizeof(ClipHeader) <= CLIP_HEADER_BYTES, "clip header");
static size_t clip_blocks(const Dims& D, const int32_t* r) {
    size_t nb = 0;
    for (int e = 0; e < D.E; ++e) nb += (size_t)((r[e] + CB - 1) / CB);
    return nb;
}
static size_t clip_gu_bytes(const Dims& D, const int32_t* r) { return clip_blocks(D, r) * D.nKB1 * WT_BYTES; }
static size_t clip_dn_bytes(const Dims& D, const int32_t* r) { return clip_blocks(D, r) * D.nDB * WT_BYTES; }
static size_t clip_total(const Dims& D, const int32_t* r) {
    return tail_map(D, CLIP_HEADER_BYTES + clip_gu_bytes(D, r) + clip_dn_bytes(D, r), false).total;
}

static int choose_tile_n(const fxm_layer* L) { return L->tile_n_override ? L->tile_n_override : PAIR_TILE_N; }
// a6: decode-sized calls (a handful of tokens per expert) go to the single-launch weight-streaming kernel
static bool use_decode(const fxm_layer* L, int T, int k) {
    const long long A = (long long)T * k;
    return L->impl == FXM_IMPL_TCGEN05 && A <= L->dec_max_A && A <= DEC_MAX_A && decode_supported(L->D);
}

// L2 prefetch distance of the decode kernel (16 KB tiles per CTA): the caller's choice (fxm_set_decode), default 0.
// Measured on B200 (L2 flushed, C4 and C2 shapes, T = 1 .. 64, every budget): a cursor of 16 or 256 tiles is 0-40 %
// SLOWER than none at every size -- prefetch requests share the SM's outstanding-request budget with the ring's own loads.
static int decode_prefetch(const fxm_layer* L, int, int) { return L->dec_pf > 0 ? L->dec_pf : 0; }

static fxm_layer* new_layer(const Dims& D, uint8_t* blob, const Tail& tl, int sms) {
    fxm_layer* L = new (std::nothrow) fxm_layer();
    if (!L) return nullptr;
    L->D = D; L->blob = blob;
    L->tables = (int*)(blob + tl.tables);
    L->state = (DevState*)(blob + tl.state);
    L->V.eblk = (const uint32_t*)(blob + tl.eblk);
    L->dec_cnt = (uint32_t*)(blob + tl.dcnt);
    L->rank_dev = nullptr; L->clipped = 0;
    L->n_registered = 0; L->current = -1; L->impl = FXM_IMPL_TCGEN05; L->num_sms = sms; L->tile_n_override = 0;
    L->host_tables.assign((size_t)MAX_TABLES * TABLE_STRIDE, 0);
    L->prof_capacity = 0; L->prof_calls = 0;
    L->x_map_ptr = nullptr; L->x_map_T = -1;
    L->h2d_stream = nullptr; L->host_calls = 0; L->ev_tail = nullptr;
    L->d2h_stream = nullptr; L->y_pending = 0; L->ev_y[0] = L->ev_y[1] = nullptr;
    L->host_ws = nullptr; L->host_ws_bytes = 0; L->host_T = -1; L->host_k = -1;
    for (int b = 0; b < 2; ++b) { L->ev_in[b] = nullptr; L->ev_done[b] = nullptr; }
    L->dec_max_A = FXM_DECODE_DEFAULT_MAX_ASSIGNMENTS; L->dec_pf = FXM_DECODE_DEFAULT_PREFETCH; L->last_launches = 0;
    L->host_flags = nullptr;
    return L;
}

// zero the tables + state of a blob and point the state's host flag at a fresh pinned word
static fxm_status init_tail(fxm_layer* L, cudaStream_t st) {
    if (cudaMemsetAsync(L->tables, 0, sizeof(int) * MAX_TABLES * TABLE_STRIDE + sizeof(DevState), st) != cudaSuccess)
        return FXM_ECUDA;
    if (cudaMemsetAsync(L->dec_cnt, 0, decode_cnt_bytes(L->D), st) != cudaSuccess) return FXM_ECUDA;
    void* hp = nullptr;
    if (cudaHostAlloc(&hp, 64, cudaHostAllocMapped) == cudaSuccess && hp) {
        std::memset(hp, 0, 64);
        void* dp = nullptr;
        if (cudaHostGetDevicePointer(&dp, hp, 0) == cudaSuccess && dp) {
            L->host_flags = (uint32_t*)hp;
            // a copy from pageable host memory is staged before the call returns, so the stack variable may go away
            if (cudaMemcpyAsync(&L->state->hflag, &dp, sizeof(dp), cudaMemcpyHostToDevice, st) != cudaSuccess) return FXM_ECUDA;
        } else {
            cudaFreeHost(hp);
        }
    } else {
        (void)cudaGetLastError();      // no mapped memory: the device flag word alone remains
    }
    return FXM_OK;
}

extern "C" {

const char* fxm_status_string(fxm_status s) {
    switch (s) {
        case FXM_OK: return "FXM_OK";
        case FXM_EINVAL: return "FXM_EINVAL: bad pointer, size or enum";
        case FXM_ESHAPE: return "FXM_ESHAPE: unsupported dimensions";
        case FXM_EPERM: return "FXM_EPERM: channel_rank row is not a permutation";
        case FXM_EBUDGET: return "FXM_EBUDGET: width outside [0, I] (or above the exported width of a clipped layer) or unknown budget index";
        case FXM_ENOTNESTED: return "FXM_ENOTNESTED: budget tables are not nested";
        case FXM_EWORKSPACE: return "FXM_EWORKSPACE: workspace too small";
        case FXM_ESTATE: return "FXM_ESTATE: no budget installed";
        case FXM_ECUDA: return "FXM_ECUDA: CUDA runtime failure";
        case FXM_ENOMEM: return "FXM_ENOMEM: host allocation failed";
        case FXM_ELIMIT: return "FXM_ELIMIT: problem larger than the fixed scratch of a no-allocation entry point";
    }
    return "FXM_?";
}

fxm_status fxm_packed_bytes(int E, int d, int I, size_t* bytes) {
    Dims D;
    if (!bytes) return FXM_EINVAL;
    if (!make_dims(E, d, I, &D)) return FXM_ESHAPE;
    *bytes = packed_total(D);
    return FXM_OK;
}

fxm_status fxm_workspace_bytes(int E, int d, int I, int T_max, int k, size_t* bytes) {
    Dims D;
    if (!bytes || T_max < 0) return FXM_EINVAL;
    if (!make_dims(E, d, I, &D)) return FXM_ESHAPE;
    if (k < 1 || k > MAX_K || k > E) return FXM_ESHAPE;
    if ((long long)T_max * k > (1LL << 30)) return FXM_ESHAPE;
    *bytes = map_workspace(D, T_max, k, nullptr).bytes;
    return FXM_OK;
}

fxm_status fxm_workspace_bytes_host(int E, int d, int I, int T_max, int k, size_t* bytes) {
    size_t inner = 0;
    fxm_status s = fxm_workspace_bytes(E, d, I, T_max, k, &inner);
    if (s != FXM_OK) return s;
    Dims D;
    make_dims(E, d, I, &D);
    *bytes = inner + host_stage_bytes(D, T_max, k);
    return FXM_OK;
}

int32_t fxm_ratio_to_width(int I, int num, int den) {
    if (I < 0 || den <= 0 || num < 0 || num > den) return -1;
    return (int32_t)(((int64_t)I * num + den - 1) / den);
}

static fxm_status device_info(int* sms) {
    int dev = 0;
    if (cudaGetDevice(&dev) != cudaSuccess) return FXM_ECUDA;
    if (cudaDeviceGetAttribute(sms, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess) return FXM_ECUDA;
    if (init_pair_kernels() != cudaSuccess || init_decode_kernel() != cudaSuccess) return FXM_ECUDA;
    return FXM_OK;
}

fxm_status fxm_pack(fxm_layer** out, int E, int d, int I, const void* W_gate, const void* W_up, const void* W_down,
                    const int32_t* channel_rank, void* packed, void* stream) {
    Dims D;
    if (!out || !W_gate || !W_up || !W_down || !packed) return FXM_EINVAL;
    if (((uintptr_t)packed & 1023u) || ((uintptr_t)W_gate & 15u) || ((uintptr_t)W_up & 15u) || ((uintptr_t)W_down & 1u))
        return FXM_EINVAL;
    if (!make_dims(E, d, I, &D)) return FXM_ESHAPE;
    if (channel_rank) {                                           // validated on the host: offline, once
        std::vector<uint8_t> seen((size_t)I);
        for (int e = 0; e < E; ++e) {
            std::fill(seen.begin(), seen.end(), 0);
            for (int p = 0; p < I; ++p) {
                const int c = channel_rank[(size_t)e * I + p];
                if (c < 0 || c >= I || seen[c]) return FXM_EPERM;
                seen[c] = 1;
            }
        }
    }
    int sms = 0;
    fxm_status s = device_info(&sms);
    if (s != FXM_OK) return s;
    cudaStream_t st = (cudaStream_t)stream;
    uint8_t* pk = (uint8_t*)packed;
    const Tail tl = tail_map(D, gu_bytes(D) + dn_bytes(D), true);
    fxm_layer* L = new_layer(D, pk, tl, sms);
    if (!L) return FXM_ENOMEM;
    L->V.gu = pk;
    L->V.dn = pk + gu_bytes(D);
    L->rank_dev = channel_rank ? (int*)(pk + tl.rank) : nullptr;
    s = init_tail(L, st);
    if (s == FXM_OK && L->rank_dev &&
        cudaMemcpyAsync(L->rank_dev, channel_rank, sizeof(int) * (size_t)E * I, cudaMemcpyHostToDevice, st) != cudaSuccess)
        s = FXM_ECUDA;
    if (s == FXM_OK && launch_pack(D, (const __nv_bfloat16*)W_gate, (const __nv_bfloat16*)W_up, (const __nv_bfloat16*)W_down,
                                   L->rank_dev, pk, (uint32_t*)(pk + tl.eblk), st) != cudaSuccess)
        s = FXM_ECUDA;
    if (s != FXM_OK) { fxm_destroy(L); return s; }
    *out = L;
    return FXM_OK;
}

void fxm_destroy(fxm_layer* L) {
    if (!L) return;
    for (cudaEvent_t ev : L->prof_events) cudaEventDestroy(ev);
    for (int b = 0; b < 2; ++b) {
        if (L->ev_in[b]) cudaEventDestroy(L->ev_in[b]);
        if (L->ev_done[b]) cudaEventDestroy(L->ev_done[b]);
    }
    if (L->ev_tail) cudaEventDestroy(L->ev_tail);
    if (L->h2d_stream) cudaStreamDestroy(L->h2d_stream);
    for (int b = 0; b < 2; ++b)
        if (L->ev_y[b]) cudaEventDestroy(L->ev_y[b]);
    if (L->d2h_stream) cudaStreamDestroy(L->d2h_stream);
    if (L->host_flags) cudaFreeHost(L->host_flags);
    delete L;
}

static fxm_status check_table(const fxm_layer* L, const int32_t* r) {
    for (int e = 0; e < L->D.E; ++e) {
        if (r[e] < 0 || r[e] > L->D.I) return FXM_EBUDGET;
        if (L->clipped && r[e] > L->r_clip[e]) return FXM_EBUDGET;      // those channels were not exported
    }
    return FXM_OK;
}

fxm_status fxm_set_budget(fxm_layer* L, const int32_t* r_host, void* stream) {
    if (!L || !r_host) return FXM_EINVAL;
    fxm_status s = check_table(L, r_host);
    if (s != FXM_OK) return s;
    const int slot = MAX_TABLES - 1;                              // the slot fxm_register_budgets never uses
    if (launch_set_table(L->tables + (size_t)slot * TABLE_STRIDE, r_host, L->D.E, (cudaStream_t)stream) != cudaSuccess)
        return FXM_ECUDA;
    std::copy(r_host, r_host + L->D.E, L->host_tables.begin() + (size_t)slot * TABLE_STRIDE);
    L->current = slot;
    return FXM_OK;
}

fxm_status fxm_register_budgets(fxm_layer* L, int B, const int32_t* r_host, int require_nested, void* stream) {
    if (!L || !r_host || B < 1 || B > FXM_MAX_BUDGETS) return FXM_EINVAL;
    const int E = L->D.E;
    for (int b = 0; b < B; ++b) {
        fxm_status s = check_table(L, r_host + (size_t)b * E);
        if (s != FXM_OK) return s;
        if (require_nested && b > 0)
            for (int e = 0; e < E; ++e)
                if (r_host[(size_t)b * E + e] > r_host[(size_t)(b - 1) * E + e]) return FXM_ENOTNESTED;
    }
    for (int b = 0; b < B; ++b) {
        if (launch_set_table(L->tables + (size_t)b * TABLE_STRIDE, r_host + (size_t)b * E, E, (cudaStream_t)stream) !=
            cudaSuccess)
            return FXM_ECUDA;
        std::copy(r_host + (size_t)b * E, r_host + (size_t)(b + 1) * E, L->host_tables.begin() + (size_t)b * TABLE_STRIDE);
    }
    L->n_registered = B;
    return FXM_OK;
}

fxm_status fxm_select_budget(fxm_layer* L, int b) {
    if (!L) return FXM_EINVAL;
    if (b < 0 || b >= L->n_registered) return FXM_EBUDGET;
    L->current = b;                                               // host-only: the next launch reads another 1 KB table
    return FXM_OK;
}

fxm_status fxm_set_impl(fxm_layer* L, int impl) {
    if (!L || (impl != FXM_IMPL_TCGEN05 && impl != FXM_IMPL_SIMT_DEBUG)) return FXM_EINVAL;
    L->impl = impl;
    return FXM_OK;
}

fxm_status fxm_set_tile_n(fxm_layer* L, int tile_n) {
    if (!L || (tile_n != 0 && tile_n != 128 && tile_n != 256 && tile_n != 512)) return FXM_EINVAL;
    L->tile_n_override = tile_n;
    return FXM_OK;
}

fxm_status fxm_set_decode(fxm_layer* L, int max_assignments, int prefetch_tiles) {
    if (!L || max_assignments < 0 || prefetch_tiles < -1 || prefetch_tiles > 4096) return FXM_EINVAL;
    L->dec_max_A = max_assignments > DEC_MAX_A ? DEC_MAX_A : max_assignments;
    L->dec_pf = prefetch_tiles;
    return FXM_OK;
}

int fxm_launches_per_ffn(const fxm_layer* L) { return L ? L->last_launches : 0; }

fxm_status fxm_profile_begin(fxm_layer* L, int max_calls) {
    if (!L || max_calls < 1 || max_calls > 4096) return FXM_EINVAL;
    for (cudaEvent_t ev : L->prof_events) cudaEventDestroy(ev);
    L->prof_events.assign((size_t)max_calls * (FXM_N_KERNELS + 1), nullptr);
    for (cudaEvent_t& ev : L->prof_events)
        if (cudaEventCreate(&ev) != cudaSuccess) return FXM_ECUDA;
    L->prof_capacity = max_calls;
    L->prof_calls = 0;
    return FXM_OK;
}

fxm_status fxm_profile_end(fxm_layer* L, float* ms_sum, int* calls) {
    if (!L || !ms_sum || !calls) return FXM_EINVAL;
    for (int j = 0; j < FXM_N_KERNELS; ++j) ms_sum[j] = 0.f;
    fxm_status rc = FXM_OK;
    for (int c = 0; c < L->prof_calls && rc == FXM_OK; ++c) {
        cudaEvent_t* ev = &L->prof_events[(size_t)c * (FXM_N_KERNELS + 1)];
        if (cudaEventSynchronize(ev[FXM_N_KERNELS]) != cudaSuccess) { rc = FXM_ECUDA; break; }
        for (int j = 0; j < FXM_N_KERNELS; ++j) {
            float ms = 0.f;
            if (cudaEventElapsedTime(&ms, ev[j], ev[j + 1]) != cudaSuccess) { rc = FXM_ECUDA; break; }
            ms_sum[j] += ms;
        }
    }
    *calls = L->prof_calls;
    for (cudaEvent_t ev : L->prof_events) cudaEventDestroy(ev);
    L->prof_events.clear();
    L->prof_capacity = 0;
    L->prof_calls = 0;
    return rc;
}

static fxm_status check_call(const fxm_layer* L, int T, int k, const void* ws, size_t ws_bytes) {
    if (!L || T < 0 || !ws || ((uintptr_t)ws & 1023u)) return FXM_EINVAL;
    if (k < 1 || k > MAX_K || k > L->D.E || (long long)T * k > (1LL << 30)) return FXM_ESHAPE;
    if (ws_bytes < map_workspace(L->D, T, k, nullptr).bytes) return FXM_EWORKSPACE;
    return FXM_OK;
}

fxm_status fxm_route(fxm_layer* L, const int32_t* topk_ids, int T, int k, int32_t* counts, int32_t* offsets,
                     int32_t* perm, int32_t* inv_perm, void* workspace, size_t workspace_bytes, void* stream) {
    fxm_status s = check_call(L, T, k, workspace, workspace_bytes);
    if (s != FXM_OK) return s;
    if (!counts || !offsets || (T > 0 && (!topk_ids || !perm || !inv_perm))) return FXM_EINVAL;
    const Workspace ws = map_workspace(L->D, T, k, workspace);
    RouteArgs a{};
    a.D = L->D; a.ids = topk_ids; a.topk_w = nullptr;
    a.r_table = L->current >= 0 ? L->tables + (size_t)L->current * TABLE_STRIDE : nullptr;
    a.T = T; a.k = k; a.tile_n = choose_tile_n(L);
    a.counts = counts; a.offsets = offsets; a.perm = perm; a.inv_perm = inv_perm;
    if (launch_route(a, ws, L->state, (cudaStream_t)stream) != cudaSuccess) return FXM_ECUDA;
    return FXM_OK;
}

// the forward with every optional input: y_add (shared-expert output, may be null); logits (router front end: then
// topk_ids / topk_w are OUTPUT buffers, or null to keep the chosen ids / weights in the workspace only)
static fxm_status ffn_impl(fxm_layer* L, const void* x, const int32_t* topk_ids, const float* topk_w, const float* logits,
                           int T, int k, const void* y_add, void* y, void* workspace, size_t workspace_bytes, void* stream) {
    fxm_status s = check_call(L, T, k, workspace, workspace_bytes);
    if (s != FXM_OK) return s;
    if (T == 0) return FXM_OK;
    if (!x || !y || ((uintptr_t)x & 15u) || ((uintptr_t)y & 15u) || ((uintptr_t)y_add & 15u)) return FXM_EINVAL;
    if (!logits && (!topk_ids || !topk_w)) return FXM_EINVAL;
    if (L->current < 0) return FXM_ESTATE;
    const Dims& D = L->D;
    cudaStream_t st = (cudaStream_t)stream;
    const Workspace ws = map_workspace(D, T, k, workspace);
    const int* table = L->tables + (size_t)L->current * TABLE_STRIDE;
    int* fe_ids = logits ? (topk_ids ? const_cast<int32_t*>(topk_ids) : ws.fe_ids) : nullptr;   // where the front end writes
    float* fe_w = logits ? (topk_w ? const_cast<float*>(topk_w) : ws.fe_w) : nullptr;
    cudaEvent_t* ev = nullptr;                                    // per-kernel timing, only between profile_begin/end
    if (L->prof_capacity > 0) {
        ev = &L->prof_events[(size_t)L->prof_calls * (FXM_N_KERNELS + 1)];
        ++L->prof_calls;
        --L->prof_capacity;
    }
#define FXM_MARK(j) if (ev && cudaEventRecord(ev[j], st) != cudaSuccess) return FXM_ECUDA;
    if (use_decode(L, T, k)) {
        // a6: one launch does a2..a5 (in-kernel grouping, weight streaming, SwiGLU, scale + combine)
        if (logits && launch_router_topk(logits, T, D.E, k, fe_ids, fe_w, st) != cudaSuccess) return FXM_ECUDA;
        for (int j = 0; j < FXM_N_KERNELS; ++j) FXM_MARK(j)
        if (launch_decode(D, L->V, table, (const __nv_bfloat16*)x, logits ? fe_ids : topk_ids, logits ? fe_w : topk_w, T, k,
                          ws.yacc, ws.dec_part, (const __nv_bfloat16*)y_add, (__nv_bfloat16*)y, L->state, L->dec_cnt, L->num_sms,
                          decode_prefetch(L, T, k), st) != cudaSuccess)
            return FXM_ECUDA;
        FXM_MARK(FXM_N_KERNELS)
        L->last_launches = logits ? 2 : 1;
        return FXM_OK;
    }
    // a2 + a3: grouping and the tile schedule for the CURRENT table, one launch
    FXM_MARK(0)
    RouteArgs ra{};
    ra.D = D; ra.ids = topk_ids; ra.topk_w = topk_w; ra.r_table = table; ra.T = T; ra.k = k; ra.tile_n = choose_tile_n(L);
    ra.logits = logits; ra.ids_out = fe_ids; ra.w_out = fe_w;      // front end fused into the route kernel (same launch count)
    ra.counts = ws.counts; ra.offsets = ws.offsets; ra.perm = ws.perm; ra.inv_perm = ws.inv_perm;
    if (launch_route(ra, ws, L->state, st) != cudaSuccess) return FXM_ECUDA;
    FXM_MARK(1)
    if (L->impl == FXM_IMPL_TCGEN05) {
        // a4 with X[pi] (Alg. 2 l.7) fused: the token rows come straight from x through a tensor map (TMA gather4)
        if (L->x_map_ptr != x || L->x_map_T != T) {
            if (encode_x_map(x, T, D.d, L->x_map) != cudaSuccess) return FXM_ECUDA;
            L->x_map_ptr = x; L->x_map_T = T;
        }
        if (launch_gemm1_pair(D, L->V, table, ws, T, L->state, L->num_sms, L->x_map, st) != cudaSuccess) return FXM_ECUDA;
        FXM_MARK(2)
        // a5: down projection, router-weight scale and scatter-add in one kernel
        if (launch_gemm2_pair(D, L->V, table, ws, L->state, L->num_sms, st) != cudaSuccess) return FXM_ECUDA;
    } else {
        if (cudaMemsetAsync(ws.yacc, 0, (size_t)T * D.d * sizeof(float), st) != cudaSuccess) return FXM_ECUDA;
        if (launch_gemm1_simt(D, L->V, table, (const __nv_bfloat16*)x, ws, st) != cudaSuccess) return FXM_ECUDA;
        FXM_MARK(2)
        if (launch_gemm2_simt(D, L->V, table, ws, st) != cudaSuccess) return FXM_ECUDA;
    }
    FXM_MARK(3)
    if (launch_finalize(D, T, ws.yacc, (const __nv_bfloat16*)y_add, (__nv_bfloat16*)y, st) != cudaSuccess) return FXM_ECUDA;
    FXM_MARK(4)
    FXM_MARK(5)
#undef FXM_MARK
    L->last_launches = 4;
    return FXM_OK;
}

fxm_status fxm_moe_ffn(fxm_layer* L, const void* x, const int32_t* topk_ids, const float* topk_w, int T, int k, void* y,
                       void* workspace, size_t workspace_bytes, void* stream) {
    return ffn_impl(L, x, topk_ids, topk_w, nullptr, T, k, nullptr, y, workspace, workspace_bytes, stream);
}

fxm_status fxm_moe_ffn_router(fxm_layer* L, const void* x, const float* router_logits, int T, int k, const void* y_shared,
                              void* y, int32_t* topk_ids_out, float* topk_w_out, void* workspace, size_t workspace_bytes,
                              void* stream) {
    if (!router_logits) return FXM_EINVAL;
    return ffn_impl(L, x, topk_ids_out, topk_w_out, router_logits, T, k, y_shared, y, workspace, workspace_bytes, stream);
}

fxm_status fxm_moe_ffn_shared(fxm_layer* L, const void* x, const int32_t* topk_ids, const float* topk_w, int T, int k,
                              const void* y_shared, void* y, void* workspace, size_t workspace_bytes, void* stream) {
    if (!y_shared) return FXM_EINVAL;
    return ffn_impl(L, x, topk_ids, topk_w, nullptr, T, k, y_shared, y, workspace, workspace_bytes, stream);
}

static fxm_status host_impl(fxm_layer* L, const void* x_host, const int32_t* topk_ids_host, const float* topk_w_host,
                            int T, int k, void* y_host, void* workspace, size_t workspace_bytes, void* stream, bool defer_y) {
    if (!L || T < 0 || !workspace || ((uintptr_t)workspace & 1023u)) return FXM_EINVAL;
    if (k < 1 || k > MAX_K || k > L->D.E || (long long)T * k > (1LL << 30)) return FXM_ESHAPE;
    const size_t inner = map_workspace(L->D, T, k, nullptr).bytes;
    const size_t stage = host_stage_bytes(L->D, T, k);
    if (workspace_bytes < inner + stage) return FXM_EWORKSPACE;
    if (T == 0) return FXM_OK;
    if (!x_host || !topk_ids_host || !topk_w_host || !y_host) return FXM_EINVAL;
    if (L->current < 0) return FXM_ESTATE;
    cudaStream_t st = (cudaStream_t)stream;
    const size_t xb = (size_t)T * L->D.d * 2, ab = (size_t)T * k * 4;
    const size_t xs = align_up(xb, 1024), as = align_up(ab, 1024);
    // the staging area sits at the END of the buffer, so it never overlaps the compute workspace of this call
    uint8_t* p = (uint8_t*)workspace + (workspace_bytes & ~(size_t)1023) - stage;
    uint8_t* yd0 = p;
    p += 2 * xs;
    // a capturing stream cannot wait on events recorded outside the capture: copy in-stream then (no overlap)
    cudaStreamCaptureStatus cap = cudaStreamCaptureStatusNone;
    if (cudaStreamIsCapturing(st, &cap) != cudaSuccess) return FXM_ECUDA;
    const bool side = cap == cudaStreamCaptureStatusNone;
    if (side && !L->h2d_stream) {
        if (cudaStreamCreateWithFlags(&L->h2d_stream, cudaStreamNonBlocking) != cudaSuccess) return FXM_ECUDA;
        for (int b = 0; b < 2; ++b)
            if (cudaEventCreateWithFlags(&L->ev_in[b], cudaEventDisableTiming) != cudaSuccess ||
                cudaEventCreateWithFlags(&L->ev_done[b], cudaEventDisableTiming) != cudaSuccess)
                return FXM_ECUDA;
        if (cudaEventCreateWithFlags(&L->ev_tail, cudaEventDisableTiming) != cudaSuccess) return FXM_ECUDA;
        if (cudaStreamCreateWithFlags(&L->d2h_stream, cudaStreamNonBlocking) != cudaSuccess) return FXM_ECUDA;
        for (int b = 0; b < 2; ++b)
            if (cudaEventCreateWithFlags(&L->ev_y[b], cudaEventDisableTiming) != cudaSuccess) return FXM_ECUDA;
    }
    cudaStream_t cs = side ? L->h2d_stream : st;
    // A different (workspace, size, T, k) than the previous host call moves the staging sets -- possibly onto memory the
    // previous call is still using (its compute workspace, its input sets, its y).  Then the copies wait for the WHOLE
    // previous call, and the set rotation starts over (both sets are free once that call is done).
    const bool same_layout = L->host_ws == workspace && L->host_ws_bytes == workspace_bytes && L->host_T == T && L->host_k == k;
    if (side && !same_layout) {
        if (L->host_ws && cudaStreamWaitEvent(cs, L->ev_tail, 0) != cudaSuccess) return FXM_ECUDA;
        // the y buffers move as well: the caller's stream must not write the new ones under a copy that still reads the old
        for (int b = 0; b < 2; ++b)
            if ((L->y_pending >> b) & 1u)
                if (cudaStreamWaitEvent(st, L->ev_y[b], 0) != cudaSuccess || cudaStreamWaitEvent(cs, L->ev_y[b], 0) != cudaSuccess)
                    return FXM_ECUDA;
        L->y_pending = 0;
        L->host_calls = 0;
    }
    const unsigned set = side ? (L->host_calls & 1u) : 0u;
    uint8_t* yd = yd0 + set * xs;
    uint8_t* xd = p + set * (xs + 2 * as);
    uint8_t* idd = xd + xs;
    uint8_t* wd = idd + as;
    // the staging set is free once the kernels of the call before last (same set) have read it
    if (side && L->host_calls >= 2 && cudaStreamWaitEvent(cs, L->ev_done[set], 0) != cudaSuccess) return FXM_ECUDA;
    if (cudaMemcpyAsync(xd, x_host, xb, cudaMemcpyHostToDevice, cs) != cudaSuccess) return FXM_ECUDA;
    if (cudaMemcpyAsync(idd, topk_ids_host, ab, cudaMemcpyHostToDevice, cs) != cudaSuccess) return FXM_ECUDA;
    if (cudaMemcpyAsync(wd, topk_w_host, ab, cudaMemcpyHostToDevice, cs) != cudaSuccess) return FXM_ECUDA;
    if (side) {
        if (cudaEventRecord(L->ev_in[set], cs) != cudaSuccess) return FXM_ECUDA;
        if (cudaStreamWaitEvent(st, L->ev_in[set], 0) != cudaSuccess) return FXM_ECUDA;
    }
    // y buffer `set` is free once the deferred copy of the call before last has read it
    if (side && ((L->y_pending >> set) & 1u)) {
        if (cudaStreamWaitEvent(st, L->ev_y[set], 0) != cudaSuccess) return FXM_ECUDA;
        L->y_pending &= ~(1u << set);
    }
    fxm_status s = fxm_moe_ffn(L, xd, (const int32_t*)idd, (const float*)wd, T, k, yd, workspace, inner, stream);
    if (s != FXM_OK) return s;
    if (side && cudaEventRecord(L->ev_done[set], st) != cudaSuccess) return FXM_ECUDA;
    if (side && defer_y) {
        // y goes back on the library's second stream, under the kernels of the next call; fxm_host_flush (or the reuse of
        // this buffer two calls on) makes the caller's stream wait for it
        if (cudaStreamWaitEvent(L->d2h_stream, L->ev_done[set], 0) != cudaSuccess) return FXM_ECUDA;
        if (cudaMemcpyAsync(y_host, yd, xb, cudaMemcpyDeviceToHost, L->d2h_stream) != cudaSuccess) return FXM_ECUDA;
        if (cudaEventRecord(L->ev_y[set], L->d2h_stream) != cudaSuccess) return FXM_ECUDA;
        L->y_pending |= 1u << set;
    } else if (cudaMemcpyAsync(y_host, yd, xb, cudaMemcpyDeviceToHost, st) != cudaSuccess) {
        return FXM_ECUDA;
    }
    if (side) {
        if (cudaEventRecord(L->ev_tail, defer_y ? L->d2h_stream : st) != cudaSuccess) return FXM_ECUDA;
        ++L->host_calls;
        L->host_ws = workspace; L->host_ws_bytes = workspace_bytes; L->host_T = T; L->host_k = k;
    }
    return FXM_OK;
}

fxm_status fxm_moe_ffn_host(fxm_layer* L, const void* x_host, const int32_t* topk_ids_host, const float* topk_w_host,
                            int T, int k, void* y_host, void* workspace, size_t workspace_bytes, void* stream) {
    return host_impl(L, x_host, topk_ids_host, topk_w_host, T, k, y_host, workspace, workspace_bytes, stream, false);
}

fxm_status fxm_moe_ffn_host_pipelined(fxm_layer* L, const void* x_host, const int32_t* topk_ids_host, const float* topk_w_host,
                                      int T, int k, void* y_host, void* workspace, size_t workspace_bytes, void* stream) {
    return host_impl(L, x_host, topk_ids_host, topk_w_host, T, k, y_host, workspace, workspace_bytes, stream, true);
}

fxm_status fxm_host_flush(fxm_layer* L, void* stream) {
    if (!L) return FXM_EINVAL;
    for (int b = 0; b < 2; ++b)
        if ((L->y_pending >> b) & 1u)
            if (cudaStreamWaitEvent((cudaStream_t)stream, L->ev_y[b], 0) != cudaSuccess) return FXM_ECUDA;
    L->y_pending = 0;
    return FXM_OK;
}

fxm_status fxm_unpack_prefix(fxm_layer* L, int e, int r, void* Wg, void* Wu, void* Wd, void* stream) {
    if (!L || e < 0 || e >= L->D.E) return FXM_EINVAL;
    if (r < 0 || r > L->D.I || (L->clipped && r > L->r_clip[e])) return FXM_EBUDGET;
    if (r == 0) return FXM_OK;
    if (!Wg || !Wu || !Wd) return FXM_EINVAL;
    if (launch_unpack_prefix(L->D, L->V, e, r, (__nv_bfloat16*)Wg, (__nv_bfloat16*)Wu, (__nv_bfloat16*)Wd,
                             (cudaStream_t)stream) != cudaSuccess)
        return FXM_ECUDA;
    return FXM_OK;
}

// ---- offline clipping (Table 2) ------------------------------------------------------

fxm_status fxm_clipped_bytes(int E, int d, int I, const int32_t* r_host, size_t* bytes) {
    Dims D;
    if (!bytes || !r_host) return FXM_EINVAL;
    if (!make_dims(E, d, I, &D)) return FXM_ESHAPE;
    for (int e = 0; e < E; ++e)
        if (r_host[e] < 0 || r_host[e] > I) return FXM_EBUDGET;
    *bytes = clip_total(D, r_host);
    return FXM_OK;
}

fxm_status fxm_export_clipped(fxm_layer* L, const int32_t* r_host, void* blob, size_t blob_bytes, void* stream) {
    if (!L || !r_host || !blob || ((uintptr_t)blob & 1023u)) return FXM_EINVAL;
    fxm_status s = check_table(L, r_host);
    if (s != FXM_OK) return s;
    const Dims& D = L->D;
    if (blob_bytes < clip_total(D, r_host)) return FXM_EWORKSPACE;
    cudaStream_t st = (cudaStream_t)stream;
    uint8_t* b = (uint8_t*)blob;
    const size_t gub = clip_gu_bytes(D, r_host), dnb = clip_dn_bytes(D, r_host);
    const Tail tl = tail_map(D, CLIP_HEADER_BYTES + gub + dnb, false);
    // header: self-description of the blob (fxm_parse_clipped_header reads it back from a host copy).  The words travel
    // in kernel arguments (two tiny launches): no pageable-memory copy, nothing synchronises.
    if (cudaMemsetAsync(b + tl.tables, 0, tl.total - tl.tables, st) != cudaSuccess) return FXM_ECUDA;
    int32_t head[8] = {(int32_t)CLIP_MAGIC, 1, D.E, D.d, D.I, 0, 0, 0};
    static_assert(offsetof(ClipHeader, r) == 32, "clip header layout");
    if (cudaMemsetAsync(b, 0, CLIP_HEADER_BYTES, st) != cudaSuccess) return FXM_ECUDA;
    if (launch_set_table((int*)b, head, 8, st) != cudaSuccess) return FXM_ECUDA;              // words 0..7, zeros up to 255
    if (launch_set_table((int*)(b + 32), r_host, D.E, st) != cudaSuccess) return FXM_ECUDA;   // r[0..E), zeros after
    int* tab0 = (int*)(b + tl.tables);                            // table slot 0 of the new blob: the widths the export kernel reads
    if (launch_set_table(tab0, r_host, D.E, st) != cudaSuccess) return FXM_ECUDA;
    if (launch_export_clipped(D, L->V, tab0, b + CLIP_HEADER_BYTES, b + CLIP_HEADER_BYTES + gub, (uint32_t*)(b + tl.eblk), st) !=
        cudaSuccess)
        return FXM_ECUDA;
    if (cudaMemsetAsync(tab0, 0, sizeof(int) * TABLE_STRIDE, st) != cudaSuccess) return FXM_ECUDA;
    return FXM_OK;
}

fxm_status fxm_parse_clipped_header(const void* host_bytes, size_t n, int* E, int* d, int* I, int32_t* r_out) {
    if (!host_bytes || n < sizeof(ClipHeader) || !E || !d || !I || !r_out) return FXM_EINVAL;
    ClipHeader h;
    std::memcpy(&h, host_bytes, sizeof(h));
    Dims D;
    if (h.magic != CLIP_MAGIC || h.version != 1 || !make_dims(h.E, h.d, h.I, &D)) return FXM_EINVAL;
    for (int e = 0; e < h.E; ++e)
        if (h.r[e] < 0 || h.r[e] > h.I) return FXM_EBUDGET;
    *E = h.E; *d = h.d; *I = h.I;
    std::copy(h.r, h.r + h.E, r_out);
    return FXM_OK;
}

fxm_status fxm_load_clipped(fxm_layer** out, int E, int d, int I, const int32_t* r_host, void* blob, size_t blob_bytes,
                            void* stream) {
    Dims D;
    if (!out || !r_host || !blob || ((uintptr_t)blob & 1023u)) return FXM_EINVAL;
    if (!make_dims(E, d, I, &D)) return FXM_ESHAPE;
    for (int e = 0; e < E; ++e)
        if (r_host[e] < 0 || r_host[e] > I) return FXM_EBUDGET;
    if (blob_bytes < clip_total(D, r_host)) return FXM_EWORKSPACE;
    int sms = 0;
    fxm_status s = device_info(&sms);
    if (s != FXM_OK) return s;
    uint8_t* b = (uint8_t*)blob;
    const size_t gub = clip_gu_bytes(D, r_host), dnb = clip_dn_bytes(D, r_host);
    const Tail tl = tail_map(D, CLIP_HEADER_BYTES + gub + dnb, false);
    fxm_layer* L = new_layer(D, b, tl, sms);
    if (!L) return FXM_ENOMEM;
    L->V.gu = b + CLIP_HEADER_BYTES;
    L->V.dn = b + CLIP_HEADER_BYTES + gub;
    L->clipped = 1;
    L->r_clip.assign(r_host, r_host + E);
    s = init_tail(L, (cudaStream_t)stream);       // tables + state start clean (a blob read back from disk carries stale ones)
    if (s == FXM_OK) s = fxm_set_budget(L, r_host, stream);       // static widths: the exported table is the current one
    if (s != FXM_OK) { fxm_destroy(L); return s; }
    *out = L;
    return FXM_OK;
}

// ---- NEXT-2: channel saliency and ranking (Eq. 2-3) ----------------------------------------------------

fxm_status fxm_saliency_workspace_bytes(int E, int d, int I, size_t* bytes) {
    Dims D;
    if (!bytes) return FXM_EINVAL;
    if (!make_dims(E, d, I, &D)) return FXM_ESHAPE;
    *bytes = saliency_workspace_bytes(D);
    return FXM_OK;
}

fxm_status fxm_saliency(int E, int d, int I, const void* W_gate, const void* W_up, const void* W_down, const void* G_gate,
                        const void* G_up, const void* G_down, int B, float* s_out, void* workspace, size_t workspace_bytes,
                        void* stream) {
    Dims D;
    if (!W_gate || !W_up || !W_down || !G_gate || !G_up || !G_down || !s_out || !workspace || B < 1) return FXM_EINVAL;
    const uintptr_t al = (uintptr_t)W_gate | (uintptr_t)W_up | (uintptr_t)W_down | (uintptr_t)G_gate | (uintptr_t)G_up |
                         (uintptr_t)G_down | (uintptr_t)workspace;
    if (al & 15u) return FXM_EINVAL;
    if (!make_dims(E, d, I, &D)) return FXM_ESHAPE;
    if (workspace_bytes < saliency_workspace_bytes(D)) return FXM_EWORKSPACE;
    if (launch_saliency(D, (const __nv_bfloat16*)W_gate, (const __nv_bfloat16*)W_up, (const __nv_bfloat16*)W_down,
                        (const __nv_bfloat16*)G_gate, (const __nv_bfloat16*)G_up, (const __nv_bfloat16*)G_down, B, s_out,
                        (float*)workspace, (cudaStream_t)stream) != cudaSuccess)
        return FXM_ECUDA;
    return FXM_OK;
}

fxm_status fxm_saliency_static(int E, int d, int I, const void* W_gate, const void* W_up, const void* W_down, const void* G_gate,
                               const void* G_up, const void* G_down, int B, float* s_out, void* stream) {
    Dims D;
    if (!W_gate || !W_up || !W_down || !G_gate || !G_up || !G_down || !s_out || B < 1) return FXM_EINVAL;
    const uintptr_t al = (uintptr_t)W_gate | (uintptr_t)W_up | (uintptr_t)W_down | (uintptr_t)G_gate | (uintptr_t)G_up |
                         (uintptr_t)G_down;
    if (al & 15u) return FXM_EINVAL;
    if (!make_dims(E, d, I, &D)) return FXM_ESHAPE;
    if (saliency_workspace_bytes(D) > SALIENCY_STATIC_BYTES) return FXM_ELIMIT;      // beyond the fixed scratch: use fxm_saliency
    if (launch_saliency_static(D, (const __nv_bfloat16*)W_gate, (const __nv_bfloat16*)W_up, (const __nv_bfloat16*)W_down,
                               (const __nv_bfloat16*)G_gate, (const __nv_bfloat16*)G_up, (const __nv_bfloat16*)G_down, B, s_out,
                               (cudaStream_t)stream) != cudaSuccess)
        return FXM_ECUDA;
    return FXM_OK;
}

fxm_status fxm_rank_channels(int E, int I, const float* s, int32_t* channel_rank_out, void* stream) {
    if (!s || !channel_rank_out) return FXM_EINVAL;
    if (E < 1 || E > MAX_E || I < 1 || !rank_supported(I)) return FXM_ESHAPE;
    if (init_rank_kernel() != cudaSuccess) return FXM_ECUDA;
    if (launch_rank(E, I, s, channel_rank_out, (cudaStream_t)stream) != cudaSuccess) return FXM_ECUDA;
    return FXM_OK;
}

// ---- NEXT-4: training-time action sampling and cost (Eq. 6-7, 10) ------------------------------------------------------

static bool check_ratios(int K, const int32_t* num, int den) {
    if (K < 1 || K > MAX_K || !num || den <= 0) return false;
    for (int k = 0; k < K; ++k)
        if (num[k] < 0 || num[k] > den) return false;
    return true;
}

fxm_status fxm_sample_budget(fxm_layer* L, const float* alpha, const float* gumbel, int K, const int32_t* num_host, int den,
                             int32_t* action_out, void* stream) {
    if (!L || !alpha || !check_ratios(K, num_host, den)) return FXM_EINVAL;
    if (L->clipped) return FXM_ESTATE;                            // a sampled width may exceed what a clipped blob holds
    const int slot = MAX_TABLES - 1;
    if (launch_sample_actions(alpha, gumbel, K, num_host, den, L->D.E, L->D.I, L->tables + (size_t)slot * TABLE_STRIDE,
                              action_out, (cudaStream_t)stream) != cudaSuccess)
        return FXM_ECUDA;
    std::fill(L->host_tables.begin() + (size_t)slot * TABLE_STRIDE, L->host_tables.begin() + (size_t)(slot + 1) * TABLE_STRIDE, -1);
    L->current = slot;
    return FXM_OK;
}

fxm_status fxm_action_cost(fxm_layer* L, const float* alpha, int K, const int32_t* num_host, int den, const int32_t* counts,
                           float* cost_out, void* stream) {
    if (!L || !alpha || !counts || !cost_out || !check_ratios(K, num_host, den)) return FXM_EINVAL;
    if (launch_action_cost(alpha, K, num_host, den, L->D.E, counts, cost_out, (cudaStream_t)stream) != cudaSuccess)
        return FXM_ECUDA;
    return FXM_OK;
}

fxm_status fxm_debug_read_h(fxm_layer* L, const int32_t* topk_ids, int T, int k, void* workspace, void* H_out, int raw,
                            void* stream) {
    if (!L || !workspace || !H_out || !topk_ids || T < 0) return FXM_EINVAL;
    if (L->current < 0) return FXM_ESTATE;
    if (T == 0) return FXM_OK;
    const Workspace ws = map_workspace(L->D, T, k, workspace);
    if (launch_read_h(L->D, T, k, topk_ids, L->tables + (size_t)L->current * TABLE_STRIDE, ws, (__nv_bfloat16*)H_out, raw,
                      (cudaStream_t)stream) != cudaSuccess)
        return FXM_ECUDA;
    return FXM_OK;
}

fxm_status fxm_device_flags(fxm_layer* L, uint32_t* flags, void* stream) {
    if (!L || !flags) return FXM_EINVAL;
    cudaStream_t st = (cudaStream_t)stream;
    uint32_t v = 0;
    const uint32_t hostbits = L->host_flags ? *(volatile uint32_t*)L->host_flags : 0u;   // survives a trapped context
    if (cudaMemcpyAsync(&v, &L->state->flags, sizeof(v), cudaMemcpyDeviceToHost, st) != cudaSuccess ||
        cudaMemsetAsync(&L->state->flags, 0, sizeof(v), st) != cudaSuccess || cudaStreamSynchronize(st) != cudaSuccess) {
        *flags = hostbits | (L->host_flags ? *(volatile uint32_t*)L->host_flags : 0u);
        if (L->host_flags && L->host_flags[1])                   // a pipeline wait timed out: say where (diagnostic)
            std::fprintf(stderr, "flexmoe: wait timed out in block %u thread %u (block size %u) on barrier 0x%x phase %u\n",
                         L->host_flags[1] >> 16, L->host_flags[1] & 0xFFFFu, L->host_flags[3] >> 8, L->host_flags[2],
                         L->host_flags[3] & 1u);
        return FXM_ECUDA;
    }
    const uint32_t hb = L->host_flags ? *(volatile uint32_t*)L->host_flags : 0u;
    if (L->host_flags) *(volatile uint32_t*)L->host_flags = 0u;
    *flags = v | hb | hostbits;
    return FXM_OK;
}

}  // extern "C"
