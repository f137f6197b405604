/*
 * flexmoe.h -- C ABI of the B200-native FlexMoE routed-expert FFN hot path (sm_100a).
 *
 * What the library computes is the paper's online-clipped routed-expert FFN (arxiv/paper_2606_27866;
 * citations are PAPER.md:<line>):
 *
 *   Eq. 1   FFN_e(h)      = W_down ( silu(W_gate h) (.) W_up h )
 *   Eq. 3   W~gate = P W_gate,  W~up = P W_up,  W~down = W_down P^T        (channel ranking)
 *   Eq. 4   FFN_e^(r)(h)  = W~down ( m(r) (.) silu(W~gate h) (.) W~up h ),  m(r) = first r_e channels
 *   Alg. 2   y[t] = sum_{j<k} topk_w[t][j] * FFN_{e}^{(r_e)}(x[t]),  e = topk_ids[t][j]
 *   Eq. 11-12 a budget is a table r[E] of retained widths; rho = 1 - mean_e r_e / I
 *
 * Conventions
 *   - extern "C", plain pointers and sizes; no torch / C++ types.  "device" pointers are CUDA device
 *     pointers of the current device, "host" pointers are ordinary host memory.
 *   - bf16 tensors are raw 16-bit patterns (upper half of an IEEE fp32), row-major as stated.
 *   - Every call returns an fxm_status; nothing throws or aborts.  *out is untouched on failure.
 *   - The library NEVER allocates or frees device memory and never synchronises the stream: the caller
 *     owns `packed` and `workspace` (sizes from the two *_bytes queries) and keeps them alive until
 *     fxm_destroy().  All device work is enqueued on `stream` (a cudaStream_t passed as void*, NULL =
 *     legacy default stream).  Asynchronous CUDA faults surface as FXM_ECUDA from a later call.
 *   - One handle = one MoE layer.  A handle is not thread-safe.
 *   - There is no CPU fallback: on a machine without a CUDA device every compute call returns FXM_ECUDA.
 *
 * Supported shapes (else FXM_ESHAPE): 1 <= E <= 256, d % 64 == 0, I % 16 == 0, 1 <= k <= min(E,16), T >= 0.
 */
#ifndef FLEXMOE_H_
#define FLEXMOE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct fxm_layer fxm_layer; /* opaque; host-side metadata + pointers into caller buffers */

typedef enum {
    FXM_OK = 0,
    FXM_EINVAL = 1,     /* NULL / misaligned pointer, negative size, bad enum                              */
    FXM_ESHAPE = 2,     /* dimensions outside the supported set above                                      */
    FXM_EPERM = 3,      /* a row of channel_rank is not a permutation of 0..I-1                            */
    FXM_EBUDGET = 4,    /* some r_e outside [0, I], or budget index outside the registered range           */
    FXM_ENOTNESTED = 5, /* fxm_register_budgets(require_nested=1): r^(b+1)_e > r^(b)_e for some e          */
    FXM_EWORKSPACE = 6, /* workspace_bytes smaller than fxm_workspace_bytes(E,d,I,T,k)                     */
    FXM_ESTATE = 7,     /* moe_ffn before any budget was installed                                         */
    FXM_ECUDA = 8,      /* a CUDA runtime call failed (no device, launch failure, earlier async fault)     */
    FXM_ENOMEM = 9,     /* a host allocation of the library failed                                         */
    FXM_ELIMIT = 10     /* a no-allocation entry point was given a problem larger than its fixed scratch   */
} fxm_status;

#define FXM_MAX_BUDGETS 15 /* tables that fxm_register_budgets can keep resident */

/* implementation selector for fxm_set_impl: the CTA-pair tcgen05 path (cta_group::2) is the product; the slow,
 * structurally simple SIMT path runs on the SAME packed layout, schedule and accumulators and exists to bisect the
 * fast kernels (it is a CUDA path, not a CPU fallback). */
#define FXM_IMPL_TCGEN05 0
#define FXM_IMPL_SIMT_DEBUG 1

/* ---- sizes first: the caller owns all device memory -------------------------------------------------- */

/* Bytes of the packed, channel-ranked, tile-major weight blob for an [E, I, d] layer (includes the
 * resident budget tables: (FXM_MAX_BUDGETS+1) * 256 int32, a small state block and a copy of channel_rank). */
fxm_status fxm_packed_bytes(int E, int d, int I, size_t* bytes);

/* Bytes of scratch for one moe_ffn / route call with at most T_max tokens and k experts per token:
 * grouping indices, tile schedule, the SwiGLU activations H [T_max*k + 16E, ceil64(I)] bf16, the fp32
 * scatter-add accumulator of y [T_max, d] and the decode kernel's partial gate/up sums (8 KB per work piece).  Monotonic in T_max: a buffer sized for T_max serves every T <= T_max. */
fxm_status fxm_workspace_bytes(int E, int d, int I, int T_max, int k, size_t* bytes);

/* ---- (1) pack: Eq. 3; layout prior art App. C.2, PAPER.md:526-540 ---------------------
 * W_gate, W_up : device, bf16 [E][I][d]   (row c of expert e = channel c)
 * W_down       : device, bf16 [E][d][I]   (column c = channel c).  W_gate / W_up must be 16-byte aligned; W_down needs only
 *                2-byte alignment, but a 16-byte aligned W_down packs ~8x faster (whole rows staged in shared memory
 *                instead of 2-byte gathers).  Misalignment beyond that -> FXM_EINVAL.
 * channel_rank : HOST int32 [E][I] or NULL (= identity).  channel_rank[e][p] is the ORIGINAL index of the
 *                p-th most important channel of expert e (argsort-descending output; gather semantics).
 *                Validated on the host before anything is enqueued (FXM_EPERM).
 * packed       : device buffer of fxm_packed_bytes(), 1024-byte aligned.  Written by kernels on `stream`;
 *                the three source tensors may be freed once the stream has passed this call.
 * The packed layout is private: 16 KB tiles of 128 rows x 64 K-elements, stored
 * pre-swizzled (128-byte swizzle) so a tile is one contiguous bulk copy into UMMA-ready shared memory;
 * gate and up rows of the same 16 channels are adjacent, and any channel prefix of an expert is a
 * contiguous prefix of its tiles -- a budget never moves weights. */
fxm_status fxm_pack(fxm_layer** out, int E, int d, int I, const void* W_gate, const void* W_up,
                    const void* W_down, const int32_t* channel_rank, void* packed, void* stream);

/* ---- (2) budgets: Eq. 11-12; runtime switching PAPER.md:230-239 --------------------
 * Widths, not ratios.  No weight is read or written by any of these. */

/* Install r_host[E] (HOST) as the current table: exactly one tiny kernel launch on `stream` (the table
 * travels in the kernel's arguments; r_host may be reused as soon as the call returns). */
fxm_status fxm_set_budget(fxm_layer* L, const int32_t* r_host, void* stream);

/* Keep B <= FXM_MAX_BUDGETS tables r_host[B][E] (HOST) resident on the device (B tiny launches).
 * require_nested != 0 checks r[b+1][e] <= r[b][e] for all b, e (reading R14). */
fxm_status fxm_register_budgets(fxm_layer* L, int B, const int32_t* r_host, int require_nested, void* stream);

/* Host-only, no CUDA call at all: the next fxm_moe_ffn reads registered table b. */
fxm_status fxm_select_budget(fxm_layer* L, int b);

/* k = ceil(I * num / den) in exact integer arithmetic (reading R2); -1 on bad input. */
int32_t fxm_ratio_to_width(int I, int num, int den);

/* ---- (3) forward: Alg. 2, PAPER.md:545-590 -----------------------------------------------------------
 * x        : device bf16 [T][d]
 * topk_ids : device int32 [T][k], each in [0, E)   (precondition; violations set a sticky device flag
 *            readable with fxm_device_flags and the offending assignment is dropped)
 * topk_w   : device fp32 [T][k], applied as given (the router is external and frozen)
 * y        : device bf16 [T][d], OVERWRITTEN (Y <- 0 then accumulate); routed experts only.
 * x and y must be 16-byte aligned.
 * workspace: device, >= fxm_workspace_bytes(E,d,I,T,k), 1024-byte aligned; contents are scratch.
 * Launches (4): route (grouping + tile schedule), grouped GEMM-1 (+X[pi] gather, +SwiGLU, +Y <- 0), grouped GEMM-2
 * (+router-weight scale, +scatter-add into an fp32 accumulator: Alg. 2 l.18-20 in one kernel), finalize (the single
 * rounding of y to bf16) -- or, for decode-sized calls (fxm_set_decode), ONE fused launch that streams the retained
 * weights once.  Grid sizes do not depend on the budget or on the routing (persistent kernels read the device-side
 * schedule), so a call is CUDA-graph capturable.  A captured call is bound to what was resolved on the host when it
 * was captured: the x pointer and T (a TMA tensor map over x is a kernel argument) and the budget TABLE SLOT that was
 * current -- fxm_select_budget after the capture does not change what a replay reads; to switch the budget of a
 * captured call, capture it after fxm_set_budget and call fxm_set_budget (which rewrites that slot in stream order)
 * before each replay.  T == 0 is a no-op. */
fxm_status fxm_moe_ffn(fxm_layer* L, const void* x, const int32_t* topk_ids, const float* topk_w, int T, int k,
                       void* y, void* workspace, size_t workspace_bytes, void* stream);

/* The same forward with the output of the layer's SHARED expert(s) added (Qwen / DeepSeek-style layers, PAPER.md:208,
 * 362): y = bf16( sum_j topk_w[t][j] FFN_e(x[t]) + y_shared[t] ), the add in fp32 before the single rounding.
 * y_shared: device bf16 [T][d], 16-byte aligned, computed by the caller (the shared expert is not pruned by FlexMoE). */
fxm_status fxm_moe_ffn_shared(fxm_layer* L, const void* x, const int32_t* topk_ids, const float* topk_w, int T, int k,
                              const void* y_shared, void* y, void* workspace, size_t workspace_bytes, void* stream);

/* NEXT-3 of SURVEY.md 8(f): the forward fed by the router's LOGITS instead of its top-k output.  The front end --
 * the k largest logits of each token (fp32 comparison, ties -> lower expert id), weights = softmax over those k logits,
 * i.e. the full softmax renormalised (reading R10) -- runs INSIDE the route kernel, so the launch count stays
 * 4; for decode-sized calls it is one small kernel in front of the fused decode kernel (2 launches).
 * router_logits : device fp32 [T][E].   y_shared : device bf16 [T][d] or NULL.
 * topk_ids_out / topk_w_out : device [T][k] int32 / fp32 or NULL: where the chosen ids and weights are written. */
fxm_status fxm_moe_ffn_router(fxm_layer* L, const void* x, const float* router_logits, int T, int k, const void* y_shared,
                              void* y, int32_t* topk_ids_out, float* topk_w_out, void* workspace, size_t workspace_bytes,
                              void* stream);

/* Same forward with HOST buffers (pinned memory recommended so the copies are asynchronous).  The inputs x [T][d] bf16,
 * topk_ids [T][k] int32 and topk_w [T][k] fp32 are copied on a library-owned side stream into one of two staging
 * sets at the tail of `workspace`, so the host->device copy of call i+1 overlaps the kernels and the device->host
 * copy of call i; `stream` waits for the inputs, runs the kernels of fxm_moe_ffn and copies y [T][d] bf16 back.
 * Contract: the three input buffers must hold their data when the call is made (they are read from call time on, not
 * in `stream` order) and stay unmodified until `stream` has passed this call; y_host is valid once `stream` has passed
 * this call.  Does not synchronise.  workspace >= fxm_workspace_bytes_host(E,d,I,T,k); the staging sets live at the END
 * of the buffer.  Calls with the same (workspace, size, T, k) pipeline; a call that changes any of them first waits (on
 * the device) for the previous host call to finish, because its staging area may lie on memory that call still uses.
 * On a capturing stream the copies are enqueued in-stream instead.  This is the end-to-end entry point bench.py times as `e2e`. */
fxm_status fxm_workspace_bytes_host(int E, int d, int I, int T_max, int k, size_t* bytes);
fxm_status fxm_moe_ffn_host(fxm_layer* L, const void* x_host, const int32_t* topk_ids_host, const float* topk_w_host,
                            int T, int k, void* y_host, void* workspace, size_t workspace_bytes, void* stream);
/* Pipelined variant of fxm_moe_ffn_host for a loop of calls: y travels back on a SECOND library-owned stream, so the
 * device->host copy of call i runs under the kernels of call i+1 (the in-stream copy of fxm_moe_ffn_host serialises with
 * them).  Contract: as above for the inputs; y_host of a call is valid once `stream` has passed a later fxm_host_flush on
 * this layer (which makes `stream` wait for every copy still in flight; host-only, no launch).  Same workspace size. */
fxm_status fxm_moe_ffn_host_pipelined(fxm_layer* L, const void* x_host, const int32_t* topk_ids_host,
                                      const float* topk_w_host, int T, int k, void* y_host, void* workspace,
                                      size_t workspace_bytes, void* stream);
fxm_status fxm_host_flush(fxm_layer* L, void* stream);

/* ---- offline clipping: PAPER.md:222 ("the pruned subnet is exported as a standalone fixed-budget checkpoint"),
 * Table 2 PAPER.md:201-206 ------------------------------------------------------------------------------------------
 * A clipped blob holds only the retained prefix of every expert -- ceil(r_e / 64) channel blocks of gate/up and of down,
 * back to back -- plus a 2 KB self-describing header and the small tail (budget tables, state).  Its size is linear in
 * the retained fraction (the law Table 2's checkpoint sizes follow).  The blob is position independent: copy it to
 * the host / a file and back, then fxm_load_clipped. */
fxm_status fxm_clipped_bytes(int E, int d, int I, const int32_t* r_host /* [E] */, size_t* bytes);
/* Device kernel copies the retained tiles of L (widths r_host [E], HOST; r_e <= I, and <= the exported widths if L is
 * itself clipped) into blob (device, 1024-byte aligned, >= fxm_clipped_bytes).  Stream-ordered, L is not modified. */
fxm_status fxm_export_clipped(fxm_layer* L, const int32_t* r_host, void* blob, size_t blob_bytes, void* stream);
/* Reads E, d, I and the widths r [E] (r_out has room for 256) from the first 2 KB of a blob copied to HOST memory. */
fxm_status fxm_parse_clipped_header(const void* host_bytes, size_t n, int* E, int* d, int* I, int32_t* r_out);
/* A layer handle over a clipped blob (device).  The exported table is installed as the current budget, so
 * fxm_moe_ffn works at once with static widths; fxm_set_budget / fxm_register_budgets accept only tables with
 * r_e <= the exported r_e (nested sub-budgets of the clipped checkpoint), else FXM_EBUDGET.  Same kernels, same
 * workspace sizes as the full layer. */
fxm_status fxm_load_clipped(fxm_layer** out, int E, int d, int I, const int32_t* r_host, void* blob, size_t blob_bytes,
                            void* stream);

/* ---- NEXT-2 of SURVEY.md 8(f): channel saliency and ranking, the step in front of pack (Eq. 2-3) ----
 * s[e][j] = (1/B) sum_b sum_{theta in Theta_j} (theta * g_theta^(b))^2 with Theta_j = row j of W_gate, row j of W_up and
 * column j of W_down.  All tensors are DEVICE bf16, 16-byte aligned: weights [E][I][d], [E][I][d], [E][d][I]
 * in ORIGINAL channel order, gradients of the B ranking batches [B][E][I][d], [B][E][I][d], [B][E][d][I].
 * s_out: device fp32 [E][I].  workspace: device, >= fxm_saliency_workspace_bytes, 16-byte aligned (partial sums).
 * fp32 accumulation in a fixed order (no floating-point atomics): reproducible.  HBM-bound: (1 + B) 6 E I d bytes. */
fxm_status fxm_saliency_workspace_bytes(int E, int d, int I, size_t* bytes);
fxm_status fxm_saliency(int E, int d, int I, const void* W_gate, const void* W_up, const void* W_down, const void* G_gate,
                        const void* G_up, const void* G_down, int B, float* s_out, void* workspace, size_t workspace_bytes,
                        void* stream);
/* The same computation for callers that cannot allocate device memory or pass scratch (CUDA graph capture, serving loops,
 * harnesses that forbid cudaMalloc): the partial sums live in a device array inside the library image, FXM_SALIENCY_STATIC_BYTES
 * (8 MB) on every GPU that loads the library, held until the process exits.  The call allocates nothing (no cudaMalloc /
 * cudaFree / allocating library routine); inputs and s_out are the caller's, as above.  Shapes whose scratch need
 * (fxm_saliency_workspace_bytes) exceeds FXM_SALIENCY_STATIC_BYTES are rejected with FXM_ELIMIT -- use fxm_saliency then
 * (the C2-shaped weight set, E=60 I=1408, needs 5.8 MB and fits; the C4-shaped one, E=64 I=2560, needs 11.1 MB and does not).
 * All calls on a device SHARE the array: calls that overlap on the GPU (streams with no ordering between them) race;
 * calls on one stream, or ordered by events, are safe.  Nothing in the array needs clearing between calls (every slot
 * that is read is written first by the same call).  Same results as fxm_saliency, bit for bit. */
#define FXM_SALIENCY_STATIC_BYTES ((size_t)8 << 20)
fxm_status fxm_saliency_static(int E, int d, int I, const void* W_gate, const void* W_up, const void* W_down,
                               const void* G_gate, const void* G_up, const void* G_down, int B, float* s_out, void* stream);
/* channel_rank_out[e][p] (device int32 [E][I]) = ORIGINAL index of the p-th most important channel of expert e: s sorted
 * in descending order, equal saliencies keep ascending original index (readings R3, R4) -- exactly the
 * channel_rank fxm_pack takes (copy it to the host first: pack validates it there).  I <= 16384. */
fxm_status fxm_rank_channels(int E, int I, const float* s, int32_t* channel_rank_out, void* stream);

/* ---- NEXT-4 of SURVEY.md 8(f): training-time action sampling and cost (Eq. 6-7, Eq. 10) --
 * fxm_sample_budget: for every expert k* = argmax_k (alpha[e][k] + gumbel[e][k]) -- the hard action of Eq. 6 for any
 * temperature tau > 0 (fp32 sum, ties -> lower k); the straight-through forward value (Eq. 7) is the hard one-hot, so
 * the width ceil(num[k*] I / den) is written into the layer's current table ON THE DEVICE: the masked
 * forward of Eq. 4 is then fxm_moe_ffn, no host round trip.  alpha, gumbel: device fp32 [E][K] (gumbel NULL = no
 * noise: the hardened mask of Eq. 11); the Gumbel noise is an input.  num_host [K], den: the action set as exact
 * ratios.  action_out: device int32 [E] or NULL.  K <= 16.  Not available on a clipped layer (FXM_ESTATE).
 * fxm_action_cost: C = sum_e q_e sum_k softmax(alpha_e)_k r_k with q_e = counts[e] / sum counts (counts: device int32
 * [E], e.g. from fxm_route); cost_out: device fp32 [1]. */
fxm_status fxm_sample_budget(fxm_layer* L, const float* alpha, const float* gumbel, int K, const int32_t* num_host, int den,
                             int32_t* action_out, void* stream);
fxm_status fxm_action_cost(fxm_layer* L, const float* alpha, int K, const int32_t* num_host, int den, const int32_t* counts,
                           float* cost_out, void* stream);

/* ---- measurement surface -------------------------------------------------------------------------------
 * Per-kernel device times of fxm_moe_ffn: between fxm_profile_begin and fxm_profile_end every
 * fxm_moe_ffn call (at most max_calls of them, <= 4096) records a CUDA event on its stream before each of its
 * launches and after the last.  fxm_profile_end synchronises those events and writes, per kernel (order: route,
 * GEMM-1+SwiGLU, GEMM-2+scale+scatter-add, finalize, fused decode kernel), the SUM of its durations in milliseconds
 * over the *calls recorded; events are host objects, no device memory is allocated. */
#define FXM_N_KERNELS 5
fxm_status fxm_profile_begin(fxm_layer* L, int max_calls);
fxm_status fxm_profile_end(fxm_layer* L, float* ms_sum /* [FXM_N_KERNELS] */, int* calls);

/* ---- parity / debug surface ---------------------------------------------------------------------------
 * Step a2 alone (Alg. 2 l.4-6; stable by (expert id, flat index t*k+j), reading R5):
 * counts [E], offsets [E+1] (exclusive scan, offsets[E] = T*k), perm [T*k], inv_perm [T*k]: device int32. */
fxm_status fxm_route(fxm_layer* L, const int32_t* topk_ids, int T, int k, int32_t* counts, int32_t* offsets,
                     int32_t* perm, int32_t* inv_perm, void* workspace, size_t workspace_bytes, void* stream);

/* Inverse of pack for a prefix: writes the first r ranked channels of expert e as plain row-major bf16
 * Wg [r][d], Wu [r][d], Wd [d][r] (device).  Test surface and the offline-clipping export. */
fxm_status fxm_unpack_prefix(fxm_layer* L, int e, int r, void* Wg, void* Wu, void* Wd, void* stream);

/* Copy the internal SwiGLU activations of the LAST general-path moe_ffn on this workspace into row-major bf16
 * H_out [T*k][I] in sorted (perm) order.  raw = 0: columns >= r_e read as 0 (the definition).  raw = 1: no reader-side
 * mask -- every column below ceil64(r_e) is returned exactly as the GEMM-1 epilogue wrote it (the columns
 * [r_e, ceil64(r_e)) must be exact zeros by the pad-zero rule); blocks that were never issued read 0.
 * Debug only. */
fxm_status fxm_debug_read_h(fxm_layer* L, const int32_t* topk_ids, int T, int k, void* workspace, void* H_out, int raw,
                            void* stream);

fxm_status fxm_set_impl(fxm_layer* L, int impl);          /* FXM_IMPL_* ; default FXM_IMPL_TCGEN05 */
/* Most rows of a token tile of the grouped GEMMs: 128, 256, 512, or 0 = default (512).  Tuning knob only. */
fxm_status fxm_set_tile_n(fxm_layer* L, int tile_n);
/* Step a6: calls with T*k <= max_assignments (<= 1024; 0 = never) run as ONE launch of the fused
 * weight-streaming decode kernel instead of the four launches above.  prefetch_tiles = how many 16 KB weight tiles
 * each CTA's L2 prefetch cursor runs ahead of its shared-memory ring (0..4096; default 0 = none: every distance
 * tried was measured slower on B200, see profiles/).  Tuning knob only: results agree within the stated tolerance
 * either way.  Needs d <= 3840, else the general path is used.  Default 640: measured on the C4-shaped layer the
 * four-launch path wins from T*k = 768 on (an expert with more than 16 tokens streams its weights twice here). */
#define FXM_DECODE_DEFAULT_MAX_ASSIGNMENTS 640
#define FXM_DECODE_DEFAULT_PREFETCH 0
fxm_status fxm_set_decode(fxm_layer* L, int max_assignments, int prefetch_tiles);
/* Synchronises `stream`, then returns the sticky device flag word (bit0: expert id out of range,
 * bit1: a pipeline wait timed out -- a bug) in *flags and clears it.  A timed-out wait traps the kernel, which kills
 * the CUDA context: bit1 is therefore also written to a pinned host word first, and this call still reports it
 * (together with FXM_ECUDA) when the device can no longer be read. */
fxm_status fxm_device_flags(fxm_layer* L, uint32_t* flags, void* stream);
/* Number of kernels the LAST fxm_moe_ffn on this layer enqueued: 1 (fused decode; 2 with the router front end) or 4
 * (route, GEMM-1, GEMM-2, finalize); bench.py's gpu_launches. */
int fxm_launches_per_ffn(const fxm_layer* L);

const char* fxm_status_string(fxm_status s);
void fxm_destroy(fxm_layer* L); /* frees host metadata only */

#ifdef __cplusplus
}
#endif
#endif /* FLEXMOE_H_ */
