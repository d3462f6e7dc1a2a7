/*
 * esc.h — C ABI of the execution-state-capsule hot path on B200 (sm_100a).
 *
 * What this boundary is.  arxiv/paper_2606_20537 puts the capsule on "a minimal execution
 * contract — three handle types, one opaque shape key, a strict mechanism-not-policy
 * boundary" that "sees only streams, graphs, events, and named buffers"
 * (Listing 1 caption; the listing body is not in PAPER.md).  The verbs and
 * their argument order follow Algorithm 1 and Listing 2
 * (PAPER.md:149-157); the scan call follows BASELINE.json north_star
 * `linattn_scan(q,k,v,g,state_in,state_out,T,chunk)` (+ the output `o`).
 *
 * Handles (3):  esc_ctx     device + library state
 *               esc_bufset  a named buffer set — either a LIVE set (the graph-bound
 *                           buffers a session runs on) or a FROZEN twin = the capsule
 *                           (bytes + boundary descriptor)
 *               esc_graph   a captured replay plan (restore + suffix scan)
 * Shape key (1): esc_shape_key, opaque to the caller.
 *
 * Conventions
 *   - Every call returns int: ESC_OK (0) or a negative ESC_ERR_*; never throws, never
 *     aborts.  Out-parameters come last and are written only on success.
 *   - "dev" pointers are CUDA device pointers, "host" pointers are ordinary host memory.
 *   - Ownership: the library NEVER allocates or frees tensor memory.  Live buffers and
 *     capsule storage slabs are caller-owned device memory (the Python binding uses
 *     torch tensors), and so is the few-KiB device scratch an esc_graph keeps its
 *     "current capsule" descriptor table in (esc_graph_scratch_bytes).  The library owns
 *     only its small host structs.
 *   - Devices: a handle belongs to its context's device.  Every verb runs on that device
 *     whatever the calling thread's current device is and leaves the current device as it
 *     found it; kernel attributes are tracked per context, so several contexts (one per GPU)
 *     may live in one process.  A context may be used from several host threads as long as
 *     calls on the same live set / graph / plan table are serialised by the caller.
 *   - Streams: every verb only ENQUEUES work on the caller's cudaStream_t (passed as
 *     void*; NULL = legacy default stream) and returns without a host sync.  Everything
 *     the host can detect (bad arguments, layout / digest mismatch, unaligned boundary,
 *     capacity) is reported BEFORE anything is enqueued: "fails loudly rather than a
 *     partial capsule".
 *   - No CPU fallback exists: without a CUDA device esc_ctx_create fails.
 */
#ifndef ESC_H_
#define ESC_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define ESC_ABI_VERSION 3u   /* 3: esc_scan_args gained `kind` (was reserved) and `beta`: gated delta-rule layers in a captured plan */

/* ---- error codes -------------------------------------------------------------------- */
#define ESC_OK               0
#define ESC_ERR_INVALID     -1   /* NULL / out-of-range argument, handle of the wrong kind    */
#define ESC_ERR_UNALIGNED   -2   /* boundary not a chunk multiple, pointer not 16-B aligned    */
#define ESC_ERR_MISMATCH    -3   /* layout digest / prefix digest / position mismatch          */
#define ESC_ERR_CAPACITY    -4   /* valid range at P exceeds a buffer, or the slab is too small */
#define ESC_ERR_UNSUPPORTED -5   /* shape / dtype / chunk the kernels do not implement          */
#define ESC_ERR_CUDA        -6   /* a CUDA runtime call failed (see esc_last_cuda_error)        */

/* Human-readable name of a return code (static string, never NULL). */
const char* esc_strerror(int code);
/* ESC_ABI_VERSION the library was built with. */
uint32_t esc_abi_version(void);
/* cudaError_t of the most recent ESC_ERR_CUDA on this host thread (0 if none). */
int esc_last_cuda_error(void);

/* ---- handles ------------------------------------------------------------------------ */
typedef struct esc_ctx    esc_ctx;
typedef struct esc_bufset esc_bufset;
typedef struct esc_graph  esc_graph;
typedef uint64_t          esc_shape_key;

/* Create / destroy the per-device context.  `device` is a CUDA ordinal.  Fails with
 * ESC_ERR_CUDA when there is no such device and ESC_ERR_UNSUPPORTED when the device is not
 * compute capability 10.x (the library holds sm_100a code only). */
int esc_ctx_create(int device, esc_ctx** out_ctx);
int esc_ctx_destroy(esc_ctx* ctx);
/* Number of SMs of the context's device (grid sizing of the persistent kernels). */
int esc_ctx_sm_count(const esc_ctx* ctx, int* out_sms);

/* ---- named buffer sets (the live set B over contiguous buffers) -- */
/*
 * One named buffer ("row").  Its valid bytes at token boundary P are, for each of its
 * n_seg segments (segment s starts at dev_ptr + s*seg_stride):
 *        fixed_bytes + P * bytes_per_token
 *   fold state (fixed size):   fixed_bytes = H*dk*dv*4, bytes_per_token = 0
 *   token-major KV [T_max, H_kv, D] ("valid over [0,P)"):
 *                                               bytes_per_token = H_kv*D*elem, n_seg = 1
 *   head-major KV [H_kv, T_max, D]:             bytes_per_token = D*elem, n_seg = H_kv,
 *                                               seg_stride = T_max*D*elem
 * `name` is copied.  dev_ptr must be 16-byte aligned for the vector path; any other
 * alignment / byte count is still copied exactly (byte path).
 */
typedef struct esc_buf_desc {
    const char* name;            /* host string, copied                                  */
    void*       dev_ptr;         /* device base address, caller-owned                    */
    uint64_t    capacity_bytes;  /* bytes allocated behind dev_ptr                       */
    uint64_t    fixed_bytes;
    uint64_t    bytes_per_token;
    uint32_t    n_seg;           /* >= 1                                                 */
    uint32_t    reserved;        /* must be 0                                            */
    uint64_t    seg_stride;      /* bytes between segment starts (ignored when n_seg==1) */
} esc_buf_desc;

#define ESC_MAX_ROWS      256u
#define ESC_POSITION_UNKNOWN UINT64_MAX

/* Register a LIVE buffer set (host side, once, off the hot path). */
int esc_bufset_create(esc_ctx* ctx, const esc_buf_desc* descs, uint32_t n_rows, esc_bufset** out_set);
/* Destroy a live set or a capsule handle (never frees device memory). */
int esc_bufset_destroy(esc_bufset* set);
/* FNV-1a-64 over (layout version, row names, fixed_bytes, bytes_per_token, n_seg): two sets
 * with the same digest have the same capsule layout (pointers, capacities and strides are
 * not part of it).  PAPER.md:121,124 "digest". */
int esc_bufset_layout_digest(const esc_bufset* set, uint64_t* out_digest);
/* Token position the live set currently holds.  Restore / fork / rollback set it to the
 * capsule's boundary; the caller advances it after appending tokens.  A fresh set is at
 * ESC_POSITION_UNKNOWN (no position checks are applied until it is set). */
int esc_bufset_set_position(esc_bufset* live, uint64_t position);
int esc_bufset_get_position(const esc_bufset* set, uint64_t* out_position);

/* Bytes of the storage slab a capsule of `set` at boundary P needs (padding included) and
 * the payload (sum of valid bytes; what Table 7's "capsule size" counts).
 * Slab layout contract: rows in table order, each row starting at the next multiple of
 * 256 B, each segment inside a row at the next multiple of 16 B; padding is don't-care.
 * ESC_ERR_CAPACITY when a valid range would exceed its buffer. */
int esc_capsule_bytes(const esc_bufset* set, uint64_t P, uint64_t* out_slab_bytes, uint64_t* out_payload_bytes);

/* P' = floor(P / chunk) * chunk  (Algorithm 1 line "align P"; §5).
 * chunk == 0 returns P. */
uint64_t esc_align_boundary(uint64_t P, uint64_t chunk);

/* ---- capsule verbs (Algorithm 1) ------------------------------------ */
#define ESC_SNAPSHOT_ALLOW_UNALIGNED 1u   /* accept P % chunk != 0 (tolerance-only restores) */

/*
 * snapshot(P): copy every row's valid bytes at boundary P from the live buffers into
 * `storage_dev` (one kernel launch on `stream`) and return a FROZEN bufset — the capsule
 * (PAPER.md:117-122).  The capsule records P, chunk, the layout digest and the caller's
 * opaque `prefix_digest`.
 *   chunk > 0 and P % chunk != 0  -> ESC_ERR_UNALIGNED unless flags has ALLOW_UNALIGNED
 *                                    (a fold state cannot be sliced after the fact,
 *                                    PAPER.md:72; the caller stops its prefill at
 *                                    esc_align_boundary(P, chunk) and snapshots there)
 *   live position known and != P  -> ESC_ERR_MISMATCH
 *   storage_bytes too small       -> ESC_ERR_CAPACITY;   storage not 256-B aligned -> ESC_ERR_UNALIGNED
 * The capsule is read-only afterwards; any number of restores / forks may read it.
 * The storage must stay allocated until the capsule handle is destroyed.
 */
int esc_snapshot(esc_bufset* live, uint64_t P, uint64_t chunk, uint64_t prefix_digest, uint32_t flags,
                 void* storage_dev, uint64_t storage_bytes, void* stream, esc_bufset** out_capsule);

/*
 * restore(cap): copy the capsule's bytes back into the live rows' valid ranges (one kernel
 * launch) and rebind the live position to the capsule's boundary.
 * Bytes beyond a row's valid range are left untouched.  If `expect_prefix_digest` is not
 * NULL it must equal the capsule's ("assert digest"), else ESC_ERR_MISMATCH.
 * Layout digests of `live` and `capsule` must match (ESC_ERR_MISMATCH); every valid range
 * must fit the live buffers (ESC_ERR_CAPACITY).
 */
int esc_restore(esc_bufset* live, const esc_bufset* capsule, const uint64_t* expect_prefix_digest, void* stream);

/*
 * fork(cap, n): restore the capsule into n live sets.  One kernel launch
 * reads each capsule byte once and writes it n times; the result is byte-identical to n
 * esc_restore calls.  1 <= n <= ESC_MAX_FORK.
 */
#define ESC_MAX_FORK 16u
int esc_fork(const esc_bufset* capsule, esc_bufset* const* lives, uint32_t n, void* stream);

/*
 * rollback(cap_earlier): restore of an earlier boundary of the same session
 * (PAPER.md:112,137).  Same as esc_restore plus: the live position, when known, must be
 * >= the capsule's boundary (ESC_ERR_MISMATCH otherwise).
 */
int esc_rollback(esc_bufset* live, const esc_bufset* capsule_earlier, void* stream);

typedef struct esc_capsule_info {
    uint64_t boundary;        /* P' the capsule was taken at                      */
    uint64_t chunk;           /* chunk it was aligned to (0 = none stated)        */
    uint64_t slab_bytes;      /* bytes of storage used, padding included          */
    uint64_t payload_bytes;   /* sum of valid bytes                               */
    uint64_t layout_digest;
    uint64_t prefix_digest;   /* opaque caller value                              */
    uint32_t n_rows;
    uint32_t n_segments;      /* rows x segments = entries of the copy table      */
    uint32_t aligned;         /* 1 when boundary % chunk == 0 (or chunk == 0)     */
    uint32_t tier;            /* ESC_TIER_GPU or ESC_TIER_HOST                     */
} esc_capsule_info;
int esc_capsule_info_get(const esc_bufset* capsule, esc_capsule_info* out_info);
/* Valid end (bytes per segment) of row `row` at the capsule's boundary (PAPER.md:86
 * "valid ends" in the descriptor). */
int esc_capsule_valid_end(const esc_bufset* capsule, uint32_t row, uint64_t* out_bytes_per_segment);

/* ---- tiers (Algorithm 1: "return tiered handle" PAPER.md:122, "promote if off-GPU" PAPER.md:125-126) ----
 * The one mechanism the capsule adds to the contract is "host-backed buffers and cross-space asynchronous
 * copy"; which capsule lives where, and when, is serving policy and stays
 * with the caller.  A capsule's storage slab is ONE contiguous range, so a tier move is one async copy.
 *   demote : GPU-tier capsule -> caller-owned PINNED host storage (cudaHostAlloc / cudaHostRegister / torch
 *            pin_memory; ESC_ERR_INVALID for pageable memory), one async D2H copy of slab_bytes on `stream`.
 *            Returns a HOST-tier capsule handle; the GPU-tier one stays valid (the caller frees its slab
 *            when it wants the memory back).
 *   promote: HOST-tier capsule -> caller-owned device storage (256-B aligned), one async H2D copy.
 * esc_restore / esc_rollback / esc_fork / esc_graph_set_capsule also take a HOST-tier capsule directly: the
 * copy kernel then reads the pinned slab over the host link (zero-copy), i.e. promotion is fused into the
 * restore and the bytes cross the link once and land in place — "promotion is the only non-sub-ms step"
 * (PAPER.md:161).  Same layout, digests, boundary and byte-exactness as the GPU tier. */
#define ESC_TIER_GPU  0u
#define ESC_TIER_HOST 1u
int esc_capsule_demote(const esc_bufset* capsule, void* storage_host, uint64_t storage_bytes, void* stream,
                       esc_bufset** out_host_capsule);
int esc_capsule_promote(const esc_bufset* host_capsule, void* storage_dev, uint64_t storage_bytes, void* stream,
                        esc_bufset** out_capsule);

/* ---- FP8 KV rows and their BF16 dequantisation stage (reading 23) -----------
 * On the long-context route the persistent KV is FP8 and a BF16 working stage is derived from it; the capsule
 * holds the FP8 bytes only ("FP8-KV roughly halves it") plus the stage's valid end as metadata,
 * and "the FP8 -> BF16 working stage is rebuilt lazily on the next read, not eagerly in restore".
 *   attach : declare that live row `row` (a pure per-token row: fixed_bytes == 0) holds FP8 E4M3 codes and has a
 *            caller-owned BF16 stage of the same shape: stage segment s starts at stage_dev + s * 2 * seg_stride,
 *            stage element i = bf16_rne(fp32(decode(code_i)) * scale); NaN codes -> 0x7FC0 | sign.  The stage is not
 *            part of the capsule or of the layout digest.  stage_capacity_bytes >= 2 x the row's capacity.
 *   valid end: tokens [0, end) of the stage are in sync with the row.  Host-tracked: esc_restore / esc_rollback /
 *            esc_fork / esc_graph_launch reset it to 0 (the paper's lazy rule); esc_dequant_stage_fill rebuilds
 *            tokens [end, upto) from the live FP8 row with one kernel launch and sets end = upto; a snapshot
 *            records the live value in the capsule (readable with the same call on the capsule handle).
 *   esc_restore_ex(flags = ESC_RESTORE_DEQUANT_EAGER): restore AND rebuild every attached stage over [0, P) in the
 *            same single kernel launch (each capsule byte is read once and written as FP8 to the row and as BF16 to
 *            the stage); sets every valid end to P.  flags = 0 is esc_restore. */
#define ESC_FORMAT_FP8_E4M3 1u
#define ESC_RESTORE_DEQUANT_EAGER 1u
#define ESC_ALL_ROWS UINT32_MAX            /* esc_dequant_stage_fill: every row that has a stage, one kernel launch */
int esc_bufset_attach_dequant_stage(esc_bufset* live, uint32_t row, void* stage_dev, uint64_t stage_capacity_bytes,
                                    uint32_t format, float scale);
int esc_dequant_stage_valid_end(const esc_bufset* set, uint32_t row, uint64_t* out_tokens);
int esc_dequant_stage_fill(esc_bufset* live, uint32_t row, uint64_t upto_tokens, void* stream);
int esc_restore_ex(esc_bufset* live, const esc_bufset* capsule, const uint64_t* expect_prefix_digest, uint32_t flags,
                   void* stream);

/* ---- restore without caller scratch and without device allocation ---------------------------------------------------
 * esc_restore_static: esc_restore (same pairing rules, same bytes written, same position / stage bookkeeping) for callers
 * that cannot call cudaMalloc or hand over scratch: code under someone else's stream capture, tight serving loops, harnesses
 * that forbid allocation.  It runs the table-in-global-memory copy kernel of the graph path (esc_graph_scratch_bytes) with
 * its descriptor tables in a static device array inside the library: 13 KiB that every GPU which loads the library holds
 * until exit.  No cudaMalloc / cudaFree / allocating routine is called; per 112 segments one table-store launch and one copy
 * launch on `stream`.
 *   Limit: the (live set, boundary) pair may have at most ESC_RESTORE_STATIC_MAX_SEGMENTS (row, segment) entries, else
 *          ESC_ERR_CAPACITY and nothing is enqueued (esc_restore has no such limit).
 *   Sharing: every call on a device uses the same tables, which keep the last call's contents (a call rewrites every word
 *          it uses; nothing needs clearing).  Calls are ordered by their stream; calls whose kernels may overlap on the GPU
 *          (different streams with no event between them, different host threads) race on the tables and must be
 *          serialised by the caller. */
#define ESC_RESTORE_STATIC_MAX_SEGMENTS 448u
uint32_t esc_restore_static_max_segments(void);
int esc_restore_static(esc_bufset* live, const esc_bufset* capsule, const uint64_t* expect_prefix_digest, void* stream);

/* ---- chunked gated linear-attention scan ---------------------------------------------- */
#define ESC_DTYPE_BF16 1u
#define ESC_DTYPE_F32  2u

/* Opaque shape key.  Encodes (B, H, d_k, d_v, in_dtype, out_dtype, chunk)
 * and nothing about T: the same key — hence the same kernel and the same arithmetic —
 * serves a cold run and a restore-then-continue run, which is what makes a chunk-aligned
 * restore + continue bit-identical to the cold run.
 * Returns 0 for a combination the library does not implement.
 * Implemented: in_dtype BF16 (q,k,v), out_dtype F32 or BF16 (o), d_k,d_v in {64,128},
 * chunk in {64,128}, 1 <= B*H <= 65535. */
esc_shape_key esc_shape_key_make(uint32_t B, uint32_t H, uint32_t d_k, uint32_t d_v,
                                 uint32_t in_dtype, uint32_t out_dtype, uint32_t chunk);

/* The d_v tile of the scan kernel for `key` on the context's device (16 or 32 columns per CTA).  It is a function of the
 * key and the device only — T never enters — which is what lets a cold run and a restore-then-continue run of one key share
 * their arithmetic bit for bit.  Informational: the tests assert the property through it. */
int esc_scan_tile_columns(const esc_ctx* ctx, esc_shape_key key, uint32_t* out_columns);

/*
 * linattn_scan: for every (b,h), with S_0 = state_in[b,h],
 *      S_t = g_t * S_{t-1} + k_t^T v_t ,   o_t = q_t S_t ,   state_out[b,h] = S_T
 * (BASELINE.json north_star; the paper only says the state is "a fold over the entire
 * prefix", folded "per chunk"), evaluated chunk by chunk:
 *      b_i = sum_{r<=i in chunk} ln g_r
 *      o_i    = exp(b_i) q_i S_prev + sum_{j<=i} exp(b_i - b_j) (q_i . k_j) v_j
 *      S_next = exp(b_C) S_prev + sum_i exp(b_C - b_i) k_i^T v_i
 * Layouts (device, contiguous innermost): q,k [B, T_stride, H, d_k] and v [B, T_stride, H, d_v]
 * in in_dtype; g [B, T_stride, H] fp32 in (0,1]; o [B, T_stride, H, d_v] in out_dtype;
 * state_in / state_out [B, H, d_k, d_v] fp32.  Pointers address the FIRST token to scan;
 * `t_stride` (>= T) is the number of tokens between consecutive batch rows.  Only tokens
 * [0,T) of each batch row are read / written.  T need not be a chunk multiple (the last
 * chunk is short).  T == 0 copies state_in to state_out.  state_in may be NULL (= zeros)
 * and may alias state_out.  q, k, v, o and the states 16-byte aligned, g 4-byte aligned
 * (ESC_ERR_UNALIGNED).
 * `chunk` must equal the key's chunk (ESC_ERR_MISMATCH): it is the alignment grid of restore boundaries the caller
 * commits to; the kernel's internal token tile is 64 for both values.  One kernel launch on `stream`.
 */
int esc_linattn_scan(esc_ctx* ctx, esc_shape_key key,
                     const void* q, const void* k, const void* v, const float* g,
                     const float* state_in, float* state_out, void* o,
                     uint64_t T, uint64_t t_stride, uint32_t chunk, void* stream);

/* ---- gated delta rule and convolution state (reading 25) -------------
 * The recurrence and the convolution window of the paper's own hybrid-model family; both are folds over the whole prefix
 * and both are capsule rows (the fold state like any esc_linattn_scan state, the convolution window as a fixed-size row).
 *
 * esc_gdn_scan: for every (b,h), S_0 = state_in[b,h]:
 *      u_t = k_t (a_t S_{t-1}) ,  S_t = a_t S_{t-1} + beta_t k_t^T (v_t - u_t) ,  o_t = q_t S_t ,  state_out = S_T
 * Layouts, alignment and aliasing rules as esc_linattn_scan; `g` holds a_t in (0,1], `beta` [B, T_stride, H] fp32 in [0,1];
 * keys are expected L2-normalised by the caller.  Evaluated in the chunked (WY) form, 64 tokens at a time, on tcgen05 tensor
 * cores (fp32 state, two-term bf16 operand splits): restore + continue is bit-identical to the cold run at every boundary
 * that is a multiple of 64 tokens from the start of the sequence of calls - in particular every boundary aligned to the
 * key's chunk - and agrees to rounding elsewhere.  out_dtype must be F32.
 *
 * esc_causal_conv: depthwise causal FIR of window W (1..8) over x [B, T_stride, C] bf16 (C % 8 == 0), weights w [C, W] fp32:
 *      y_t[c] = sum_{i<W} w[c][i] * x_{t-W+1+i}[c]      (+ SiLU with ESC_CONV_SILU),   y [B, T, C] fp32 (dense in T)
 * where x_s for s < 0 is the carried window state_in [B, C, W-1] fp32 (oldest first; NULL = zeros); state_out receives the
 * last W-1 inputs after the call and may alias state_in. */
#define ESC_CONV_SILU 1u
int esc_gdn_scan(esc_ctx* ctx, esc_shape_key key, const void* q, const void* k, const void* v, const float* g,
                 const float* beta, const float* state_in, float* state_out, void* o, uint64_t T, uint64_t t_stride,
                 void* stream);
int esc_causal_conv(esc_ctx* ctx, const void* x, const float* w, const float* state_in, float* state_out, float* y,
                    uint32_t B, uint64_t T, uint64_t t_stride, uint32_t C, uint32_t W, uint32_t flags, void* stream);

/* ---- captured replay plan ("replay Graph[key] — never a recapture") -- */
typedef struct esc_scan_args {
    esc_shape_key key;
    const void*  q; const void* k; const void* v; const float* g;
    const float* state_in; float* state_out; void* o;
    uint64_t T; uint64_t t_stride; uint32_t chunk;
    uint32_t kind;        /* ESC_SCAN_LINATTN (0): esc_linattn_scan;  ESC_SCAN_GDN (1): esc_gdn_scan (out_dtype F32) */
    const float* beta;    /* ESC_SCAN_GDN: [B, T_stride, H] fp32 as in esc_gdn_scan; must be NULL for ESC_SCAN_LINATTN */
} esc_scan_args;
#define ESC_SCAN_LINATTN 0u
#define ESC_SCAN_GDN 1u

/*
 * Capture ONE CUDA graph = [restore node: capsule -> `live`] -> [scan node per layer, in
 * order].  A layer is a linear-attention scan or a gated delta-rule scan (`kind`; a plan may mix
 * them); the scan nodes chain by programmatic dependent launch.  `live` may be NULL (no restore
 * node: a cold plan).  The restore node reads its
 * copy table from a device-resident descriptor, so the capsule can be swapped between replays
 * WITHOUT recapturing (the paper's "host overwrites a bound sub-buffer between replays" idiom,
 * PAPER.md:110).  That descriptor lives in `scratch_dev`: caller-owned device memory of at least
 * esc_graph_scratch_bytes() bytes, 16-byte aligned (ESC_ERR_CAPACITY / ESC_ERR_UNALIGNED), which
 * must stay allocated, and untouched by the caller, until the graph is destroyed; a cold plan
 * (live == NULL) takes NULL / 0.  `max_boundary` bounds the capsules that may later be bound
 * (it sizes the restore node's grid; esc_graph_set_capsule refuses a later boundary with
 * ESC_ERR_CAPACITY).  `stream` is used for the capture and for one small kernel ahead of it that
 * stores an empty table (a launch before any capsule is bound is refused on the host anyway).
 * Lifetimes: `live`, the layers' buffers and the scratch are referenced, not copied — they must
 * outlive the graph (destroy the graph before the live set).
 */
uint64_t esc_graph_scratch_bytes(void);
int esc_graph_capture(esc_ctx* ctx, esc_bufset* live, uint64_t max_boundary,
                      const esc_scan_args* layers, uint32_t n_layers,
                      void* scratch_dev, uint64_t scratch_bytes, void* stream, esc_graph** out_graph);
/* Bind the capsule the next launches restore from: host rebuilds the table and enqueues one
 * small kernel on `stream` that stores it to the graph's device-resident copy (the table travels as a
 * kernel parameter: no copy engine, no host-side wait; the call may be repeated at any rate).  Same layout / capacity checks as esc_restore. */
int esc_graph_set_capsule(esc_graph* graph, const esc_bufset* capsule, void* stream);
/* One cudaGraphLaunch on `stream`.  ESC_ERR_INVALID if the plan has a restore node and no
 * capsule is bound. */
int esc_graph_launch(esc_graph* graph, void* stream);
/* ESC_ERR_INVALID for a plan the context's Graph[key] table owns (the table destroys it on eviction / esc_ctx_destroy). */
int esc_graph_destroy(esc_graph* graph);

/* ---- Graph[key] table ("replay Graph[key]"; "a bounded set of shape variants
 * (the ShapeKey table with LRU eviction) and a fixed maximum sequence length") -------------------------------------
 * Mechanism only: a bounded map  plan key -> captured esc_graph  kept in the context, least-recently-used eviction.
 * Which suffix lengths / boundaries get a bucket is the caller's policy; the helpers below give the usual choice.
 *   esc_suffix_bucket(T, chunk): the smallest chunk * 2^k >= T (0 for T == 0).  A plan captured for the bucket serves
 *       any suffix T' <= bucket whose tail the caller pads with k = v = 0, g = 1 tokens (reading 13: the state
 *       and the real tokens' outputs are bit-identical to a T'-token scan, the chunk grid being the same).
 *   esc_plan_key_make(shape key, suffix bucket, max boundary, n_layers): opaque 64-bit key (FNV-1a of the four).
 *   put: the table takes ownership of `graph` (esc_graph_destroy on it then fails); inserting into a full table destroys
 *        the least recently used plan; putting an existing key replaces (and destroys) the old plan; a graph already held
 *        under another key is refused (ESC_ERR_INVALID).  capacity >= 1 (default 8).
 *   contains: whether a key is present, without touching the LRU order or the statistics (lets a binding drop its
 *        references to evicted plans).
 *   get: ESC_OK and the plan (now most recently used), or ESC_ERR_MISMATCH when the key is absent — "a new shape
 *        needing capture": the caller captures and puts.  The table still owns the plan.
 *   stats: hits, misses, evictions since the context was created. */
uint64_t esc_suffix_bucket(uint64_t T, uint64_t chunk);
uint64_t esc_plan_key_make(esc_shape_key key, uint64_t suffix_bucket, uint64_t max_boundary, uint32_t n_layers);
int esc_plan_table_set_capacity(esc_ctx* ctx, uint32_t capacity);
int esc_plan_table_put(esc_ctx* ctx, uint64_t plan_key, esc_graph* graph);
int esc_plan_table_get(esc_ctx* ctx, uint64_t plan_key, esc_graph** out_graph);
int esc_plan_table_contains(const esc_ctx* ctx, uint64_t plan_key, uint32_t* out_present);
int esc_plan_table_stats(const esc_ctx* ctx, uint32_t* out_size, uint64_t* out_hits, uint64_t* out_misses,
                         uint64_t* out_evictions);

#ifdef __cplusplus
}
#endif
#endif /* ESC_H_ */
