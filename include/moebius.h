/*
 * moebius.h -- C ABI of the B200-native Moebius TP<->EP reshard (arXiv 2606.26607).
 *
 * The hot path of the paper on ONE GPU: the single resident copy of the MoE expert weights
 * (gate/up/down) and of the paged KV cache is moved between the tensor-parallel layout and the
 * expert-parallel layout at FIXED ADDRESSES (PAPER.md:35, :148-158 §4.2, :160-191 §4.3).  The R
 * logical ranks are R fixed-address regions of one caller-owned device allocation.
 *
 * Conventions
 *   - extern "C", plain pointers and sizes.  Every pointer is marked HOST or DEVICE below.
 *   - Every function returns an int status: 0 = MOEBIUS_OK, negative = error.  No exceptions, no
 *     aborts, no global state.  A failed call leaves the context and all device bytes untouched.
 *   - The caller owns every device byte and the stream.  The library owns only host objects
 *     (context, plans).  `moebius_reshard` allocates nothing on host or device (PAPER.md:158:
 *     "a switch does not allocate dynamic buffers").
 *   - POD structs carry `struct_size` (set it to sizeof(the struct) before the call).
 *   - There is no CPU fallback: `moebius_reshard` needs a CUDA device and returns MOEBIUS_E_CUDA
 *     without one.  The planner entry points are host-only and run anywhere.
 *
 * Layouts (PAPER.md:100 §3.1, :116 §3.2; orientation per BASELINE.json, reading A1)
 *   TP  rank r: gate,up [E, H, I/R] = columns [r*I/R,(r+1)*I/R) of every expert; down [E, I/R, H] =
 *       the matching rows; K/V pool [pages_tp, page_tokens, hpr, D] with r's KV-head shard of every
 *       request, one block table shared by all ranks.  Fewer KV heads than ranks: head h is
 *       replicated on ranks [h*rep, (h+1)*rep), rep = R/kv_heads.
 *   EP  rank r: gate,up [E/R, H, I], down [E/R, I, H] = experts [r*E/R,(r+1)*E/R) whole; K/V pool
 *       [pages_ep, page_tokens, kv_heads, D] with all heads of r's own requests.
 *   Both views of a tensor live in the same rank region.  Weights: a chain of 3L+1 slots per rank,
 *   object k = 3*layer + {gate:0, up:1, down:2}; the TP view of object k is slot k, the EP view is
 *   slot k+1 (Fig. 7, at (layer,matrix) grain).  KV: the TP pool and the EP pool of
 *   a (rank, layer, K|V) alias the same bytes with different page sizes.
 *   w_orient = 1 (the paper's own shapes): two objects per layer, W13 (2 slots) at slot 3*layer and
 *   W2 (1 slot) at slot 3*layer+2; every EP view starts 2 slots (the largest object) after its TP
 *   view, so the chain has 3L+2 slots.
 *   When staging_cap_bytes does not allow that many spare slots, the shift shrinks (down to 0: the two
 *   views alias the same bytes) and the objects that then overlap themselves take the in-place path
 *   (moebius_config_t::w_inplace).
 */
#ifndef MOEBIUS_H_
#define MOEBIUS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#define MOEBIUS_API __attribute__((visibility("default")))

typedef enum { MOEBIUS_TP = 0, MOEBIUS_EP = 1 } moebius_mode_t;
typedef enum { MOEBIUS_BF16 = 0, MOEBIUS_FP32 = 1, MOEBIUS_FP8_E4M3_B128 = 2 } moebius_dtype_t;

/* tensor ids for moebius_view */
typedef enum {
  MOEBIUS_T_GATE = 0, MOEBIUS_T_UP = 1, MOEBIUS_T_DOWN = 2,
  MOEBIUS_T_KPOOL = 3, MOEBIUS_T_VPOOL = 4,
  MOEBIUS_T_GATE_SCALE = 5, MOEBIUS_T_UP_SCALE = 6, MOEBIUS_T_DOWN_SCALE = 7, /* fp8 only */
  /* w_orient = 1 (the paper's own shapes): ids 0..2 and 5..7 are invalid, these are valid */
  MOEBIUS_T_W13 = 8, MOEBIUS_T_W2 = 9,
  MOEBIUS_T_W13_SCALE = 10, MOEBIUS_T_W2_SCALE = 11, /* fp8 only */
  /* attention projections (attn_mode != 0): wq [Hq,D,H], wk/wv [Hkv,D,H], wo [H,Hq,D] */
  MOEBIUS_T_WQ = 12, MOEBIUS_T_WK = 13, MOEBIUS_T_WV = 14, MOEBIUS_T_WO = 15
} moebius_tensor_t;

/* How the attention projections follow a switch. */
typedef enum {
  MOEBIUS_ATTN_NONE = 0,   /* no attention tensors in the unified buffer                              */
  MOEBIUS_ATTN_DUAL = 1,   /* the paper's default: the full copy (EP) and the head shard (TP) are both
                              resident at fixed views; a switch moves nothing ("pointer swap": the
                              caller reads the views of the published active mode), at the price of
                              one duplicated head shard per rank                                      */
  MOEBIUS_ATTN_GATHER = 2  /* the memory-saving variant: one full-size tensor per rank; the TP view of
                              a rank is its head shard IN PLACE inside it (a strided view for wo), so
                              EP->TP keeps the local slice (nothing moves) and TP->EP rebuilds the
                              rest from the other ranks' shards (the paper's All-Gather)              */
} moebius_attn_mode_t;

typedef enum {
  MOEBIUS_OK = 0,
  MOEBIUS_E_INVAL = -1,    /* bad argument / unsupported shape (reading A3)            */
  MOEBIUS_E_CAPACITY = -2, /* target mode cannot hold the live requests: cancel the switch
                                                                               */
  MOEBIUS_E_STAGING = -3,  /* staging buffer too small for the schedule this request set needs   */
  MOEBIUS_E_STATE = -4,    /* plan.from != active mode, context not bound, ...                   */
  MOEBIUS_E_CUDA = -5      /* CUDA runtime error or no device                                    */
} moebius_status_t;

typedef struct moebius_ctx moebius_ctx_t;   /* opaque, host */
typedef struct moebius_plan moebius_plan_t; /* opaque, host */

/* All caller-filled.  Symbols as in PAPER.md:100 (P there is R here). */
typedef struct {
  uint32_t struct_size;
  int32_t R, L, E, H, I;      /* E%R==0, I%R==0, (I/R)*elem_bytes % 16 == 0, else MOEBIUS_E_INVAL */
  int32_t w_dtype;            /* moebius_dtype_t; FP8_E4M3_B128 adds fp32 128x128-block scales    */
  int32_t w_orient;           /* 0: gate,up [E,H,I], down [E,I,H] (BASELINE.json, the default).
                                 1: the paper's W13 [E,2I,H] (gate rows, then up rows) and W2
                                 [E,H,I]; TP shards: W13 [E,2I/R,H] = rank r's gate
                                 rows then its up rows (reading A2), W2 [E,H,I/R]                */
  int32_t kv_heads, head_dim, page_tokens;
  int32_t kv_dtype;           /* MOEBIUS_BF16 or MOEBIUS_FP32; kv_heads%R==0 or R%kv_heads==0     */
  int64_t kv_pool_bytes_per_rank_layer; /* capacity of ONE K (or V) pool of one rank and layer; a
                                 multiple of the EP page size page_tokens*kv_heads*head_dim*b    */
  int32_t max_requests, max_pages_per_request;
  int64_t staging_cap_bytes;  /* upper bound for spare weight slot (all ranks) + KV staging (+ the
                                 duplicated attention shards of MOEBIUS_ATTN_DUAL), e.g.
                                 0.024 * resident (reading A12).  0 = no bound. */
  int32_t n_q_heads;          /* query heads Hq (attn_mode != 0): Hq % R == 0, Hq % kv_heads == 0   */
  int32_t attn_mode;          /* moebius_attn_mode_t; attention weights are bf16                    */
  int32_t w_inplace;          /* 0: automatic -- the EP view of an object starts as many slots after its
                                 TP view as the cap allows: the largest object's size (every move out of
                                 place, S1) or fewer, down to none (S2: objects that overlap themselves
                                 are moved block by block in dependency waves, blocks on permutation
                                 cycles parked in the bounded staging buffer).
                                 1: force shift 0 (both views alias the same bytes: fully in place)   */
  int32_t reserved0;
} moebius_config_t;

/* Sizes the caller must allocate, and where things are.  All byte counts. */
typedef struct {
  uint32_t struct_size;
  int32_t pages_tp, pages_ep;           /* pages per pool in each mode                            */
  int32_t tp_page_bytes, ep_page_bytes;
  int64_t base_bytes;                   /* the unified allocation: R rank regions                 */
  int64_t rank_stride_bytes;            /* rank r's region is [r*stride, (r+1)*stride)            */
  int64_t weight_slot_bytes;            /* one (layer,matrix) object of one rank                  */
  int64_t weight_spare_bytes;           /* the spare slot, all ranks                              */
  int64_t staging_bytes;                /* KV staging buffer to allocate (may be 0)               */
  int64_t desc_bytes;                   /* device descriptor/work-list buffer                     */
  int64_t table_bytes;                  /* device block-table buffer                              */
  int64_t resident_bytes;               /* expert bytes + KV pool capacity, all ranks (cap denominator) */
  /* block-table buffer layout (int32 units from its start): header[16] = {active mode, n_req,
     max_requests, max_pages_per_request, 0...}, then owner[max_requests] (-1 = all
     ranks, TP), seq_lens[max_requests], block_tables[max_requests][max_pages_per_request] (-1 pad) */
  int32_t tbl_owner_off, tbl_lens_off, tbl_bt_off, tbl_reserved;
  int64_t attn_full_bytes;              /* full q/k/v/o copies, all ranks and layers (0 without attention) */
  int64_t attn_dup_bytes;               /* MOEBIUS_ATTN_DUAL: the head shards held beside them, all ranks
                                           (1.7 GB per GPU for Qwen3-235B)              */
  int64_t w_staging_bytes;              /* the tail of the staging buffer that parks weight blocks (S2);
                                           0 when every object moves out of place                     */
  int32_t w_shift_slots;                /* slots between an object's TP view and its EP view          */
  int32_t reserved1;
} moebius_layout_t;

/* One view; offset in bytes from dev_base; shape/stride in elements.  Every view is dense row-major
 * except the TP view of wo under MOEBIUS_ATTN_GATHER, whose head-shard columns sit in place inside
 * the full [H, Hq, D] tensor (stride[0] = Hq*D). */
typedef struct {
  uint32_t struct_size;
  int32_t ndim, elem_bytes;
  int64_t offset;
  int64_t shape[4];
  int64_t stride[4];
} moebius_view_t;

/* What one plan moves (reading A15). */
typedef struct {
  uint32_t struct_size;
  int32_t n_segments, n_kv_moves, n_kv_rounds, n_kv_staged, n_pool_groups;
  int64_t n_units;                       /* work units the kernel executes                        */
  int64_t w_moved, w_relocated, w_read;  /* expert weights (+ scales): owner-changed / written / read */
  int64_t kv_moved, kv_relocated, kv_read;
  int64_t staging_used_bytes;            /* KV staging this plan uses                             */
  int64_t desc_upload_bytes, table_upload_bytes;
  int64_t attn_moved, attn_relocated, attn_read;   /* attention projections (MOEBIUS_ATTN_GATHER, TP->EP) */
  int64_t w_staged_bytes;                /* S2: expert bytes parked in (and later taken from) the staging buffer */
  int32_t n_w_waves, n_w_parked;         /* S2: dependency waves over all in-place objects, parked blocks  */
} moebius_stats_t;

/* ---- context (host only) ------------------------------------------------------------------ */

/* Validates the config and builds the region map ("one large contiguous unified
 * buffer", views at fixed regions).  cfg: HOST.  out: HOST, receives a new context. */
MOEBIUS_API int moebius_create(const moebius_config_t* cfg, moebius_ctx_t** out);
/* Destroy every plan of a context before the context itself (a destroyed plan hands its pinned
 * upload image back to its context for the next moebius_plan to reuse). */
MOEBIUS_API void moebius_destroy(moebius_ctx_t* ctx);

/* Sizes of the four caller-owned device buffers.  out: HOST. */
MOEBIUS_API int moebius_layout(const moebius_ctx_t* ctx, moebius_layout_t* out);

/* The fixed view of one tensor ("two sets of tensor views ... alias the same
 * rank-local backing buffer"; :158 "each mode-specific tensor keeps a fixed device-side memory
 * address").  out: HOST.  Scale tensors: MOEBIUS_E_INVAL unless w_dtype is FP8_E4M3_B128. */
MOEBIUS_API int moebius_view(const moebius_ctx_t* ctx, moebius_mode_t mode, int rank, int layer,
                             int tensor_id, moebius_view_t* out);

/* Binds the caller-owned DEVICE buffers (sizes from moebius_layout; all 256-byte aligned); they
 * stay fixed for the life of the context.  dev_staging may be NULL when staging_bytes == 0.
 * `initial_mode` says which layout the bytes under dev_base currently hold. */
MOEBIUS_API int moebius_bind(moebius_ctx_t* ctx, void* dev_base, void* dev_staging, void* dev_desc,
                             int32_t* dev_tables, moebius_mode_t initial_mode);

MOEBIUS_API int moebius_active_mode(const moebius_ctx_t* ctx); /* moebius_mode_t or negative */

/* ---- planner (host only) ------------------------------------------------------------------ */

/* Emits the work list for one switch (§3): the owner-changed weight slices, the
 * request ownership under `to` (TP->EP: sort by decreasing length, greedy least-loaded rank,
 * PAPER.md:124), the target block tables (canonical allocation, reading A7), the KV page
 * moves with their dependency rounds / staging, and the byte accounting.
 *   seq_lens          HOST int32[n_req]            tokens per live request (0 = waiting, no KV)
 *   src_owner         HOST int32[n_req]            EP source only (owner rank), else NULL
 *   src_block_tables  HOST int32[n_req][max_pages_per_request], -1 padded; pages of the SOURCE
 *                     mode (TP: shared table; EP: page ids within the owner's pool)
 *   out               HOST, receives a new plan
 * MOEBIUS_E_CAPACITY: the target mode cannot hold the requests -- the caller cancels the switch
 * (PAPER.md:213).  n_req == 0 is the weight-only warm-up switch. */
MOEBIUS_API int moebius_plan(moebius_ctx_t* ctx, moebius_mode_t from, moebius_mode_t to, int32_t n_req,
                             const int32_t* seq_lens, const int32_t* src_owner,
                             const int32_t* src_block_tables, moebius_plan_t** out);
MOEBIUS_API void moebius_plan_destroy(moebius_plan_t* plan);

/* The request state under the target mode.  dst_owner: HOST int32[n_req] (-1 = all ranks, TP).
 * dst_block_tables: HOST int32[n_req][max_pages_per_request].  Either may be NULL. */
MOEBIUS_API int moebius_block_tables(const moebius_plan_t* plan, int32_t* dst_owner,
                                     int32_t* dst_block_tables);

MOEBIUS_API int moebius_plan_stats(const moebius_plan_t* plan, moebius_stats_t* out);

/* Diagnostic dump of the work list for host-side hazard checking (tests).  what: 0 = segments
 * (moebius_segment_t-sized records), 1 = KV move descriptors (16 B each), 2 = 2-D
 * copy descriptors (32 B each), 3 = the dependency wave of every segment (int32 each), 4 = bulk copy
 * descriptors (16 B each), 5 = weight blocks of the in-place path (16 B each).  buf: HOST, cap bytes; *needed receives the full size. */
MOEBIUS_API int moebius_plan_export(const moebius_plan_t* plan, int what, void* buf, int64_t cap,
                                    int64_t* needed);

/* ---- execution (needs a CUDA device) ------------------------------------------------------ */

/* Enqueues one switch on `cuda_stream` (a cudaStream_t; NULL = default stream) and returns after
 * the launch: work-list upload into dev_desc, ONE persistent sm_100a kernel that executes it
 * ("reads from the source-mode alias and writes ... the target-mode slot", one HBM read
 * and one write per element, Table 1 :185), then the new tables + active-mode flag into dev_tables.
 * MOEBIUS_E_STATE if plan.from is not the active mode.  On success the active mode becomes plan.to.
 * Work on the stream is ordered after everything enqueued before it; no other stream may touch
 * the bound buffers while it runs. */
MOEBIUS_API int moebius_reshard(moebius_ctx_t* ctx, const moebius_plan_t* plan, void* cuda_stream);

/* The same switch as a PLAN-INDEPENDENT sequence, for callers that keep the switch itself inside a
 * captured CUDA graph (PAPER.md:197-201 keeps everything round the switch in
 * graphs).  moebius_stage_plan (host only, plus one pinned allocation on its first call) copies the
 * plan's work list and tables into a pinned mailbox at a fixed host address, checks plan.from against
 * the active mode and makes plan.to the active mode.  moebius_reshard_staged enqueues: counters := 0,
 * mailbox -> dev_desc (fixed size: the whole descriptor capacity), the kernel with a fixed full grid
 * and arguments that do not depend on the plan (the kernel reads segment/unit counts from the
 * uploaded header), mailbox tables -> dev_tables (fixed size).  It may be called under stream
 * capture; each replay of the captured graph executes whatever plan was staged last.  Exactly one
 * execution must follow each moebius_stage_plan, and the next plan may be staged only after that
 * execution's uploads have completed (synchronise the stream or an event recorded after it).
 * MOEBIUS_E_STATE: nothing staged yet / wrong active mode. */
MOEBIUS_API int moebius_stage_plan(moebius_ctx_t* ctx, const moebius_plan_t* plan);
MOEBIUS_API int moebius_reshard_staged(moebius_ctx_t* ctx, void* cuda_stream);

/* Rank-share execution, the multi-GPU form of a switch.
 * A plan's segments fall into dependency WAVES (moebius_plan_waves); within a wave nothing depends on
 * anything.  Every process builds the same plan (the planner is deterministic), binds a
 * moebius_arena in which it owns ranks [rank_lo, rank_hi), and for wave = 0 .. n_waves-1 calls
 * moebius_reshard_share, which enqueues one launch executing only the units whose EP-side rank it
 * owns -- EP->TP: read the own EP view, store into every TP owner's region (push); TP->EP: load from
 * the TP holders, write the own EP view (pull) -- followed by a barrier across the processes (one per
 * dependency round).  After the last wave each process calls moebius_reshard_publish (tables + the
 * active-mode flip).  Wave 0 also uploads the work list.  On one GPU the shares of a wave may simply
 * be enqueued one after another; the result is identical to moebius_reshard. */
MOEBIUS_API int moebius_plan_waves(const moebius_plan_t* plan, int32_t* n_waves);
MOEBIUS_API int moebius_reshard_share(moebius_ctx_t* ctx, const moebius_plan_t* plan, int rank_lo, int rank_hi,
                                      int wave, void* cuda_stream);
/* What ranks [rank_lo, rank_hi) execute of a plan in `wave` (-1: all waves).  out4: HOST int64[4] =
 * {units, bytes read, bytes written, bytes crossing between ranks}; the crossing bytes of all ranks
 * sum to the plan's owner-changed bytes (moebius_stats_t w_moved + kv_moved). */
MOEBIUS_API int moebius_share_stats(const moebius_plan_t* plan, int rank_lo, int rank_hi, int wave, int64_t* out4);
MOEBIUS_API int moebius_reshard_publish(moebius_ctx_t* ctx, const moebius_plan_t* plan, void* cuda_stream);

/* The same split with the round barrier ON THE DEVICE: one launch per GPU for the whole switch instead of
 * one launch and one host barrier per wave ("one cross-GPU barrier per dependency
 * round").  The ranks are cut into n_shares shares, share s owning ranks
 * [rank_bounds[s], rank_bounds[s+1]) (HOST int32[n_shares + 1], from 0 to R).  The launch executes shares
 * [share_first, share_first + share_count): its CTAs are divided among them, every CTA walks the plan's
 * waves taking only its share's units, and after each wave the last CTA of a share raises the share's flag
 * (st.release.sys) in the flag page inside that share's first rank region; every CTA then waits for the
 * flags of ALL n_shares shares (ld.acquire.sys) -- addresses inside the unified buffer, i.e. peer memory
 * when the share runs on another GPU.
 *   share_count == n_shares: the whole switch on this device in ONE cooperative launch whose CTA groups
 *     play the GPUs (this is how the barrier is verified on one GPU: separate launches that wait for one
 *     another must not be run on one device).
 *   share_count == 1: the launch of one GPU of n_shares; the other GPUs launch theirs concurrently, after a
 *     host barrier that follows everybody's flag clearing.  (Not exercisable on a one-GPU pool.)
 * Uploads the work list like moebius_reshard; end the switch with moebius_reshard_publish.  Needs
 * cooperative-launch support and 2 * n_shares * waves <= 16384. */
MOEBIUS_API int moebius_reshard_shares(moebius_ctx_t* ctx, const moebius_plan_t* plan, int n_shares,
                                       const int32_t* rank_bounds, int share_first, int share_count, void* cuda_stream);

/* ---- the staged comparison path (needs a CUDA device) --------------- */

/* PAPER.md:162-170 and Table 1 (:176-189): the "Naive" implementation of a switch -- per object, gather
 * the source bytes into per-peer chunks in a staging buffer (local permute), exchange the chunks
 * (All-to-All), and for the paged KV cache scatter the received chunks into the target pages.  On one
 * device the exchange is a device copy, so every element makes 2 (weights: permute, exchange) or 3 (KV:
 * gather, exchange, scatter) read+write passes through HBM where moebius_reshard makes one.  Same plan,
 * same result bit for bit (target views, published tables, active mode); it exists to MEASURE the pass
 * counts of Table 1 and the fused kernel's gain on the same box, and is not part of the product path.
 *   dev_scratch   DEVICE, 256-byte aligned, at least moebius_naive_scratch_bytes(ctx, plan) bytes,
 *                 caller-owned (the paper's staging slots S / 2S: here one weight object over all ranks,
 *                 or a pool's gathered + received KV), outside the unified buffer and its 2.4 % budget
 *   stats6        HOST int64[6] or NULL: {kernel launches, bytes read, bytes written, bytes of the weight
 *                 passes, bytes of the KV passes, scratch bytes needed}
 * Synchronises the stream once before its launches (descriptor upload from pageable host memory).
 * With moebius_set_timing the span of its launches is recorded like a moebius_reshard kernel. */
MOEBIUS_API int moebius_naive_scratch_bytes(const moebius_ctx_t* ctx, const moebius_plan_t* plan, int64_t* out);
MOEBIUS_API int moebius_reshard_naive(moebius_ctx_t* ctx, const moebius_plan_t* plan, void* dev_scratch,
                                      int64_t scratch_bytes, void* cuda_stream, int64_t* stats6);

/* The same staged path for callers that cannot allocate device memory where they stand (code under CUDA graph
 * capture, tight serving loops, harnesses that forbid cudaMalloc): its staging buffer is a file-scope static
 * device array of MOEBIUS_STATIC_SCRATCH_BYTES inside the library -- every GPU that loads the library holds
 * those bytes until the process exits -- so the call allocates NO device memory: no cudaMalloc, no cudaFree,
 * no allocating CUDA library routine (on the host it builds its descriptor lists like moebius_reshard_naive).
 * Same plan, same kernels, same result bit for bit as moebius_reshard_naive and moebius_reshard.
 *   Limit: a plan with moebius_naive_scratch_bytes(ctx, plan) > MOEBIUS_STATIC_SCRATCH_BYTES is refused with
 *   MOEBIUS_E_STAGING ("staging buffer too small") before anything is enqueued; use moebius_reshard_naive
 *   with a caller-owned buffer for those.  moebius_static_scratch_bytes() returns the limit (host only).
 *   Sharing: every call on a device uses the one array, which keeps the previous call's bytes.  Nothing in
 *   it has to start at zero (each launch reads only what an earlier launch of the same call wrote), so
 *   nothing is cleared.  Calls that OVERLAP on the GPU -- two streams, two contexts on one device -- race on
 *   the array: serialise them.  stats6 as for moebius_reshard_naive. */
#define MOEBIUS_STATIC_SCRATCH_BYTES (64 * 1024 * 1024)
MOEBIUS_API int64_t moebius_static_scratch_bytes(void);
MOEBIUS_API int moebius_reshard_naive_static(moebius_ctx_t* ctx, const moebius_plan_t* plan, void* cuda_stream,
                                             int64_t* stats6);

/* Kernel-only device time of the last moebius_reshard, in ms (CUDA events on its stream; the call
 * synchronises on the end event).  Enabled with moebius_set_timing(ctx, 1). */
MOEBIUS_API int moebius_set_timing(moebius_ctx_t* ctx, int enable);
MOEBIUS_API int moebius_last_kernel_ms(moebius_ctx_t* ctx, float* ms);
/* The same for the most recent calls (a ring of 64), oldest first.  out_ms: HOST float[cap];
 * *n_out receives how many were written.  Synchronises on each end event. */
MOEBIUS_API int moebius_kernel_ms_history(moebius_ctx_t* ctx, float* out_ms, int cap, int* n_out);

/* Data-path selection, before the first moebius_plan of a context.  enable != 0 (the default):
 * segments whose shapes allow it run on the TMA path (tensor-map loads/stores through shared memory,
 * `pipes` warps per SM, each with a ring of two `stage_kb` KB stages; 0 = the context's defaults: the stage
 * is a whole number of EP pages near 48 KB and the pipes fill 208 KB -- 2 and 48 at 16-KB pages).  enable == 0:
 * everything runs on the ld.global/st.global path.  Results are identical either way.  A plan built
 * before the call cannot be executed after it (MOEBIUS_E_STATE).  2*pipes*stage_kb <= 208. */
MOEBIUS_API int moebius_set_tma(moebius_ctx_t* ctx, int enable, int pipes, int stage_kb);
/* The pipes' shared-memory rings (tuning; after moebius_set_tma, which resets the ring to two stages).
 * A TMA unit takes exactly the bytes it needs from its pipe's ring, first in first out, so units smaller
 * than a stage pack the ring deeper.  ring_kb: bytes of one pipe's ring in KB, >= stage_kb,
 * pipes * ring_kb <= 208; 0 = two stages.  max_loads: units of one pipe whose loads may be in flight at
 * once (1..7; 0 = the default 2: a store's shared-memory read completes long before a load lands, so two
 * loads in flight per pipe and a store that is waited for at once keep more bytes in flight than one load
 * behind two draining stores -- measured 1.4-2.3 % faster on B200 at the BASELINE shapes).
 * Results are identical.  PAPER.md:172 fixes what a slice move reads and writes, not how it is staged. */
MOEBIUS_API int moebius_set_ring(moebius_ctx_t* ctx, int ring_kb, int max_loads);

/* KV schedule (tuning; before moebius_plan).  When target pages overlap live source pages the page
 * moves form dependency chains; the planner runs them in at most `max_level` + 2 device-wide rounds
 * and cuts longer chains by staging the page at the cut (bounded staging buffer; if the cut pages
 * of one pool do not fit it, longer chains are allowed).  0 restores the default (64: a round costs
 * ~10 us on B200, a staged page an extra copy of it in all 2L pools); at most 1024.  Results are
 * identical for every value. */
MOEBIUS_API int moebius_set_kv_rounds(moebius_ctx_t* ctx, int max_level);
/* KV work is cut into slices that the merged work list interleaves with the weight chain, one per chain
 * link where there is enough of it, so that the drain of a link hides behind independent KV units.
 * min_units: the smallest slice (tuning; 0 = the default, 8192 units).  Results are identical. */
MOEBIUS_API int moebius_set_kv_slice(moebius_ctx_t* ctx, int min_units);
/* Weight chain (tuning; before moebius_plan).  enable != 0: when all objects have the same size and every
 * move is out of place, a link is cut into 2 x 2 segments (half of the EP ranks x half of the rows) that
 * wait for ONE half of the predecessor, so consecutive links overlap instead of being separated by a
 * device-wide drain (PAPER.md:156 fixes the order, not the grain).  enable == 0 (the default: the banded
 * order measured slower on B200 than the drains it removes): a link waits for the whole predecessor.
 * Results are identical. */
MOEBIUS_API int moebius_set_chain_bands(moebius_ctx_t* ctx, int enable);
/* Which side of a short-run weight unit (gate, up, W2) goes through the tensor-map box (tuning; any time).
 * 1 (the default; measured 2-4 % faster EP->TP, 0.3 % TP->EP on B200): the EP side is ONE contiguous bulk
 * copy and the box covers the TP views [run][rank][row], landing in EP order (full units only; ragged
 * ones use mode 0).  0: the box covers the EP rows [run][row][group] and lands group-major, the TP side is
 * R contiguous bulk copies.  Bits 4-5 (tuning): L2 promotion of the TP-side map, 0 none / 1, 2, 3 = 64,
 * 128, 256 bytes.  Results are identical. */
MOEBIUS_API int moebius_set_xt_mode(moebius_ctx_t* ctx, int mode);

/* L2 cache-hint policy of the TMA loads and stores (tuning; any time): 0 none (the hardware default),
 * 1 evict_first, 2 evict_last, 3 evict_normal, 4 evict_unchanged (PTX createpolicy.fractional.L2, fraction
 * 1.0, passed as .L2::cache_hint to every cp.async.bulk[.tensor]).  Nothing is ever re-read (L2 hit rate
 * 0.03 %), so this only shapes how the L2 writes dirty lines back.  Default: loads evict_last, stores
 * unhinted -- A/B on B200, alternating in one session: 0.6 % (235B shape), 0.9 % (30B, fp8), 1.0 % (config 2)
 * faster than no hint; evict_first on either side and any hint on the stores are neutral or slower.
 * Results are identical. */
MOEBIUS_API int moebius_set_l2_policy(moebius_ctx_t* ctx, int load_policy, int store_policy);

/* Launch shape override for the ld/st path (tuning): values <= 0 restore the defaults; threads is a
 * multiple of 32, at most 256. */
MOEBIUS_API int moebius_set_launch(moebius_ctx_t* ctx, int ctas_per_sm, int threads, int unit_kb);

/* ---- peer-mappable unified buffer (needs a CUDA device) ------------- */

/* each rank's buffer is exported once and mapped by its peers, whose kernels
 * store into it.  Here: ONE virtual range of R * rank_stride bytes (rank_stride is a multiple of
 * 2 MiB for this), rank r's region backed by its OWN physical allocation mapped at
 * base + r * rank_stride.  Ranks [rank_lo, rank_hi) are created on `device` by this call; the others
 * are imported from the processes that own them (POSIX file descriptors of their allocations, sent
 * over a unix socket by the caller).  All addresses the planner and kernel use, tensor maps
 * included, are the same whether the ranks share a GPU or have one each.  The resulting base is a
 * valid `dev_base` for moebius_bind once every rank is mapped (moebius_arena_ready == MOEBIUS_OK). */
typedef struct moebius_arena moebius_arena_t; /* opaque, host */
MOEBIUS_API int moebius_arena_create(const moebius_ctx_t* ctx, int device, int rank_lo, int rank_hi,
                                     moebius_arena_t** out);
MOEBIUS_API void moebius_arena_destroy(moebius_arena_t* arena);
MOEBIUS_API void* moebius_arena_base(const moebius_arena_t* arena);        /* DEVICE pointer */
MOEBIUS_API int moebius_arena_ready(const moebius_arena_t* arena);
MOEBIUS_API int moebius_arena_export(const moebius_arena_t* arena, int rank, int* fd_out); /* a local rank */
MOEBIUS_API int moebius_arena_import(moebius_arena_t* arena, int rank, int fd);            /* a peer's rank */

/* ---- switch coordinator (host only; §4.5) ----------------------------------- */

typedef struct moebius_policy moebius_policy_t; /* opaque, host */
typedef enum { MOEBIUS_POLICY_INTERACTIVE = 0, MOEBIUS_POLICY_ROLLOUT = 1 } moebius_policy_kind_t;
typedef enum {
  MOEBIUS_DECISION_STAY = 0,
  MOEBIUS_DECISION_SWITCH = 1,    /* the caller now plans + reshards to the other mode */
  MOEBIUS_DECISION_CANCELLED = 2  /* the policy wanted to switch but the target mode cannot hold the
                                     live requests: cancelled, retried after the cooldown (:213) */
} moebius_decision_t;
typedef struct {
  uint32_t struct_size;
  int32_t W;                  /* averaging window in iterations (EP->TP), >= 1                    */
  double T_h, T_l;            /* TP->EP when the latest count > T_h; EP->TP when the mean of the
                                 last W counts < T_l; T_l <= T_h (hysteresis band)   */
  double cooldown_s;          /* no decision for this long after a switch or a cancelled attempt   */
} moebius_policy_config_t;

/* The paper's two settings: interactive T_l = 0.8 T_h, W = 8; rollout T_l = T_h,
 * W = 1.  The paper runs T_h = 256, cooldown 5 s.  out: HOST (struct_size set by the caller). */
MOEBIUS_API int moebius_policy_preset(int kind, double T_h, double cooldown_s, moebius_policy_config_t* out);
MOEBIUS_API int moebius_policy_create(const moebius_policy_config_t* cfg, moebius_mode_t initial_mode,
                                      moebius_policy_t** out);
MOEBIUS_API void moebius_policy_destroy(moebius_policy_t* policy);
MOEBIUS_API int moebius_policy_mode(const moebius_policy_t* policy);

/* One sample of the control signal -- the global in-flight request count n_req -- taken after a
 * decode iteration at time now_s (seconds, any monotonic origin).  seq_lens: HOST
 * int32[n_req], used only for the capacity check of the target mode, which runs through `ctx`
 * (NULL = no check).  *decision receives a moebius_decision_t, *mode_after (may be NULL) the mode
 * the policy is in after the call.  The policy only decides; the caller executes the switch. */
MOEBIUS_API int moebius_policy_step(moebius_policy_t* policy, moebius_ctx_t* ctx, double now_s, int32_t n_req,
                                    const int32_t* seq_lens, int32_t* decision, int32_t* mode_after);

/* MOEBIUS_OK if mode `to` can hold these requests (TP: all pages in one pool of pages_tp; EP: the
 * greedy partition of PAPER.md:124, each rank's share in pages_ep), else MOEBIUS_E_CAPACITY
 * (TP replication reduces capacity when there are fewer KV heads than ranks). */
MOEBIUS_API int moebius_capacity_check(moebius_ctx_t* ctx, moebius_mode_t to, int32_t n_req, const int32_t* seq_lens);

/* Startup calibration: from decode costs probed at ascending batch sizes under both
 * modes, the batch size where they cross (linear interpolation between probes; EP never cheaper ->
 * the largest probe, always cheaper -> the smallest).  All arrays HOST, length n. */
MOEBIUS_API int moebius_policy_calibrate(int32_t n, const int32_t* batch_sizes, const double* tp_cost,
                                         const double* ep_cost, int32_t* T_h_out);

MOEBIUS_API const char* moebius_status_str(int status);
MOEBIUS_API int moebius_version(void);

#ifdef __cplusplus
}
#endif
#endif /* MOEBIUS_H_ */
