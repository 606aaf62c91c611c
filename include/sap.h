/* sap.h — C ABI of the B200-native SAP attention hot path.
 *
 * Exact causal attention over a packed ("hybrid-context") sequence with no cross-document
 * contamination, computed as partial attention between P sequence chunks (the paper's per-rank Q
 * shards against incoming K/V shards, emulated on one GPU as chunks in HBM) and merged exactly
 * through log-sum-exp.
 *
 * Citations are to /root/reference/PAPER.md (HSAP, arxiv/paper_2606_30460):
 *   attention definition          §2.2.1, eq. at PAPER.md:55  Softmax(QK^T/sqrt(d))V, Q,K,V in R^{N x H x d} (:53)
 *   packing / cu_len masking      §2.1, PAPER.md:39-45        "only compute attention within each segment", causal
 *   chunks + online merge         §2.2.1, PAPER.md:59         blocks Q_i,K_i,V_i of n = N/P rows, merged "in an online manner"
 *   JIT compile -> code lists     §3.1-3.2, Table 1 (:85-98): the `computing` instruction
 *   "copy and rescale" fused      §6, PAPER.md:239 (the paper's stated future work; done in the kernel epilogue here)
 *   backward tensors dq,dkv,do    Table 1
 *
 * Conventions
 *   - Every function returns an int status (0 = SAP_OK); nothing throws, nothing aborts.
 *   - "host" / "device" is stated per pointer.  Device buffers are owned by the caller; the library
 *     allocates device memory only for a plan's device mirror (sap_plan_upload, and the range-restricted
 *     programs of the partial / per-rank / per-item calls, built on first use of a range and uploaded on
 *     the caller's stream) and frees it in sap_plan_destroy.  Only sap_plan_upload and sap_plan_destroy
 *     synchronise the device; every other call is asynchronous on its stream.
 *   - Range-restricted programs are cached with the plan, 64 per kind of call; beyond that the least recently used
 *     one is freed, stream-ordered behind the last kernels that read it on every stream that used it.  Building one
 *     allocates (cudaMallocAsync) and copies from pageable host memory, so the FIRST use of a range (or the first
 *     after its eviction) cannot be recorded into a CUDA graph: during stream capture such a call returns
 *     SAP_ERR_UNSUPPORTED and leaves the capture intact - make the call once outside capture first.  A program a
 *     graph has recorded a launch on is kept until sap_plan_destroy.
 *   - A plan's device mirror lives on one device (the current device of its first upload); every attention call takes
 *     the caller's token count n_tokens and fails with SAP_ERR_PLAN_MISMATCH when it differs from the plan's (the kernels
 *     index the tensors by the plan's token ranges) or when the current device is another one.
 *   - Layouts (packed "thd"): q/out/dout/dq  [N, Hq,  d] bf16, contiguous;
 *     k/v/dk/dv [N, Hkv, d] bf16, contiguous; lse [Hq, N] fp32 (natural log of the sum of
 *     exp(scale * q.k) over the visible keys); cu_seqlens int32 [D+1], cu[0] = 0, non-decreasing,
 *     cu[D] = N.  q-head h reads kv-head h / (Hq/Hkv).
 *   - Visibility: key s is visible to row t iff both lie in the same document and s <= t.
 *   - head_dim in {64, 128}; Hq % Hkv == 0; N % n_chunks == 0 (contiguous equal chunks).
 *   - All device pointers must be 16-byte aligned.
 */
#ifndef SAP_H_
#define SAP_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- status codes (every call returns one; the paper's executor has no error model, this is the library's) ---- */
enum {
  SAP_OK = 0,
  SAP_ERR_INVALID_ARG = 1,        /* null pointer, n_chunks < 1, n_docs < 1, bad range               */
  SAP_ERR_BAD_CU_SEQLENS = 2,     /* cu[0] != 0, decreasing, or total length 0                        */
  SAP_ERR_INDIVISIBLE = 3,        /* N % n_chunks != 0                                                */
  SAP_ERR_UNSUPPORTED = 4,        /* head_dim not in {64,128}, Hq % Hkv != 0, misaligned pointer      */
  SAP_ERR_WORKSPACE_TOO_SMALL = 5,
  SAP_ERR_WRONG_ARCH = 6,         /* current device is not compute capability 10.x                    */
  SAP_ERR_CUDA = 7,               /* a CUDA runtime/driver call failed; see sap_last_cuda_error()     */
  SAP_ERR_NO_DEVICE = 8,          /* no CUDA device / driver available                                */
  SAP_ERR_PLAN_MISMATCH = 9,      /* n_tokens != the plan's token count, or the plan's mirror is on another device */
  SAP_ERR_STATIC_LIMIT = 10       /* sap_attn_bwd_static: the problem does not fit the library's built-in scratch memory */
};

/* ---- plan (host-side JIT planner; §3.2 Step 1, :106-:108) ------------------------- */
enum { SAP_MASK_SKIP = 0, SAP_MASK_FULL = 1, SAP_MASK_DIAG = 2 };

/* One `computing` work item (Table 1): partial attention of q-chunk i against
 * kv-chunk j.  10 x int32, no padding, memcmp-comparable. */
typedef struct {
  int32_t q_chunk, kv_chunk;     /* i, j (j <= i)                                                   */
  int32_t doc_lo, doc_hi;        /* inclusive range of contributing documents                        */
  int32_t mask_kind;             /* SAP_MASK_FULL (no element masked inside the item's rectangle)    */
                                 /* or SAP_MASK_DIAG (j == i: block-diagonal causal)                 */
  int32_t step;                  /* ring step i - j                                                  */
  int32_t q_begin, q_end;        /* absolute token range of rows that have visible keys, half-open   */
  int32_t kv_begin, kv_end;      /* absolute token range of keys that are visible to some row        */
} sap_item_t;

typedef struct sap_plan sap_plan_t; /* opaque; immutable after creation except for the lazy device mirror */

/* Build the plan for `cu_seqlens_host` (host, int32[n_docs+1]) split into `n_chunks` equal chunks.
 * Keeps only chunk pairs whose documents intersect under causality, in ring order per q-chunk
 * (step 0 = diagonal, then j = i-1, i-2, ...), and compiles the per-tile work lists the kernels
 * walk.  Pure host code: works without a GPU.  *out is set only on SAP_OK. */
int sap_plan_create(const int32_t* cu_seqlens_host, int32_t n_docs, int32_t n_chunks, sap_plan_t** out);
void sap_plan_destroy(sap_plan_t* plan); /* frees host memory and the device mirror; NULL is a no-op */

int32_t sap_plan_n_items(const sap_plan_t* plan);               /* number of non-SKIP items          */
int32_t sap_plan_n_chunks(const sap_plan_t* plan);
int32_t sap_plan_n_tokens(const sap_plan_t* plan);
const sap_item_t* sap_plan_items(const sap_plan_t* plan);       /* host, plan-owned, [n_items]       */
const int32_t* sap_plan_chunk_offsets(const sap_plan_t* plan);  /* host, [P+1], CSR by q_chunk       */
const int32_t* sap_plan_kv_offsets(const sap_plan_t* plan);     /* host, [P+1], CSR by kv_chunk      */
const int32_t* sap_plan_kv_index(const sap_plan_t* plan);       /* host, [n_items], item ids by kv_chunk */
const uint8_t* sap_plan_kind_map(const sap_plan_t* plan);       /* host, [P*P] row-major, SKIP above diag */
int64_t sap_plan_useful_pairs(const sap_plan_t* plan);          /* sum over documents of L(L+1)/2    */
/* Number of 128x128 score tiles the forward kernel issues per q-head (for issue-efficiency reports). */
int64_t sap_plan_fwd_tiles(const sap_plan_t* plan);

/* Compile Steps 2-3 (§3.2, :110-:118): which rank computes each item and at which stage, for P real ranks
 * (one chunk per rank).  Host only; does not change what the single-GPU kernels do.
 *   policy SAP_SCHED_RING     : item (i, j) on rank i at stage i - j (plain ring attention, :59).
 *   policy SAP_SCHED_BALANCED : Step 2, per causal region (= document spanning chunks a..b, m = b-a+1): the diagonal
 *       item stays on its rank at stage 0; a FULL item (i, j) stays on rank i at regional stage i-j when
 *       i-j <= m/2, else it is computed by the idle early rank j (Q_i travels to the K/V, the partial travels back)
 *       at regional stage m-(i-j) — the LightSeq / DistFlashAttn balancing the paper refers to (:116).
 *       Step 3: a rank that sits in two regions is over-subscribed.  (a) While the busiest rank holds a FULL item
 *       whose other end (rank i or j) has at least two items fewer, the item whose other end is least loaded moves
 *       there.  (b) At most one item per rank per stage: a rank runs its items back to back in order of
 *       (regional stage, q_chunk, kv_chunk); stage = position in that list (shards travel point to point, so any
 *       order is legal).
 * slots: host, [sap_plan_n_items], written in item order.  *n_stages = 1 + the largest stage.  The paper's Fig. 3 is
 * missing from the extracted text; this is the reading recorded in DESIGN.md (R-5). */
enum { SAP_SCHED_RING = 0, SAP_SCHED_BALANCED = 1 };
typedef struct { int32_t rank, stage; } sap_slot_t;
int sap_plan_schedule(const sap_plan_t* plan, int32_t policy, sap_slot_t* slots, int32_t* n_stages);

/* Jitted code generation (§3.2 :120-:124, instruction set of Table 1 :85-:98), forward pass: the
 * instruction list of one rank for a schedule made by sap_plan_schedule.  One code = 5 x int32, memcmp-comparable:
 *   stage   -1 (prologue) .. n_stages (epilogue); a rank walks its list in order, one stage after the other
 *   opcode  SAP_OP_SEND / SAP_OP_RECV  create $send-op / $recv-op {tensor} %peer: all SEND/RECV codes of one stage form
 *                                      ONE batched isend/irecv that is in flight while the stage's block is computed
 *                                      (:122-:124); every SEND has its RECV at the same stage on the peer
 *           SAP_OP_COMPUTING           partial attention of plan item `item` on the compute buffers (:102)
 *           SAP_OP_COPY                after the stage's batch completed: received q / kv -> compute buffer; received
 *                                      o -> merged into this rank's running (O, LSE) ("copy and rescale", :239)
 *   tensor  SAP_T_Q / SAP_T_KV / SAP_T_O (o = a partial result: normalised output + LSE)
 *   peer    the other rank (SEND: destination, RECV / COPY: source); -1 for COMPUTING
 *   item    the plan item the data belongs to
 * Rule: an item computed on the rank of its Q gets K/V_j sent j -> i one stage earlier; an item computed on the rank
 * of its K/V (a helper, Step 2) gets Q_i sent i -> j one stage earlier and its partial result sent back j -> i one
 * stage later.  Inside a stage: SEND / RECV codes ordered by (opcode, tensor, peer, item), then COMPUTING, then COPY
 * codes ordered by (tensor, peer, item).
 * codes: host, capacity `cap` codes; returns the number of codes of `rank` (call with cap = 0 to size), < 0 on error. */
enum { SAP_OP_SEND = 0, SAP_OP_RECV = 1, SAP_OP_COMPUTING = 2, SAP_OP_COPY = 3 };
enum { SAP_T_Q = 0, SAP_T_KV = 1, SAP_T_O = 2 };
typedef struct { int32_t stage, opcode, tensor, peer, item; } sap_code_t;
int32_t sap_plan_codegen(const sap_plan_t* plan, const sap_slot_t* slots, int32_t rank, sap_code_t* codes, int32_t cap);

/* The same for the backward pass (tensors do / dq / dkv of Table 1).  An item computed on the rank of
 * its Q (which also holds dO, LSE and D of those rows) gets K/V_j sent j -> i one stage earlier and sends its dK/dV
 * contribution (`dkv`) back j <- i one stage later; an item computed on the rank of its K/V gets Q_i and dO_i (`do`
 * carries LSE and D along) one stage earlier and sends its dQ contribution (`dq`) back to i one stage later.  COPY of
 * a received dq / dkv adds it into the owner's gradient.  Same code format, order and return value as
 * sap_plan_codegen; tensors SAP_T_Q, SAP_T_KV, SAP_T_DO, SAP_T_DQ, SAP_T_DKV. */
enum { SAP_T_DO = 3, SAP_T_DQ = 4, SAP_T_DKV = 5 };
int32_t sap_plan_codegen_bwd(const sap_plan_t* plan, const sap_slot_t* slots, int32_t rank, sap_code_t* codes, int32_t cap);

/* Copy the compiled work lists to the current CUDA device (cudaMalloc + synchronous cudaMemcpy): the "compile" side
 * runs "ahead of the communication and computation".  Called implicitly by the first sap_attn_* call that
 * uses the plan; call it yourself to keep that cost out of a timed region.  Idempotent; serialised per plan by a mutex;
 * a failed upload frees what it had allocated.  SAP_ERR_PLAN_MISMATCH if the plan is already on another device. */
int sap_plan_upload(sap_plan_t* plan);

/* ---- attention ------------------------------------------------------------------------------ */
enum { SAP_PASS_FWD = 0, SAP_PASS_BWD = 1 };

/* Bytes of caller-provided device workspace a pass needs (fwd: 0; bwd: D = rowsum(dO*O), fp32 [Hq,N], padded to
 * 256 B, followed by the fp32 dQ accumulator [N,Hq,d] the fused backward kernel reduces into).  A buffer of fixed,
 * known size that the caller allocates once: the paper's "fixed global buffer ... no memory jitter". */
size_t sap_workspace_bytes(const sap_plan_t* plan, int n_q_heads, int n_kv_heads, int head_dim, int pass);

/* Forward: for every row, attention over the visible keys, walking the row's
 * q-chunk items in plan order and merging the per-item partials on chip (running max / sum / O).
 * q,k,v,cu_seqlens_dev: device, read.  out: device bf16 [N,Hq,d], written.  lse: device fp32 [Hq,N], written.
 * cuda_stream: a cudaStream_t (NULL = legacy default stream).  Asynchronous.
 * workspace / workspace_bytes: not used (the forward needs no workspace: sap_workspace_bytes(..., SAP_PASS_FWD) = 0); kept
 * so that the two passes have the same signature.  Pass NULL, 0.
 * With an even Hq/Hkv the launch is persistent (one CTA per SM; work items = (Q tile, pair of q-heads of a group) taken
 * in order off a device counter).  Each launch needs a counter pair of its own while it runs.  The pairs come from two
 * per-device pools of 4096 that launches take round-robin and leave zeroed: one pool for ordinary launches, one for
 * launches recorded during stream capture (a captured launch keeps its pair for the life of the graph, so graph replays
 * never meet ordinary launches on a pair).  Calls may therefore overlap freely on different streams and with graph
 * replays, within two limits: fewer than 4096 forward launches of one process in flight on one device at a time, and
 * at most 4096 forward launches captured into graphs that can run concurrently with each other.  A kernel that finds
 * its pair was shared traps (the launch fails with a CUDA error) instead of returning wrong output. */
int sap_attn_fwd(const void* q, const void* k, const void* v, const int32_t* cu_seqlens_dev,
                 sap_plan_t* plan, int64_t n_tokens, void* out, float* lse,
                 int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale,
                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/* Partial forward over plan items [item_begin, item_end) only (ids index sap_plan_items).
 * out_f32: device fp32 [N,Hq,d], normalised partial output; lse: device fp32 [Hq,N].
 * Rows with no visible key among those items get out = 0, lse = -inf.  Items of one q-chunk cover
 * disjoint key sets, so partials of disjoint item sets merge exactly with sap_lse_merge. */
int sap_attn_fwd_partial(const void* q, const void* k, const void* v, const int32_t* cu_seqlens_dev,
                         sap_plan_t* plan, int64_t n_tokens, int32_t item_begin, int32_t item_end,
                         float* out_f32, float* lse,
                         int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale,
                         void* cuda_stream);

/* Exact merge of two partials over disjoint key sets (online softmax; "rescale", :239):
 *   L = max(La,Lb) + ln(e^{La-max} + e^{Lb-max});  O = e^{La-L} Oa + e^{Lb-L} Ob;  (-inf, 0) is the identity.
 * o_a,o_b: device fp32 [N,Hq,d]; lse_a,lse_b: device fp32 [Hq,N]; o_out: device, fp32 or bf16
 * (out_is_bf16 != 0) [N,Hq,d]; lse_out: device fp32 [Hq,N].  Outputs may alias the `a` inputs.
 * Only rows [row_begin,row_end) are read and written. */
int sap_lse_merge(const float* o_a, const float* lse_a, const float* o_b, const float* lse_b,
                  void* o_out, int out_is_bf16, float* lse_out,
                  int64_t n_tokens, int n_q_heads, int head_dim, int64_t row_begin, int64_t row_end,
                  void* cuda_stream);

/* Backward (Table 1 tensors do/dq/dkv).  With P = exp(scale*QK^T - LSE) on the visible
 * pairs: D_t = sum_c dO_tc O_tc; dP = dO V^T; dS = P*(dP - D); dQ = scale dS K; dK = scale dS^T Q;
 * dV = P^T dO; dK/dV are summed over the Hq/Hkv q-heads of a group.
 * dout,q,k,v,out,lse,cu_seqlens_dev: device, read (out/lse as written by sap_attn_fwd).
 * dq [N,Hq,d], dk,dv [N,Hkv,d]: device bf16, written (every element).  workspace: device, at least
 * sap_workspace_bytes(plan, ..., SAP_PASS_BWD) bytes.  dQ is reduced in fp32 with atomic adds, so its low
 * bits may differ from run to run (any accumulation order is correct, A-14); dK, dV are deterministic. */
int sap_attn_bwd(const void* dout, const void* q, const void* k, const void* v, const void* out,
                 const float* lse, const int32_t* cu_seqlens_dev, sap_plan_t* plan, int64_t n_tokens,
                 void* dq, void* dk, void* dv,
                 int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale,
                 void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- backward without allocation --------------------------------------------------------------------------------
 * The same backward pass as sap_attn_bwd (same kernels, same arguments and layouts, same results) for callers that
 * have no way to obtain device memory at the point where they need the gradients: code that runs under a framework
 * whose memory pool is the only permitted allocator and is not reachable from there, a callback or plug-in that is
 * handed tensors but no allocator, a real-time or already memory-budgeted process in which cudaMalloc (a device-wide
 * synchronisation that can also fail late) is ruled out after start-up.  sap_attn_bwd asks such a caller for two
 * things it cannot give: a workspace buffer, and - on the first use of a plan - sap_plan_upload, which calls
 * cudaMalloc.  This entry point needs neither.  The tile program and the workspace (D and the fp32 dQ accumulator)
 * live in a fixed array that is part of the library image on the device: SAP_STATIC_WORKSPACE_BYTES + 256 KiB per GPU
 * that loads the library, held until the process exits whether or not this function is ever called.
 *   - The call itself runs no cudaMalloc, cudaFree, or any other allocating routine, and never uploads the plan's
 *     device mirror; the tile program is copied from the plan's host memory on cuda_stream at every call.
 *   - Limit: sap_workspace_bytes(plan, Hq, Hkv, d, SAP_PASS_BWD) <= SAP_STATIC_WORKSPACE_BYTES, i.e. about
 *     N * Hq * (d + 1) * 4 bytes <= 16 MiB (4096 tokens x 8 q-heads at d = 128), and a tile program of at most 256 KiB
 *     (not reached by plans within the first limit unless they hold thousands of documents).  Anything larger returns
 *     SAP_ERR_STATIC_LIMIT before the device is touched; use sap_attn_bwd with your own workspace then.
 *   - The first call on each device also does that device's one-time set-up (kernel attributes, looking up the
 *     array's device address, and the driver loading the kernels).  Make that first call before any stream capture.
 *   - All calls of a process on one device share the one array.  It keeps what the previous call left; each call
 *     rewrites the program and D and clears the accumulator on cuda_stream before its kernels run.  Calls on the same
 *     stream are therefore safe back to back; two calls that can overlap on the GPU (different streams without an
 *     ordering between them, or different host threads) race on the array and give wrong gradients with no error.
 *     sap_attn_bwd with separate workspaces is the form for concurrent use.
 *   - Returns SAP_ERR_UNSUPPORTED while a non-default sap_debug_set_bwd_stages mask is in force.  Otherwise errors and
 *     asynchrony as sap_attn_bwd; dq, dk, dv are outputs the caller owns. */
#define SAP_STATIC_WORKSPACE_BYTES ((size_t)16 << 20)
int sap_attn_bwd_static(const void* dout, const void* q, const void* k, const void* v, const void* out,
                        const float* lse, const int32_t* cu_seqlens_dev, sap_plan_t* plan, int64_t n_tokens,
                        void* dq, void* dk, void* dv,
                        int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale, void* cuda_stream);

/* ---- per-rank launches ------------------------------------------------------------------
 * The same kernels restricted to the chunks one rank owns (rank i holds Q_i, K_i, V_i).  Token indices
 * stay global: every pointer is the base of the WHOLE [N, H, d] tensor, of which a launch reads the rows the plan
 * names and writes only the rows of its own chunks.  With the tensors laid out across GPUs (peer-mapped virtual
 * memory), a rank's forward streams the K/V tiles of other ranks through TMA while it computes, and a rank's
 * backward adds its dQ contributions into the owner's accumulator with red.global - the transfer is inside the
 * kernel, tile by tile.  On one GPU the chunk ranges simply partition one launch into P launches.
 *
 * sap_attn_fwd_chunks : forward of q-chunks [q_chunk_begin, q_chunk_end): writes out / lse rows of those chunks only.
 * Backward in three phases that ranks run with a barrier in between (workspace as for sap_attn_bwd; all three take
 * the base of the whole workspace):
 *   sap_attn_bwd_begin  : D = rowsum(dO * O) for the rows of q-chunks [begin, end) and zeroes their dQ accumulator rows
 *   sap_attn_bwd_chunks : fused kernel for the K/V tiles of kv-chunks [begin, end): writes dk / dv rows of those
 *                         chunks, adds dQ contributions into the accumulator rows of every q-chunk that attends them;
 *                         needs chunk_len % 128 == 0 (SAP_ERR_UNSUPPORTED otherwise)
 *   sap_attn_bwd_end    : dq rows of q-chunks [begin, end) = bf16(scale * accumulator)
 * All asynchronous on cuda_stream; device pointers as in sap_attn_fwd / sap_attn_bwd. */
int sap_attn_fwd_chunks(const void* q, const void* k, const void* v, const int32_t* cu_seqlens_dev, sap_plan_t* plan,
                        int64_t n_tokens, int32_t q_chunk_begin, int32_t q_chunk_end, void* out, float* lse,
                        int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale, void* cuda_stream);
int sap_attn_bwd_begin(const void* dout, const void* out, sap_plan_t* plan, int64_t n_tokens, int32_t q_chunk_begin, int32_t q_chunk_end,
                       int n_q_heads, int n_kv_heads, int head_dim, void* workspace, size_t workspace_bytes,
                       void* cuda_stream);
int sap_attn_bwd_chunks(const void* dout, const void* q, const void* k, const void* v, const float* lse,
                        const int32_t* cu_seqlens_dev, sap_plan_t* plan, int64_t n_tokens, int32_t kv_chunk_begin, int32_t kv_chunk_end,
                        void* dk, void* dv, int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale,
                        void* workspace, size_t workspace_bytes, void* cuda_stream);
int sap_attn_bwd_end(sap_plan_t* plan, int64_t n_tokens, int32_t q_chunk_begin, int32_t q_chunk_end, void* dq,
                     int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale,
                     void* workspace, size_t workspace_bytes, void* cuda_stream);

/* ---- per-item launches: the `computing` instruction of the backward pass -------------------
 * sap_attn_bwd_items: the fused backward kernel restricted to plan items [item_begin, item_end) (Table 1, PAPER.md:85-98:
 * one `computing` code = one item; the tensors it reads are q / do of the item's rows and kv of its keys, the ones it
 * produces are the dq and dkv CONTRIBUTIONS of that item, :87-96).  K/V-stationary over the 256-key (head_dim 128) or
 * 128-key tiles that intersect the items' key ranges:
 *   dk, dv : device bf16 [N,Hkv,d]; rows of every touched tile are written with the items' contribution (zero where no
 *            item contributes), rows of untouched tiles are left alone - pass scratch buffers and take
 *            [kv_begin, kv_end) of each item;
 *   dQ     : contributions are ADDED into the fp32 accumulator of `workspace` (rows [q_begin, q_end) of each item),
 *            which sap_attn_bwd_begin zeroes (and fills D for) and sap_attn_bwd_end converts.
 * Other arguments, errors and asynchrony as sap_attn_bwd_chunks. */
/* sap_attn_fwd_items: the forward `computing` instruction: as sap_attn_fwd_partial, but only the 128-row Q tiles that
 * intersect the items' row ranges are computed and written (rows of a touched tile without a visible key among the items
 * get out = 0, lse = -inf); rows of other tiles are left alone.  With tensors addressed through shard-sized buffers
 * (base pointer moved back by the shard's first row) a rank therefore needs memory for one shard of q / out and one of
 * k / v, not for the sequence.
 * Shard-pointer contract (both items entry points): the library checks pointers, not what lies behind them.  The
 * kernels move whole tiles with TMA - 128-row boxes that start on multiples of 128 (q, k, v, dout), 256 keys per K/V
 * pair-tile in the head_dim-128 backward - and a box is read in full even where the mask then drops its rows.  A
 * buffer that holds only rows [r0, r0 + n) of a tensor (pointer = buffer - r0 * H * d elements) is therefore legal
 * only if r0 and n are multiples of 128 (256 for k / v / dk / dv of the head_dim-128 backward); with any other shard
 * length pass full-length tensors (rows outside the shard may hold anything finite).  executor.shard_view_ok is the
 * same rule on the Python side; ring.cuda_fns and executor.LocalExecutor apply it. */
int sap_attn_fwd_items(const void* q, const void* k, const void* v, const int32_t* cu_seqlens_dev,
                       sap_plan_t* plan, int64_t n_tokens, int32_t item_begin, int32_t item_end,
                       float* out_f32, float* lse,
                       int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale, void* cuda_stream);
int sap_attn_bwd_items(const void* dout, const void* q, const void* k, const void* v, const float* lse,
                       const int32_t* cu_seqlens_dev, sap_plan_t* plan, int64_t n_tokens, int32_t item_begin, int32_t item_end,
                       void* dk, void* dv, int n_q_heads, int n_kv_heads, int head_dim, float softmax_scale,
                       void* workspace, size_t workspace_bytes, void* cuda_stream);

/* dst = (accumulate ? dst : 0) + alpha * src, elementwise over n_elems values; dst, src: device, fp32 or bf16 each
 * (*_is_bf16), 16-byte aligned, n_elems % 8 == 0.  The COPY instruction for received gradient contributions
 * ("copy-dq / copy-dkv src_buf dst_buf", Table 1: a received dq / dkv is added into the owner's
 * gradient) and the conversion of an fp32 gradient total to bf16.  Asynchronous on cuda_stream. */
int sap_axpy(void* dst, int dst_is_bf16, const void* src, int src_is_bf16, int64_t n_elems, float alpha, int accumulate,
             void* cuda_stream);

/* ---- stitched allocation: the data plane of real ranks ------------------------------ */
/* One device virtual address range of n_chunks * chunk_bytes bytes whose chunk c is physical memory of device
 * device_of_chunk[c], readable and writable by every device in access_devices - the layout that lets a rank's launch
 * (sap_attn_fwd_chunks, sap_attn_bwd_chunks) read the K/V shards its plan names where they live and add its dQ
 * contributions into their owner's accumulator, instead of the grouped send / recv of PAPER.md:59, :100-102, :124 (inside
 * an NVLink / NVSwitch domain).  A tensor [N, H, d] placed at sap_stitched_ptr has rows [c n, (c+1) n) of chunk c in
 * device_of_chunk[c]'s memory when chunk_bytes = n * H * d * sizeof(element).
 * chunk_bytes must be a multiple of sap_stitched_granularity of every owner (2 MiB on B200), else SAP_ERR_UNSUPPORTED.
 * All arrays are host arrays, read.  Synchronous (CUDA virtual-memory API); several devices need P2P access between them
 * (SAP_ERR_CUDA with the CUresult in sap_last_cuda_error otherwise).  The range belongs to the handle: sap_stitched_free
 * unmaps and releases it (NULL is a no-op); the caller must have finished all work that uses it.
 * This call is the form for one process driving several devices; sap_stitched_create_local below is the one for one
 * process per GPU. */
typedef struct sap_stitched sap_stitched_t;
int sap_stitched_granularity(int device, size_t* bytes);
int sap_stitched_alloc(int32_t n_chunks, size_t chunk_bytes, const int32_t* device_of_chunk, int32_t n_access,
                       const int32_t* access_devices, sap_stitched_t** out);
void* sap_stitched_ptr(const sap_stitched_t* s);            /* device pointer of the range (NULL for NULL) */
size_t sap_stitched_bytes(const sap_stitched_t* s);         /* n_chunks * chunk_bytes */
int32_t sap_stitched_owner(const sap_stitched_t* s, int32_t chunk);   /* device that holds chunk, -1 if out of range */
void sap_stitched_free(sap_stitched_t* s);
/* The same range with one process per GPU (the launch model of torch.distributed): every process reserves the whole
 * range on its `device`, creates and maps the chunks c with own[c] != 0 (host array [n_chunks]) as exportable allocations,
 * hands a POSIX file descriptor of each to the other processes (sap_stitched_export_fd; the descriptor travels over a Unix
 * socket with SCM_RIGHTS, the receiver closes it after the import) and maps theirs (sap_stitched_import_fd, chunk not yet
 * mapped).  A chunk that is not mapped must not be touched.  sap_stitched_owner is -1 for imported chunks.  Synchronous. */
int sap_stitched_create_local(int32_t n_chunks, size_t chunk_bytes, int device, const uint8_t* own, sap_stitched_t** out);
int sap_stitched_export_fd(const sap_stitched_t* s, int32_t chunk, int* fd);
int sap_stitched_import_fd(sap_stitched_t* s, int32_t chunk, int fd);

/* ---- diagnostics ---------------------------------------------------------------------------- */
const char* sap_strerror(int status);
int sap_last_cuda_error(void);      /* the cudaError_t / CUresult of the last SAP_ERR_CUDA on this thread */
/* Number of kernels the library has launched in this process (all streams); for launch accounting. */
int64_t sap_launch_count(void);
/* Diagnostic (host only, no GPU): the tile program the kernels walk, as flat int32 records - tiles [n][4] = (row0, rows,
 * seg_begin, seg_end) of each stationary tile, segs [n][8] = (t_begin, t_end, q_lo, q_hi, kv_lo, kv_hi, item, 0) of each
 * run of streamed tiles: element (row t, key s) of a (tile, segment) is computed iff t (Q-stationary) or s
 * (K/V-stationary) lies in the tile, the other index in [t_begin, t_end), q_lo <= t < q_hi, kv_lo <= s < kv_hi, both in
 * one document and s <= t.  kind: 0 forward (Q-stationary), 1 / 2 backward K/V-stationary with 128- / 256-key tiles;
 * 3 / 4 items [a, b) Q-stationary (all tiles / touched tiles: sap_attn_fwd_partial / sap_attn_fwd_items); 5 q-chunks
 * [a, b) (sap_attn_fwd_chunks); 6 / 7 kv-chunks [a, b) with 128- / 256-key tiles (sap_attn_bwd_chunks); 8 / 9 items
 * [a, b) K/V-stationary (sap_attn_bwd_items); 10 forward with 256-row Q tiles (two 128-row units of one head per work
 * item: the forward of odd Hq/Hkv, e.g. MHA).  Returns the number of tiles (call with null buffers to size), *n_segs
 * the number of segments; < 0 on error.  Buffers are filled only when large enough. */
int32_t sap_debug_tile_program(const sap_plan_t* plan, int32_t kind, int32_t a, int32_t b, int32_t* tiles, int32_t tiles_cap,
                               int32_t* segs, int32_t segs_cap, int32_t* n_segs);
/* Diagnostic: which forward kernel the forward calls launch.  0 (default): the persistent pair kernel on head pairs (two
 * q-heads of one GQA group per work item, sharing the K/V tiles) whenever Hq/Hkv is even; for odd Hq/Hkv (MHA) the same
 * kernel on row pairs (two 128-row halves of a 256-row tile of one q-head) in sap_attn_fwd when the launch has at least
 * 16 work items per SM, the one-head kernel otherwise; 1: always the one-head kernel; 2: row pairs in sap_attn_fwd whatever
 * the size and Hq/Hkv.  Process-wide; returns the previous value. */
int sap_debug_set_fwd_form(int form);
/* Diagnostic: which fused backward main kernel runs at head_dim 128.  0 (default): the CTA-pair kernel (tcgen05
 * cta_group::2 over 256-key pair-tiles); 1: the one-CTA kernel (always used at head_dim 64).  Process-wide; returns the
 * previous value. */
int sap_debug_set_bwd_form(int form);
/* Diagnostic: which kernels sap_attn_bwd launches, so each can be timed alone and the two forms of the main
 * pass compared.  Bits: 1 = D pre-pass, 8 = fused main kernel (dK, dV, fp32 dQ accumulator; 5 GEMMs per tile
 * pair; zeroes the accumulator first), 16 = dQ post pass (bf16(scale * accumulator)); 2 = split dK/dV kernel,
 * 4 = split dQ kernel (the deterministic, atomics-free form: 7 GEMMs per tile pair).  Default 1|8|16; a negative
 * mask restores the default.  Process-wide; returns the previous mask.  With a partial mask the skipped outputs
 * are left untouched. */
int sap_debug_set_bwd_stages(int mask);

#ifdef __cplusplus
}
#endif
#endif /* SAP_H_ */
