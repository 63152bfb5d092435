/*
 * cocoscale.h -- C ABI of the B200-native replicated decoder-layer hot path of CoCoScale
 * (arxiv/paper_2607_04181, "layer-wise scaling"; PAPER.md = the paper text as surveyed).
 *
 * What this library is: the forward of ONE hot decoder layer over a decode batch that is split
 * across that layer's replicas (section 3.1), on ONE GPU, where a replica is an
 * extra byte copy of the layer's weights held in reclaimed HBM; plus creating / retiring such
 * replicas without ever re-capturing the CUDA Graph that replays the forward (the paper
 * re-captures when the configuration vector v changes; here a device-resident
 * replica table is read by the kernels instead).
 *
 * Layer arithmetic (BASELINE.json north_star; the paper gives none):  RMSNorm -> QKV projection
 * -> RoPE (rotate-half, position seq_len-1) -> KV append -> paged GQA decode attention
 * -> O projection + residual -> RMSNorm -> SwiGLU MLP -> down projection + residual.
 * bf16 storage, fp32 accumulation.  Readings of every point the paper leaves open: DESIGN.md.
 *
 * Conventions
 *   - All pointers named *_dev / documented "device" are device memory of the context's GPU;
 *     everything else is host memory.  The library never takes ownership of caller memory.
 *   - `stream` arguments are a `cudaStream_t` passed as `void*` (NULL = legacy default stream).
 *   - Every call returns a cc_status; on failure cc_last_error() (thread-local) says why.
 *     No exception or abort crosses this boundary.
 *   - One control thread per cc_ctx.  cc_forward only ENQUEUES work (no allocation, no
 *     synchronisation, no host read of device data) and is safe inside stream capture.
 *   - Forwards of one context must not overlap on the device: enqueue them on ONE stream (or
 *     order the streams with events).  The GEMM kernels are persistent (one CTA per SM) and their
 *     CTAs wait for one another in the stream-K fixup; two such grids sharing the SMs could
 *     starve each other.  Replica copies on the side stream may overlap freely.
 *   - Caller-owned buffers handed to cc_forward (hidden, KV pools, block table, seq_lens,
 *     replica_assign) must keep their addresses while a captured graph that contains the call is
 *     alive ("tensor memory addresses remain constant across iterations").
 *   - There is no CPU fallback: without a usable CUDA device every compute entry point fails
 *     with CC_ERR_CUDA.
 */
#ifndef COCOSCALE_H_
#define COCOSCALE_H_

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif
#if defined(__GNUC__)
#pragma GCC visibility push(default)   /* the library is built with -fvisibility=hidden */
#endif

#define CC_MAX_REPLICAS 4   /* P_max = 4 */
#define CC_PAGE_SIZE 16     /* tokens per KV page (BASELINE.json configs) */
#define CC_MAX_LAYERS 128   /* rows of the device replica table per context */

typedef enum {
    CC_OK = 0,
    CC_ERR_INVALID = 1,  /* bad argument / unsupported shape                                  */
    CC_ERR_NO_SLOT = 2,  /* no donated range can hold another replica (infeasible Delta_res,  */
                         /* PAPER.md:320-323)                                                 */
    CC_ERR_CUDA = 3,     /* a CUDA call failed, or no device                                  */
    CC_ERR_BUSY = 4,     /* range still holds a live slot / replica still copying             */
    CC_ERR_STATE = 5     /* e.g. releasing replica 0 or a replica that is not live            */
} cc_status;

/* Bits of the sticky device error word (cc_poll_device_error). Set by kernels on contract
 * violations that are only visible on the device inside a graph; never a fault. */
#define CC_DEVERR_BAD_REPLICA 1u   /* replica_assign[b] not an active replica: row ran on replica 0 */
#define CC_DEVERR_BAD_PAGE 2u      /* block-table entry < 0 or >= n_pages inside seq_len: row skipped */
#define CC_DEVERR_BAD_SEQLEN 4u    /* seq_len > max_position or needs > max_blocks_per_seq: row skipped */
#define CC_DEVERR_HANG 8u          /* reserved: an internal wait gave up (the kernel traps instead)       */
#define CC_DEVERR_TOO_MANY_DECODE 32u /* a step of more than 256 rows holds more than 256 decode rows, 64 prompt chunks or
                                      * 1024 query tiles: the surplus is skipped */
#define CC_DEVERR_SPLIT_REQUEST 16u /* rows of one request (same first page) name different replicas: each row
                                      still runs on the replica it names, but the request's KV then spans two
                                      partitions -- not what PAPER.md:103 "each replica maintains its own
                                      partition" allows                                                     */

typedef struct cc_ctx cc_ctx;     /* device, side stream, donated ranges, replica table, error word */
typedef struct cc_layer cc_layer; /* one decoder layer: slot 0 blob, replica slots, workspace        */

typedef struct {
    int32_t hidden;              /* d; multiple of 64, at most 8192                             */
    int32_t n_q_heads;           /* Hq                                                          */
    int32_t n_kv_heads;          /* Hkv in {1, 2, 4, 8}; Hq % Hkv == 0 and Hq / Hkv <= 8        */
    int32_t head_dim;            /* Dh: 64 or 128                                               */
    int32_t ffn;                 /* F (SwiGLU width)                                            */
    float rms_eps;
    float rope_base;
    int32_t page_size;           /* must be CC_PAGE_SIZE                                        */
    int32_t max_batch;           /* rows per cc_forward call, 1..256                            */
    int32_t max_blocks_per_seq;  /* row width of the block table                                */
    int32_t max_position;        /* largest seq_len accepted (RoPE table rows)                  */
} cc_layer_desc;

/* bf16, DEVICE, each matrix [out][in] row-major (y = W x), gains [hidden].
 * wq [Hq*Dh][d], wk/wv [Hkv*Dh][d], wo [d][Hq*Dh], wgate/wup [F][d], wdown [d][F]. */
typedef struct {
    const void *g1, *wq, *wk, *wv, *wo, *g2, *wgate, *wup, *wdown;
} cc_layer_weights;

/* Paged KV cache of this layer (caller-owned, DEVICE).
 * k_pool / v_pool: bf16 [n_pages][n_kv_heads][CC_PAGE_SIZE][head_dim]; K is stored post-RoPE.
 * block_table: int32 [max_batch][max_blocks_per_seq]; entry j of row b is the page holding
 * tokens [16j, 16j+16) of request b; padding = -1 (never dereferenced below seq_len). The caller
 * has already placed the page that holds position seq_len-1. */
typedef struct {
    void *k_pool;
    void *v_pool;
    const int32_t *block_table;
    int32_t n_pages;
} cc_kv_pages;

/* ---- context ------------------------------------------------------------------------------ */
cc_status cc_ctx_create(int device, cc_ctx **out);
cc_status cc_ctx_destroy(cc_ctx *ctx); /* all layers must have been destroyed */

/* "Reclaimed HBM": lend [dev_base, dev_base+bytes) (device memory the caller keeps owning) as
 * replica slot space.  Trimmed to 1024-byte boundaries.  CC_ERR_INVALID if it overlaps a range
 * already donated.  cc_ctx_reclaim takes it back; CC_ERR_BUSY while any live slot lies in it. */
cc_status cc_ctx_donate(cc_ctx *ctx, void *dev_base, size_t bytes);
cc_status cc_ctx_reclaim(cc_ctx *ctx, void *dev_base);

/* Chunk size of the replica copy ("fine-grained chunked transfer"); one kernel
 * launch per chunk on the context's side stream.  Default 32 MiB; multiple of 1 MiB. */
cc_status cc_ctx_set_copy_chunk(cc_ctx *ctx, size_t chunk_bytes);

/* Programmatic dependent launch between the kernels of one cc_forward (default on; the
 * environment variable CC_PDL=0 turns it off at cc_ctx_create).  A launch attribute only: the
 * kernels and their results are the same either way. */
cc_status cc_ctx_set_pdl(cc_ctx *ctx, int enabled);

/* GEMM operand format of the layers created AFTER this call (the blob is packed at cc_create_layer).  The paper fixes
 * no arithmetic ("Transformer layers"); north_star fixes bf16 storage and the tolerance.
 *   CC_OPERAND_F16    the bf16 weights are converted to fp16 when packed (exact for 2^-17 <= |w| <= 65504, rounded to
 *                     the 2^-24 grid below that) and every GEMM operand is ONE fp16 plane (11 significand bits);
 *                     cc_create_layer fails with CC_ERR_INVALID if a weight exceeds the fp16 range;
 *   CC_OPERAND_BF16X2 weights stay bf16, operands are TWO bf16 planes hi + lo (16 bits; twice the tensor work);
 *   CC_OPERAND_AUTO   (default) F16, falling back to BF16X2 for a layer with a weight outside the fp16 range.
 * The environment variable CC_OPERAND_FORMAT=f16|bf16x2 sets the same at cc_ctx_create. */
enum { CC_OPERAND_AUTO = 0, CC_OPERAND_F16 = 1, CC_OPERAND_BF16X2 = 2 };
cc_status cc_ctx_set_operand_format(cc_ctx *ctx, int format);

/* Activation planes of the four GEMM operands (x: QKV input, o: O input, y: gate/up input, a: down input) of
 * CC_OPERAND_F16 layers, chosen per step: a step of at most `rows` rows takes planes_upto_rows[4], a larger one
 * planes_above[4]; each entry 1 (one fp16 plane, 11 significand bits) or 2 (hi + lo fp16 planes, twice the tensor
 * work of that projection, and a larger activation slab per pipeline stage).  The default is {2,1,1,1} for every step
 * size (rows = 64): the QKV input is the operand whose rounding shows (DESIGN.md "Precision" has the measured errors of
 * every choice).  The choice depends on the step's
 * row count only, never on replica_assign, so outputs stay bit-identical across replica counts.  The environment
 * variable CC_PLANES="xoya,xoya[,rows]" sets the same at cc_ctx_create.  BF16X2 layers always use two planes. */
cc_status cc_ctx_set_operand_planes(cc_ctx *ctx, int rows, const int *planes_upto_rows, const int *planes_above);

/* Sticky device error word (CC_DEVERR_* bits); reading clears it. Synchronises the device. */
cc_status cc_poll_device_error(cc_ctx *ctx, uint32_t *bits);

/* ---- layer lifecycle ------------------------------------------------------------------------ */
/* Re-packs the nine weight tensors into one library-owned blob ("slot 0": tcgen05 operand tile
 * images + gains), allocates the layer's workspace and its replica-table row.  Everything the
 * layer will ever need is allocated here (PAPER.md:393 persistent pool); later calls allocate
 * nothing on the device.  Synchronous. */
cc_status cc_create_layer(cc_ctx *ctx, const cc_layer_desc *desc, const cc_layer_weights *weights_dev,
                          cc_layer **out);
cc_status cc_destroy_layer(cc_layer *layer);

/* The operand format this layer was packed in: CC_OPERAND_F16 or CC_OPERAND_BF16X2. */
cc_status cc_layer_operand_format(const cc_layer *layer, int *format);

/* Bytes of one replica slot of this layer (= bytes cc_scale_layer copies per new replica). */
cc_status cc_layer_blob_bytes(const cc_layer *layer, size_t *bytes);

/* Set the TARGET replica count, 1..CC_MAX_REPLICAS (a replica is a copy of the
 * layer's weights).  Growing: takes the lowest free slot(s) from the donated ranges and enqueues
 * the chunked in-HBM copy of slot 0 on the side stream; returns at once (CC_ERR_NO_SLOT if no
 * range fits; nothing changes then).  Shrinking: marks the highest-numbered live replicas for
 * retirement.  Nothing becomes visible to cc_forward until cc_commit. */
cc_status cc_scale_layer(cc_layer *layer, int n_replicas);

/* Publish: makes `stream` wait for the finished copies, then enqueues the replica-table update
 * (new rows / retired rows) on `stream`, so that forwards enqueued or replayed on `stream`
 * AFTER this call see the new replica set and earlier ones the old.  Retired slots return to
 * the allocator once the work enqueued before the flip has finished (checked lazily by later
 * calls).  Never captures or re-captures anything; must be called outside stream capture.
 * No-op when nothing is pending. */
cc_status cc_commit(cc_layer *layer, void *stream);

/* Retire one live replica (1..CC_MAX_REPLICAS-1); takes effect at the next cc_commit.
 * CC_ERR_STATE for replica 0 or a replica that is not live / already retiring. */
cc_status cc_release_replica(cc_layer *layer, int replica);

/* n_active: replicas visible to forwards enqueued now; n_pending: copies enqueued by
 * cc_scale_layer and not yet committed. Either pointer may be NULL. */
cc_status cc_query(cc_layer *layer, int *n_active, int *n_pending);

/* A replica's own KV partition ("a replica holds a copy of the weights AND the KV of its requests",
 * PAPER.md:103 "each replica maintains its own partition"): from now on the rows that replica_assign gives to
 * `replica` append and read their K/V in THESE pools ([n_pages][n_kv_heads][16][head_dim] bf16, device memory the
 * caller owns, 16-byte aligned), and the page ids in their block-table rows are relative to them; replicas without a
 * partition keep using the pools passed to cc_forward.  k_pool_dev = v_pool_dev = NULL removes the partition.  The
 * base pointers go into the layer's row of the device replica table (enqueued on `stream`; the QKV epilogue reads them
 * there); the attention kernels take one TMA descriptor per replica as launch parameters, so a CAPTURED graph keeps
 * the pools it was captured with: set partitions before capturing.  All rows of one request must name one replica. */
cc_status cc_layer_set_kv_partition(cc_layer *layer, int replica, void *k_pool_dev, void *v_pool_dev, int32_t n_pages,
                                    void *stream);

/* Which replica indices forwards enqueued now may name: bit r of *mask set <=> replica r is live and
 * published.  After cc_release_replica(layer, 1) with three live replicas the set is {0, 2}: indices are
 * not compacted (a captured graph and the caller's replica_assign keep their meaning), so a caller that
 * splits a batch must split it over THESE indices -- naming a retired index sets CC_DEVERR_BAD_REPLICA
 * and the row runs on replica 0. */
cc_status cc_active_replicas(cc_layer *layer, uint32_t *mask);

/* Device address and size of replica r's blob (for byte-exact checks of the copy). */
cc_status cc_replica_blob(cc_layer *layer, int replica, const void **blob_dev, size_t *bytes);

/* ---- the hot path --------------------------------------------------------------------------- */
/* One decode step of the layer over `batch` rows (batch <= max_batch), in place on hidden_dev.
 *   hidden_dev      bf16 [batch][hidden], DEVICE; row b is replaced by the layer's output for
 *                   request b (original request order: PAPER.md:101 gather + concat).
 *   kv              see cc_kv_pages; the step appends request b's new K/V at position
 *                   seq_lens[b]-1 and attends over positions [0, seq_lens[b]).
 *   seq_lens_dev    int32 [batch], DEVICE: tokens attended INCLUDING the one being decoded.
 *                   seq_lens[b] <= 0 marks a padding row: left untouched, no KV write.
 *   replica_assign_dev  int32 [batch], DEVICE: which replica's weights serve row b
 *                   (PAPER.md:93 sub-batches; any assignment, any group sizes including 0).
 * Several rows may belong to ONE request (a prompt chunk): they carry copies of its block-table row and
 * consecutive seq_lens t+1, t+2, ...; every row's K/V is appended before any row attends, so the row
 * of token t attends exactly positions <= t (causal prefill through the decode kernels; such rows must
 * name the same replica if the caller keeps KV partitions).  tests/test_prefill_chunk.py.
 * Rows are grouped by replica on the device; each group streams ITS replica's weight slot, read
 * through the device replica table, so a graph captured around this call keeps working across
 * cc_commit.  Results are bit-identical for any assignment and replica count. */
cc_status cc_forward(cc_layer *layer, void *hidden_dev, const cc_kv_pages *kv, const int32_t *seq_lens_dev,
                     const int32_t *replica_assign_dev, int batch, void *stream);

/* Same step with HOST buffers for the per-step inputs: copies block table, seq_lens and
 * replica_assign to library-owned device staging (through a pinned mirror, one transfer; the
 * three buffers may be pageable), runs the step and synchronises `stream`; on
 * return hidden_host holds the result rows (padding rows untouched).  When hidden_host is pinned
 * memory mapped into the device's address space (cudaHostAlloc / cudaHostRegister, 16-byte
 * aligned) the kernels read and write it in place: the first kernel fetches the rows over PCIe
 * (keeping a device copy for the residual) and the last epilogue stores the result rows to it.
 * Otherwise hidden is staged through two copies.  Same results bit for bit either way.  The KV
 * pools stay on the device (they are state, like the weights).  block_table_host is
 * [batch][max_blocks_per_seq]. */
cc_status cc_forward_host(cc_layer *layer, void *hidden_host, void *k_pool_dev, void *v_pool_dev,
                          int32_t n_pages, const int32_t *block_table_host, const int32_t *seq_lens_host,
                          const int32_t *replica_assign_host, int batch, void *stream);

/* The same, ENQUEUE-ONLY: returns once the copies and kernels are on `stream`; hidden_host holds the result after the
 * caller has synchronised the stream (or an event recorded behind the call).  Lets consecutive steps overlap their host
 * work (table marshalling, launches) with the device work of the step before.  Needs the pinned, mapped hidden_host of
 * the in-place path (CC_ERR_INVALID otherwise) and batch <= 256; hidden_host must stay untouched until the step has run;
 * block_table_host / seq_lens_host / replica_assign_host are consumed before the call returns. */
cc_status cc_forward_host_async(cc_layer *layer, void *hidden_host, void *k_pool_dev, void *v_pool_dev,
                          int32_t n_pages, const int32_t *block_table_host, const int32_t *seq_lens_host,
                          const int32_t *replica_assign_host, int batch, void *stream);

/* The same step, launched kernel by kernel with a CUDA event between consecutive kernels (so
 * without programmatic dependent launch), synchronised; stage_ms_host[i] (host, fp32
 * [CC_MAX_PROFILE_STAGES], unused entries 0) receives the device time of kernel i in milliseconds, in launch
 * order: grouping + input norm, QKV GEMM (+RoPE, KV append), attention (+chunk merge), O GEMM
 * (+residual, norm statistics), gate/up GEMM (+norm scale, SwiGLU), down GEMM (+residual, request
 * order); for a step of more than 256 rows: grouping, input norm, QKV GEMM, decode attention, chunk-prefill
 * attention, O GEMM, row statistics, gate/up GEMM, down GEMM.  For per-kernel roofline accounting; not capture-safe.  hidden_dev may also be the pinned
 * host buffer of cc_forward_host (its in-place path is then what is timed). */
#define CC_MAX_PROFILE_STAGES 10
cc_status cc_forward_profiled(cc_layer *layer, void *hidden_dev, const cc_kv_pages *kv, const int32_t *seq_lens_dev,
                              const int32_t *replica_assign_dev, int batch, void *stream, float *stage_ms_host);

/* Grid of the four projection kernels (QKV, O, gate/up, down) of a SMALL step (<= 80 rows) of this layer: ctas[4] CTAs
 * each, in clusters of cluster[4] CTAs (0 = the stream-K kernel, one CTA per SM; > 0 = the cluster split-K kernel, one
 * cluster per 256 output features).  A function of the layer shape and the device, fixed at cc_create_layer. */
cc_status cc_layer_gemm_grids(const cc_layer *layer, int *ctas, int *cluster);

/* Kernel launches one cc_forward enqueues (for launch accounting). */
cc_status cc_forward_launch_count(const cc_layer *layer, int *n);

/* The vectorised chunked copy kernel on its own: dst/src DEVICE, 32-byte aligned (256-bit
 * accesses), bytes % 16 == 0, else CC_ERR_INVALID; chunk_bytes = 0 uses the context's chunk size.
 * Enqueue-only on `stream`. */
cc_status cc_replica_copy(cc_ctx *ctx, void *dst_dev, const void *src_dev, size_t bytes, size_t chunk_bytes,
                          void *stream);

/* ---- KV partition per replica (a replica holds its requests' KV; PAPER.md:103, 119:
 * the cache is redistributed, chunk by chunk, when the parallelism degree changes) --------------- */
/* Host-only planner.  The page pool [0, n_pages) is cut into n_replicas equal partitions, partition r =
 * pages [r * (n_pages / n_replicas), (r + 1) * (n_pages / n_replicas)).  For the rows in increasing
 * order and their pages in increasing order (only pages below ceil(seq_len / 16), rows with
 * seq_len <= 0 are skipped), every page that lies outside the partition of the row's replica moves to
 * the LOWEST page of that partition that no live row referenced before the call and no earlier move
 * took.  Outputs: the re-mapped block table (same shape; untouched entries copied), the move list
 * src -> dst in that order, its length.  CC_ERR_NO_SLOT (outputs unspecified) when a partition has too
 * few free pages; CC_ERR_INVALID on a bad table (entry out of range or referenced twice). */
cc_status cc_kv_plan_migration(const int32_t *block_table_host, const int32_t *seq_lens_host,
                               const int32_t *replica_assign_host, int batch, int max_blocks_per_seq, int n_pages,
                               int n_replicas, int32_t *new_block_table_host, int32_t *src_pages_host,
                               int32_t *dst_pages_host, int *n_moves);

/* Pre-copy migration, second half (the transfer is chunked and fitted between decode steps, so
 * decoding goes on -- with the OLD table -- while the bulk of a plan is copied on a side stream).  Once that copy
 * has finished, this plans what the steps wrote meanwhile.  seq_lens_planned is the seq_lens array the first
 * plan was made with (of the last step enqueued before it, or of the next one: a step writes position
 * seq_len - 1, so either way only positions >= seq_lens_planned - 1 can have changed).  For every row, pages
 * with index < (seq_lens_planned - 1) / 16 keep the place `planned_block_table` gave them; the tail page of
 * then and every page added since are taken from `block_table_now` and planned by cc_kv_plan_migration's
 * rule over that hybrid table.  seq_lens_now[b] >= seq_lens_planned[b], or 0 for a row
 * that finished (a slot re-used by a new request passes seq_lens_planned[b] = 0).  The caller must not have
 * handed out a destination of the first plan as a new page meanwhile (CC_ERR_INVALID: referenced twice).
 * Outputs as cc_kv_plan_migration: `final_block_table` is the table to swap in after the returned moves ran. */
cc_status cc_kv_plan_catchup(const int32_t *block_table_now_host, const int32_t *seq_lens_planned_host,
                             const int32_t *seq_lens_now_host, const int32_t *planned_block_table_host,
                             const int32_t *replica_assign_host, int batch, int max_blocks_per_seq, int n_pages,
                             int n_replicas, int32_t *final_block_table_host, int32_t *src_pages_host,
                             int32_t *dst_pages_host, int *n_moves);

/* Copies page src[i] -> dst[i] (all kv heads, page_bytes = n_kv_heads * 16 * head_dim * 2) in both pools,
 * for i < n_moves; src/dst lists are DEVICE int32.  Sources and destinations must be disjoint sets (the
 * planner guarantees it).  Enqueue-only on `stream`: put it between decode steps, or on a side stream
 * ordered before the step that uses the new block table. */
cc_status cc_kv_migrate(cc_ctx *ctx, void *k_pool_dev, void *v_pool_dev, size_t page_bytes,
                        const int32_t *src_pages_dev, const int32_t *dst_pages_dev, int n_moves, void *stream);

/* ---- the paper's cost / speed-up model and scaling decision (host only; Eq. 1-10,
 * PAPER.md:290-353 Algorithm 2).  The hot path takes replica counts and replica_assign from its caller;
 * this is the piece that would choose them.  Readings: DESIGN.md 7c. -------------------------------- */
typedef struct {
    int32_t L;                    /* layers of the model                                             */
    int32_t P_max;                /* largest parallelism degree considered, <= CC_MAX_REPLICAS        */
    double slo;                   /* latency objective                                               */
    double delta;                 /* tolerance band |latency - SLO| / SLO <= delta: no action          */
    double beta[CC_MAX_REPLICAS + 1]; /* beta(P) = T(P) / (L * t_comp), index P (beta[1] = 0)          */
    double cost_per_device;       /* Cost(N, P) = cost_per_device * (P - 1) + cost_per_layer_copy * N * (P - 1) */
    double cost_per_layer_copy;
} cc_ctl_params;
typedef enum { CC_CTL_NONE = 0, CC_CTL_UPDATED = 1, CC_CTL_INSTANCE_SCALE = 2 } cc_ctl_action;

double cc_ctl_mem_bytes(int N, int P, int bs, int l, int d_hidden, double kappa);             /* Eq. 1 */
double cc_ctl_flops(int N, int P, int bs, int l, int d_hidden);                               /* Eq. 2 */
double cc_ctl_comm_seconds(int P, int bs, int l, int d_hidden, double kappa, double bandwidth_bytes_per_s); /* Eq. 5 */
double cc_ctl_speedup(int L, int N, int P, double beta);                                      /* Eq. 7 */
double cc_ctl_speedup_vec(const int32_t *v, int L, int bs, double t_comp_s, int d_hidden, double kappa,
                          double bandwidth_bytes_per_s);                                      /* Eq. 8-10 */
int cc_ctl_distance(int N0, int P0, int N1, int P1);                  /* Dist of Algorithm 2, nested segments */
int cc_ctl_candidate_count(int L, int P_max);                         /* L * P_max            */
/* One pass of Algorithm 2's body for one instance: on CC_CTL_UPDATED the new (N, P) is written and
 * *cold_capacity reduced by the resource difference (increased when it is negative). */
cc_status cc_ctl_decide(const cc_ctl_params *p, int N_cur, int P_cur, double latency, double *cold_capacity,
                        int *N_new, int *P_new, cc_ctl_action *action);

/* Algorithm 1, initial global placement: instances in descending Priority = load - capacity
 * (Eq. 11) each take, among the (N, P) with 1 <= N <= L, 2 <= P <= P_max whose per-device memory C_mem(N, P)
 * (Eq. 1) fits on at least P - 1 devices of the pool (Load < tau_idle, not yet taken), the one of largest S(N, P)
 * (Eq. 7 with p->beta; ties: fewer devices, then fewer layers) and the P - 1 fitting devices of largest free
 * memory (ties: lower index).  Only P_max and beta of `p` are used.  `out` has room for n_inst entries;
 * instances that fit nowhere get none.  On one GPU there is nothing to place: this is the paper's bootstrap
 * step stated for completeness of the controller. */
typedef struct {
    int32_t L, bs, l, d_hidden;   /* layers, batch size, sequence length, hidden size (Eq. 1)            */
    double kappa;                 /* bytes per element                                                   */
    double load, capacity;        /* current load and sustainable load of the instance (Eq. 11)          */
} cc_ctl_instance;
typedef struct {
    double load;                  /* compute utilisation of the device, same unit as tau_idle            */
    double free_mem_bytes;
} cc_ctl_device;
typedef struct {
    int32_t instance, N, P;
    int32_t devices[CC_MAX_REPLICAS - 1];   /* P - 1 device indices, then -1                              */
    double speedup;
} cc_ctl_placement;
cc_status cc_ctl_place(const cc_ctl_params *p, const cc_ctl_instance *instances, int n_instances,
                       const cc_ctl_device *devices, int n_devices, double tau_idle, cc_ctl_placement *out,
                       int *n_out);

/* ---- timeline of a tracing build (measurement aid) ---------------------------------------------
 * A library built with -DCC_TRACE (python -m paper_2607_04181_b200.build --trace) records, for every kernel of
 * cc_forward and every trace point in it, the earliest and latest %globaltimer value (ns) over the CTAs that
 * passed the point.  out_host (may be NULL): uint64 [16][8][2] = [kernel][point][min, max]; kernel 0 = prologue
 * (points: entry, dependency wait done, end), 1 = attention (entry, dependency wait done, consumers saw the end),
 * 2..5 = QKV / O / gate-up / down GEMM (entry, dependency wait done, producer issued all, mainloop drained and
 * partials stored, first fixup wait done, end); 8..11 = min / max duration of a CTA's first ([0]) and second ([1])
 * stream-K fixup pass of those GEMMs, 12..15 = [0..1][max] number of such passes, [2..3][max] their summed
 * duration.  reset != 0 re-arms the buffer after the read.  Synchronises the device.  CC_ERR_STATE in a product
 * build (the points compile to nothing there).  Driver: python -m paper_2607_04181_b200.timeline. */
cc_status cc_debug_trace(cc_ctx *ctx, uint64_t *out_host, int reset);

/* ---- stage taps (tests only; reads the workspace left by the last cc_forward) ---------------- */
typedef enum {
    CC_TAP_X = 0,   /* [batch][hidden]      input RMSNorm output (GEMM operand, layer format)    */
    CC_TAP_Q = 1,   /* [batch][Hq*Dh]       q after RoPE (fp32)                                 */
    CC_TAP_O = 2,   /* [batch][Hq*Dh]       attention output (GEMM operand, layer format)        */
    CC_TAP_H1 = 3,  /* [batch][hidden]      hidden + O-projection (fp32)                        */
    CC_TAP_Y = 4,   /* [batch][hidden]      post-attention RMSNorm output (operand x its row scale) */
    CC_TAP_A = 5    /* [batch][ffn]         silu(gate)*up (GEMM operand, layer format)          */
} cc_tap;
/* out_host: fp32 [batch][dim] in ORIGINAL row order; padding rows are zero. Synchronous. */
cc_status cc_debug_tap(cc_layer *layer, cc_tap which, float *out_host, int batch);
/* perm_host[pos] (int32, length >= max_batch + 64): original row at grouped position pos or -1;
 * counts_host[CC_MAX_REPLICAS]: rows per replica group, from the last cc_forward. Synchronous. */
cc_status cc_debug_grouping(cc_layer *layer, int32_t *perm_host, int32_t *counts_host, int32_t *n_pos);

/* ---- host-only slot allocator (the same code cc_ctx uses; exposed so it can be tested without
 * a GPU).  Addresses are plain integers here. ---------------------------------------------------- */
typedef struct cc_slotalloc cc_slotalloc;
cc_slotalloc *cc_slotalloc_create(void);
void cc_slotalloc_destroy(cc_slotalloc *a);
cc_status cc_slotalloc_donate(cc_slotalloc *a, uint64_t base, uint64_t bytes);
cc_status cc_slotalloc_reclaim(cc_slotalloc *a, uint64_t base);
cc_status cc_slotalloc_alloc(cc_slotalloc *a, uint64_t bytes, uint64_t *addr); /* lowest address that fits */
cc_status cc_slotalloc_free(cc_slotalloc *a, uint64_t addr);
uint64_t cc_slotalloc_free_bytes(const cc_slotalloc *a);

/* ---- an entry point that allocates nothing ---------------------------------------------------------------------
 * Paged GQA decode attention as a stand-alone call for callers that cannot
 * allocate device memory: it needs no cc_ctx and no layer and calls no cudaMalloc / cudaFree / allocating library
 * routine.  Its split-KV partial results live in ONE file-scope device array of CC_STATIC_SCRATCH_BYTES that every GPU
 * which loads the library holds until the process exits (cc_forward keeps the same partials in the layer workspace that
 * cc_create_layer allocates, and is the fast path: TMA page boxes, one CTA per SM).
 *   q           device, fp32 [batch][n_q_heads][head_dim], post-RoPE, unscaled (the 1/sqrt(head_dim) is applied here)
 *   k_pool,     device, bf16 [n_pages][n_kv_heads][16][head_dim] (the layout of cc_forward's pools), read only
 *   v_pool
 *   block_table device, int32 [batch][max_blocks]; entries below ceil(seq_len / 16) must be valid page ids (an id
 *               outside [0, n_pages) is read as page 0, never out of bounds)
 *   seq_lens    device, int32 [batch]; row b attends positions 0 .. seq_lens[b] - 1; a row with seq_lens[b] <= 0 gives zeros
 *   out         device, fp32 [batch][n_q_heads][head_dim], written
 *   stream      a cudaStream_t of the CURRENT device (NULL = the default stream); the call only enqueues
 * head_dim 64 or 128; n_q_heads a multiple of n_kv_heads, at most 16 times it.  Sizes whose partial results do not fit
 * the array even with one range per row (64 KiB + batch * n_q_heads * (head_dim + 2) * 4 bytes > CC_STATIC_SCRATCH_BYTES,
 * or batch * n_kv_heads > 16384) are rejected with CC_ERR_INVALID and a message naming the limit.  The first call on a
 * device takes the array's address (cudaGetSymbolAddress with that device current): make it outside a stream capture.
 * Every call on a device shares the array: calls that OVERLAP on the GPU race -- use one stream, or order them with
 * events.  The result does not depend on which block finishes last (ranges are merged in range order). */
#define CC_STATIC_SCRATCH_BYTES ((size_t)8 << 20)
size_t cc_static_scratch_bytes(void);
cc_status cc_attention_decode_static(const float *q, const void *k_pool, const void *v_pool, const int32_t *block_table,
                                     const int32_t *seq_lens, float *out, int batch, int n_q_heads, int n_kv_heads,
                                     int head_dim, int max_blocks, int n_pages, void *stream);

const char *cc_last_error(void);
const char *cc_version(void);

#if defined(__GNUC__)
#pragma GCC visibility pop
#endif
#ifdef __cplusplus
}
#endif
#endif /* COCOSCALE_H_ */
