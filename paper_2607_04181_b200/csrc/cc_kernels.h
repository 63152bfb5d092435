// cc_kernels.h -- host-callable launchers of the sm_100a kernels (product code).
#pragma once
#include "cc_common.cuh"

struct CcBigSched;
// Device workspace of one layer (allocated once at cc_create_layer; PAPER.md:393 persistent pool).
struct CcWork {
    CcSched* sched;
    int* perm;           // [Mpad] original row at grouped position, or -1
    int* pg_prefix;      // [max_batch + 1] pages of the rows before row b, request order (attention work split)
    int* pos_of;         // [max_batch] grouped position of row b, or -1
    int* first_wr;       // [max_batch] lowest page index of row b's request that some row of this step appends to
    uint8_t* x_act;      // packed GEMM operands, [K/64][Mpad/8][planes][8][128 B swizzled]: one fp16 plane or bf16 hi|lo
    uint8_t* o_act;
    uint8_t* y_act;
    uint8_t* a_act;
    float* qkv_part;     // stream-K partial sums, [(P + ST) * CC_G][Mpad][128] fp32 (piece-major)
    float* o_part;
    float* gu_part;
    float* d_part;
    float* q_rot;        // [Mpad][Hq*Dh] fp32, q after RoPE
    float* h1;           // [Mpad][d]     fp32, hidden + O projection
    float* ssq;          // [d/128][Mpad] fp32, per-tile sum of squares of h1 (post-attention RMSNorm statistic)
    float* inv_in;       // [Mpad] 1/rms of the input row (k_prologue): the O epilogue stores y' = h1 * g2 * inv_in so that the
                         // operand stays O(1) whatever the scale of `hidden` (fp16 range); the gate/up epilogue divides it out
    int* flags;          // [4][CC_FLAG_STRIDE] stream-K fixup counters, zeroed by k_prologue every step
    int* attn_cnt;       // [Mpad][Hkv] pieces finished per (row, kv head); the last finisher merges and resets
    float* att_o;        // [max_batch + SMs][Hq][Dh] fp32 un-normalised piece outputs (slot = row + CTA)
    float2* att_ml;      // [max_batch + SMs][Hq] (max in log2 units, sum)
    // ---- large-M path (layers created with max_batch > 256; steps of more than 256 rows: DESIGN.md "Mixed steps") ----
    CcBigSched* bs;      // counts of the step: decode rows, prompt chunks, prefill work items, the work counter
    int* row_pos;        // [Mpad] position s-1 of grouped row p, or -1
    int* row_page;       // [Mpad] page that holds that position, or -1
    float* gu_scale;     // [Mpad] rms of the input row over rms of h1 (the gate/up epilogue's row scale)
    int* dec_rows;       // [CC_BIG_MAX_DEC] original row of decode row i (a row outside every prompt chunk)
    int* chunk_row0;     // [CC_BIG_MAX_CHUNKS] first original row of prompt chunk c (its rows are consecutive)
    int* chunk_len;      // [CC_BIG_MAX_CHUNKS] rows (tokens) of chunk c
    int* item_chunk;     // [CC_BIG_MAX_ITEMS] prefill work item -> chunk
    int* item_tile;      // [CC_BIG_MAX_ITEMS] prefill work item -> query tile of that chunk
    const float2* rope_cs;  // [max_position][Dh/2] (cos, sin), built in fp64 on the host
    uint32_t* err;       // sticky device error word (context-owned)
    unsigned long long* trace;   // CC_TRACE builds: [CC_TRACE_KERNELS][CC_TRACE_POINTS][min, max] of %globaltimer; else null
};

#define CC_BIG_MAX_DEC 256       // decode rows of a large step (they go through k_attn's page-range split)
#define CC_BIG_MAX_CHUNKS 64     // prompt chunks of a large step
#define CC_BIG_MAX_ITEMS 1024    // (chunk, query tile) items of a large step
struct CcBigSched {
    int n_dec, n_chunks, n_items, work;
    int n_dec_pages;             // KV pages of the decode rows (the attention work axis of the large step)
    int pad_[3];
};

// ---- tracing build (python -m paper_2607_04181_b200.build --trace; read with cc_debug_trace / timeline.py) ----
// A CC_TRACE build records, per kernel and trace point, the earliest and the latest %globaltimer value over the
// CTAs that pass it (one thread per CTA); the product build compiles the points away.
#define CC_TRACE_KERNELS 16
#define CC_TRACE_POINTS 8
#if defined(CC_TRACE) && defined(__CUDACC__)
__device__ __forceinline__ unsigned long long cc_gtime() {
    unsigned long long t;
    asm volatile("mov.u64 %0, %%globaltimer;" : "=l"(t)::"memory");
    return t;
}
__device__ __forceinline__ void cc_trace_minmax(unsigned long long* tr, int k, int pt, unsigned long long v) {
    if (tr == nullptr) return;
    atomicMin(tr + ((size_t)k * CC_TRACE_POINTS + pt) * 2, v);
    atomicMax(tr + ((size_t)k * CC_TRACE_POINTS + pt) * 2 + 1, v);
}
#define CC_TP(W, k, pt) cc_trace_minmax((W).trace, (k), (pt), cc_gtime())
#else
#define CC_TP(W, k, pt) ((void)0)
#endif
// kernel ids of the trace: 0 prologue, 1 attention, 2..5 the four GEMMs (2 + KIND); 8 + KIND: duration of the
// first ([0]) and second ([1]) stream-K fixup pass of a CTA, 12 + KIND: [0][max] passes counted / [2][max] their sum

struct CcKv {
    __nv_bfloat16* k_pool;        // the pools passed to cc_forward: every replica without a partition of its own
    __nv_bfloat16* v_pool;
    const int* block_table;
    int n_pages;
    // resolved on the host per forward: the pools replica r's rows live in (its partition, else the pools above); the
    // attention launchers build one TMA descriptor pair per replica from them, the kernels bound page ids by n_pages_r
    const void* k_pool_r[CC_MAXR];
    const void* v_pool_r[CC_MAXR];
    int n_pages_r[CC_MAXR];
};


// Launch options shared by the forward chain.
struct CcLaunch {
    cudaStream_t st;
    int n_sms;
    bool pdl;            // programmatic dependent launch between the kernels of the chain
};


// cc_forward_host with a pinned hidden buffer: the prologue reads the rows straight from mapped host memory and
// leaves a device copy for the O epilogue's residual (null: hidden is device memory, nothing staged).
struct CcStageOut {
    __nv_bfloat16* hidden = nullptr;   // [batch][d]
};

cudaError_t cc_launch_prologue(const int* assign, const int* seq_lens, const int* block_table, int batch,
                               const __nv_bfloat16* hidden, const CcDims& D, const CcLayerTable* tab, const CcWork& W,
                               const CcLaunch& L, const CcStageOut& so = CcStageOut());
// which: 0 = QKV, 1 = O, 2 = gate/up, 3 = down
cudaError_t cc_launch_gemm(int which, const CcDims& D, const CcLayerTable* tab, const CcWork& W, const int* seq_lens,
                           const int* assign, int batch, const CcKv& kv, __nv_bfloat16* hidden, const CcLaunch& L);
// rowmap (large steps): original row of entry i of the attention work axis (the decode rows); null = row i itself
// small steps (at most cc_gemm_cl_max_rows() grouped rows) of QKV / O / down as a cluster split-K (cc_gemm.cu: k_gemm_cl)
cudaError_t cc_launch_gemm_cl(int which, const CcDims& D, const CcLayerTable* tab, const CcWork& W, const int* seq_lens,
                              const int* assign, int batch, const CcKv& kv, __nv_bfloat16* hidden, const CcLaunch& L);
void cc_gemm_cl_geometry(int which, CcGemmGeo& g, int n_sms);   // sets g.S and g.cl_tiles
int cc_gemm_cl_max_rows();
cudaError_t cc_launch_attention(const int* seq_lens, const CcKv& kv, const CcDims& D, const CcLayerTable* tab,
                                const CcWork& W, const CcLaunch& L, const int* rowmap = nullptr);
// ---- large steps (cc_big.cu, cc_big_gemm.cu, cc_prefill.cu) ----
cudaError_t cc_launch_big_group(const int* assign, const int* seq_lens, const int* block_table, int batch, const CcDims& D,
                                const CcLayerTable* tab, const CcWork& W, cudaStream_t st);
cudaError_t cc_launch_big_norm(const __nv_bfloat16* hidden, int batch, const CcDims& D, const CcLayerTable* tab, const CcWork& W,
                               cudaStream_t st);
cudaError_t cc_launch_big_rowstat(const CcDims& D, const CcWork& W, cudaStream_t st);
cudaError_t cc_launch_big_gemm(int which, const CcDims& D, const CcLayerTable* tab, const CcWork& W, const int* seq_lens,
                               const int* assign, int batch, const CcKv& kv, __nv_bfloat16* hidden, const CcLaunch& L);
cudaError_t cc_launch_prefill_attention(const int* seq_lens, const CcKv& kv, const CcDims& D, const CcWork& W, const CcLaunch& L);

cudaError_t cc_launch_copy(void* dst, const void* src, size_t bytes, int n_sms, cudaStream_t st);
cudaError_t cc_launch_page_copy(void* k_pool, void* v_pool, size_t page_bytes, const int* src, const int* dst, int n_moves,
                                cudaStream_t st);
cudaError_t cc_launch_publish(CcLayerTable* row_dev, const CcLayerTable& value, cudaStream_t st);
// mode 0: rows of src0, then src1, then src2 (concatenated); mode 1: rows alternate src0[j], src1[j].
// fmt = CC_FMT_F16 converts the bf16 weights to fp16; *overflow_dev is set when a weight does not fit (|w| > 65504 or not finite).
cudaError_t cc_launch_pack(uint8_t* dst, const __nv_bfloat16* src0, const __nv_bfloat16* src1,
                           const __nv_bfloat16* src2, int rows0, int rows1, int rows2, int mode, int K, int n_tiles,
                           int k_blocks, int fmt, uint32_t* overflow_dev, cudaStream_t st);
// which: 1 = fp32 row buffer [Mpad][dim], 2 = packed operand in the layer's format,
// 3 = packed operand times the row's 1/rms from W.ssq over W.inv_in (the y' operand is stored before its statistic is known)
cudaError_t cc_launch_tap(const void* src, int which, int planes, int dim, const CcDims& D, const CcWork& W,
                          float* out_dev, int batch, cudaStream_t st);
int cc_max_hidden();

// Generic launcher: plain <<<>>> semantics, plus the PDL attribute when asked for.
template <typename... KArgs, typename... Args>
static inline cudaError_t cc_launch_kernel(void (*kern)(KArgs...), dim3 grid, dim3 block, size_t smem,
                                           const CcLaunch& L, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = grid;
    cfg.blockDim = block;
    cfg.dynamicSmemBytes = smem;
    cfg.stream = L.st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[0].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = L.pdl ? 1 : 0;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}
