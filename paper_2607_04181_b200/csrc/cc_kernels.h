// cc_kernels.h -- host-callable launchers of the sm_100a kernels (product code).
#pragma once
#include "cc_common.cuh"

// Device workspace of one layer (allocated once at cc_create_layer; PAPER.md:393 persistent pool).
struct CcWork {
    CcSched* sched;
    int* perm;           // [Mpad] original row at grouped position, or -1
    int* pg_prefix;      // [max_batch + 1] pages of the rows before row b, request order (attention work split)
    int* pos_of;         // [max_batch] grouped position of row b, or -1
    int* first_wr;       // [max_batch] lowest page index of row b's request that some row of this step appends to
    uint8_t* x_act;      // packed bf16 GEMM operands, [K/64][Mpad/8][plane hi|lo][8][128 B swizzled]
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
    int* flags;          // [4][CC_FLAG_STRIDE] stream-K fixup counters, zeroed by k_prologue every step
    int* attn_cnt;       // [Mpad][Hkv] pieces finished per (row, kv head); the last finisher merges and resets
    float* att_o;        // [max_batch + SMs][Hq][Dh] fp32 un-normalised piece outputs (slot = row + CTA)
    float2* att_ml;      // [max_batch + SMs][Hq] (max in log2 units, sum)
    const float2* rope_cs;  // [max_position][Dh/2] (cos, sin), built in fp64 on the host
    uint32_t* err;       // sticky device error word (context-owned)
    unsigned long long* trace;   // CC_TRACE builds: [CC_TRACE_KERNELS][CC_TRACE_POINTS][min, max] of %globaltimer; else null
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
    __nv_bfloat16* k_pool;
    __nv_bfloat16* v_pool;
    const int* block_table;
    int n_pages;
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
cudaError_t cc_launch_attention(const int* seq_lens, const CcKv& kv, const CcDims& D, const CcLayerTable* tab,
                                const CcWork& W, const CcLaunch& L);

cudaError_t cc_launch_copy(void* dst, const void* src, size_t bytes, int n_sms, cudaStream_t st);
cudaError_t cc_launch_page_copy(void* k_pool, void* v_pool, size_t page_bytes, const int* src, const int* dst, int n_moves,
                                cudaStream_t st);
cudaError_t cc_launch_publish(CcLayerTable* row_dev, const CcLayerTable& value, cudaStream_t st);
// mode 0: rows of src0, then src1, then src2 (concatenated); mode 1: rows alternate src0[j], src1[j].
cudaError_t cc_launch_pack(uint8_t* dst, const __nv_bfloat16* src0, const __nv_bfloat16* src1,
                           const __nv_bfloat16* src2, int rows0, int rows1, int rows2, int mode, int K, int n_tiles,
                           int k_blocks, cudaStream_t st);
// which: 0 = one packed bf16 plane (K = dim), 1 = fp32 row buffer [Mpad][dim], 2 = hi + lo planes,
// 3 = hi + lo planes scaled by the row's 1/rms from W.ssq (the un-normalised y' operand)
cudaError_t cc_launch_tap(const void* src, int which, int dim, const CcDims& D, const CcWork& W,
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
