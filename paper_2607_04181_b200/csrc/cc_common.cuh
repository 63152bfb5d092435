// cc_common.cuh -- device-side structures and sm_100a PTX wrappers shared by the kernels of
// libcocoscale.  (Product code; shares nothing with oracle/.)
#pragma once
#include <cuda_runtime.h>
#include <cuda_bf16.h>
#include <cuda_fp16.h>
#include <stdint.h>

#define CC_MAXR 4              // CC_MAX_REPLICAS
#define CC_PAGE 16             // tokens per KV page
#define CC_TILE_N 128          // weight rows per GEMM tile (UMMA M)
#define CC_TILE_K 64           // K elements per pipeline stage (one 128B-swizzle atom of bf16)
#define CC_A_TILE_BYTES (CC_TILE_N * CC_TILE_K * 2)   // 16 KiB packed weight tile
#define CC_ROW_ALIGN 16        // group offsets are multiples of this (UMMA N granularity)
#define CC_MAX_MPAD 320        // (256 rows + 16 * CC_MAXR group padding): upper bound of CcDims::Mpad
#define CC_FLAG_STRIDE 256     // stream-K fixup counters per projection (>= super tiles of any projection)

// GEMM operand formats (chosen per layer at cc_create_layer).  F16: the bf16 weights are converted to fp16 when they
// are packed (exact for 2^-17 <= |w| <= 65504) and the activations are ONE fp16 plane (11 significand bits).
// BF16X2: weights stay bf16, activations are two bf16 planes hi + lo (16 bits) -- twice the tensor work and slab
// traffic; the fallback for weights outside the fp16 range.  tcgen05 kind::f16 needs A and B in the SAME format.
#define CC_FMT_BF16X2 0
#define CC_FMT_F16 1

#define CC_DEVERR_BAD_REPLICA 1u
#define CC_DEVERR_BAD_PAGE 2u
#define CC_DEVERR_BAD_SEQLEN 4u
#define CC_DEVERR_HANG 8u         // an mbarrier wait gave up (kernel bug); the kernel trapped
#define CC_DEVERR_SPLIT_REQUEST 16u   // rows of one request name different replicas
#define CC_DEVERR_TOO_MANY_DECODE 32u  // a large step holds more decode rows, prompt chunks or prefill tiles than its tables
#define CC_BIG_MAX_ROWS 8192          // rows of a large step (cc_layer_desc.max_batch of a large layer)

// ---- device replica table -----------------------------------------
// One row per layer, at a fixed device address for the life of the context.  Kernels read the
// weight-blob base of replica r from here at run time, so a captured graph survives flips.
struct CcReplicaRow {
    const uint8_t* blob;   // packed weight blob of replica r (slot base), or nullptr
    void* k_pool;          // replica r's own KV partition, or nullptr = the pools passed to cc_forward;
    void* v_pool;          //   page ids in the block-table rows of r's requests are relative to it
    int n_pages;
    int pad_;
};
struct CcLayerTable {
    CcReplicaRow rep[CC_MAXR];
    uint32_t active_mask;  // bit r set <=> replica r may be named by replica_assign
    uint32_t pad_[3];
};

// Geometry of one weight-streaming GEMM (swap-AB: packed weight tiles are the UMMA A operand,
// M = 128 output features; the activations are the B operand, N = rows of one replica group).
// CC_G adjacent tiles (a "super tile" of CC_G * 128 output features) are streamed together: one
// pipeline stage holds the CC_G weight atoms of one k-block (contiguous in the blob, ONE bulk
// copy of CC_G * 16 KiB) plus the activation slab of that k-block (ONE bulk copy), so the slab
// is fetched from L2 once per CC_G atoms and the single producer thread issues two copies per
// 32 KiB of weights (measured: the copy-issue rate, not HBM, bounded the one-atom-per-stage
// version).
// The (super tile, k-block) "units" are numbered super-tile-major and cut into P contiguous
// ranges, range i owned by CTA i.  P and the cut points depend on the layer shape and the SM
// count only -- never on the batch split -- so every output element is summed in one fixed
// order whatever the replica count (PAPER.md:385 bit-wise consistency).
#define CC_G 2
struct CcGemmGeo {
    int ST;       // super tiles of CC_G * 128 output features
    int KB;       // k-blocks of 64 per tile
    int P;        // CTAs (ranges)
    int S;        // cluster size of the small-step cluster split-K kernel (k_gemm_cl), 0 = stream-K only
    int cl_tiles; // tiles of 128 output features per cluster of that kernel: 2 (a super tile) or 1
    int pad_;
    size_t w_off; // byte offset of the packed matrix inside a replica blob
};
// Range of CTA i: units [cc_range_begin(i), cc_range_begin(i+1)).
__host__ __device__ __forceinline__ long long cc_range_begin(const CcGemmGeo& g, int i) {
    return (long long)i * g.ST * g.KB / g.P;
}
// CTA whose range holds unit u (inverse of cc_range_begin).
__host__ __device__ __forceinline__ int cc_range_of_unit(const CcGemmGeo& g, long long u) {
    return (int)(((u + 1) * g.P - 1) / ((long long)g.ST * g.KB));
}
// A "piece" is the part of one 128-feature tile that one CTA accumulated.  Piece slot of
// (CTA c, super tile st, tile j of the super tile) = (c + st) * CC_G + j: unique, and increasing
// along the unit axis.  Partial sums live at part[slot][pos][128] fp32.  The pieces of tile t
// are `count` slots starting at `first`, CC_G apart, to be added in that order.
__host__ __device__ __forceinline__ void cc_tile_pieces(const CcGemmGeo& g, int t, int& first, int& count) {
    const int st = t / CC_G, j = t - st * CC_G;
    const int c0 = cc_range_of_unit(g, (long long)st * g.KB);
    const int c1 = cc_range_of_unit(g, (long long)(st + 1) * g.KB - 1);
    first = (c0 + st) * CC_G + j;
    count = c1 - c0 + 1;
}
// Byte offset of packed weight atom (tile t, k-block kb) inside its matrix.
__host__ __device__ __forceinline__ size_t cc_atom_off(int KB, int t, int kb) {
    return (((size_t)(t / CC_G) * KB + kb) * CC_G + (t % CC_G)) * (size_t)CC_A_TILE_BYTES;
}

// Static per-layer geometry, passed to kernels by value.
struct CcDims {
    int d, Hq, Hkv, Dh, G, F;
    int QD, KD;                 // Hq*Dh, Hkv*Dh
    int Mpad;                   // rows of every grouped workspace buffer (multiple of 16)
    int Mpart;                  // rows of the stream-K partial buffers (small steps only: min(Mpad, CC_MAX_MPAD))
    int fmt;                    // GEMM operand format of this layer: CC_FMT_F16 or CC_FMT_BF16X2
    int pl[4];                  // activation planes of the four GEMM operands (x, o, y, a): 1 = one plane, 2 = hi + lo; set per
                                // step by the host (cc_api.cu plane policy); BF16X2 layers always use 2
    int max_batch, max_blocks, max_position;
    float eps;
    float qk_scale_log2;        // log2(e) / sqrt(Dh)
    int pf_next, pf_self;       // small steps on the cluster GEMMs: weight stages a kernel prefetches into L2 for every CTA of the
                                // NEXT projection once its own copies are issued / of its own range while it waits for its
                                // predecessor (cc_prefetch_weights); 0 = off; set per step by the host
    CcGemmGeo qkv, o, gu, dn;   // the four projections
    size_t off_g1, off_g2;      // gains inside the blob (bf16 [d])
};

// Per-forward schedule, rebuilt on the device by k_prologue every step (row a0).
struct CcSched {
    int cnt[CC_MAXR];      // rows in replica group r
    int goff[CC_MAXR];     // first grouped position of group r (multiple of 16)
    int n_pos;             // grouped positions in use (end of the last group, multiple of 16)
    int n_items;           // KV pages of the whole batch (the attention work axis)
    int nmax;              // largest padded group size (UMMA N of the widest group)
    int pad_[5];
};

// Replica that serves row b, or -1 for a row that does not run (padding, bad seq_len); `err` collects the
// CC_DEVERR_* bits.  The ONE statement of the row-validity rules: the grouping kernel and the QKV GEMM
// (which counts the groups itself, because it starts before the grouping kernel has finished) both use it.
__device__ __forceinline__ int cc_row_replica_of(int s, int rep, const CcDims& D, uint32_t active_mask, uint32_t& err) {
    if (s <= 0) return -1;
    if (s > D.max_position || (s + CC_PAGE - 1) / CC_PAGE > D.max_blocks) {
        err |= CC_DEVERR_BAD_SEQLEN;
        return -1;
    }
    if (rep < 0 || rep >= CC_MAXR || !((active_mask >> rep) & 1u)) {
        err |= CC_DEVERR_BAD_REPLICA;
        rep = 0;
    }
    return rep;
}
__device__ __forceinline__ int cc_row_replica(const int* __restrict__ assign, const int* __restrict__ seq_lens, int b,
                                              int batch, const CcDims& D, uint32_t active_mask, uint32_t& err) {
    if (b >= batch) return -1;
    const int s = seq_lens[b];
    if (s <= 0) return -1;
    return cc_row_replica_of(s, assign[b], D, active_mask, err);
}

// Replica group that holds grouped position `pos` (groups are laid out in replica order).
__device__ __forceinline__ int replica_of_pos(const int* cnt, const int* goff, int pos) {
    int r = 0;
#pragma unroll
    for (int i = 1; i < CC_MAXR; ++i)
        if (cnt[i] > 0 && pos >= goff[i]) r = i;
    return r;
}

// ---- small helpers -----------------------------------------------------------------------
__device__ __forceinline__ float bf16lo(uint32_t w) { return __uint_as_float(w << 16); }
__device__ __forceinline__ float bf16hi(uint32_t w) { return __uint_as_float(w & 0xffff0000u); }
__device__ __forceinline__ uint32_t pack_bf16(float lo, float hi) {
    __nv_bfloat162 v = __floats2bfloat162_rn(lo, hi);   // .x = lo (low 16 bits)
    return *reinterpret_cast<uint32_t*>(&v);
}
// two floats -> fp16x2 bits (round to nearest even, clamped to the finite fp16 range so that a drifting benchmark
// input saturates instead of turning into inf - inf = NaN)
__device__ __forceinline__ uint32_t pack_f16(float lo, float hi) {
    lo = fminf(fmaxf(lo, -65504.f), 65504.f);
    hi = fminf(fmaxf(hi, -65504.f), 65504.f);
    __half2 v = __floats2half2_rn(lo, hi);   // .x = lo (low 16 bits)
    return *reinterpret_cast<uint32_t*>(&v);
}
__device__ __forceinline__ void split_hilo(float v0, float v1, uint32_t& hi, uint32_t& lo) {
    hi = pack_bf16(v0, v1);
    lo = pack_bf16(v0 - bf16lo(hi), v1 - bf16hi(hi));
}
__device__ __forceinline__ uint32_t smem_u32(const void* p) {
    return static_cast<uint32_t>(__cvta_generic_to_shared(p));
}
// Byte offset of the 16-byte chunk holding element (row, k) of plane `pl` inside a packed
// activation buffer [K/64][Mpad/8][planes][8 rows][128 B]: 8-row groups of the hi and lo planes
// alternate, so the slab of one k-block and one row group (rows goff .. goff+n, both multiples of
// 8) is ONE contiguous range holding both planes; inside an 8-row group the 128-byte rows are
// stored in the 128B-swizzle pattern (16-byte chunk c of row r at c ^ (r & 7)).  The UMMA
// descriptor of a plane uses a stride of planes * 1024 bytes between 8-row groups.
__device__ __forceinline__ size_t act_chunk_off(int row, int k, int Mpad, int planes, int pl) {
    const int kb = k >> 6, c = (k >> 3) & 7;
    return ((((size_t)kb * (Mpad >> 3) + (row >> 3)) * planes + pl) << 10) + (size_t)((row & 7) << 7) +
           (size_t)((c ^ (row & 7)) << 4);
}

// Stores N = 2, 4 or 8 consecutive operand values (k a multiple of N) of grouped row `row` in the layer's element
// format, as `planes` planes: one plane = the rounded value, two = hi + lo (lo = the rounded remainder).
enum { CC_OP_X = 0, CC_OP_O = 1, CC_OP_Y = 2, CC_OP_A = 3 };
template <int N>
__device__ __forceinline__ void act_store(uint8_t* act, const CcDims& D, int planes, int row, int k, const float (&v)[N]) {
    uint8_t* dst = act + act_chunk_off(row, k, D.Mpad, planes, 0) + (k & 7) * 2;
    uint32_t a[N / 2], b[N / 2] = {};
    if (D.fmt == CC_FMT_F16) {
#pragma unroll
        for (int i = 0; i < N / 2; ++i) {
            a[i] = pack_f16(v[2 * i], v[2 * i + 1]);
            if (planes == 2) {
                const float2 h = __half22float2(*reinterpret_cast<const __half2*>(&a[i]));
                b[i] = pack_f16(v[2 * i] - h.x, v[2 * i + 1] - h.y);
            }
        }
    } else {
#pragma unroll
        for (int i = 0; i < N / 2; ++i) split_hilo(v[2 * i], v[2 * i + 1], a[i], b[i]);
    }
    if constexpr (N == 2) {
        *reinterpret_cast<uint32_t*>(dst) = a[0];
        if (planes == 2) *reinterpret_cast<uint32_t*>(dst + 1024) = b[0];
    } else if constexpr (N == 4) {
        *reinterpret_cast<uint2*>(dst) = make_uint2(a[0], a[1]);
        if (planes == 2) *reinterpret_cast<uint2*>(dst + 1024) = make_uint2(b[0], b[1]);
    } else {
        static_assert(N == 8, "act_store: N must be 2, 4 or 8");
        *reinterpret_cast<uint4*>(dst) = make_uint4(a[0], a[1], a[2], a[3]);
        if (planes == 2) *reinterpret_cast<uint4*>(dst + 1024) = make_uint4(b[0], b[1], b[2], b[3]);
    }
}

// ---- mbarrier / bulk-copy / TMA ----------------------------------------------------------
__device__ __forceinline__ void mbar_init(uint64_t* bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(smem_u32(bar)), "r"(count));
}
__device__ __forceinline__ void fence_mbar_init() {
    asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
}
__device__ __forceinline__ void fence_proxy_async_smem() {
    asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
}
__device__ __forceinline__ void mbar_expect_tx(uint64_t* bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(smem_u32(bar)), "r"(bytes)
                 : "memory");
}
__device__ __forceinline__ void mbar_arrive(uint64_t* bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(smem_u32(bar)) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint64_t* bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(ok)
        : "r"(smem_u32(bar)), "r"(parity)
        : "memory");
    return ok != 0;
}
// Bounded wait: try_wait suspends in hardware for a while per call, so this limit is seconds of
// real time; a kernel bug then traps (CUDA error at the next sync) instead of hanging the GPU.
__device__ __forceinline__ void mbar_wait(uint64_t* bar, uint32_t parity) {
    uint32_t spins = 0;
    while (!mbar_try_wait(bar, parity)) {
        if (++spins > (1u << 26)) __trap();
    }
}
// One lane of a fully converged warp (elect.sync).  Code under `if (elect_one())` in warp-uniform
// control flow keeps its operands in uniform registers, so single-thread instructions (UBLKCP,
// UTCHMMA, UTCBAR) are issued directly; under `if (lane == 0)` the compiler wraps every one of them
// in an ELECT / R2UR.BROADCAST / BRA.U.ANY waterfall loop (~100 cycles per tcgen05.mma, measured).
__device__ __forceinline__ bool elect_one() {
    uint32_t pred;
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "elect.sync _|p, 0xffffffff;\n\t"
        "selp.u32 %0, 1, 0, p;\n\t}"
        : "=r"(pred));
    return pred != 0;
}
// Tell the compiler a value is warp-uniform (broadcast from lane 0).
__device__ __forceinline__ int uniform(int v) { return __shfl_sync(0xffffffffu, v, 0); }
__device__ __forceinline__ uint32_t uniform(uint32_t v) { return __shfl_sync(0xffffffffu, v, 0); }
__device__ __forceinline__ const uint8_t* uniform(const uint8_t* p) {
    return reinterpret_cast<const uint8_t*>(__shfl_sync(0xffffffffu, reinterpret_cast<unsigned long long>(p), 0));
}
// Programmatic dependent launch: wait for the preceding kernel's memory / let the next one start.
__device__ __forceinline__ void pdl_wait() { asm volatile("griddepcontrol.wait;" ::: "memory"); }
__device__ __forceinline__ void pdl_launch_dependents() { asm volatile("griddepcontrol.launch_dependents;" ::: "memory"); }
// cp.async (LDGSTS) 16 bytes, L2 only.
__device__ __forceinline__ void cp_async16(uint32_t dst_smem, const void* src) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst_smem), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }
// 1-D bulk copy global -> shared (TMA engine, no descriptor); completes `bytes` on the mbarrier.
__device__ __forceinline__ void bulk_g2s(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(
                     smem_u32(dst_smem)),
                 "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar))
                 : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(void* dst_smem, const void* src_gmem, uint32_t bytes, uint64_t* bar,
                                              uint64_t policy) {
    asm volatile(
        "cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::
            "r"(smem_u32(dst_smem)),
        "l"(src_gmem), "r"(bytes), "r"(smem_u32(bar)), "l"(policy)
        : "memory");
}
// 2-D tensor-map TMA load (box of the map's shape at element coordinates (c0, c1)) -> shared memory;
// completes the box's bytes on the mbarrier.  `tmap` must live in kernel parameter / constant space.
__device__ __forceinline__ void tma_load_2d(uint32_t dst_smem, const void* tmap, int c0, int c1, uint32_t bar_smem) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3}], [%4];" ::"r"(dst_smem),
        "l"(tmap), "r"(c0), "r"(c1), "r"(bar_smem)
        : "memory");
}
__device__ __forceinline__ void tma_load_2d_hint(uint32_t dst_smem, const void* tmap, int c0, int c1, uint32_t bar_smem,
                                                 uint64_t policy) {
    asm volatile(
        "cp.async.bulk.tensor.2d.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1, {%2, %3}], [%4], %5;" ::
            "r"(dst_smem),
        "l"(tmap), "r"(c0), "r"(c1), "r"(bar_smem), "l"(policy)
        : "memory");
}
// L2 prefetch of a contiguous global range (16-byte granules): no shared memory, no barrier, fire and forget.
__device__ __forceinline__ void bulk_prefetch_l2(const void* src_gmem, uint32_t bytes) {
    asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(src_gmem), "r"(bytes) : "memory");
}
// CTA c' = (cluster unit, rank) of the small-step cluster GEMM with geometry N (k_gemm_cl) copies, for every replica that has
// rows, the weight stages of k-blocks [rank KB / S, (rank + 1) KB / S) of its (super) tile, in that order.  This prefetches
// stages [skip, skip + n) of that sequence into L2 for the CTAs c' = c, c + step, ... of N.  Called by one whole warp: the
// kernel BEFORE N calls it once its own copies are issued (its exchange and epilogue would leave HBM idle otherwise, and
// N's CTAs cannot start on an SM whose shared memory the predecessor still holds), N itself while it waits for that kernel.
__device__ __forceinline__ void cc_prefetch_weights(const CcGemmGeo& N, const uint8_t* const* blob, const int* cnt, int c,
                                                    int step, int skip, int n, int lane) {
    if (N.S <= 0 || n <= 0) return;
    const int n_cta = N.ST * CC_G / N.cl_tiles * N.S;
    const uint32_t wbytes = (uint32_t)N.cl_tiles * CC_A_TILE_BYTES;
    const size_t wstage = (size_t)CC_G * CC_A_TILE_BYTES;
    for (int cc = c; cc < n_cta; cc += step) {
        const int unit = cc / N.S, rank = cc % N.S;
        const int st = N.cl_tiles == 2 ? unit : unit / CC_G;
        const int kb0 = (int)((long long)rank * N.KB / N.S), len = (int)((long long)(rank + 1) * N.KB / N.S) - kb0;
        const size_t off = N.w_off + ((size_t)st * N.KB + kb0) * wstage + (N.cl_tiles == 2 ? 0 : (size_t)(unit % CC_G) * CC_A_TILE_BYTES);
        for (int i = skip + lane; i < skip + n; i += 32) {
            int ri = i / len;
            const int kb = i - ri * len;
            int r = 0;
            for (; r < CC_MAXR; ++r)
                if (cnt[r] > 0 && ri-- == 0) break;                // the ri-th replica that has rows
            if (r < CC_MAXR) bulk_prefetch_l2(blob[r] + off + (size_t)kb * wstage, wbytes);
        }
    }
}
__device__ __forceinline__ uint64_t policy_evict_first() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(p));
    return p;
}
__device__ __forceinline__ uint64_t policy_evict_last() {
    uint64_t p;
    asm volatile("createpolicy.fractional.L2::evict_last.b64 %0, 1.0;" : "=l"(p));
    return p;
}
// ---- tcgen05 / TMEM --------------------------------------------------------------------------
template <int kCols>
__device__ __forceinline__ void tmem_alloc(uint32_t* dst_smem) {   // one full warp
    asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst_smem)),
                 "n"(kCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
}
template <int kCols>
__device__ __forceinline__ void tmem_dealloc(uint32_t taddr) {     // the same warp
    asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(kCols) : "memory");
}
__device__ __forceinline__ void tc_fence_before() { asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory"); }
__device__ __forceinline__ void tc_fence_after() { asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory"); }
// D[tmem] (+)= A[smem desc] * B[smem desc]; bf16 x bf16 -> fp32; issued by ONE thread.
__device__ __forceinline__ void umma_bf16(uint32_t d_tmem, uint64_t a_desc, uint64_t b_desc, uint32_t idesc,
                                          uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t"
        "setp.ne.b32 p, %4, 0;\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], %1, %2, %3, p;\n\t}" ::"r"(d_tmem),
        "l"(a_desc), "l"(b_desc), "r"(idesc), "r"(accumulate)
        : "memory");
}
// Same, with the two descriptors given as 32-bit low words plus their (loop-invariant) high words:
// all the fields that change from MMA to MMA -- the start address -- live in the low word.
__device__ __forceinline__ void umma_bf16_lo(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t a_hi, uint32_t b_hi,
                                             uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .b64 da, db;\n\t"
        "setp.ne.b32 p, %6, 0;\n\t"
        "mov.b64 da, {%1, %3};\n\t"
        "mov.b64 db, {%2, %4};\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], da, db, %5, p;\n\t}" ::"r"(d_tmem),
        "r"(a_lo), "r"(b_lo), "r"(a_hi), "r"(b_hi), "r"(idesc), "r"(accumulate)
        : "memory");
}
// mbarrier arrive once all previously issued tcgen05.mma of this thread have completed.
__device__ __forceinline__ void umma_commit(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::1.mbarrier::arrive::one.shared::cluster.b64 [%0];" ::"r"(smem_u32(bar))
                 : "memory");
}
// TMEM -> registers: this warp's 32 lanes x 16 consecutive fp32 columns.
__device__ __forceinline__ void tmem_ld_32x32b_x16(uint32_t taddr, uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x16.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15}, [%16];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15])
        : "r"(taddr)
        : "memory");
}
__device__ __forceinline__ void tmem_ld_wait() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }

// Shared-memory matrix descriptor: K-major operand, 128B swizzle, rows of 128 bytes, 8-row
// groups 1024 bytes apart (SBO), descriptor version 1 (sm_100).  Tile base must be 1024-aligned;
// advancing K by 16 bf16 inside the swizzle atom adds 32 bytes to the start address.
__device__ __forceinline__ uint64_t umma_desc_sw128(uint32_t smem_addr, uint32_t sbo_bytes = 1024) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);   // start address  [0,14)
    d |= (uint64_t)1 << 16;                          // LBO (unused for swizzled K-major) [16,30)
    d |= (uint64_t)(sbo_bytes >> 4) << 32;           // SBO: bytes between 8-row groups [32,46)
    d |= (uint64_t)1 << 46;                          // version = 1    [46,48)
    d |= (uint64_t)2 << 61;                          // SWIZZLE_128B   [61,64)
    return d;
}
// Instruction descriptor, kind::f16: D = fp32 (bits 4-5 = 1), A format at bits 7-9 and B format at bits 10-12
// (0 = fp16, 1 = bf16), both K-major, N >> 3 at bit 17, M >> 4 at bit 24.  A and B must have the SAME format:
// bf16 x fp16 raises an illegal-instruction fault on sm_100a (measured in round 1 and again in round 2 with a
// one-MMA probe, either operand order), although the descriptor has separate fields.
__device__ __forceinline__ uint32_t umma_idesc_m128(uint32_t n, int fmt) {
    const uint32_t ab = fmt == CC_FMT_F16 ? 0u : 1u;
    return (1u << 4) | (ab << 7) | (ab << 10) | ((n >> 3) << 17) | ((128u >> 4) << 24);
}

// ---- thread-block clusters / CTA pairs (cta_group::2) -------------------------------------------------
__device__ __forceinline__ uint32_t cluster_ctarank() {
    uint32_t r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ void cluster_sync_all() {
    asm volatile("barrier.cluster.arrive.release.aligned;" ::: "memory");
    asm volatile("barrier.cluster.wait.acquire.aligned;" ::: "memory");
}
// shared::cluster address of `local_smem_addr` in CTA `cta` of the cluster
__device__ __forceinline__ uint32_t mapa_u32(uint32_t local_smem_addr, uint32_t cta) {
    uint32_t r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(local_smem_addr), "r"(cta));
    return r;
}
// (default semantics: release at CTA scope.  With .release.cluster the compiler emits MEMBAR.ALL.GPU in front of every
// arrive -- measured: ~1300 cycles per k-block in the relay warp of the large-M GEMM, the kernel's whole bound.  What
// the arrivals order here was written by the async proxy (TMA) or read through TMEM, not by this thread's stores.)
__device__ __forceinline__ void mbar_arrive_cluster(uint32_t cluster_addr) {
    asm volatile("mbarrier.arrive.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
template <int kCols>
__device__ __forceinline__ void tmem_alloc_pair(uint32_t* dst_smem) {   // one full warp in EACH CTA of the pair
    asm volatile("tcgen05.alloc.cta_group::2.sync.aligned.shared::cta.b32 [%0], %1;" ::"r"(smem_u32(dst_smem)), "n"(kCols)
                 : "memory");
    asm volatile("tcgen05.relinquish_alloc_permit.cta_group::2.sync.aligned;" ::: "memory");
}
template <int kCols>
__device__ __forceinline__ void tmem_dealloc_pair(uint32_t taddr) {
    asm volatile("tcgen05.dealloc.cta_group::2.sync.aligned.b32 %0, %1;" ::"r"(taddr), "n"(kCols) : "memory");
}
// D[tmem of both CTAs] (+)= A * B over the CTA pair: M = 256 (128 rows of A from each CTA), N = n (n / 2 rows of B
// from each CTA); issued by ONE thread of the leader CTA (rank 0); descriptors are smem offsets valid in both CTAs.
__device__ __forceinline__ void umma_pair_lo(uint32_t d_tmem, uint32_t a_lo, uint32_t b_lo, uint32_t a_hi, uint32_t b_hi,
                                             uint32_t idesc, uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .b64 da, db;\n\t"
        "setp.ne.b32 p, %6, 0;\n\t"
        "mov.b64 da, {%1, %3};\n\t"
        "mov.b64 db, {%2, %4};\n\t"
        "tcgen05.mma.cta_group::2.kind::f16 [%0], da, db, %5, p;\n\t}" ::"r"(d_tmem),
        "r"(a_lo), "r"(b_lo), "r"(a_hi), "r"(b_hi), "r"(idesc), "r"(accumulate)
        : "memory");
}
// mbarrier arrive in BOTH CTAs of the pair (same smem offset) once all previously issued MMAs have completed
__device__ __forceinline__ void umma_commit_pair(uint64_t* bar) {
    asm volatile("tcgen05.commit.cta_group::2.mbarrier::arrive::one.shared::cluster.multicast::cluster.b64 [%0], %1;" ::"r"(
                     smem_u32(bar)),
                 "h"((uint16_t)3)
                 : "memory");
}
__device__ __forceinline__ uint32_t umma_idesc_pair_m256(uint32_t n, int fmt) {
    const uint32_t ab = fmt == CC_FMT_F16 ? 0u : 1u;
    return (1u << 4) | (ab << 7) | (ab << 10) | ((n >> 3) << 17) | ((256u >> 4) << 24);
}
// TMEM -> registers: this warp's 32 lanes x 32 consecutive fp32 columns.
__device__ __forceinline__ void tmem_ld_32x32b_x32(uint32_t taddr, uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.ld.sync.aligned.32x32b.x32.b32 "
        "{%0, %1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, "
        "%16, %17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31}, [%32];"
        : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]), "=r"(r[8]),
          "=r"(r[9]), "=r"(r[10]), "=r"(r[11]), "=r"(r[12]), "=r"(r[13]), "=r"(r[14]), "=r"(r[15]), "=r"(r[16]),
          "=r"(r[17]), "=r"(r[18]), "=r"(r[19]), "=r"(r[20]), "=r"(r[21]), "=r"(r[22]), "=r"(r[23]), "=r"(r[24]),
          "=r"(r[25]), "=r"(r[26]), "=r"(r[27]), "=r"(r[28]), "=r"(r[29]), "=r"(r[30]), "=r"(r[31])
        : "r"(taddr)
        : "memory");
}

// ---- legacy tensor path used by decode attention (HBM-bound, tiny M): mma.sync + ldmatrix ----
__device__ __forceinline__ void ldsm_x4(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr));
}
__device__ __forceinline__ void ldsm_x4_trans(uint32_t addr, uint32_t& r0, uint32_t& r1, uint32_t& r2, uint32_t& r3) {
    asm volatile("ldmatrix.sync.aligned.m8n8.x4.trans.shared.b16 {%0,%1,%2,%3}, [%4];"
                 : "=r"(r0), "=r"(r1), "=r"(r2), "=r"(r3)
                 : "r"(addr));
}
// D(16x8, fp32) += A(16x16, bf16, row) * B(16x8, bf16, col)
__device__ __forceinline__ void mma_bf16_16816(float (&c)[4], uint32_t a0, uint32_t a1, uint32_t a2, uint32_t a3,
                                               uint32_t b0, uint32_t b1) {
    asm volatile(
        "mma.sync.aligned.m16n8k16.row.col.f32.bf16.bf16.f32 {%0,%1,%2,%3}, {%4,%5,%6,%7}, {%8,%9}, {%0,%1,%2,%3};"
        : "+f"(c[0]), "+f"(c[1]), "+f"(c[2]), "+f"(c[3])
        : "r"(a0), "r"(a1), "r"(a2), "r"(a3), "r"(b0), "r"(b1));
}
__device__ __forceinline__ void named_bar_sync(int id, int nthreads) {
    asm volatile("bar.sync %0, %1;" ::"r"(id), "r"(nthreads) : "memory");
}
