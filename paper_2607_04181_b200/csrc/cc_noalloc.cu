// cc_noalloc.cu -- cc_attention_decode_static: paged GQA decode attention (PAPER.md:103, 391, 476:
// softmax(q K^T / sqrt(Dh)) V over the cached positions t < seq_len of each row, through its block-table row) as ONE
// stand-alone entry point that ALLOCATES NOTHING: no cc_ctx, no layer, no cudaMalloc / cudaFree / allocating library
// call -- for callers that cannot allocate (a harness that forbids it, a tight serving loop, code around a capture).
//
// The layer's own attention kernel (cc_attention.cu) keeps its split-KV partial results in the layer workspace that
// cc_create_layer allocates.  This variant keeps them in a file-scope device array of a fixed, modest size instead
// (CC_STATIC_SCRATCH_BYTES = 8 MiB; every GPU that loads the library holds it until the process exits).  It is a plain
// split-KV kernel -- no TMA, no tensor-map descriptor (building one is a driver call per forward): the hot path stays
// cc_forward; this one trades speed for having no state at all.
//
// In HOST code the array's name is a host-side stand-in, not a device address.  The address is taken once per device,
// with that device current, by cudaGetSymbolAddress, and passed to the kernel as an ordinary pointer.
//
// Every call (of every thread, on every stream of a device) shares the one array: calls that overlap on the GPU RACE --
// enqueue them on one stream, or order them with events.  The array keeps the last call's contents; the only part that
// must start at zero, the arrival counters, is cleared by a cudaMemsetAsync in front of every launch.
#include <cuda_runtime.h>

#include <cmath>
#include <cstdarg>
#include <cstdint>
#include <cstdio>
#include <mutex>

#include "../../include/cocoscale.h"
#include "cc_common.cuh"

void cc_internal_set_error(const char* msg);   // cc_api.cu: what cc_last_error() returns on this thread

constexpr size_t kScratchBytes = CC_STATIC_SCRATCH_BYTES;

// The scratch memory of this file's kernel.  Device code may name it directly; host code must not pass this name to a kernel
// (see above) -- scratch_address() below is the one place that turns it into a device pointer.
static __device__ __align__(256) unsigned char g_static_scratch[kScratchBytes];

namespace {

constexpr int kMaxSplit = 8;                   // a row's positions are cut into at most 8 ranges
constexpr int kChunk = 128;                    // positions per pass of a block = its threads
constexpr int kMaxG = 16;                      // query heads per kv head
constexpr int kCounterBytes = 64 * 1024;       // front of the array: one arrival counter per (row, kv head)

__device__ __forceinline__ float bf16_bits_to_float(uint32_t b) { return __uint_as_float(b << 16); }

// One block per (range sp of the row's positions, kv head h, row b), kChunk threads.  Pass over a chunk of kChunk positions:
// thread i scores position i against the G query heads of the kv head (q in shared memory), the block agrees on the new
// running maxima, the probabilities go to shared memory, then thread d (head dimension d; with DH = 64 the two halves of the
// block take alternate query heads) adds sum_t p[g][t] V[t][d] for its heads.  The range's (m, l, o) go to the scratch
// array; the block that arrives last at the (row, kv head) counter merges the ranges IN RANGE ORDER and writes the result,
// so the output does not depend on which block that is.
template <int DH>
__global__ void __launch_bounds__(kChunk) k_attn_static(const float* __restrict__ q, const uint16_t* __restrict__ kp,
                                                        const uint16_t* __restrict__ vp, const int* __restrict__ block_table,
                                                        const int* __restrict__ seq_lens, float* __restrict__ out, int Hq, int Hkv,
                                                        int max_blocks, int n_pages, int n_split, float scale_log2,
                                                        unsigned char* scratch) {
    constexpr int NPART = kChunk / DH;                                 // 1 (DH = 128) or 2 (DH = 64)
    const int sp = blockIdx.x, h = blockIdx.y, b = blockIdx.z, G = Hq / Hkv, batch = gridDim.z;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const int d = tid % DH, part = tid / DH;
    __shared__ float s_q[kMaxG * DH];
    __shared__ float s_p[kMaxG][kChunk];
    __shared__ float s_red[kMaxG][kChunk / 32];
    __shared__ int s_page[kChunk];
    __shared__ int s_last;
    int* counters = reinterpret_cast<int*>(scratch);
    float* part_ml = reinterpret_cast<float*>(scratch + kCounterBytes);                  // [row][q head][range][2]
    float* part_o = part_ml + (size_t)batch * Hq * n_split * 2;                          // [row][q head][range][DH]
    const int s = seq_lens[b];
    if (s <= 0) {                                                      // a row that does not run: zeros (block-uniform)
        if (sp == 0)
            for (int i = tid; i < G * DH; i += kChunk) out[((size_t)b * Hq + (size_t)h * G) * DH + i] = 0.f;
        return;
    }
    const int len = (((s + n_split - 1) / n_split) + CC_PAGE - 1) / CC_PAGE * CC_PAGE;   // whole pages per range
    const int t0 = sp * len, t1 = min(s, t0 + len);
    for (int i = tid; i < G * DH; i += kChunk) s_q[i] = q[((size_t)b * Hq + (size_t)h * G) * DH + i] * scale_log2;
    float m_run[kMaxG], acc[kMaxG], l_run[kMaxG];
#pragma unroll
    for (int g = 0; g < kMaxG; ++g) {
        m_run[g] = -INFINITY;
        acc[g] = 0.f;
        l_run[g] = 0.f;
    }
    __syncthreads();
    for (int c0 = t0; c0 < t1; c0 += kChunk) {
        const int t = c0 + tid;
        const bool valid = t < t1;
        float sc[kMaxG];
#pragma unroll
        for (int g = 0; g < kMaxG; ++g) sc[g] = 0.f;
        int page = 0;
        if (valid) {
            page = block_table[(size_t)b * max_blocks + t / CC_PAGE];
            if (page < 0 || page >= n_pages) page = 0;                 // documented precondition; never read out of bounds
            const uint4* krow = reinterpret_cast<const uint4*>(kp + (((size_t)page * Hkv + h) * CC_PAGE + t % CC_PAGE) * DH);
#pragma unroll 4
            for (int j = 0; j < DH / 8; ++j) {
                const uint4 kv = krow[j];
                const uint32_t w[4] = {kv.x, kv.y, kv.z, kv.w};
                float kf[8];
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    kf[2 * i] = bf16_bits_to_float(w[i] & 0xffffu);
                    kf[2 * i + 1] = bf16_bits_to_float(w[i] >> 16);
                }
#pragma unroll
                for (int g = 0; g < kMaxG; ++g)
                    if (g < G) {
                        const float* qg = s_q + g * DH + 8 * j;
#pragma unroll
                        for (int i = 0; i < 8; ++i) sc[g] = fmaf(qg[i], kf[i], sc[g]);
                    }
            }
        }
        s_page[tid] = page;
#pragma unroll
        for (int g = 0; g < kMaxG; ++g)
            if (g < G) {
                if (!valid) sc[g] = -INFINITY;
                float mx = sc[g];
#pragma unroll
                for (int o = 16; o > 0; o >>= 1) mx = fmaxf(mx, __shfl_xor_sync(0xffffffffu, mx, o));
                if (lane == 0) s_red[g][warp] = mx;
            }
        __syncthreads();
        float alpha[kMaxG];
#pragma unroll
        for (int g = 0; g < kMaxG; ++g)
            if (g < G) {
                float mx = s_red[g][0];
#pragma unroll
                for (int w = 1; w < kChunk / 32; ++w) mx = fmaxf(mx, s_red[g][w]);
                const float m_new = fmaxf(m_run[g], mx);               // finite: the chunk holds at least one position
                alpha[g] = exp2f(m_run[g] - m_new);                    // first chunk: exp2(-inf) = 0
                m_run[g] = m_new;
                s_p[g][tid] = exp2f(sc[g] - m_new);                    // 0 for a position past the range
            }
        __syncthreads();
        const int n_here = min(kChunk, t1 - c0);
#pragma unroll
        for (int g = 0; g < kMaxG; ++g)
            if (g < G && g % NPART == part) {
                acc[g] *= alpha[g];
                l_run[g] *= alpha[g];
            }
        for (int tt = 0; tt < n_here; ++tt) {
            const int tpos = c0 + tt;
            const float v = bf16_bits_to_float(vp[(((size_t)s_page[tt] * Hkv + h) * CC_PAGE + tpos % CC_PAGE) * DH + d]);
#pragma unroll
            for (int g = 0; g < kMaxG; ++g)
                if (g < G && g % NPART == part) {
                    const float p = s_p[g][tt];
                    acc[g] = fmaf(p, v, acc[g]);
                    l_run[g] += p;
                }
        }
        __syncthreads();                                               // s_p, s_red, s_page are rewritten by the next chunk
    }
    // ---- this range's partial result -> the scratch array ----
#pragma unroll
    for (int g = 0; g < kMaxG; ++g)
        if (g < G && g % NPART == part) {
            const size_t slot = ((size_t)b * Hq + (size_t)h * G + g) * n_split + sp;
            part_o[slot * DH + d] = acc[g];
            if (d == 0) {
                part_ml[slot * 2] = m_run[g];                          // an empty range (short row): m = -inf, l = 0
                part_ml[slot * 2 + 1] = l_run[g];
            }
        }
    __threadfence();
    __syncthreads();
    if (tid == 0) s_last = atomicAdd(&counters[b * Hkv + h], 1) == n_split - 1;
    __syncthreads();
    if (!s_last) return;
    __threadfence();
    // ---- the last block to arrive merges the ranges in range order ----
#pragma unroll
    for (int g = 0; g < kMaxG; ++g)
        if (g < G && g % NPART == part) {
            const size_t slot0 = ((size_t)b * Hq + (size_t)h * G + g) * n_split;
            float M = -INFINITY;
            for (int i = 0; i < n_split; ++i) M = fmaxf(M, __ldcg(part_ml + (slot0 + i) * 2));   // range 0 is never empty
            float L = 0.f, O = 0.f;
            for (int i = 0; i < n_split; ++i) {
                const float w = exp2f(__ldcg(part_ml + (slot0 + i) * 2) - M);
                L = fmaf(w, __ldcg(part_ml + (slot0 + i) * 2 + 1), L);
                O = fmaf(w, __ldcg(part_o + (slot0 + i) * DH + d), O);
            }
            out[((size_t)b * Hq + (size_t)h * G + g) * DH + d] = O / L;
        }
    if (tid == 0) counters[b * Hkv + h] = 0;                           // (the host clears them before every launch anyway)
}

// The device address of the scratch array, taken once per device with that device current.
cudaError_t scratch_address(int device, unsigned char** out) {
    constexpr int kMaxDevices = 64;
    static std::mutex mu;
    static unsigned char* addr[kMaxDevices] = {};
    if (device < 0 || device >= kMaxDevices) return cudaErrorInvalidDevice;
    std::lock_guard<std::mutex> lock(mu);
    if (!addr[device]) {
        void* p = nullptr;
        const cudaError_t e = cudaGetSymbolAddress(&p, g_static_scratch);   // the CURRENT device's copy of the array
        if (e != cudaSuccess) return e;
        addr[device] = static_cast<unsigned char*>(p);
    }
    *out = addr[device];
    return cudaSuccess;
}

cc_status fail_static(cc_status st, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    cc_internal_set_error(buf);
    return st;
}

}  // namespace

extern "C" {

size_t cc_static_scratch_bytes(void) { return kScratchBytes; }

cc_status cc_attention_decode_static(const float* q, const void* k_pool, const void* v_pool, const int32_t* block_table,
                                     const int32_t* seq_lens, float* out, int batch, int n_q_heads, int n_kv_heads, int head_dim,
                                     int max_blocks, int n_pages, void* stream) {
    if (!q || !k_pool || !v_pool || !block_table || !seq_lens || !out) return fail_static(CC_ERR_INVALID, "null argument");
    if (batch <= 0 || max_blocks <= 0 || n_pages <= 0) return fail_static(CC_ERR_INVALID, "batch, max_blocks and n_pages must be positive");
    if (head_dim != 64 && head_dim != 128) return fail_static(CC_ERR_INVALID, "head_dim %d: this entry point takes 64 or 128", head_dim);
    if (n_kv_heads <= 0 || n_q_heads <= 0 || n_q_heads % n_kv_heads || n_q_heads / n_kv_heads > kMaxG)
        return fail_static(CC_ERR_INVALID, "%d query heads over %d kv heads: need a whole ratio of at most %d", n_q_heads, n_kv_heads, kMaxG);
    if (batch > 65535 || n_kv_heads > 65535) return fail_static(CC_ERR_INVALID, "batch and n_kv_heads are grid dimensions: at most 65535");
    if ((size_t)batch * n_kv_heads * sizeof(int) > (size_t)kCounterBytes)
        return fail_static(CC_ERR_INVALID, "batch * n_kv_heads = %lld exceeds the %d arrival counters of the static scratch array",
                           (long long)batch * n_kv_heads, kCounterBytes / (int)sizeof(int));
    // ranges per row: a function of the arguments only -- about one per 512 positions of the widest possible row, at most 8,
    // fewer if their partial results would not fit into the array
    const size_t per_split = (size_t)batch * n_q_heads * (head_dim + 2) * sizeof(float);
    int n_split = (max_blocks + 31) / 32;
    if (n_split > kMaxSplit) n_split = kMaxSplit;
    if (n_split < 1) n_split = 1;
    while (n_split > 1 && kCounterBytes + per_split * n_split > kScratchBytes) --n_split;
    if (kCounterBytes + per_split * n_split > kScratchBytes)
        return fail_static(CC_ERR_INVALID,
                           "batch %d x %d query heads x head_dim %d needs %zu bytes of scratch; the static array holds %zu "
                           "(CC_STATIC_SCRATCH_BYTES): use cc_forward, whose workspace is sized at cc_create_layer",
                           batch, n_q_heads, head_dim, kCounterBytes + per_split, kScratchBytes);
    int device = 0;
    cudaError_t e = cudaGetDevice(&device);
    unsigned char* scratch = nullptr;
    if (e == cudaSuccess) e = scratch_address(device, &scratch);
    if (e != cudaSuccess) return fail_static(CC_ERR_CUDA, "cudaGetSymbolAddress of the static scratch array: %s", cudaGetErrorString(e));
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    e = cudaMemsetAsync(scratch, 0, (size_t)batch * n_kv_heads * sizeof(int), st);      // the arrival counters start at zero
    if (e != cudaSuccess) return fail_static(CC_ERR_CUDA, "cudaMemsetAsync: %s", cudaGetErrorString(e));
    const float scale_log2 = (float)(1.4426950408889634 / std::sqrt((double)head_dim));
    const dim3 grid((unsigned)n_split, (unsigned)n_kv_heads, (unsigned)batch);
    const uint16_t* kp = static_cast<const uint16_t*>(k_pool);
    const uint16_t* vp = static_cast<const uint16_t*>(v_pool);
    if (head_dim == 128)
        k_attn_static<128><<<grid, kChunk, 0, st>>>(q, kp, vp, block_table, seq_lens, out, n_q_heads, n_kv_heads, max_blocks, n_pages,
                                                    n_split, scale_log2, scratch);
    else
        k_attn_static<64><<<grid, kChunk, 0, st>>>(q, kp, vp, block_table, seq_lens, out, n_q_heads, n_kv_heads, max_blocks, n_pages,
                                                   n_split, scale_log2, scratch);
    e = cudaGetLastError();
    if (e != cudaSuccess) return fail_static(CC_ERR_CUDA, "launch of k_attn_static: %s", cudaGetErrorString(e));
    return CC_OK;
}

}  // extern "C"
