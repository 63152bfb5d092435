// cc_rowwise.cu -- the small memory-bound kernels around the GEMMs of the replicated decoder layer
// (sm_100a):
//   k_group        a0     micro-batch grouping + attention work list (device-built, graph-safe)
//   k_rmsnorm_in   a1     input RMSNorm -> GEMM operand
// The split-KV merge is done by the attention kernel itself (cc_attention.cu); RoPE + KV append, residual + post-attention norm, SwiGLU and the final residual are the fused
// epilogues of the stream-K fixup inside the GEMM kernel (cc_gemm.cu).  Every reduction order in
// this file is a function of the layer shape and seq_len only (never of the batch split), which
// is what makes outputs bit-identical across replica counts.
//
// GEMM operands are written as TWO bf16 planes, hi = bf16(v) and lo = bf16(v - hi): the tensor
// core multiplies the bf16 weights by both and accumulates in fp32, so the activations carry
// ~16 mantissa bits.  One bf16 plane alone costs ~6e-3 rms on the layer output at d = 4096,
// too close to the 1e-2 absolute tolerance.
#include "cc_kernels.h"

namespace {

__device__ __forceinline__ int replica_of_pos(const CcSched* s, int pos) {
    int r = 0;
#pragma unroll
    for (int i = 1; i < CC_MAXR; ++i)
        if (s->cnt[i] > 0 && pos >= s->goff[i]) r = i;
    return r;
}

// Deterministic block-wide sum (same value in every thread).
__device__ __forceinline__ float block_sum(float v, float* red) {
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) v += __shfl_xor_sync(0xffffffffu, v, o);
    const int w = threadIdx.x >> 5, l = threadIdx.x & 31;
    __syncthreads();
    if (l == 0) red[w] = v;
    __syncthreads();
    float t = 0.f;
    const int nw = blockDim.x >> 5;
    for (int i = 0; i < nw; ++i) t += red[i];
    return t;
}

// hi/lo split of two values -> packed bf16x2 words of the two planes.
__device__ __forceinline__ void split_hilo(float v0, float v1, uint32_t& hi, uint32_t& lo) {
    hi = pack_bf16(v0, v1);
    lo = pack_bf16(v0 - bf16lo(hi), v1 - bf16hi(hi));
}

// ---------------------------------------------------------------------------------------------
// a0: grouping.  One block; thread b owns row b.  Stable partition by replica,
// groups start at multiples of 16 rows; builds the split-KV work list (pos, chunk).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(256) k_group(const int* __restrict__ assign, const int* __restrict__ seq_lens,
                                               int batch, CcDims D, const CcLayerTable* __restrict__ tab, CcWork W) {
    __shared__ int s_wcnt[8][CC_MAXR];     // rows of replica r in warp w
    __shared__ int s_wnch[8];              // KV pages of the rows of warp w
    __shared__ int s_goff[CC_MAXR + 1], s_cnt[CC_MAXR];
    const int b = threadIdx.x, warp = b >> 5, lane = b & 31;
    pdl_wait();
    pdl_launch_dependents();
    const uint32_t mask = tab->active_mask;
    int rep = -1;
    if (b < batch) {
        const int s = seq_lens[b];
        if (s > 0) {
            if (s > D.max_position || (s + CC_PAGE - 1) / CC_PAGE > D.max_blocks) {
                atomicOr(W.err, CC_DEVERR_BAD_SEQLEN);
            } else {
                rep = assign[b];
                if (rep < 0 || rep >= CC_MAXR || !((mask >> rep) & 1u)) {
                    atomicOr(W.err, CC_DEVERR_BAD_REPLICA);
                    rep = 0;
                }
            }
        }
    }
    for (int i = b; i < D.Mpad; i += blockDim.x) W.perm[i] = -1;
    for (int i = b; i < 4 * CC_FLAG_STRIDE; i += blockDim.x) W.flags[i] = 0;   // stream-K fixup counters of this step
    // rank of this row among the rows of its replica: ballots inside the warp + warp prefix
    uint32_t bal[CC_MAXR];
#pragma unroll
    for (int r = 0; r < CC_MAXR; ++r) bal[r] = __ballot_sync(0xffffffffu, rep == r);
    // attention chunks ahead of this row inside the warp (rows keep request order in the work list
    // only within a replica group, so the list is ordered by grouped position below)
    if (lane == 0) {
#pragma unroll
        for (int r = 0; r < CC_MAXR; ++r) s_wcnt[warp][r] = __popc(bal[r]);
    }
    __syncthreads();
    if (b == 0) {
        int off = 0;
        for (int r = 0; r < CC_MAXR; ++r) {
            int c = 0;
            for (int w = 0; w < 8; ++w) c += s_wcnt[w][r];
            s_cnt[r] = c;
            s_goff[r] = off;
            off += (c + CC_ROW_ALIGN - 1) / CC_ROW_ALIGN * CC_ROW_ALIGN;
        }
        s_goff[CC_MAXR] = off;
    }
    __syncthreads();
    int pos = -1;
    if (rep >= 0) {
        uint32_t mine = 0;
#pragma unroll
        for (int r = 0; r < CC_MAXR; ++r)
            if (rep == r) mine = bal[r];
        int rank = __popc(mine & ((1u << lane) - 1u));
        for (int w = 0; w < warp; ++w) rank += s_wcnt[w][rep];
        pos = s_goff[rep] + rank;
        W.perm[pos] = b;
    }
    // attention work split: pages of the rows in request order (prefix sums); the attention CTAs cut this
    // page axis into equal contiguous ranges -- a function of the batch, never of the replica split
    if (b < D.max_batch) W.pos_of[b] = pos;
    const int npg = (rep >= 0) ? (seq_lens[b] + CC_PAGE - 1) / CC_PAGE : 0;
    int pre = npg;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, pre, o);
        if (lane >= o) pre += v;
    }
    if (lane == 31) s_wnch[warp] = pre;
    __syncthreads();
    int base = pre - npg, total = 0;
    for (int w = 0; w < 8; ++w) {
        if (w < warp) base += s_wnch[w];
        total += s_wnch[w];
    }
    if (b < D.max_batch) W.pg_prefix[b] = base;
    if (b == 0) W.pg_prefix[D.max_batch] = total;
    if (b == 0) {
        int nmax = 0;
        for (int r = 0; r < CC_MAXR; ++r) {
            W.sched->cnt[r] = s_cnt[r];
            W.sched->goff[r] = s_goff[r];
            nmax = max(nmax, (s_cnt[r] + CC_ROW_ALIGN - 1) / CC_ROW_ALIGN * CC_ROW_ALIGN);
        }
        W.sched->n_pos = s_goff[CC_MAXR];
        W.sched->n_items = total;
        W.sched->nmax = nmax;
    }
}

// ---------------------------------------------------------------------------------------------
// a1: x = h * rsqrt(mean(h^2) + eps) * g1  ->  hi/lo operand planes.  One block per position.
// ---------------------------------------------------------------------------------------------
constexpr int kNormThreads = 512;
__global__ void __launch_bounds__(kNormThreads) k_rmsnorm_in(const __nv_bfloat16* __restrict__ hidden, CcDims D,
                                                             const CcLayerTable* __restrict__ tab, CcWork W) {
    __shared__ float red[kNormThreads / 32];
    const int pos = blockIdx.x;
    pdl_wait();
    pdl_launch_dependents();
    if (threadIdx.x == 0) {   // warm L2 with the head of the QKV weight stream of the first non-empty group
        int r0 = 0;
        while (r0 < CC_MAXR - 1 && W.sched->cnt[r0] == 0) ++r0;
        for (int c = blockIdx.x; c < D.qkv.P; c += gridDim.x) cc_prefetch_gemm_head(D.qkv, tab->rep[r0].blob, c);
    }
    if (pos >= W.sched->n_pos) return;
    const int b = W.perm[pos];
    if (b < 0) return;
    const int r = replica_of_pos(W.sched, pos);
    const uint4* g = reinterpret_cast<const uint4*>(tab->rep[r].blob + D.off_g1);
    const uint4* row = reinterpret_cast<const uint4*>(hidden + (size_t)b * D.d);
    const int nchunk = D.d >> 3;
    float ss = 0.f;
    for (int c = threadIdx.x; c < nchunk; c += kNormThreads) {
        const uint4 v = row[c];
        const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float a = bf16lo(w[i]), bb = bf16hi(w[i]);
            ss += a * a + bb * bb;
        }
    }
    ss = block_sum(ss, red);
    const float inv = rsqrtf(ss / (float)D.d + D.eps);
    for (int c = threadIdx.x; c < nchunk; c += kNormThreads) {
        const uint4 v = row[c], gv = g[c];
        const uint32_t w[4] = {v.x, v.y, v.z, v.w}, gw[4] = {gv.x, gv.y, gv.z, gv.w};
        uint32_t hi[4], lo[4];
#pragma unroll
        for (int i = 0; i < 4; ++i)
            split_hilo(bf16lo(w[i]) * inv * bf16lo(gw[i]), bf16hi(w[i]) * inv * bf16hi(gw[i]), hi[i], lo[i]);
        uint8_t* dst = W.x_act + act_chunk_off(pos, c << 3, D.Mpad, 2, 0);
        *reinterpret_cast<uint4*>(dst) = make_uint4(hi[0], hi[1], hi[2], hi[3]);
        *reinterpret_cast<uint4*>(dst + 1024) = make_uint4(lo[0], lo[1], lo[2], lo[3]);
    }
}

constexpr int kMaxVecPerThread = 4;   // hidden <= 4 * 4 * 512 = 8192 (operand layout and epilogue limits)

// Test tap: widen a workspace buffer to fp32 [batch][dim] in original row order.
// which: 0 = one bf16 plane, 1 = fp32 rows, 2 = hi + lo planes, 3 = hi + lo planes times the row's
// 1/rms (the y' operand is stored un-normalised; its statistic lives in W.ssq).
__global__ void __launch_bounds__(256) k_tap(const void* __restrict__ src, int which, int dim, CcDims D,
                                             CcWork W, float* __restrict__ out, int batch) {
    const int pos = blockIdx.x;
    if (pos >= W.sched->n_pos) return;
    const int b = W.perm[pos];
    if (b < 0 || b >= batch) return;
    float scale = 1.f;
    if (which == 3) {
        float ss = 0.f;
        for (int t = 0; t < (D.d + 127) / 128; ++t) ss += W.ssq[(size_t)t * D.Mpad + pos];
        scale = rsqrtf(ss / (float)D.d + D.eps);
    }
    for (int k = threadIdx.x; k < dim; k += blockDim.x) {
        float v;
        if (which == 1) {
            v = reinterpret_cast<const float*>(src)[(size_t)pos * dim + k];
        } else {
            const uint8_t* p = reinterpret_cast<const uint8_t*>(src) + act_chunk_off(pos, k, D.Mpad, which >= 2 ? 2 : 1, 0) + (k & 7) * 2;
            v = __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(p));
            if (which >= 2) v += __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(p + 1024));
            v *= scale;
        }
        out[(size_t)b * dim + k] = v;
    }
}

}  // namespace

// ---- launchers ---------------------------------------------------------------------------------
cudaError_t cc_launch_group(const int* assign, const int* seq_lens, int batch, const CcDims& D,
                            const CcLayerTable* tab, const CcWork& W, const CcLaunch& L) {
    return cc_launch_kernel(k_group, dim3(1), dim3(256), 0, L, assign, seq_lens, batch, D, tab, W);
}
cudaError_t cc_launch_rmsnorm_in(const __nv_bfloat16* hidden, const CcDims& D, const CcLayerTable* tab,
                                 const CcWork& W, const CcLaunch& L) {
    return cc_launch_kernel(k_rmsnorm_in, dim3(D.Mpad), dim3(kNormThreads), 0, L, hidden, D, tab, W);
}
cudaError_t cc_launch_tap(const void* src, int which, int dim, const CcDims& D, const CcWork& W,
                          float* out_dev, int batch, cudaStream_t st) {
    k_tap<<<D.Mpad, 256, 0, st>>>(src, which, dim, D, W, out_dev, batch);
    return cudaGetLastError();
}
int cc_max_hidden() { return kMaxVecPerThread * 4 * kNormThreads; }
