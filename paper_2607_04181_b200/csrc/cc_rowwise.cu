// cc_rowwise.cu -- the small memory-bound kernels around the GEMMs of the replicated decoder layer
// (sm_100a):
//   k_prologue     a0+a1  micro-batch grouping, page prefix of the attention split, input RMSNorm -> operand
// The split-KV merge is done by the attention kernel itself (cc_attention.cu); RoPE + KV append,
// residual + post-attention norm, SwiGLU and the final residual are the fused epilogues of the
// stream-K fixup inside the GEMM kernel (cc_gemm.cu).  Every reduction order in
// this file is a function of the layer shape and seq_len only (never of the batch split), which
// is what makes outputs bit-identical across replica counts.
//
// GEMM operands are written in the layer's operand format (act_store, cc_common.cuh): ONE fp16 plane
// (11 significand bits) against fp16 weights, or TWO bf16 planes hi = bf16(v), lo = bf16(v - hi) against
// bf16 weights.  One bf16 plane alone costs ~6e-3 rms on the layer output at d = 4096, too close to the
// 1e-2 absolute tolerance.
#include "cc_kernels.h"

namespace {

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

// ---------------------------------------------------------------------------------------------
// a0 + a1 in one kernel, one block per request row (+ two blocks for the tables).
// a0: grouping.  Every block repeats it (256 rows: a few ballots), thread b owns row b.  Stable partition
// by replica, groups start at multiples of 16 rows; page prefix of the attention work
// split.  Block 0 publishes the tables; each block learns the grouped position of its own row.
// a1: x = h * rsqrt(mean(h^2) + eps) * g1  ->  hi/lo operand planes of that row.  The row is requested before
// the grouping (its address does not depend on it) and stays in registers between the two passes.
// ---------------------------------------------------------------------------------------------
constexpr int kNormThreads = 512;
constexpr int kNormVec = 2;            // uint4 (8 bf16) per thread: hidden <= 8 * 2 * 512 = 8192
__global__ void __launch_bounds__(kNormThreads) k_prologue(const int* __restrict__ assign, const int* __restrict__ seq_lens,
                                                           const int* __restrict__ block_table, int batch,
                                                           const __nv_bfloat16* __restrict__ hidden, CcDims D,
                                                           const CcLayerTable* __restrict__ tab, CcWork W, CcStageOut so) {
    __shared__ int s_wcnt[8][CC_MAXR];     // rows of replica r in warp w
    __shared__ int s_wnch[8];              // KV pages of the rows of warp w
    __shared__ int s_goff[CC_MAXR + 1], s_cnt[CC_MAXR];
    __shared__ int s_mypos, s_myrep;
    __shared__ int s_key[256], s_wpg[256];   // first page id of row b (names its request), page index row b appends to
    __shared__ signed char s_rep[256];       // replica that serves row b (scan block only)
    __shared__ float red[kNormThreads / 32];
    const int b = threadIdx.x, warp = b >> 5, lane = b & 31;
    // grid = batch + 2: block b < batch normalises row b; the two extra blocks only publish the tables and look for the
    // rows that share a request, so that no row's block carries that work on top of its own (it was the slowest block
    // of the kernel by ~3 us, and the QKV GEMM waits for the last one)
    const bool pub = blockIdx.x == gridDim.x - 2;    // this block writes the tables
    const bool scan = blockIdx.x == gridDim.x - 1;   // this one finds the rows that share a request (prompt chunks)
    const bool has_row = (int)blockIdx.x < batch;
    if (b == 0) CC_TP(W, 0, 0);
    pdl_wait();
    if (b == 0) CC_TP(W, 0, 1);
    pdl_launch_dependents();
    if (b == 0) s_mypos = -1;
    const int my_b = blockIdx.x;
    const int nchunk = D.d >> 3;
    uint4 v[kNormVec];
    {
        const uint4* row = reinterpret_cast<const uint4*>(hidden + (size_t)my_b * D.d);
#pragma unroll
        for (int j = 0; j < kNormVec; ++j) {
            const int c = threadIdx.x + j * kNormThreads;
            v[j] = (has_row && c < nchunk) ? row[c] : make_uint4(0, 0, 0, 0);
        }
    }
    int rep = -1, pos = -1;
    if (b < 256) {
        uint32_t err = 0;
        rep = cc_row_replica(assign, seq_lens, b, batch, D, tab->active_mask, err);
        if (pub && err) atomicOr(W.err, err);
        if (scan) {
            // rows of one request carry copies of its block-table row, so its first page id names the request
            s_key[b] = rep >= 0 ? block_table[(size_t)b * D.max_blocks] : -1 - b;
            s_wpg[b] = rep >= 0 ? (seq_lens[b] - 1) / CC_PAGE : 0x7fffffff;
            s_rep[b] = (signed char)rep;
        }
        uint32_t bal[CC_MAXR];
#pragma unroll
        for (int r = 0; r < CC_MAXR; ++r) bal[r] = __ballot_sync(0xffffffffu, rep == r);
        if (lane == 0) {
#pragma unroll
            for (int r = 0; r < CC_MAXR; ++r) s_wcnt[warp][r] = __popc(bal[r]);
        }
        __syncwarp();
        if (pub) {
            for (int i = b; i < D.Mpad; i += 256) W.perm[i] = -1;
            for (int i = b; i < 4 * CC_FLAG_STRIDE; i += 256) W.flags[i] = 0;   // stream-K fixup counters of this step
        }
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
    if (scan) {
        // The attention kernel streams a row's pages before this step's appends are finished, up to the first page
        // some row of the step writes.  For a lone decode row that is its last page; for the rows of a prompt chunk
        // (one request, consecutive positions) it is the lowest page any of them appends to.  One warp per row, the
        // lanes share the comparisons (a thread per row walking all rows took 3 us at batch 64, and the QKV GEMM
        // waits for this block).
        for (int rb = warp; rb < batch; rb += kNormThreads / 32) {
            const int key = s_key[rb], rrep = s_rep[rb];
            int m = 0x7fffffff;
            bool split = false;
            for (int j = lane; j < batch; j += 32)
                if (s_key[j] == key) {
                    m = min(m, s_wpg[j]);
                    split |= s_rep[j] != rrep;
                }
            m = __reduce_min_sync(0xffffffffu, m);
            split = __any_sync(0xffffffffu, split);
            if (lane == 0 && rrep >= 0) {
                W.first_wr[rb] = m;
                if (split) atomicOr(W.err, CC_DEVERR_SPLIT_REQUEST);   // one request served by two replicas
            }
        }
    }
    if (b < 256) {
        // rank of this row among the rows of its replica: ballot of its warp + the warps before it
        // (the ballots are taken again -- cheaper than keeping four of them alive across the barriers)
        uint32_t mine = 0;
#pragma unroll
        for (int r = 0; r < CC_MAXR; ++r) {
            const uint32_t br = __ballot_sync(0xffffffffu, rep == r);
            if (rep == r) mine = br;
        }
        if (rep >= 0) {
            int rank = __popc(mine & ((1u << lane) - 1u));
            for (int w = 0; w < warp; ++w) rank += s_wcnt[w][rep];
            pos = s_goff[rep] + rank;
            if (pub) W.perm[pos] = b;
            if (b == my_b) { s_mypos = pos; s_myrep = rep; }
        }
        // attention work split: pages of the rows in request order (prefix sums); the attention CTAs cut this
        // page axis into equal contiguous ranges -- a function of the batch, never of the replica split
        if (pub) {
            if (b < D.max_batch) W.pos_of[b] = pos;
            const int npg = (rep >= 0) ? (seq_lens[b] + CC_PAGE - 1) / CC_PAGE : 0;
            int pre = npg;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int v = __shfl_up_sync(0xffffffffu, pre, o);
                if (lane >= o) pre += v;
            }
            if (lane == 31) s_wnch[warp] = pre;
            named_bar_sync(1, 256);
            int base = pre - npg, total = 0;
            for (int w = 0; w < 8; ++w) {
                if (w < warp) base += s_wnch[w];
                total += s_wnch[w];
            }
            if (b < D.max_batch) W.pg_prefix[b] = base;
            if (b == 0) {
                W.pg_prefix[D.max_batch] = total;
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
    }
    __syncthreads();
    const int mypos = s_mypos;
    if (mypos < 0) {                       // block-uniform: padding row, or one of the two table blocks
        if (b == 0 && (pub || scan)) CC_TP(W, 0, 2);
        return;
    }
    const uint4* g = reinterpret_cast<const uint4*>(tab->rep[s_myrep].blob + D.off_g1);
    uint4 gv[kNormVec];
    float ss = 0.f;
#pragma unroll
    for (int j = 0; j < kNormVec; ++j) {
        const int c = threadIdx.x + j * kNormThreads;
        gv[j] = make_uint4(0, 0, 0, 0);
        if (c < nchunk) {
            gv[j] = g[c];
            if (so.hidden != nullptr) reinterpret_cast<uint4*>(so.hidden + (size_t)my_b * D.d)[c] = v[j];
        }
        const uint32_t w[4] = {v[j].x, v[j].y, v[j].z, v[j].w};
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float a = bf16lo(w[i]), bb = bf16hi(w[i]);
            ss += a * a + bb * bb;
        }
    }
    ss = block_sum(ss, red);
    const float inv = rsqrtf(ss / (float)D.d + D.eps);
#pragma unroll
    for (int j = 0; j < kNormVec; ++j) {
        const int c = threadIdx.x + j * kNormThreads;
        if (c >= nchunk) break;
        const uint32_t w[4] = {v[j].x, v[j].y, v[j].z, v[j].w}, gw[4] = {gv[j].x, gv[j].y, gv[j].z, gv[j].w};
        float x[8];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            x[2 * i] = bf16lo(w[i]) * inv * bf16lo(gw[i]);
            x[2 * i + 1] = bf16hi(w[i]) * inv * bf16hi(gw[i]);
        }
        act_store<8>(W.x_act, D, D.pl[CC_OP_X], mypos, c << 3, x);
    }
    if (threadIdx.x == 0) W.inv_in[mypos] = inv;
    if (b == 0) CC_TP(W, 0, 2);
}

// Test tap: widen a workspace buffer to fp32 [batch][dim] in original row order.
// which: 1 = fp32 rows, 2 = packed operand (the layer's format), 3 = packed operand times the row's
// 1/rms over the input row's 1/rms (the y' operand is stored before its statistic, W.ssq, is known).
__global__ void __launch_bounds__(256) k_tap(const void* __restrict__ src, int which, int planes, int dim, CcDims D,
                                             CcWork W, float* __restrict__ out, int batch) {
    const int pos = blockIdx.x;
    if (pos >= W.sched->n_pos) return;
    const int b = W.perm[pos];
    if (b < 0 || b >= batch) return;
    float scale = 1.f;
    if (which == 3) {
        float ss = 0.f;
        for (int t = 0; t < (D.d + 127) / 128; ++t) ss += W.ssq[(size_t)t * D.Mpad + pos];
        scale = rsqrtf(ss / (float)D.d + D.eps) / W.inv_in[pos];
    }
    for (int k = threadIdx.x; k < dim; k += blockDim.x) {
        float v;
        if (which == 1) {
            v = reinterpret_cast<const float*>(src)[(size_t)pos * dim + k];
        } else {
            const uint8_t* p = reinterpret_cast<const uint8_t*>(src) + act_chunk_off(pos, k, D.Mpad, planes, 0) + (k & 7) * 2;
            if (D.fmt == CC_FMT_F16) {
                v = __half2float(*reinterpret_cast<const __half*>(p));
                if (planes == 2) v += __half2float(*reinterpret_cast<const __half*>(p + 1024));
            } else {
                v = __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(p));
                v += __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(p + 1024));
            }
            v *= scale;
        }
        out[(size_t)b * dim + k] = v;
    }
}

}  // namespace

// ---- launchers ---------------------------------------------------------------------------------
cudaError_t cc_launch_prologue(const int* assign, const int* seq_lens, const int* block_table, int batch,
                               const __nv_bfloat16* hidden, const CcDims& D, const CcLayerTable* tab, const CcWork& W,
                               const CcLaunch& L, const CcStageOut& so) {
    return cc_launch_kernel(k_prologue, dim3(batch + 2), dim3(kNormThreads), 0, L, assign, seq_lens, block_table, batch, hidden, D, tab,
                            W, so);
}
cudaError_t cc_launch_tap(const void* src, int which, int planes, int dim, const CcDims& D, const CcWork& W,
                          float* out_dev, int batch, cudaStream_t st) {
    k_tap<<<D.Mpad, 256, 0, st>>>(src, which, planes, dim, D, W, out_dev, batch);
    return cudaGetLastError();
}
int cc_max_hidden() { return kNormVec * 8 * kNormThreads; }
