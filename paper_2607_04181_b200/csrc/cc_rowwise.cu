// cc_rowwise.cu -- the small memory-bound kernels between the GEMMs of the replicated decoder
// layer (sm_100a).  Each one is the fused epilogue of the GEMM before it and the prologue of
// the GEMM after it:
//   k_group        a0     micro-batch grouping + attention work list (device-built, graph-safe)
//   k_rmsnorm_in   a1     input RMSNorm -> GEMM operand
//   k_rope_append  a3+a4  QKV piece reduce, RoPE, KV append into the paged cache
//   k_attn_combine a5     fixed-order merge of the split-KV partials -> GEMM operand
//   k_resid_norm   a6+a7  O-proj piece reduce + residual, RMSNorm -> GEMM operand
//   k_swiglu       a8     gate/up piece reduce, silu(gate)*up -> GEMM operand
//   k_final        a9     down piece reduce + residual, rows back in request order
// "Piece reduce": the stream-K GEMM leaves, per tile of 128 output features, a few fp32 partial
// sums; they are added here in increasing piece order.  That order, like every other reduction
// order in this file, is a function of the layer shape only (never of the batch split), which is
// what makes outputs bit-identical across replica counts.
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
    __shared__ int s_wnch[8];              // attention chunks in warp w
    __shared__ int s_goff[CC_MAXR + 1], s_cnt[CC_MAXR];
    const int b = threadIdx.x, warp = b >> 5, lane = b & 31;
    pdl_wait();
    pdl_launch_dependents();
    const uint32_t mask = tab->active_mask;
    int rep = -1, nch = 0;
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
                nch = (s + CC_ATTN_CHUNK - 1) / CC_ATTN_CHUNK;
            }
        }
    }
    for (int i = b; i < D.Mpad; i += blockDim.x) W.perm[i] = -1;
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
    // work list ordered by request index b (any fixed order is fine: items are independent)
    int pre = nch;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int v = __shfl_up_sync(0xffffffffu, pre, o);
        if (lane >= o) pre += v;
    }
    if (lane == 31) s_wnch[warp] = pre;
    __syncthreads();
    int base = pre - nch;
    for (int w = 0; w < warp; ++w) base += s_wnch[w];
    for (int c = 0; c < nch; ++c) W.items[base + c] = make_int2(pos, c);
    if (b == 0) {
        int total = 0, nmax = 0;
        for (int w = 0; w < 8; ++w) total += s_wnch[w];
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

// ---------------------------------------------------------------------------------------------
// a3 + a4: reduce the QKV pieces (fixed order), rotate q and k at position s-1 (rotate-half pairs
// (i, i+Dh/2), cos/sin from the fp64-built table), keep q in fp32, store bf16(k), bf16(v) into the
// page slot of position s-1 (PAPER.md:103 local append).
// grid (tile, row group); block (64, 4): thread x owns the column pair (f0, f0 + Dh/2) of its tile.
// ---------------------------------------------------------------------------------------------
constexpr int kRopeRows = 4;
__global__ void __launch_bounds__(64 * kRopeRows) k_rope_append(const int* __restrict__ seq_lens, CcKv kv, CcDims D,
                                                                CcWork W) {
    const int t = blockIdx.x, pos = blockIdx.y * kRopeRows + threadIdx.y;
    pdl_wait();
    pdl_launch_dependents();
    if (pos >= W.sched->n_pos) return;
    const int b = W.perm[pos];
    if (b < 0) return;
    const int half = D.Dh >> 1;
    const int j = threadIdx.x;
    const int f0 = (j / half) * D.Dh + (j % half);         // first column of the pair inside the tile
    int p0, np;
    cc_tile_pieces(D.qkv, t, p0, np);
    float a = 0.f, bb = 0.f;
    for (int i = 0; i < np; ++i) {
        const float* src = W.qkv_part + ((size_t)(p0 + i * CC_G) * D.Mpad + pos) * 128;
        a += src[f0];
        bb += src[f0 + half];
    }
    const int col = t * 128 + f0;                          // column of `a` in [q | k | v]
    if (col >= D.QD + 2 * D.KD) return;                    // padding columns of the last tile
    const int s = seq_lens[b], p = s - 1;
    const int i = col % D.Dh;                              // index inside the head, < half
    if (col < D.QD + D.KD) {                               // q or k: rotate
        const float2 c = W.rope_cs[(size_t)p * half + i];
        const float ra = a * c.x - bb * c.y, rb = bb * c.x + a * c.y;
        if (col < D.QD) {
            W.q_rot[(size_t)pos * D.QD + col] = ra;
            W.q_rot[(size_t)pos * D.QD + col + half] = rb;
            return;
        }
        a = ra;
        bb = rb;
    }
    const int page = kv.block_table[(size_t)b * D.max_blocks + p / CC_PAGE];
    if (page < 0 || page >= kv.n_pages) {
        if (j == 0) atomicOr(W.err, CC_DEVERR_BAD_PAGE);
        return;
    }
    const bool is_k = col < D.QD + D.KD;
    const int kc = col - D.QD - (is_k ? 0 : D.KD);         // column inside K (or V)
    const int hk = kc / D.Dh;
    __nv_bfloat16* dst = (is_k ? kv.k_pool : kv.v_pool) + (((size_t)page * D.Hkv + hk) * CC_PAGE + p % CC_PAGE) * D.Dh;
    dst[i] = __float2bfloat16_rn(a);
    dst[i + half] = __float2bfloat16_rn(bb);
}

// ---------------------------------------------------------------------------------------------
// a5 (second half): merge the split-KV partials of one (row, head) in chunk order -> bf16 operand
// (one plane: the O projection does not need more).
// grid (Hq, row); block = Dh/2 threads, two dims each.
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(64) k_attn_combine(const int* __restrict__ seq_lens, CcDims D, CcWork W) {
    const int hq = blockIdx.x, pos = blockIdx.y;
    pdl_wait();
    pdl_launch_dependents();
    if (pos >= W.sched->n_pos) return;
    const int b = W.perm[pos];
    if (b < 0) return;
    const int nch = (seq_lens[b] + CC_ATTN_CHUNK - 1) / CC_ATTN_CHUNK;
    const int dim = threadIdx.x * 2;
    if (dim >= D.Dh) return;
    const size_t row = ((size_t)pos * D.Hq + hq) * W.nch_max;
    float M = -INFINITY;
    for (int c = 0; c < nch; ++c) M = fmaxf(M, W.att_ml[row + c].x);
    float L = 0.f, a0 = 0.f, a1 = 0.f;
    for (int c = 0; c < nch; ++c) {
        const float2 ml = W.att_ml[row + c];
        const float w = exp2f(ml.x - M);
        const float2 o = *reinterpret_cast<const float2*>(W.att_o + (row + c) * D.Dh + dim);
        L += w * ml.y;
        a0 += w * o.x;
        a1 += w * o.y;
    }
    const float inv = 1.f / L;
    const int e = hq * D.Dh + dim;
    uint8_t* dst = W.o_act + act_chunk_off(pos, e, D.Mpad, 1, 0) + (e & 7) * 2;
    *reinterpret_cast<uint32_t*>(dst) = pack_bf16(a0 * inv, a1 * inv);
}

// ---------------------------------------------------------------------------------------------
// a6 (reduce + residual) and a7 (RMSNorm): h1 = h + sum of pieces ; y = rmsnorm(h1) * g2.
// One block per position; thread owns float4 column groups (kept in registers, <= 4 per thread).
// ---------------------------------------------------------------------------------------------
constexpr int kMaxVecPerThread = 4;   // hidden <= 4 * 4 * 512 = 8192
__global__ void __launch_bounds__(kNormThreads) k_resid_norm(const __nv_bfloat16* __restrict__ hidden, CcDims D,
                                                             const CcLayerTable* __restrict__ tab, CcWork W) {
    __shared__ float red[kNormThreads / 32];
    const int pos = blockIdx.x;
    pdl_wait();
    pdl_launch_dependents();
    if (pos >= W.sched->n_pos) return;
    const int b = W.perm[pos];
    if (b < 0) return;
    const int r = replica_of_pos(W.sched, pos);
    const __nv_bfloat16* g = reinterpret_cast<const __nv_bfloat16*>(tab->rep[r].blob + D.off_g2);
    float4 v[kMaxVecPerThread];
    float ss = 0.f;
#pragma unroll
    for (int it = 0; it < kMaxVecPerThread; ++it) {
        const int col = (it * kNormThreads + threadIdx.x) * 4;
        if (col >= D.d) break;
        const int t = col >> 7, f = col & 127;
        int p0, np;
        cc_tile_pieces(D.o, t, p0, np);
        float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
        for (int i = 0; i < np; ++i) {
            const float4 q = *reinterpret_cast<const float4*>(W.o_part + ((size_t)(p0 + i * CC_G) * D.Mpad + pos) * 128 + f);
            acc.x += q.x; acc.y += q.y; acc.z += q.z; acc.w += q.w;
        }
        const uint2 hb = *reinterpret_cast<const uint2*>(hidden + (size_t)b * D.d + col);
        acc.x += bf16lo(hb.x); acc.y += bf16hi(hb.x); acc.z += bf16lo(hb.y); acc.w += bf16hi(hb.y);
        v[it] = acc;
        *reinterpret_cast<float4*>(W.h1 + (size_t)pos * D.d + col) = acc;
        ss += (acc.x * acc.x + acc.y * acc.y) + (acc.z * acc.z + acc.w * acc.w);
    }
    ss = block_sum(ss, red);
    const float inv = rsqrtf(ss / (float)D.d + D.eps);
#pragma unroll
    for (int it = 0; it < kMaxVecPerThread; ++it) {
        const int col = (it * kNormThreads + threadIdx.x) * 4;
        if (col >= D.d) break;
        const uint2 gb = *reinterpret_cast<const uint2*>(g + col);
        uint32_t hi0, lo0, hi1, lo1;
        split_hilo(v[it].x * inv * bf16lo(gb.x), v[it].y * inv * bf16hi(gb.x), hi0, lo0);
        split_hilo(v[it].z * inv * bf16lo(gb.y), v[it].w * inv * bf16hi(gb.y), hi1, lo1);
        uint8_t* dst = W.y_act + act_chunk_off(pos, col, D.Mpad, 2, 0) + (col & 7) * 2;
        *reinterpret_cast<uint2*>(dst) = make_uint2(hi0, hi1);
        *reinterpret_cast<uint2*>(dst + 1024) = make_uint2(lo0, lo1);
    }
}

// ---------------------------------------------------------------------------------------------
// a8: a_j = silu(gate_j) * up_j with gate_j, up_j at interleaved columns 2j, 2j+1 of the gate/up
// GEMM output.  grid (tile, row group); block (32, 8): thread x owns 4 columns = 2 outputs.
// ---------------------------------------------------------------------------------------------
constexpr int kEpiRows = 8;
__global__ void __launch_bounds__(32 * kEpiRows) k_swiglu(CcDims D, CcWork W) {
    const int t = blockIdx.x, pos = blockIdx.y * kEpiRows + threadIdx.y;
    pdl_wait();
    pdl_launch_dependents();
    if (pos >= W.sched->n_pos) return;
    if (W.perm[pos] < 0) return;
    const int f = threadIdx.x * 4;
    int p0, np;
    cc_tile_pieces(D.gu, t, p0, np);
    float4 acc = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int i = 0; i < np; ++i) {
        const float4 q = *reinterpret_cast<const float4*>(W.gu_part + ((size_t)(p0 + i * CC_G) * D.Mpad + pos) * 128 + f);
        acc.x += q.x; acc.y += q.y; acc.z += q.z; acc.w += q.w;
    }
    const float a0 = acc.x / (1.f + __expf(-acc.x)) * acc.y;
    const float a1 = acc.z / (1.f + __expf(-acc.z)) * acc.w;
    uint32_t hi, lo;
    split_hilo(a0, a1, hi, lo);
    const int k = t * 64 + threadIdx.x * 2;                 // output index (K index of the down GEMM)
    if (k >= D.dn.KB * CC_TILE_K) return;                   // padding tiles of the last super tile
    uint8_t* dst = W.a_act + act_chunk_off(pos, k, D.Mpad, 2, 0) + (k & 7) * 2;
    *reinterpret_cast<uint32_t*>(dst) = hi;
    *reinterpret_cast<uint32_t*>(dst + 1024) = lo;
}

// ---------------------------------------------------------------------------------------------
// a9 (reduce + residual): out[b] = bf16(h1 + sum of pieces), written to row b = original order
// (PAPER.md:101 gather + concat along batch).  grid (tile, row group); block (32, 8).
// ---------------------------------------------------------------------------------------------
__global__ void __launch_bounds__(32 * kEpiRows) k_final(__nv_bfloat16* __restrict__ hidden, CcDims D, CcWork W) {
    const int t = blockIdx.x, pos = blockIdx.y * kEpiRows + threadIdx.y;
    pdl_wait();
    pdl_launch_dependents();
    if (pos >= W.sched->n_pos) return;
    const int b = W.perm[pos];
    if (b < 0) return;
    const int f = threadIdx.x * 4, col = t * 128 + f;
    if (col >= D.d) return;
    int p0, np;
    cc_tile_pieces(D.dn, t, p0, np);
    float4 acc = *reinterpret_cast<const float4*>(W.h1 + (size_t)pos * D.d + col);
    float4 sum = make_float4(0.f, 0.f, 0.f, 0.f);
    for (int i = 0; i < np; ++i) {
        const float4 q = *reinterpret_cast<const float4*>(W.d_part + ((size_t)(p0 + i * CC_G) * D.Mpad + pos) * 128 + f);
        sum.x += q.x; sum.y += q.y; sum.z += q.z; sum.w += q.w;
    }
    uint2 o;
    o.x = pack_bf16(acc.x + sum.x, acc.y + sum.y);
    o.y = pack_bf16(acc.z + sum.z, acc.w + sum.w);
    *reinterpret_cast<uint2*>(hidden + (size_t)b * D.d + col) = o;
}

// Test tap: widen a workspace buffer to fp32 [batch][dim] in original row order.
// which: 0 = one bf16 plane, 1 = fp32 rows, 2 = hi + lo planes.
__global__ void __launch_bounds__(256) k_tap(const void* __restrict__ src, int which, int dim, CcDims D,
                                             CcWork W, float* __restrict__ out, int batch) {
    const int pos = blockIdx.x;
    if (pos >= W.sched->n_pos) return;
    const int b = W.perm[pos];
    if (b < 0 || b >= batch) return;
    for (int k = threadIdx.x; k < dim; k += blockDim.x) {
        float v;
        if (which == 1) {
            v = reinterpret_cast<const float*>(src)[(size_t)pos * dim + k];
        } else {
            const uint8_t* p = reinterpret_cast<const uint8_t*>(src) + act_chunk_off(pos, k, D.Mpad, which == 2 ? 2 : 1, 0) + (k & 7) * 2;
            v = __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(p));
            if (which == 2) v += __bfloat162float(*reinterpret_cast<const __nv_bfloat16*>(p + 1024));
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
cudaError_t cc_launch_rope_append(const int* seq_lens, const CcKv& kv, const CcDims& D, const CcWork& W,
                                  const CcLaunch& L) {
    const dim3 grid(D.qkv.ST * CC_G, (D.Mpad + kRopeRows - 1) / kRopeRows), block(64, kRopeRows);
    return cc_launch_kernel(k_rope_append, grid, block, 0, L, seq_lens, kv, D, W);
}
cudaError_t cc_launch_attn_combine(const int* seq_lens, const CcDims& D, const CcWork& W, const CcLaunch& L) {
    return cc_launch_kernel(k_attn_combine, dim3(D.Hq, D.Mpad), dim3(64), 0, L, seq_lens, D, W);
}
cudaError_t cc_launch_resid_norm(const __nv_bfloat16* hidden, const CcDims& D, const CcLayerTable* tab,
                                 const CcWork& W, const CcLaunch& L) {
    return cc_launch_kernel(k_resid_norm, dim3(D.Mpad), dim3(kNormThreads), 0, L, hidden, D, tab, W);
}
cudaError_t cc_launch_swiglu(const CcDims& D, const CcWork& W, const CcLaunch& L) {
    const dim3 grid(D.gu.ST * CC_G, (D.Mpad + kEpiRows - 1) / kEpiRows), block(32, kEpiRows);
    return cc_launch_kernel(k_swiglu, grid, block, 0, L, D, W);
}
cudaError_t cc_launch_final(__nv_bfloat16* hidden, const CcDims& D, const CcWork& W, const CcLaunch& L) {
    const dim3 grid(D.dn.ST * CC_G, (D.Mpad + kEpiRows - 1) / kEpiRows), block(32, kEpiRows);
    return cc_launch_kernel(k_final, grid, block, 0, L, hidden, D, W);
}
cudaError_t cc_launch_tap(const void* src, int which, int dim, const CcDims& D, const CcWork& W,
                          float* out_dev, int batch, cudaStream_t st) {
    k_tap<<<D.Mpad, 256, 0, st>>>(src, which, dim, D, W, out_dev, batch);
    return cudaGetLastError();
}
int cc_max_hidden() { return kMaxVecPerThread * 4 * kNormThreads; }
