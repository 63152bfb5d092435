// cc_big.cu -- the row-wise kernels of a LARGE step (more than 256 rows: prompt chunks + decode rows; SURVEY.md 8(f)
// NEXT-2, BASELINE.json configs[3]):
//   k_big_group    a0  stable partition of up to CC_BIG_MAX_ROWS rows by replica, per-row position / page tables,
//                      the prompt chunks of the step (runs of rows that share a block-table row at consecutive
//                      seq_lens), the decode rows outside them with the page prefix of their attention split, and
//                      the work items of the chunk-prefill attention kernel
//   k_big_norm     a1  input RMSNorm -> GEMM operand, one block per row
//   k_big_rowstat  a7  per-row scale of the gate/up epilogue from the O epilogue's per-tile sums of squares
// The small-step kernels (cc_rowwise.cu) hold a row per thread and stop at 256 rows; these walk the rows in strides.
// Nothing here depends on the replica assignment except the grouping itself (PAPER.md:385 bit-wise consistency).
#include "cc_kernels.h"

namespace {

constexpr int kGroupThreads = 1024;

// exclusive prefix of v over the block (all threads call); *total = sum
__device__ __forceinline__ int block_scan_excl(int v, int* s_w, int* total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    int inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const int t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();
    if (lane == 31) s_w[w] = inc;
    __syncthreads();
    int base = 0, tot = 0;
    for (int i = 0; i < kGroupThreads / 32; ++i) {
        if (i < w) base += s_w[i];
        tot += s_w[i];
    }
    *total = tot;
    return base + inc - v;
}

__global__ void __launch_bounds__(kGroupThreads) k_big_group(const int* __restrict__ assign, const int* __restrict__ seq_lens,
                                                             const int* __restrict__ block_table, int batch, CcDims D,
                                                             const CcLayerTable* __restrict__ tab, CcWork W) {
    __shared__ signed char s_rep[CC_BIG_MAX_ROWS];
    __shared__ unsigned char s_cont[CC_BIG_MAX_ROWS + 1];     // row b continues the chunk of row b - 1
    __shared__ int s_w[kGroupThreads / 32];
    __shared__ int s_cnt[CC_MAXR], s_goff[CC_MAXR + 1], s_run[CC_MAXR];
    __shared__ int s_ndec, s_nchunk, s_ntail, s_pages, s_pages_dec;
    __shared__ int s_head[CC_BIG_MAX_CHUNKS], s_tail[CC_BIG_MAX_CHUNKS], s_ntile[CC_BIG_MAX_CHUNKS];
    const int tid = threadIdx.x;
    const uint32_t mask = tab->active_mask;
    uint32_t err = 0;
    if (tid < CC_MAXR) s_cnt[tid] = 0;
    for (int i = tid; i < D.Mpad; i += kGroupThreads) {
        W.perm[i] = -1;
        W.row_pos[i] = -1;
        W.row_page[i] = -1;
    }
    __syncthreads();
    // ---- pass 1: the replica of every row, chunk continuation flags, rows per replica ----
    for (int b0 = 0; b0 < batch; b0 += kGroupThreads) {
        const int b = b0 + tid;
        int rep = -1;
        if (b < batch) rep = cc_row_replica(assign, seq_lens, b, batch, D, mask, err);
        if (b < batch) s_rep[b] = (signed char)rep;
        bool cont = false;
        if (b < batch && b > 0 && rep >= 0) {
            uint32_t e2 = 0;                                           // (row b - 1 reports its own errors)
            cont = cc_row_replica(assign, seq_lens, b - 1, batch, D, mask, e2) >= 0 && seq_lens[b] == seq_lens[b - 1] + 1 &&
                   block_table[(size_t)b * D.max_blocks] == block_table[(size_t)(b - 1) * D.max_blocks];
        }
        if (b < batch) s_cont[b] = cont ? 1 : 0;
#pragma unroll
        for (int r = 0; r < CC_MAXR; ++r) {
            const uint32_t bal = __ballot_sync(0xffffffffu, rep == r);
            if ((tid & 31) == 0 && bal) atomicAdd(&s_cnt[r], __popc(bal));
        }
    }
    if (tid == 0) s_cont[batch] = 0;
    __syncthreads();
    if (tid == 0) {
        int off = 0;
        for (int r = 0; r < CC_MAXR; ++r) {
            s_goff[r] = off;
            s_run[r] = 0;
            off += (s_cnt[r] + CC_ROW_ALIGN - 1) / CC_ROW_ALIGN * CC_ROW_ALIGN;
        }
        s_goff[CC_MAXR] = off;
        s_ndec = 0;
        s_nchunk = 0;
        s_ntail = 0;
        s_pages = 0;
        s_pages_dec = 0;
    }
    __syncthreads();
    // ---- pass 2: grouped positions (stable), per-row tables, decode-row list with its page prefix ----
    for (int b0 = 0; b0 < batch; b0 += kGroupThreads) {
        const int b = b0 + tid;
        const int rep = b < batch ? s_rep[b] : -1;
        int pos = -1;
#pragma unroll
        for (int r = 0; r < CC_MAXR; ++r) {
            int tot;
            const int ex = block_scan_excl(rep == r ? 1 : 0, s_w, &tot);
            if (rep == r) pos = s_goff[r] + s_run[r] + ex;
            __syncthreads();
            if (tid == 0) s_run[r] += tot;
        }
        if (b < batch) {
            W.pos_of[b] = pos;
            if (pos >= 0) {
                const int p = seq_lens[b] - 1;
                W.perm[pos] = b;
                W.row_pos[pos] = p;
                W.row_page[pos] = block_table[(size_t)b * D.max_blocks + p / CC_PAGE];
                W.first_wr[b] = p / CC_PAGE;
                if (s_cont[b] && s_rep[b - 1] != rep) err |= CC_DEVERR_SPLIT_REQUEST;   // one request, two replicas
            }
        }
        // decode rows: live rows that neither continue a chunk nor start one
        const bool dec = rep >= 0 && !s_cont[b] && !s_cont[b + 1];
        const int npg = dec ? (seq_lens[b] + CC_PAGE - 1) / CC_PAGE : 0;
        int n_here, pg_here;
        const int di = block_scan_excl(dec ? 1 : 0, s_w, &n_here);
        const int pg = block_scan_excl(npg, s_w, &pg_here);
        if (dec) {
            const int i = s_ndec + di;
            if (i < CC_BIG_MAX_DEC) {
                W.dec_rows[i] = b;
                W.pg_prefix[i] = s_pages + pg;
                if (i == CC_BIG_MAX_DEC - 1 || (di == n_here - 1)) atomicMax(&s_pages_dec, s_pages + pg + npg);   // end of the list so far
            } else {
                err |= CC_DEVERR_TOO_MANY_DECODE;
            }
        }
        __syncthreads();
        if (tid == 0) {
            s_ndec += n_here;
            s_pages += pg_here;
        }
        __syncthreads();
    }
    // chunks: a head is a live row that does not continue a chunk but whose successor does; a tail is a row that
    // continues one and whose successor does not.  Runs are disjoint and ordered, so head c pairs with tail c.
    for (int b0 = 0; b0 < batch; b0 += kGroupThreads) {
        const int b = b0 + tid;
        const bool head = b < batch && s_rep[b] >= 0 && !s_cont[b] && s_cont[b + 1];
        const bool tail = b < batch && s_cont[b] && !s_cont[b + 1];
        int n_here, t_here;
        const int ci = block_scan_excl(head ? 1 : 0, s_w, &n_here);
        const int ti = block_scan_excl(tail ? 1 : 0, s_w, &t_here);
        if (head) {
            if (s_nchunk + ci < CC_BIG_MAX_CHUNKS) s_head[s_nchunk + ci] = b; else err |= CC_DEVERR_TOO_MANY_DECODE;
        }
        if (tail && s_ntail + ti < CC_BIG_MAX_CHUNKS) s_tail[s_ntail + ti] = b;
        __syncthreads();
        if (tid == 0) {
            s_nchunk += n_here;
            s_ntail += t_here;
        }
        __syncthreads();
    }
    if (err) atomicOr(W.err, err);
    const int n_chunks = min(s_nchunk, CC_BIG_MAX_CHUNKS);
    const int T = 128 / D.G;                                           // tokens of a query tile
    if (tid < n_chunks) {
        const int len = s_tail[tid] - s_head[tid] + 1;
        W.chunk_row0[tid] = s_head[tid];
        W.chunk_len[tid] = len;
        s_ntile[tid] = (len + T - 1) / T;
    }
    __syncthreads();
    // prefill work items (chunk, query tile): the late (long-prefix, expensive) tiles first.  Thread t owns tile index
    // j = jmax - 1 - t of every chunk that has one; a scan over t gives its items their places.
    int jmax = 0;
    for (int c = 0; c < n_chunks; ++c) jmax = max(jmax, s_ntile[c]);
    int n_items_tot = 0;
    for (int t0 = 0; t0 < jmax; t0 += kGroupThreads) {
        const int j = jmax - 1 - (t0 + tid);
        int cntj = 0;
        if (j >= 0)
            for (int c = 0; c < n_chunks; ++c) cntj += s_ntile[c] > j;
        int here;
        int at = n_items_tot + block_scan_excl(cntj, s_w, &here);
        if (j >= 0)
            for (int c = 0; c < n_chunks; ++c)
                if (s_ntile[c] > j) {
                    if (at < CC_BIG_MAX_ITEMS) {
                        W.item_chunk[at] = c;
                        W.item_tile[at] = j;
                    }
                    ++at;
                }
        n_items_tot += here;
        __syncthreads();
    }
    if (n_items_tot > CC_BIG_MAX_ITEMS && tid == 0) atomicOr(W.err, CC_DEVERR_TOO_MANY_DECODE);
    if (tid == 0) {
        const int n_dec = min(s_ndec, CC_BIG_MAX_DEC);
        const int n_items = min(n_items_tot, CC_BIG_MAX_ITEMS);
        // the page prefix of the unused decode slots = the total (k_attn reads CC_BIG_MAX_DEC + 1 entries)
        const int total = s_pages_dec;
        for (int i = n_dec; i <= CC_BIG_MAX_DEC; ++i) W.pg_prefix[i] = total;
        int nmax = 0;
        for (int r = 0; r < CC_MAXR; ++r) {
            W.sched->cnt[r] = s_cnt[r];
            W.sched->goff[r] = s_goff[r];
            nmax = max(nmax, (s_cnt[r] + CC_ROW_ALIGN - 1) / CC_ROW_ALIGN * CC_ROW_ALIGN);
        }
        W.sched->n_pos = s_goff[CC_MAXR];
        W.sched->n_items = total;
        W.sched->nmax = nmax;
        W.bs->n_dec = n_dec;
        W.bs->n_chunks = n_chunks;
        W.bs->n_items = n_items;
        W.bs->work = 0;
        W.bs->n_dec_pages = total;
    }
}

// a1 for large steps: one block per row, the grouped position comes from k_big_group.
constexpr int kNormThreads = 512;
__global__ void __launch_bounds__(kNormThreads) k_big_norm(const __nv_bfloat16* __restrict__ hidden, CcDims D,
                                                           const CcLayerTable* __restrict__ tab, CcWork W) {
    __shared__ float red[kNormThreads / 32];
    const int b = blockIdx.x;
    const int pos = W.pos_of[b];
    if (pos < 0) return;
    const int rep = replica_of_pos(W.sched->cnt, W.sched->goff, pos);
    const int nchunk = D.d >> 3;
    const uint4* row = reinterpret_cast<const uint4*>(hidden + (size_t)b * D.d);
    const uint4* g = reinterpret_cast<const uint4*>(tab->rep[rep].blob + D.off_g1);
    uint4 v[2], gv[2];
    float ss = 0.f;
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const int c = threadIdx.x + j * kNormThreads;
        v[j] = c < nchunk ? row[c] : make_uint4(0, 0, 0, 0);
        gv[j] = c < nchunk ? g[c] : make_uint4(0, 0, 0, 0);
        const uint32_t w[4] = {v[j].x, v[j].y, v[j].z, v[j].w};
#pragma unroll
        for (int i = 0; i < 4; ++i) ss += bf16lo(w[i]) * bf16lo(w[i]) + bf16hi(w[i]) * bf16hi(w[i]);
    }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = ss;
    __syncthreads();
    float t = 0.f;
    for (int i = 0; i < kNormThreads / 32; ++i) t += red[i];
    const float inv = rsqrtf(t / (float)D.d + D.eps);
#pragma unroll
    for (int j = 0; j < 2; ++j) {
        const int c = threadIdx.x + j * kNormThreads;
        if (c >= nchunk) break;
        const uint32_t w[4] = {v[j].x, v[j].y, v[j].z, v[j].w}, gw[4] = {gv[j].x, gv[j].y, gv[j].z, gv[j].w};
        float x[8];
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            x[2 * i] = bf16lo(w[i]) * inv * bf16lo(gw[i]);
            x[2 * i + 1] = bf16hi(w[i]) * inv * bf16hi(gw[i]);
        }
        act_store<8>(W.x_act, D, D.pl[CC_OP_X], pos, c << 3, x);
    }
    if (threadIdx.x == 0) W.inv_in[pos] = inv;
}

// a7 for large steps: scale of the gate/up epilogue = (1/rms of h1) / (1/rms of the input row); tile order fixed.
__global__ void __launch_bounds__(256) k_big_rowstat(CcDims D, CcWork W) {
    const int p = blockIdx.x * blockDim.x + threadIdx.x;
    if (p >= W.sched->n_pos) return;
    float s = 0.f;
    if (W.perm[p] >= 0) {
        float ss = 0.f;
        const int nt = (D.d + 127) >> 7;
        for (int t = 0; t < nt; ++t) ss += W.ssq[(size_t)t * D.Mpad + p];
        s = rsqrtf(ss / (float)D.d + D.eps) / W.inv_in[p];
    }
    W.gu_scale[p] = s;
}

}  // namespace

cudaError_t cc_launch_big_group(const int* assign, const int* seq_lens, const int* block_table, int batch, const CcDims& D,
                                const CcLayerTable* tab, const CcWork& W, cudaStream_t st) {
    k_big_group<<<1, kGroupThreads, 0, st>>>(assign, seq_lens, block_table, batch, D, tab, W);
    return cudaGetLastError();
}
cudaError_t cc_launch_big_norm(const __nv_bfloat16* hidden, int batch, const CcDims& D, const CcLayerTable* tab, const CcWork& W,
                               cudaStream_t st) {
    k_big_norm<<<batch, kNormThreads, 0, st>>>(hidden, D, tab, W);
    return cudaGetLastError();
}
cudaError_t cc_launch_big_rowstat(const CcDims& D, const CcWork& W, cudaStream_t st) {
    k_big_rowstat<<<(D.Mpad + 255) / 256, 256, 0, st>>>(D, W);
    return cudaGetLastError();
}
