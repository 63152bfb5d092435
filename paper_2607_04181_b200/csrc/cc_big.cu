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

// exclusive prefix of v over the block (all threads call); *total = sum.  v may pack several counters in bit fields
// that cannot carry into one another.  Two levels of shuffles: the warps' totals are scanned by warp 0.
__device__ __forceinline__ unsigned long long block_scan_excl(unsigned long long v, unsigned long long* s_w, unsigned long long* total) {
    const int lane = threadIdx.x & 31, w = threadIdx.x >> 5;
    unsigned long long inc = v;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) {
        const unsigned long long t = __shfl_up_sync(0xffffffffu, inc, o);
        if (lane >= o) inc += t;
    }
    __syncthreads();                                                   // the previous call's readers are done with s_w
    if (lane == 31) s_w[w] = inc;
    __syncthreads();
    if (w == 0) {
        static_assert(kGroupThreads == 1024, "one warp total per lane");
        unsigned long long x = s_w[lane];
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned long long t = __shfl_up_sync(0xffffffffu, x, o);
            if (lane >= o) x += t;
        }
        s_w[lane] = x;
    }
    __syncthreads();
    *total = s_w[kGroupThreads / 32 - 1];
    return (w ? s_w[w - 1] : 0ull) + inc - v;
}

__global__ void __launch_bounds__(kGroupThreads) k_big_group(const int* __restrict__ assign, const int* __restrict__ seq_lens,
                                                             const int* __restrict__ block_table, int batch, CcDims D,
                                                             const CcLayerTable* __restrict__ tab, CcWork W) {
    __shared__ signed char s_rep[CC_BIG_MAX_ROWS];
    __shared__ unsigned char s_cont[CC_BIG_MAX_ROWS + 1];     // row b continues the chunk of row b - 1
    __shared__ unsigned long long s_w[kGroupThreads / 32];
    __shared__ int s_cnt[CC_MAXR], s_goff[CC_MAXR + 1];
    __shared__ int s_pages_dec;
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
    // Every global read of the grouping is issued up front, eight rows per thread (a row at a time, the dependent reads of the
    // three passes cost ~30 memory latencies: 60-90 us of a step): the row's and its predecessor's seq_len, replica and
    // first page id now, the page its token is appended to once the seq_len is there.
    constexpr int kIt = CC_BIG_MAX_ROWS / kGroupThreads;
    int seqv[kIt], repv[kIt], lpv[kIt];
    bool contv[kIt];
    {
        int asg[kIt], fpv[kIt], seqp[kIt], asgp[kIt], fpp[kIt];
#pragma unroll
        for (int k = 0; k < kIt; ++k) {
            const int b = k * kGroupThreads + tid;
            const bool in = b < batch, inp = in && b > 0;
            seqv[k] = in ? seq_lens[b] : 0;
            asg[k] = in ? assign[b] : 0;
            fpv[k] = in ? block_table[(size_t)b * D.max_blocks] : -1;
            seqp[k] = inp ? seq_lens[b - 1] : 0;
            asgp[k] = inp ? assign[b - 1] : 0;
            fpp[k] = inp ? block_table[(size_t)(b - 1) * D.max_blocks] : -2;
        }
#pragma unroll
        for (int k = 0; k < kIt; ++k) {
            const int b = k * kGroupThreads + tid;
            repv[k] = b < batch ? cc_row_replica_of(seqv[k], asg[k], D, mask, err) : -1;
            uint32_t e2 = 0;                                           // (row b - 1 reports its own errors)
            contv[k] = repv[k] >= 0 && b > 0 && cc_row_replica_of(seqp[k], asgp[k], D, mask, e2) >= 0 && seqv[k] == seqp[k] + 1 &&
                       fpv[k] == fpp[k];
            lpv[k] = repv[k] >= 0 ? block_table[(size_t)b * D.max_blocks + (seqv[k] - 1) / CC_PAGE] : -1;
        }
    }
    // ---- pass 1: the replica of every row, chunk continuation flags, rows per replica ----
#pragma unroll
    for (int k = 0; k < kIt; ++k) {
        const int b = k * kGroupThreads + tid;
        if (k * kGroupThreads >= batch) break;
        const int rep = repv[k];
        if (b < batch) {
            s_rep[b] = (signed char)rep;
            s_cont[b] = contv[k] ? 1 : 0;
        }
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
            off += (s_cnt[r] + CC_ROW_ALIGN - 1) / CC_ROW_ALIGN * CC_ROW_ALIGN;
        }
        s_goff[CC_MAXR] = off;
        s_pages_dec = 0;
    }
    __syncthreads();
    // ---- pass 2: grouped positions (stable), per-row tables, decode-row list with its page prefix ----
    // (every thread keeps the running totals: the scans hand the iteration's totals to all)
    int run[CC_MAXR] = {0, 0, 0, 0}, n_dec_run = 0, pages_run = 0;
#pragma unroll
    for (int k = 0; k < kIt; ++k) {
        if (k * kGroupThreads >= batch) break;
        const int b = k * kGroupThreads + tid;
        const int rep = repv[k];
        int pos = -1;
        {   // rank among the rows of the same replica: the four counters of an iteration (<= 1024 each) in 16-bit fields
            unsigned long long tot;
            const unsigned long long ex = block_scan_excl(rep >= 0 ? 1ull << (16 * rep) : 0ull, s_w, &tot);
            if (rep >= 0) pos = s_goff[rep] + run[rep] + (int)((ex >> (16 * rep)) & 0xffffull);
#pragma unroll
            for (int r = 0; r < CC_MAXR; ++r) run[r] += (int)((tot >> (16 * r)) & 0xffffull);
        }
        if (b < batch) {
            W.pos_of[b] = pos;
            if (pos >= 0) {
                const int p = seqv[k] - 1;
                W.perm[pos] = b;
                W.row_pos[pos] = p;
                W.row_page[pos] = lpv[k];
                W.first_wr[b] = p / CC_PAGE;
                if (s_cont[b] && s_rep[b - 1] != rep) err |= CC_DEVERR_SPLIT_REQUEST;   // one request, two replicas
            }
        }
        // decode rows: live rows that neither continue a chunk nor start one; their count (low 16 bits) and pages together
        const bool dec = rep >= 0 && !s_cont[b] && !s_cont[b + 1];
        const int npg = dec ? (seqv[k] + CC_PAGE - 1) / CC_PAGE : 0;
        unsigned long long dtot;
        const unsigned long long dex = block_scan_excl((dec ? 1ull : 0ull) | ((unsigned long long)npg << 16), s_w, &dtot);
        const int di = (int)(dex & 0xffffull), pg = (int)(dex >> 16), n_here = (int)(dtot & 0xffffull);
        if (dec) {
            const int i = n_dec_run + di;
            if (i < CC_BIG_MAX_DEC) {
                W.dec_rows[i] = b;
                W.pg_prefix[i] = pages_run + pg;
                if (i == CC_BIG_MAX_DEC - 1 || (di == n_here - 1)) atomicMax(&s_pages_dec, pages_run + pg + npg);   // end of the list so far
            } else {
                err |= CC_DEVERR_TOO_MANY_DECODE;
            }
        }
        n_dec_run += n_here;
        pages_run += (int)(dtot >> 16);
    }
    // chunks: a head is a live row that does not continue a chunk but whose successor does; a tail is a row that
    // continues one and whose successor does not.  Runs are disjoint and ordered, so head c pairs with tail c.
    int n_chunk_run = 0, n_tail_run = 0;
    for (int b0 = 0; b0 < batch; b0 += kGroupThreads) {
        const int b = b0 + tid;
        const bool head = b < batch && s_rep[b] >= 0 && !s_cont[b] && s_cont[b + 1];
        const bool tail = b < batch && s_cont[b] && !s_cont[b + 1];
        unsigned long long tot;
        const unsigned long long ex = block_scan_excl((head ? 1ull : 0ull) | (tail ? 1ull << 16 : 0ull), s_w, &tot);
        const int ci = (int)(ex & 0xffffull), ti = (int)(ex >> 16);
        if (head) {
            if (n_chunk_run + ci < CC_BIG_MAX_CHUNKS) s_head[n_chunk_run + ci] = b; else err |= CC_DEVERR_TOO_MANY_DECODE;
        }
        if (tail && n_tail_run + ti < CC_BIG_MAX_CHUNKS) s_tail[n_tail_run + ti] = b;
        n_chunk_run += (int)(tot & 0xffffull);
        n_tail_run += (int)(tot >> 16);
    }
    __syncthreads();
    if (err) atomicOr(W.err, err);
    const int n_chunks = min(n_chunk_run, CC_BIG_MAX_CHUNKS);
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
        unsigned long long here64;
        int at = n_items_tot + (int)block_scan_excl((unsigned long long)cntj, s_w, &here64);
        const int here = (int)here64;
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
        const int n_dec = min(n_dec_run, CC_BIG_MAX_DEC);
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
