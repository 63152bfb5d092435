// cc_attention.cu -- paged GQA decode attention, split-KV (the KV cache
// partitioning the paper relies on: PAPER.md:103, 391, 476).
//
// HBM-bound: every cached K/V byte of a request is read exactly once per step.  What was measured on
// the way here: per-(page, head) 4 KiB requests from four warps
// per CTA, by per-lane cp.async or by small TMA boxes alike, stream at 4.7 TB/s even with the math
// removed, and the ragged end of a 256-token work list costs another ~9 us; whole pages (all kv
// heads, 2 x 32 KiB contiguous) staged by one producer warp stream at 5.3 TB/s, 6.1 TB/s with an L2
// evict-first policy, and a static equal split of the page axis removes the ragged end.  Hence:
//   * the work axis is the list of KV pages of the whole batch (rows in request order); it is cut
//     into equal contiguous ranges, one per persistent CTA (one CTA per SM), so every CTA streams
//     the same number of bytes (+- one page) whatever the context lengths are.  A row that spans
//     several ranges is split there ("pieces"); the split is a function of the batch only, never
//     of the replica assignment;
//   * a producer warp stages whole pages by TMA: one cp.async.bulk.tensor box of
//     (Hkv * 16 rows) x 128 bytes per half page through a tensor map of the caller's pool (built
//     on the host per forward), 128-byte swizzle, into a ring of 64 KiB stages (K + V of 8 / Hkv
//     pages), "full" mbarrier per stage, "empty" mbarrier released by the consumers;
//   * eight consumer warps: warp w owns kv head w % Hkv of page w / Hkv of the stage.  The G query
//     heads that share a kv head are the (zero-padded) 16 rows of an mma.sync m16n8k16 tile, so
//     one KV read serves the whole GQA group.  (M <= 8 real rows: the warp-level tensor path is
//     ample; tcgen05 needs M >= 64.)  ldmatrix reads of the swizzled rows are conflict-free;
//   * softmax is online per warp (running max / sum in log2 units, fp32).  At the end of a chunk
//     piece the warps that share a kv head (Hkv < 8) are merged in fixed order through smem; the
//     piece partials of one (row, kv head) are merged in piece order by the warp that finishes the
//     pair's last piece (a counter per pair), so no separate combine kernel runs.  Every merge
//     order is fixed => bit-identical across replicas, whatever CTA finishes last.
//   * KV loads carry an L2 evict-first policy (measured: +12 % stream rate; the data is used once).
#include "cc_kvmaps.h"

namespace {

constexpr int kCW = 8;                                  // consumer warps
constexpr int kAttnThreads = (kCW + 1) * 32;            // + the producer warp (warp kCW)
constexpr int kAttnStages = 3;
constexpr int kBarMerge = 1;                            // named barrier of the consumer warps

enum { kMetaFirst = 1, kMetaLast = 2, kMetaEnd = 4 };
struct StageMeta {          // written by the producer before it arms the stage's "full" barrier
    int pos;                // grouped position of the row (Q, outputs)
    int s;                  // its seq_len
    int flags;              // kMetaFirst / kMetaLast group of the piece, kMetaEnd
    int pg;                 // index (within the row) of the stage's first page
    int slot;               // partial-result slot of this piece = row + CTA
    int slot0, n_pieces;    // the row's pieces are slots slot0 .. slot0 + n_pieces - 1
    int n_in;               // pages of the piece in this stage (<= pages per stage)
};

template <int DH>
struct AttnCfg {
    static constexpr int kUnitBytes = CC_PAGE * DH * 2;            // K (or V) of one (page, kv head)
    static constexpr int kStageBytes = 2 * kCW * kUnitBytes;       // K + V of kCW (page, head) units
    static constexpr int kMergeStride = DH + 4;                    // floats per (warp, q head): o[DH], m, l, pad (16-byte rows)
    static constexpr size_t kCtrlBytes = kAttnStages * sizeof(StageMeta) + 2 * kAttnStages * 8 + 260 * 4;
    static size_t smem_bytes(int G) {
        return (size_t)kAttnStages * kStageBytes + (size_t)kCW * G * kMergeStride * 4 + kCtrlBytes;
    }
};

template <int DH>
__global__ void __launch_bounds__(kAttnThreads, 1)
k_attn(const int* __restrict__ seq_lens, CcKv kv, CcDims D, CcWork W, const CcLayerTable* __restrict__ tab,
       const int* __restrict__ rowmap, const __grid_constant__ CcKvMaps maps) {
    using C = AttnCfg<DH>;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const int warp = uniform((int)(threadIdx.x >> 5)), lane = threadIdx.x & 31;
    const int G = D.G, Hkv = D.Hkv;
    const int PPS = kCW / Hkv;                                     // pages per stage
    float* merge = reinterpret_cast<float*>(smem_raw + (size_t)kAttnStages * C::kStageBytes);
    StageMeta* meta = reinterpret_cast<StageMeta*>(merge + (size_t)kCW * G * C::kMergeStride);
    uint64_t* full = reinterpret_cast<uint64_t*>(meta + kAttnStages);
    uint64_t* empty = full + kAttnStages;
    const uint32_t ring_u32 = smem_u32(smem_raw);
    // stage layout: [page of the stage][K | V][half of Dh (64 dims = 128 bytes)][Hkv * 16 rows][128 B]
    const uint32_t half_bytes = (uint32_t)Hkv * CC_PAGE * 128u;
    const uint32_t kv_bytes = half_bytes * (DH / 64);              // K (or V) of one page, all heads
    const uint32_t page_bytes = 2u * kv_bytes;

    if (threadIdx.x == 0) {
        for (int i = 0; i < kAttnStages; ++i) {
            mbar_init(&full[i], 1);
            mbar_init(&empty[i], kCW);
        }
        fence_mbar_init();
    }
    __syncthreads();
    // The grouping tables (k_prologue) were complete two kernels back, seq_lens and the block table are
    // inputs: only q and the K/V of the token being decoded come from the predecessor (the QKV GEMM).
    // So the producer starts streaming the OLD pages at once -- while the predecessor's CTAs on other
    // SMs are still in their fixup -- and waits for it only before the first stage that holds a page
    // this step appends to (the last page of a lone row; for the rows of a prompt chunk the lowest page
    // any of them writes: W.first_wr from the prologue); the consumers wait before they read q.
    if (threadIdx.x == 0) CC_TP(W, 1, 0);
    pdl_launch_dependents();
    const int T = W.sched->n_items;                               // KV pages of the batch
    int* s_prefix = reinterpret_cast<int*>(empty + kAttnStages);  // [max_batch + 1]
    for (int i = threadIdx.x; i <= D.max_batch; i += kAttnThreads) s_prefix[i] = W.pg_prefix[i];
    __syncthreads();

    if (warp == kCW) {
        // ===================== producer: whole pages by TMA =====================
        // CTAs in use: every one of them gets at least one page, so the CTAs that share a row are consecutive
        const long long n_cta = min((int)gridDim.x, max(T, 1));
        auto cta_of_page = [&](int x) { return (int)((((long long)x + 1) * n_cta - 1) / T); };   // inverse of the cut
        const bool idle = (long long)blockIdx.x >= n_cta;
        const int P0 = idle ? 0 : (int)((long long)T * blockIdx.x / n_cta);
        const int P1 = idle ? 0 : (int)((long long)T * (blockIdx.x + 1) / n_cta);
        const uint64_t pol = policy_evict_first();
        int stage = 0;
        uint32_t ph = 0;
        bool waited = false;
        int b = 0;
        if (P0 < P1) {                                            // row that holds page P0
            int cntb = 0;
            for (int i = lane; i < D.max_batch; i += 32) cntb += (s_prefix[i + 1] <= P0);
#pragma unroll
            for (int sft = 16; sft > 0; sft >>= 1) cntb += __shfl_xor_sync(0xffffffffu, cntb, sft);
            b = cntb;
        }
        int p = P0;
        while (p < P1) {
            const int r0 = s_prefix[b], r1 = s_prefix[b + 1];
            if (r1 <= p) { ++b; continue; }                       // rows without pages (padding)
            const int q0 = p - r0, q1 = min(r1, P1) - r0;         // this CTA's pages of row b
            // large steps: the work axis runs over the decode rows only, b indexes that list (k_big_group)
            const int rb = rowmap ? rowmap[b] : b;
            const int pos = W.pos_of[rb], s = seq_lens[rb], first_wr = W.first_wr[rb];
            const int rep = replica_of_pos(W.sched->cnt, W.sched->goff, pos);   // whose KV partition the row's pages are in
            const CUtensorMap* tmK = &maps.k[rep];
            const CUtensorMap* tmV = &maps.v[rep];
            const int n_pool_pages = kv.n_pages_r[rep];
            const int slot0 = b + cta_of_page(r0), n_pieces = cta_of_page(r1 - 1) - cta_of_page(r0) + 1;
            const int slot = b + (int)blockIdx.x;
            const int n_groups = (q1 - q0 + PPS - 1) / PPS;
            int id = 0, id_base = -32;                            // lane l: id of page q0 + id_base + l of the row
            for (int g = 0; g < n_groups; ++g) {
                const int rel = g * PPS, qg = q0 + rel;           // first page of the group
                if (rel >= id_base + 32) {                        // next 32 page ids (32 % PPS == 0: groups never straddle)
                    id_base = rel;
                    const int q = qg + lane;
                    id = 0;
                    if (q < q1) {
                        id = kv.block_table[(size_t)rb * D.max_blocks + q];
                        if (id < 0 || id >= n_pool_pages) {
                            atomicOr(W.err, CC_DEVERR_BAD_PAGE);
                            id = 0;
                        }
                    }
                }
                mbar_wait(&empty[stage], ph ^ 1);
                const int in_grp = min(PPS, q1 - qg);
                if (!waited && qg + in_grp > first_wr) {          // the stage holds a page this step appends to
                    pdl_wait();
                    waited = true;
                }
                int pid[kCW];
#pragma unroll
                for (int pp = 0; pp < kCW; ++pp) pid[pp] = __shfl_sync(0xffffffffu, id, (rel - id_base + pp) & 31);
                if (elect_one()) {
                    StageMeta m;
                    m.pos = pos; m.s = s; m.pg = qg; m.slot = slot; m.slot0 = slot0; m.n_pieces = n_pieces; m.n_in = in_grp;
                    m.flags = (g == 0 ? kMetaFirst : 0) | (g == n_groups - 1 ? kMetaLast : 0);
                    meta[stage] = m;
                    mbar_expect_tx(&full[stage], (uint32_t)in_grp * page_bytes);
                    const uint32_t bar = smem_u32(&full[stage]);
                    const uint32_t dst0 = ring_u32 + (uint32_t)stage * C::kStageBytes;
#pragma unroll
                    for (int pp = 0; pp < kCW; ++pp) {
                        if (pp < in_grp) {
                            const int row0 = pid[pp] * Hkv * CC_PAGE;  // the pool seen as [pages * Hkv * 16 rows][DH]
                            const uint32_t dst = dst0 + (uint32_t)pp * page_bytes;
#pragma unroll
                            for (int h = 0; h < DH / 64; ++h) {
                                tma_load_2d_hint(dst + h * half_bytes, tmK, h * 64, row0, bar, pol);
                                tma_load_2d_hint(dst + kv_bytes + h * half_bytes, tmV, h * 64, row0, bar, pol);
                            }
                        }
                    }
                }
                if (++stage == kAttnStages) { stage = 0; ph ^= 1; }
            }
            p = r0 + q1;
            ++b;
        }
        // my pages are on their way; the consumers still work on them: the first weight stages of the O projection's CTAs go
        // to L2 meanwhile (small steps on the cluster GEMMs only: D.pf_next)
        if (D.pf_next > 0) {
            const uint8_t* blobs[CC_MAXR];
#pragma unroll
            for (int r = 0; r < CC_MAXR; ++r) blobs[r] = tab->rep[r].blob;
            cc_prefetch_weights(D.o, blobs, W.sched->cnt, (int)blockIdx.x, (int)gridDim.x, 0, D.pf_next, lane);
        }
        // end marker for the consumers
        if (!waited) pdl_wait();
        mbar_wait(&empty[stage], ph ^ 1);
        if (elect_one()) {
            meta[stage].flags = kMetaEnd;
            mbar_arrive(&full[stage]);
        }
        return;
    }

    // ===================== consumers: warp w = kv head w % Hkv of page w / Hkv of the stage =====================
    const int h = warp % Hkv, pp = warp / Hkv;
    const int g = lane >> 2, t4 = lane & 3;
    float* my_merge = merge + (size_t)warp * G * C::kMergeStride;
    int stage = 0;
    uint32_t ph = 0;
    // Q fragments, scaled by log2(e)/sqrt(Dh), as bf16 hi + lo (q = hi + lo to ~16 bits): row g < G of the 16-row mma
    // tile carries hi, row g + 8 carries lo (G <= 8 leaves the upper eight rows free), so ONE mma.sync yields both
    // partial products and their sum is exact to ~16 bits against the bf16 K; the probabilities are split the same
    // way against the bf16 V.  With single bf16 planes the attention output carried a 2e-3 relative error, at SHORT
    // contexts (|o| ~ 0.4) the largest error of the whole layer: single output elements of 16-token rows at the
    // cfg2 layer shape sat on the tolerance (tests/test_gpu_long.py).
    uint32_t qa0[DH / 16], qa2[DH / 16], ql0[DH / 16], ql2[DH / 16];
    float o[DH / 8][4];
    float m_run = -INFINITY, l_run = 0.f;
#pragma unroll
    for (int nt = 0; nt < DH / 8; ++nt) o[nt][0] = o[nt][1] = o[nt][2] = o[nt][3] = 0.f;
    pdl_wait();                                         // q (and the new K/V) come from the QKV GEMM
    if (threadIdx.x == 32) CC_TP(W, 1, 1);

    for (;;) {
        mbar_wait(&full[stage], ph);
        const StageMeta m = meta[stage];
        if (m.flags & kMetaEnd) {
            if (threadIdx.x == 32) CC_TP(W, 1, 2);
            break;
        }
        if (m.flags & kMetaFirst) {   // new item: Q fragments, reset the running softmax state
            const float* qrow = W.q_rot + (size_t)m.pos * D.QD + (size_t)(h * G + g) * DH;
#pragma unroll
            for (int ks = 0; ks < DH / 16; ++ks) {
                float2 x0 = make_float2(0.f, 0.f), x1 = make_float2(0.f, 0.f);
                if (g < G) {
                    x0 = *reinterpret_cast<const float2*>(qrow + ks * 16 + 2 * t4);
                    x1 = *reinterpret_cast<const float2*>(qrow + ks * 16 + 8 + 2 * t4);
                }
                x0.x *= D.qk_scale_log2; x0.y *= D.qk_scale_log2; x1.x *= D.qk_scale_log2; x1.y *= D.qk_scale_log2;
                qa0[ks] = pack_bf16(x0.x, x0.y);
                qa2[ks] = pack_bf16(x1.x, x1.y);
                ql0[ks] = pack_bf16(x0.x - bf16lo(qa0[ks]), x0.y - bf16hi(qa0[ks]));
                ql2[ks] = pack_bf16(x1.x - bf16lo(qa2[ks]), x1.y - bf16hi(qa2[ks]));
            }
        }
        const int tok0 = (m.pg + pp) * CC_PAGE;
        if (pp < m.n_in) {   // (then tok0 < s: the piece only holds pages of the context)
            const int valid = min(CC_PAGE, m.s - tok0);
            const uint32_t sK = ring_u32 + (uint32_t)stage * C::kStageBytes + (uint32_t)pp * page_bytes + (uint32_t)h * 2048u;
            const uint32_t sV = sK + kv_bytes;
            if (valid < CC_PAGE) {   // ragged last page: the V rows past seq_len hold other data; p = 0 must meet 0
                for (int q = lane; q < (CC_PAGE - valid) * (DH / 8); q += 32) {
                    const int r = valid + q / (DH / 8), c = q % (DH / 8);
                    asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(sV + (c >> 3) * half_bytes + r * 128 + ((c & 7) << 4)), "r"(0) : "memory");
                }
                fence_proxy_async_smem();   // the TMA refill of this stage must not pass these stores
                __syncwarp();
            }
            // ---- scores: S[16 x 16] = Q[16 x DH] . K^T
            float s0[4] = {0.f, 0.f, 0.f, 0.f}, s1[4] = {0.f, 0.f, 0.f, 0.f};
            {
                const int mi = lane >> 3, rr = lane & 7;
                const int tok = ((mi >> 1) << 3) + rr;
                const uint32_t rowaddr = sK + (uint32_t)tok * 128;
#pragma unroll
                for (int ks = 0; ks < DH / 16; ++ks) {
                    const int ch = ks * 2 + (mi & 1);
                    uint32_t r0, r1, r2, r3;
                    ldsm_x4(rowaddr + (uint32_t)(ch >> 3) * half_bytes + (uint32_t)(((ch & 7) ^ (tok & 7)) << 4), r0, r1, r2, r3);
                    mma_bf16_16816(s0, qa0[ks], ql0[ks], qa2[ks], ql2[ks], r0, r1);   // c[0..1]: hi . K, c[2..3]: lo . K
                    mma_bf16_16816(s1, qa0[ks], ql0[ks], qa2[ks], ql2[ks], r2, r3);
                }
            }
            // ---- online softmax on row g (tokens 2t,2t+1 and 8+2t,8+2t+1 of the page)
            s0[0] += s0[2]; s0[1] += s0[3]; s1[0] += s1[2]; s1[1] += s1[3];   // hi + lo rows of q
            const int c0 = 2 * t4;
            float v00 = (c0 < valid) ? s0[0] : -INFINITY, v01 = (c0 + 1 < valid) ? s0[1] : -INFINITY;
            float v10 = (c0 + 8 < valid) ? s1[0] : -INFINITY, v11 = (c0 + 9 < valid) ? s1[1] : -INFINITY;
            float pmax = fmaxf(fmaxf(v00, v01), fmaxf(v10, v11));
            pmax = fmaxf(pmax, __shfl_xor_sync(0xffffffffu, pmax, 1));
            pmax = fmaxf(pmax, __shfl_xor_sync(0xffffffffu, pmax, 2));
            const float m_new = fmaxf(m_run, pmax);        // finite: token 0 of the page is valid
            const float alpha = exp2f(m_run - m_new);
            const float p00 = exp2f(v00 - m_new), p01 = exp2f(v01 - m_new);
            const float p10 = exp2f(v10 - m_new), p11 = exp2f(v11 - m_new);
            l_run = l_run * alpha + ((p00 + p01) + (p10 + p11));
            m_run = m_new;
            const uint32_t pa0 = pack_bf16(p00, p01), pa2 = pack_bf16(p10, p11);   // probabilities: bf16 hi (rows g) + lo (rows g + 8)
            const uint32_t pl0 = pack_bf16(p00 - bf16lo(pa0), p01 - bf16hi(pa0)), pl2 = pack_bf16(p10 - bf16lo(pa2), p11 - bf16hi(pa2));
            // ---- O[16 x DH] = alpha * O + P[16 x 16] . V[16 x DH]
            {
                const int mi = lane >> 3, rr = lane & 7;
                const int tok = ((mi & 1) << 3) + rr;
                const uint32_t rowaddr = sV + (uint32_t)tok * 128;
#pragma unroll
                for (int jn = 0; jn < DH / 16; ++jn) {
                    const int ch = jn * 2 + (mi >> 1);
                    uint32_t r0, r1, r2, r3;
                    ldsm_x4_trans(rowaddr + (uint32_t)(ch >> 3) * half_bytes + (uint32_t)(((ch & 7) ^ (tok & 7)) << 4), r0, r1, r2, r3);
                    o[2 * jn][0] *= alpha; o[2 * jn][1] *= alpha; o[2 * jn][2] *= alpha; o[2 * jn][3] *= alpha;
                    o[2 * jn + 1][0] *= alpha; o[2 * jn + 1][1] *= alpha; o[2 * jn + 1][2] *= alpha; o[2 * jn + 1][3] *= alpha;
                    mma_bf16_16816(o[2 * jn], pa0, pl0, pa2, pl2, r0, r1);             // c[0..1] += hi . V, c[2..3] += lo . V
                    mma_bf16_16816(o[2 * jn + 1], pa0, pl0, pa2, pl2, r2, r3);
                }
            }
        }
        __syncwarp();                                  // every lane is done with the stage
        if (lane == 0) mbar_arrive(&empty[stage]);
        if (++stage == kAttnStages) { stage = 0; ph ^= 1; }
        if (!(m.flags & kMetaLast)) continue;

        // ---------------- end of the chunk: merge, write the partial (or the final operand) ----------------
        float l_tot = l_run;
        l_tot += __shfl_xor_sync(0xffffffffu, l_tot, 1);
        l_tot += __shfl_xor_sync(0xffffffffu, l_tot, 2);
        if (g < G) {
            float* mrow = my_merge + (size_t)g * C::kMergeStride;
#pragma unroll
            for (int nt = 0; nt < DH / 8; ++nt)
                *reinterpret_cast<float2*>(mrow + nt * 8 + 2 * t4) = make_float2(o[nt][0] + o[nt][2], o[nt][1] + o[nt][3]);
            if (t4 == 0) {
                mrow[DH] = m_run;
                mrow[DH + 1] = l_tot;
            }
        }
        // the accumulators are dead now: reset them here, so that nothing of the chunk loop stays live
        // through the code below (the next stage of this warp starts a new item)
#pragma unroll
        for (int nt = 0; nt < DH / 8; ++nt) o[nt][0] = o[nt][1] = o[nt][2] = o[nt][3] = 0.f;
        m_run = -INFINITY;
        l_run = 0.f;
        if (PPS > 1) named_bar_sync(kBarMerge, kCW * 32); else __syncwarp();
        // the first warp of each kv head combines the PPS warps of that head (fixed order); from here on
        // lane l owns dims 4l .. 4l+3 of every q head of the group
        const int dim = lane * 4;
        const int nch = m.n_pieces;
        auto store_operand = [&](int q, float4 v, float inv) {   // row of the O-projection operand, in the layer's operand format
            const float x[4] = {v.x * inv, v.y * inv, v.z * inv, v.w * inv};
            act_store<4>(W.o_act, D, D.pl[CC_OP_O], m.pos, (h * G + q) * DH + dim, x);
        };
        if (pp == 0 && dim < DH) {
#pragma unroll 1
            for (int q = 0; q < G; ++q) {
                float M = -INFINITY;
                for (int p = 0; p < PPS; ++p) M = fmaxf(M, merge[(size_t)((h + p * Hkv) * G + q) * C::kMergeStride + DH]);
                float4 a = make_float4(0.f, 0.f, 0.f, 0.f);
                float L = 0.f;
                for (int p = 0; p < PPS; ++p) {
                    const float* mr = merge + (size_t)((h + p * Hkv) * G + q) * C::kMergeStride;
                    const float sc = exp2f(mr[DH] - M);
                    const float4 v = *reinterpret_cast<const float4*>(mr + dim);
                    a.x += sc * v.x; a.y += sc * v.y; a.z += sc * v.z; a.w += sc * v.w;
                    L += sc * mr[DH + 1];
                }
                if (nch == 1) {   // the only chunk of this row: normalise and write the operand
                    store_operand(q, a, 1.f / L);
                } else {
                    const size_t row = (size_t)m.slot * D.Hq + h * G + q;
                    *reinterpret_cast<float4*>(W.att_o + row * DH + dim) = a;
                    if (lane == 0) W.att_ml[row] = make_float2(M, L);
                }
            }
        }
        if (PPS > 1) named_bar_sync(kBarMerge, kCW * 32); else __syncwarp();   // merge rows may be rewritten
        if (pp != 0 || nch == 1) continue;
        // ---- the warp that finishes the pair's last piece merges all of them, in piece order
        __syncwarp();
        int last = 0;
        if (lane == 0) {
            __threadfence();                                    // cumulative over the warp's partial stores (ordered by the __syncwarp)
            int* cnt = W.attn_cnt + m.pos * Hkv + h;
            last = atomicAdd(cnt, 1) == nch - 1;
            if (last) *cnt = 0;                                 // ready for the next step
        }
        last = __shfl_sync(0xffffffffu, last, 0);
        if (!last) continue;
        __threadfence();
        for (int q0 = 0; q0 < G; q0 += 4) {                         // four q heads x two chunks in flight
            size_t row[4];
            float M[4], L[4];
            float4 a[4];
#pragma unroll
            for (int u = 0; u < 4; ++u) {
                row[u] = (size_t)m.slot0 * D.Hq + h * G + min(q0 + u, G - 1);   // piece c of the row: + c * Hq
                M[u] = -INFINITY; L[u] = 0.f; a[u] = make_float4(0.f, 0.f, 0.f, 0.f);
            }
            for (int c = lane; c < nch; c += 32) {
#pragma unroll
                for (int u = 0; u < 4; ++u) M[u] = fmaxf(M[u], __ldcg(&W.att_ml[row[u] + (size_t)c * D.Hq]).x);
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
#pragma unroll
                for (int sft = 16; sft > 0; sft >>= 1) M[u] = fmaxf(M[u], __shfl_xor_sync(0xffffffffu, M[u], sft));
            for (int c0 = 0; c0 < nch; c0 += 2) {               // added in piece order
                float2 ml[4][2];
                float4 v[4][2];
#pragma unroll
                for (int u = 0; u < 4; ++u)
#pragma unroll
                    for (int cc = 0; cc < 2; ++cc) {
                        const bool ok = c0 + cc < nch;
                        ml[u][cc] = ok ? __ldcg(&W.att_ml[row[u] + (size_t)(c0 + cc) * D.Hq]) : make_float2(-INFINITY, 0.f);
                        v[u][cc] = (ok && dim < DH) ? __ldcg(reinterpret_cast<const float4*>(W.att_o + (row[u] + (size_t)(c0 + cc) * D.Hq) * DH + dim))
                                                    : make_float4(0.f, 0.f, 0.f, 0.f);
                    }
#pragma unroll
                for (int u = 0; u < 4; ++u)
#pragma unroll
                    for (int cc = 0; cc < 2; ++cc) {
                        const float w = exp2f(ml[u][cc].x - M[u]);
                        L[u] += w * ml[u][cc].y;
                        a[u].x += w * v[u][cc].x; a[u].y += w * v[u][cc].y; a[u].z += w * v[u][cc].z; a[u].w += w * v[u][cc].w;
                    }
            }
#pragma unroll
            for (int u = 0; u < 4; ++u)
                if (q0 + u < G && dim < DH) store_operand(q0 + u, a[u], 1.f / L[u]);
        }
    }
}

}  // namespace

cudaError_t cc_attn_configure() {
    cudaError_t e = cudaFuncSetAttribute(k_attn<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AttnCfg<128>::smem_bytes(8));
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_attn<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)AttnCfg<64>::smem_bytes(8));
}

// Tensor map of a caller-owned KV pool seen as a 2-D bf16 tensor [n_pages * Hkv * 16 rows][Dh], boxes of
// box_rows rows (one page of all kv heads: Hkv * 16; one page of one head: 16) x 64 elements (128 bytes) with the 128-byte swizzle.  cuTensorMapEncodeTiled is
// a driver entry point; it is looked up once through the runtime, so the library needs no link against libcuda.
cudaError_t cc_make_kv_tensor_map(CUtensorMap* out, const void* pool, int n_pages, int Hkv, int Dh, int box_rows) {
    typedef CUresult (*EncodeFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                 const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                 CUtensorMapL2promotion, CUtensorMapFloatOOBfill);
    static EncodeFn encode = nullptr;
    if (!encode) {
        void* fn = nullptr;
        cudaDriverEntryPointQueryResult qr;
        cudaError_t e = cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &fn, cudaEnableDefault, &qr);
        if (e != cudaSuccess) return e;
        if (qr != cudaDriverEntryPointSuccess || !fn) return cudaErrorNotSupported;
        encode = (EncodeFn)fn;
    }
    const cuuint64_t dims[2] = {(cuuint64_t)Dh, (cuuint64_t)n_pages * Hkv * CC_PAGE};
    const cuuint64_t strides[1] = {(cuuint64_t)Dh * 2};
    const cuuint32_t box[2] = {64, (cuuint32_t)box_rows};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(pool), dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t cc_launch_attention(const int* seq_lens, const CcKv& kv, const CcDims& D, const CcLayerTable* tab,
                                const CcWork& W, const CcLaunch& L, const int* rowmap) {
    CcKvMaps maps;
    cudaError_t e = cc_make_kv_maps(&maps, kv, D.Hkv, D.Dh, D.Hkv * CC_PAGE);
    if (e != cudaSuccess) return e;
    const dim3 grid(L.n_sms), block(kAttnThreads);
    if (D.Dh == 128)
        return cc_launch_kernel(k_attn<128>, grid, block, AttnCfg<128>::smem_bytes(D.G), L, seq_lens, kv, D, W, tab, rowmap, maps);
    return cc_launch_kernel(k_attn<64>, grid, block, AttnCfg<64>::smem_bytes(D.G), L, seq_lens, kv, D, W, tab, rowmap, maps);
}

// One descriptor pair per replica; replicas that share a pool share the encoding.
cudaError_t cc_make_kv_maps(CcKvMaps* out, const CcKv& kv, int Hkv, int Dh, int box_rows) {
    for (int r = 0; r < CC_MAXR; ++r) {
        int same = -1;
        for (int q = 0; q < r; ++q)
            if (kv.k_pool_r[q] == kv.k_pool_r[r] && kv.v_pool_r[q] == kv.v_pool_r[r] && kv.n_pages_r[q] == kv.n_pages_r[r]) same = q;
        if (same >= 0) {
            out->k[r] = out->k[same];
            out->v[r] = out->v[same];
            continue;
        }
        cudaError_t e = cc_make_kv_tensor_map(&out->k[r], kv.k_pool_r[r], kv.n_pages_r[r], Hkv, Dh, box_rows);
        if (e == cudaSuccess) e = cc_make_kv_tensor_map(&out->v[r], kv.v_pool_r[r], kv.n_pages_r[r], Hkv, Dh, box_rows);
        if (e != cudaSuccess) return e;
    }
    return cudaSuccess;
}
