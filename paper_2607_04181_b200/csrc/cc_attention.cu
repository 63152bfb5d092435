// cc_attention.cu -- paged GQA decode attention, split-KV (the KV cache
// partitioning the paper relies on: PAPER.md:103, 391, 476).
//
// HBM-bound: every cached K/V byte of a request is read exactly once per step.  Work item =
// (grouped row, kv head, chunk of 256 tokens = 16 pages); the G query heads that share the kv
// head are the (zero-padded) 16 rows of an mma.sync m16n8k16 tile, so one KV read serves the
// whole GQA group.  This is a memory kernel with M <= 8 real rows: the legacy warp-level
// tensor path is ample here (tcgen05 needs M >= 64), the design effort goes into the stream:
//   * each warp owns every 4th page of the chunk (w, w+4, ...) and a private ring of stages (one
//     stage = one K page + one V page of one kv head = 2 x 16 x Dh bf16) filled by TMA: one elected
//     lane issues cp.async.bulk.tensor boxes of 16 tokens x 128 bytes through a tensor map of the
//     caller's pool (built on the host per forward), completion on one mbarrier per stage; loads of
//     the next pages -- and of the next work item -- are in flight while a page is being used.
//     (The earlier per-lane 16-byte cp.async path topped out at 4.7 TB/s with the math removed.)
//   * the tensor map's 128-byte swizzle lands the rows so that the ldmatrix reads of the K
//     (B operand of q.K^T) and V (transposed B operand of p.V) fragments are conflict-free;
//   * softmax is online per warp (running max / sum in log2 units, fp32), the 4 warps of a CTA
//     are merged in fixed order through smem; the chunk partials of one (row, kv head) are merged
//     in chunk order by whichever CTA finishes that pair's last chunk (a counter per pair), so no
//     separate combine kernel runs.  The chunking depends on seq_len only and every merge order
//     is fixed => bit-identical across replicas, whatever CTA does the work.
//   * CTAs draw work items from a device counter (first item static), full chunks first and the
//     ragged last chunks at the end of the list, which evens out the tail of the kernel.
#include "cc_kernels.h"
#include <cuda.h>

namespace {

constexpr int kAttnWarps = 4;
constexpr int kAttnThreads = kAttnWarps * 32;
constexpr int kAttnStages = 3;
constexpr int kPagesPerChunk = CC_ATTN_CHUNK / CC_PAGE;       // 16
constexpr int kSlotsPerItem = kPagesPerChunk / kAttnWarps;    // 4 page slots per warp per item

template <int DH>
struct AttnCfg {
    static constexpr int kRowBytes = DH * 2;
    static constexpr int kPageBytes = CC_PAGE * kRowBytes;     // one K (or V) page of one kv head
    static constexpr int kStageBytes = 2 * kPageBytes;
    static constexpr int kMergeStride = DH + 2;                // floats per (warp, head): o[DH], m, l
    static size_t smem_bytes(int G) {
        return (size_t)kAttnWarps * kAttnStages * kStageBytes + (size_t)kAttnWarps * G * kMergeStride * 4 + 32 + (size_t)kAttnWarps * kAttnStages * 8;
    }
};

struct ItemMeta {
    int pos, chunk, b, s;     // s <= 0 marks "no item"
};

template <int DH>
__global__ void __launch_bounds__(kAttnThreads, 2)
k_attn(const int* __restrict__ seq_lens, CcKv kv, CcDims D, CcWork W, const CcLayerTable* __restrict__ tab,
       const __grid_constant__ CUtensorMap tmK, const __grid_constant__ CUtensorMap tmV) {
    using C = AttnCfg<DH>;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    const int warp = uniform((int)(threadIdx.x >> 5)), lane = threadIdx.x & 31;
    const int g = lane >> 2, t4 = lane & 3;
    uint8_t* ring = smem_raw + (size_t)warp * kAttnStages * C::kStageBytes;
    float* merge = reinterpret_cast<float*>(smem_raw + (size_t)kAttnWarps * kAttnStages * C::kStageBytes);
    const uint32_t ring_u32 = smem_u32(ring);

    int* s_seq = reinterpret_cast<int*>(merge + (size_t)kAttnWarps * D.G * C::kMergeStride);   // [4] item ids + [1] flag
    uint64_t* bars = reinterpret_cast<uint64_t*>(s_seq + 8) + warp * kAttnStages;              // "stage full", per warp
    if (lane == 0) {
#pragma unroll
        for (int i = 0; i < kAttnStages; ++i) mbar_init(&bars[i], 1);
        fence_mbar_init();
    }
    __syncwarp();
    pdl_wait();
    pdl_launch_dependents();

    const int G = D.G, Hkv = D.Hkv;
    const int n_total = W.sched->n_items * Hkv;
    // item sequence of this CTA: seq[0] = blockIdx.x, later ones from the counter; seq[n + 2] is drawn
    // while item n runs, so the loads of the next item can be in flight before the current one ends
    if (threadIdx.x == 0) {
        s_seq[0] = (int)blockIdx.x;
        s_seq[1] = (int)gridDim.x + atomicAdd(W.attn_ctr, 1);
    }
    __syncthreads();

    // ---- producer side: issue the cp.async copies of page slot k of this warp -------------------
    ItemMeta pm = {0, 0, 0, 0};
    int p_hk = 0, p_item = -1, p_page_id[2] = {0, 0};   // lane l holds the ids of pages l and l + 32 of the chunk
    static_assert(kPagesPerChunk <= 64, "two page ids per lane");
    auto prefetch = [&](int k) {
        const int it = k / kSlotsPerItem, i = k % kSlotsPerItem;
        if (it != p_item) {
            p_item = it;
            const int j = s_seq[it & 3];
            if (j >= n_total) {
                pm.s = 0;
                return;
            }
            const int base = j / Hkv;
            p_hk = j - base * Hkv;
            const int2 rec = W.items[base];
            pm.pos = rec.x;
            pm.chunk = rec.y;
            pm.b = W.perm[rec.x];
            pm.s = seq_lens[pm.b];
            const int n_row_pages = (pm.s + CC_PAGE - 1) / CC_PAGE;
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                const int pg = pm.chunk * kPagesPerChunk + lane + 32 * h;
                int id = 0;
                if (lane + 32 * h < kPagesPerChunk && pg < n_row_pages) {
                    id = kv.block_table[(size_t)pm.b * D.max_blocks + pg];
                    if (id < 0 || id >= kv.n_pages) {
                        atomicOr(W.err, CC_DEVERR_BAD_PAGE);
                        id = 0;
                    }
                }
                p_page_id[h] = id;
            }
        }
        const int pl = warp + i * kAttnWarps;                       // page within the chunk
        const int tok0 = pm.chunk * CC_ATTN_CHUNK + pl * CC_PAGE;   // first token of the page
        const int page0 = __shfl_sync(0xffffffffu, p_page_id[0], pl & 31), page1 = __shfl_sync(0xffffffffu, p_page_id[1], pl & 31);
        const int page = pl < 32 ? page0 : page1;
        // warp-uniform values + elect.sync keep the TMA issue on the uniform datapath (no per-lane waterfall)
        const int do_load = uniform((int)(tok0 < pm.s));
        const int row0 = uniform((page * Hkv + p_hk) * CC_PAGE);     // row of the pool seen as [pages*Hkv*16][DH]
        const int st = k % kAttnStages;
        if (do_load && elect_one()) {
            const uint32_t dstK = ring_u32 + (uint32_t)st * C::kStageBytes, dstV = dstK + C::kPageBytes;
            const uint32_t bar = smem_u32(&bars[st]);
            mbar_expect_tx(&bars[st], C::kStageBytes);
#pragma unroll
            for (int h = 0; h < DH / 64; ++h) {                       // boxes of 16 tokens x 64 dims (128 bytes)
                tma_load_2d(dstK + h * 2048, &tmK, h * 64, row0, bar);
                tma_load_2d(dstV + h * 2048, &tmV, h * 64, row0, bar);
            }
        }
    };

    for (int k = 0; k < kAttnStages - 1; ++k) prefetch(k);
    uint32_t phases = 0;                                   // bit st = parity of the next completion of stage st

    // ---- consumer state ----------------------------------------------------------------------
    ItemMeta cm = {0, 0, 0, 0};
    int c_hk = 0;
    uint32_t qa0[DH / 16], qa2[DH / 16];   // Q fragments (rows g < G), scaled by log2(e)/sqrt(Dh)
    float o[DH / 8][4];
    float m_run = -INFINITY, l_run = 0.f;

    int next_id = 0;                                       // thread 0: the id drawn for seq[it + 2]
    for (int k = 0;; ++k) {
        const int it = k / kSlotsPerItem, i = k % kSlotsPerItem;
        if (i == 0 && s_seq[it & 3] >= n_total) break;     // CTA-uniform: the list is exhausted
        prefetch(k + kAttnStages - 1);

        if (i == 0) {   // new item: metadata, Q fragments, reset the running softmax state
            if (threadIdx.x == 0) next_id = (int)gridDim.x + atomicAdd(W.attn_ctr, 1);
            const int j = s_seq[it & 3];
            const int base = j / Hkv;
            c_hk = j - base * Hkv;
            const int2 rec = W.items[base];
            cm.pos = rec.x;
            cm.chunk = rec.y;
            cm.b = W.perm[rec.x];
            cm.s = seq_lens[cm.b];
            const float* qrow = W.q_rot + (size_t)cm.pos * D.QD + (size_t)(c_hk * G + g) * DH;
#pragma unroll
            for (int ks = 0; ks < DH / 16; ++ks) {
                float2 x0 = make_float2(0.f, 0.f), x1 = make_float2(0.f, 0.f);
                if (g < G) {
                    x0 = *reinterpret_cast<const float2*>(qrow + ks * 16 + 2 * t4);
                    x1 = *reinterpret_cast<const float2*>(qrow + ks * 16 + 8 + 2 * t4);
                }
                qa0[ks] = pack_bf16(x0.x * D.qk_scale_log2, x0.y * D.qk_scale_log2);
                qa2[ks] = pack_bf16(x1.x * D.qk_scale_log2, x1.y * D.qk_scale_log2);
            }
#pragma unroll
            for (int nt = 0; nt < DH / 8; ++nt) o[nt][0] = o[nt][1] = o[nt][2] = o[nt][3] = 0.f;
            m_run = -INFINITY;
            l_run = 0.f;
        }

        const int pl = warp + i * kAttnWarps;
        const int tok0 = cm.chunk * CC_ATTN_CHUNK + pl * CC_PAGE;
        if (tok0 < cm.s) {
            const int valid = min(CC_PAGE, cm.s - tok0);
            const int st = k % kAttnStages;
            const uint32_t sK = ring_u32 + (uint32_t)st * C::kStageBytes;
            const uint32_t sV = sK + C::kPageBytes;
            mbar_wait(&bars[st], (phases >> st) & 1u);
            phases ^= 1u << st;
            if (valid < CC_PAGE) {   // ragged last page: the V rows past seq_len hold other data; p = 0 must meet 0
                for (int q = lane; q < (CC_PAGE - valid) * (DH / 8); q += 32) {
                    const int r = valid + q / (DH / 8), c = q % (DH / 8);
                    asm volatile("st.shared.v4.b32 [%0], {%1, %1, %1, %1};" ::"r"(sV + (c >> 3) * 2048 + r * 128 + ((c & 7) << 4)), "r"(0) : "memory");
                }
                fence_proxy_async_smem();   // a later TMA refill of this stage must not pass these stores
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
                    ldsm_x4(rowaddr + (uint32_t)((ch >> 3) * 2048 + (((ch & 7) ^ (tok & 7)) << 4)), r0, r1, r2, r3);
                    mma_bf16_16816(s0, qa0[ks], 0u, qa2[ks], 0u, r0, r1);
                    mma_bf16_16816(s1, qa0[ks], 0u, qa2[ks], 0u, r2, r3);
                }
            }
            // ---- online softmax on row g (tokens 2t,2t+1 and 8+2t,8+2t+1 of the page)
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
            const uint32_t pa0 = pack_bf16(p00, p01), pa2 = pack_bf16(p10, p11);
            // ---- O[16 x DH] = alpha * O + P[16 x 16] . V[16 x DH]
            {
                const int mi = lane >> 3, rr = lane & 7;
                const int tok = ((mi & 1) << 3) + rr;
                const uint32_t rowaddr = sV + (uint32_t)tok * 128;
#pragma unroll
                for (int jn = 0; jn < DH / 16; ++jn) {
                    const int ch = jn * 2 + (mi >> 1);
                    uint32_t r0, r1, r2, r3;
                    ldsm_x4_trans(rowaddr + (uint32_t)((ch >> 3) * 2048 + (((ch & 7) ^ (tok & 7)) << 4)), r0, r1, r2, r3);
                    o[2 * jn][0] *= alpha; o[2 * jn][1] *= alpha;
                    o[2 * jn + 1][0] *= alpha; o[2 * jn + 1][1] *= alpha;
                    mma_bf16_16816(o[2 * jn], pa0, 0u, pa2, 0u, r0, r1);
                    mma_bf16_16816(o[2 * jn + 1], pa0, 0u, pa2, 0u, r2, r3);
                }
            }
        }
        __syncwarp();   // all lanes are done with this stage before a later prefetch overwrites it

        if (i == kSlotsPerItem - 1) {
            // ---- merge the 4 warps of the CTA in fixed order, write the chunk partial
            float l_tot = l_run;
            l_tot += __shfl_xor_sync(0xffffffffu, l_tot, 1);
            l_tot += __shfl_xor_sync(0xffffffffu, l_tot, 2);
            if (g < G) {
                float* mrow = merge + (size_t)(warp * G + g) * C::kMergeStride;
#pragma unroll
                for (int nt = 0; nt < DH / 8; ++nt)
                    *reinterpret_cast<float2*>(mrow + nt * 8 + 2 * t4) = make_float2(o[nt][0], o[nt][1]);
                if (t4 == 0) {
                    mrow[DH] = m_run;
                    mrow[DH + 1] = l_tot;
                }
            }
            if (threadIdx.x == 0) s_seq[(it + 2) & 3] = next_id;
            __syncthreads();
            const int nch = (cm.s + CC_ATTN_CHUNK - 1) / CC_ATTN_CHUNK;     // CTA-uniform
            for (int e = 2 * threadIdx.x; e < G * DH; e += 2 * kAttnThreads) {
                const int hg = e / DH, dim = e - hg * DH;
                float M = -INFINITY;
#pragma unroll
                for (int w = 0; w < kAttnWarps; ++w) M = fmaxf(M, merge[(size_t)(w * G + hg) * C::kMergeStride + DH]);
                float a0 = 0.f, a1 = 0.f, L = 0.f;
#pragma unroll
                for (int w = 0; w < kAttnWarps; ++w) {
                    const float* mr = merge + (size_t)(w * G + hg) * C::kMergeStride;
                    const float sc = exp2f(mr[DH] - M);
                    a0 += sc * mr[dim];
                    a1 += sc * mr[dim + 1];
                    L += sc * mr[DH + 1];
                }
                const int hq = c_hk * G + hg;
                if (nch == 1) {   // the only chunk of this row: normalise and write the O-projection operand
                    const float inv = 1.f / L;
                    const int col = hq * DH + dim;
                    uint8_t* dst = W.o_act + act_chunk_off(cm.pos, col, D.Mpad, 1, 0) + (col & 7) * 2;
                    *reinterpret_cast<uint32_t*>(dst) = pack_bf16(a0 * inv, a1 * inv);
                } else {
                    const size_t row = ((size_t)cm.pos * D.Hq + hq) * W.nch_max + cm.chunk;
                    *reinterpret_cast<float2*>(W.att_o + row * DH + dim) = make_float2(a0, a1);
                    if (dim == 0) W.att_ml[row] = make_float2(M, L);
                }
            }
            if (nch > 1) {
                // ---- the CTA that finishes the pair's last chunk merges all of them, in chunk order
                __threadfence();
                __syncthreads();
                if (threadIdx.x == 0) {
                    int* cnt = W.attn_cnt + cm.pos * Hkv + c_hk;
                    const int last = atomicAdd(cnt, 1) == nch - 1;
                    if (last) *cnt = 0;                             // ready for the next step
                    s_seq[4] = last;
                }
                __syncthreads();
                if (s_seq[4]) {
                    __threadfence();
                    for (int e = 2 * threadIdx.x; e < G * DH; e += 2 * kAttnThreads) {
                        const int hg = e / DH, dim = e - hg * DH, hq = c_hk * G + hg;
                        const size_t row = ((size_t)cm.pos * D.Hq + hq) * W.nch_max;
                        float M = -INFINITY;
                        for (int c = 0; c < nch; ++c) M = fmaxf(M, __ldcg(&W.att_ml[row + c]).x);
                        float L = 0.f, a0 = 0.f, a1 = 0.f;
                        for (int c = 0; c < nch; ++c) {
                            const float2 ml = __ldcg(&W.att_ml[row + c]);
                            const float w = exp2f(ml.x - M);
                            const float2 ov = __ldcg(reinterpret_cast<const float2*>(W.att_o + (row + c) * DH + dim));
                            L += w * ml.y;
                            a0 += w * ov.x;
                            a1 += w * ov.y;
                        }
                        const float inv = 1.f / L;
                        const int col = hq * DH + dim;
                        uint8_t* dst = W.o_act + act_chunk_off(cm.pos, col, D.Mpad, 1, 0) + (col & 7) * 2;
                        *reinterpret_cast<uint32_t*>(dst) = pack_bf16(a0 * inv, a1 * inv);
                    }
                }
            }
            __syncthreads();   // merge buffer and flags are reused by the next item
        }
    }
    // out of items: warm L2 with the head of the O-projection weight stream of the first non-empty group
    if (threadIdx.x == 0) {
        int r0 = 0;
        while (r0 < CC_MAXR - 1 && W.sched->cnt[r0] == 0) ++r0;
        cc_prefetch_gemm_head(D.o, tab->rep[r0].blob, (int)blockIdx.x);
    }
}

}  // namespace

cudaError_t cc_attn_configure() {
    cudaError_t e = cudaFuncSetAttribute(k_attn<128>, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024);
    if (e != cudaSuccess) return e;
    return cudaFuncSetAttribute(k_attn<64>, cudaFuncAttributeMaxDynamicSharedMemorySize, 112 * 1024);
}

// Tensor map of a caller-owned KV pool seen as a 2-D bf16 tensor [n_pages * Hkv * 16 rows][Dh], boxes of
// 16 rows x 64 elements (128 bytes) with the 128-byte swizzle.  cuTensorMapEncodeTiled is a driver entry
// point; it is looked up once through the runtime, so the library needs no link against libcuda.
static cudaError_t make_kv_tensor_map(CUtensorMap* out, const void* pool, int n_pages, int Hkv, int Dh) {
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
    const cuuint32_t box[2] = {64, CC_PAGE};
    const cuuint32_t estr[2] = {1, 1};
    const CUresult r = encode(out, CU_TENSOR_MAP_DATA_TYPE_BFLOAT16, 2, const_cast<void*>(pool), dims, strides, box, estr,
                              CU_TENSOR_MAP_INTERLEAVE_NONE, CU_TENSOR_MAP_SWIZZLE_128B, CU_TENSOR_MAP_L2_PROMOTION_L2_256B,
                              CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    return r == CUDA_SUCCESS ? cudaSuccess : cudaErrorInvalidValue;
}

cudaError_t cc_launch_attention(const int* seq_lens, const CcKv& kv, const CcDims& D, const CcLayerTable* tab,
                                const CcWork& W, const CcLaunch& L) {
    CUtensorMap tmK, tmV;
    cudaError_t e = make_kv_tensor_map(&tmK, kv.k_pool, kv.n_pages, D.Hkv, D.Dh);
    if (e == cudaSuccess) e = make_kv_tensor_map(&tmV, kv.v_pool, kv.n_pages, D.Hkv, D.Dh);
    if (e != cudaSuccess) return e;
    const dim3 grid(2 * L.n_sms), block(kAttnThreads);
    if (D.Dh == 128)
        return cc_launch_kernel(k_attn<128>, grid, block, AttnCfg<128>::smem_bytes(D.G), L, seq_lens, kv, D, W, tab, tmK, tmV);
    return cc_launch_kernel(k_attn<64>, grid, block, AttnCfg<64>::smem_bytes(D.G), L, seq_lens, kv, D, W, tab, tmK, tmV);
}
