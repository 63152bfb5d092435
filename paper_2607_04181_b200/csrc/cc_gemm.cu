// cc_gemm.cu -- the weight-streaming projection GEMM of the replicated decoder layer (sm_100a).
//
// SURVEY.md 8(a) rows a2 (QKV), a6 (O), a8 (gate/up), a9 (down); replica indirection row a10.
// Decode is HBM-bound: every weight byte is read once per replica group, so the kernel is built
// around the weight stream, not around the MMA:
//   * swap-AB: a packed weight tile (128 output features x 64 k, a 16 KiB pre-swizzled image
//     made once at cc_create_layer) is the tcgen05 A operand (M = 128); the activations of one
//     replica group (n rows, n = multiple of 16, <= 256) are the B operand (N = n): one fp16 plane
//     against fp16 weight images, or two bf16 planes hi + lo that are both multiplied into the
//     same accumulator against bf16 images (CcDims::fmt).
//   * CC_G = 2 adjacent tiles form a super tile: one pipeline stage = the two weight atoms of
//     one k-block (32 KiB, contiguous in the blob, one bulk copy) + the activation slab of that
//     k-block (both planes, one bulk copy), feeding two fp32 accumulators D[128][n] in TMEM
//     (double-buffered while 2 * CC_G * n <= 512 columns).
//   * one persistent CTA per SM, stream-K: the (super tile, k-block) units are cut into P
//     contiguous ranges fixed by the layer shape (cc_common.cuh); CTA i streams range i of
//     EVERY active replica's blob, whose base it reads from the device replica table at run
//     time (PAPER.md:391-393 re-captures a graph when the replica set changes; here nothing does).
//   * warp 0 = producer: 1-D bulk copies (TMA engine, no tensor map) into a ring of smem stages
//     guarded by mbarriers; warp 1 = MMA issuer (one elected thread, tcgen05.commit frees the
//     stage); warps 2..5 = epilogue (tcgen05.ld -> fp32 partials in global memory).
//   * stream-K fixup inside the kernel: when a CTA has streamed its whole range it signals a
//     per-super-tile counter; the m CTAs that share a super tile then each add up the m fp32
//     partials ("pieces", fixed order 0..m-1) of every m-th row and apply the fused epilogue of
//     the projection (RoPE + KV append | residual + norm statistics + operand packing | SwiGLU |
//     residual + write-back in request order), so no separate reduce kernel runs between GEMMs.
#include "cc_epilogue.cuh"
#include <cstdio>

namespace {

constexpr int kGemmThreads = 512;         // warp 0 producer, 1 MMA, 2..5 TMEM epilogue, 6..15 row tables; all 16 in the fixup
constexpr int kHdrBytes = 8192;           // barriers + per-row tables in front of the stage ring
constexpr int kMaxStages = 5;            // deeper rings do not stream faster (measured again in round 2: 5 stages no change, 6 stages slower at R = 4)
constexpr int kGemmSmem = 225 * 1024;     // dynamic shared memory per CTA
constexpr int kTmemCols = 512;
constexpr uint32_t kWStage = CC_G * CC_A_TILE_BYTES;   // weight bytes per stage (32 KiB)

struct GemmSmemHdr {                      // lives at the start of dynamic smem
    uint64_t full[12];                    // kMaxStages (k_gemm, two-tile k_gemm_cl) or kClMaxStages (one-tile k_gemm_cl) in use
    uint64_t empty[12];
    uint64_t tmem_full[2];
    uint64_t tmem_empty[2];
    uint32_t tmem_base;
    int cnt[CC_MAXR];
    int goff[CC_MAXR];
    const uint8_t* blob[CC_MAXR];
    __nv_bfloat16* kpool[CC_MAXR];        // the KV pools replica r's rows append to (its partition, else the call's pools)
    __nv_bfloat16* vpool[CC_MAXR];
    int kvpages[CC_MAXR];
    int perm[CC_MAX_MPAD];                // original row at grouped position, or -1
    int aux[CC_MAX_MPAD];                 // QKV: position s-1; O: bits of 1/rms of the input row; gate/up: bits of rms_in/rms of h1
    int page[CC_MAX_MPAD];                // QKV: page that holds position s-1, or -1
};
static_assert(sizeof(GemmSmemHdr) <= kHdrBytes, "header does not fit");

// per-row tables of the fused epilogues, held in shared memory (built by the helper warps)
struct SmemTab {
    const GemmSmemHdr* H;
    __device__ __forceinline__ int aux(int p) const { return H->aux[p]; }
    __device__ __forceinline__ int page(int p) const { return H->page[p]; }
    __device__ __forceinline__ const uint8_t* blob(int p) const { return H->blob[replica_of_pos(H->cnt, H->goff, p)]; }
    __device__ __forceinline__ __nv_bfloat16* k_pool(int p) const { return H->kpool[replica_of_pos(H->cnt, H->goff, p)]; }
    __device__ __forceinline__ __nv_bfloat16* v_pool(int p) const { return H->vpool[replica_of_pos(H->cnt, H->goff, p)]; }
    __device__ __forceinline__ int kv_pages(int p) const { return H->kvpages[replica_of_pos(H->cnt, H->goff, p)]; }
};

// Slice of the fixup of super tile `st` done by contributor k of m: rows k, k + m, ... of both tiles.
// KI items (row, tile) per warp iteration, QU pieces of each loaded per round trip (KI * QU loads in
// flight per lane); pieces are added in the order 0..m-1 whatever KI and QU are.
template <int KIND, int KI, int QU>
__device__ __forceinline__ void fixup_tile(const float* __restrict__ part, const CcEpi& E, const CcDims& D, const CcWork& W,
                                           const GemmSmemHdr* H, int st, int c0, int m, int k, int n_pos, int warp,
                                           int lane) {
    constexpr int kWarps = kGemmThreads / 32;
    const int Mpad = D.Mpart;
    const int my_rows = (n_pos - k + m - 1) / m;
    const int n_items = my_rows * CC_G;
    const size_t piece_stride = (size_t)CC_G * Mpad * 128;     // floats between consecutive pieces of a tile
    for (int it0 = warp * KI; it0 < n_items; it0 += kWarps * KI) {
        const float* src[KI];
        int pp[KI], bb[KI], tt[KI];
        float4 acc[KI];
        EpiPre pre[KI];
#pragma unroll
        for (int u = 0; u < KI; ++u) {
            const int it = it0 + u;
            const int row = it / CC_G, j = it - row * CC_G;
            pp[u] = k + row * m;
            tt[u] = st * CC_G + j;
            bb[u] = (it < n_items) ? H->perm[pp[u]] : -1;
            src[u] = part + ((size_t)((c0 + st) * CC_G + j) * Mpad + pp[u]) * 128 + 4 * lane;
            acc[u] = make_float4(0.f, 0.f, 0.f, 0.f);
            if (bb[u] >= 0) epi_pre<KIND>(pre[u], E, D, W, SmemTab{H}, tt[u], pp[u], bb[u], lane);
        }
        for (int q0 = 0; q0 < m; q0 += QU) {
            float4 v[KI][QU];
#pragma unroll
            for (int u = 0; u < KI; ++u)
#pragma unroll
                for (int qq = 0; qq < QU; ++qq)
                    v[u][qq] = (bb[u] >= 0 && q0 + qq < m)
                                   ? __ldcg(reinterpret_cast<const float4*>(src[u] + (size_t)(q0 + qq) * piece_stride))
                                   : make_float4(0.f, 0.f, 0.f, 0.f);
#pragma unroll
            for (int u = 0; u < KI; ++u)
#pragma unroll
                for (int qq = 0; qq < QU; ++qq) {
                    acc[u].x += v[u][qq].x; acc[u].y += v[u][qq].y; acc[u].z += v[u][qq].z; acc[u].w += v[u][qq].w;
                }
        }
#pragma unroll
        for (int u = 0; u < KI; ++u)
            if (bb[u] >= 0) epi_fin<KIND>(pre[u], E, D, W, SmemTab{H}, tt[u], pp[u], bb[u], acc[u], lane);   // warp-uniform branch
    }
}

__device__ __forceinline__ int ld_acquire(const int* p) {
    int v;
    asm volatile("ld.acquire.gpu.global.s32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}

template <int KIND>
__global__ void __launch_bounds__(kGemmThreads, 1)
k_gemm(CcGemmGeo G, const uint8_t* __restrict__ act, float* __restrict__ part, int* __restrict__ flags,
       CcEpi E, CcDims D, CcWork W, const CcLayerTable* __restrict__ tab) {
    const int planes = D.pl[KIND];             // operand of projection KIND: x, o, y, a
    const CcSched* __restrict__ sched = W.sched;
    const int Mpad = D.Mpad;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    GemmSmemHdr* H = reinterpret_cast<GemmSmemHdr*>(smem_raw);
    const int warp = uniform((int)(threadIdx.x >> 5)), lane = threadIdx.x & 31;

    if (threadIdx.x == 0) CC_TP(W, 2 + KIND, 0);
    // ---- one-time setup (independent of the previous kernel: overlaps its tail under PDL) ----
    if (threadIdx.x == 0) {
        for (int i = 0; i < kMaxStages; ++i) {
            mbar_init(&H->full[i], 1);
            mbar_init(&H->empty[i], 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&H->tmem_full[i], 1);
            mbar_init(&H->tmem_empty[i], 4);
        }
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc<kTmemCols>(&H->tmem_base);
    // The replica table was written long ago; the grouping tables (k_prologue) were complete two kernels
    // back for every projection but the first: the QKV GEMM starts while k_prologue may still be running
    // (programmatic dependent launch), so it counts the groups from the inputs itself -- the same rule,
    // cc_row_replica -- to know which replica's weights to stream first and how wide the row groups are.
    if (KIND == EPI_QKV) {
        int* wcnt = H->aux;                                   // [8 warps][CC_MAXR], free until the helper warps run
        if (threadIdx.x < 256) {
            uint32_t err = 0;
            const int rep = cc_row_replica(E.assign, E.seq_lens, threadIdx.x, E.batch, D, tab->active_mask, err);
#pragma unroll
            for (int r = 0; r < CC_MAXR; ++r) {
                const uint32_t bal = __ballot_sync(0xffffffffu, rep == r);
                if (lane == 0) wcnt[warp * CC_MAXR + r] = __popc(bal);
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int off = 0;
            for (int r = 0; r < CC_MAXR; ++r) {
                int c = 0;
                for (int w = 0; w < 8; ++w) c += wcnt[w * CC_MAXR + r];
                H->cnt[r] = c;
                H->goff[r] = off;
                off += (c + CC_ROW_ALIGN - 1) / CC_ROW_ALIGN * CC_ROW_ALIGN;
            }
        }
        if (threadIdx.x < CC_MAXR) {
            const CcReplicaRow rr = tab->rep[threadIdx.x];
            H->blob[threadIdx.x] = rr.blob;
            H->kpool[threadIdx.x] = rr.k_pool ? (__nv_bfloat16*)rr.k_pool : E.kv.k_pool;
            H->vpool[threadIdx.x] = rr.k_pool ? (__nv_bfloat16*)rr.v_pool : E.kv.v_pool;
            H->kvpages[threadIdx.x] = rr.k_pool ? rr.n_pages : E.kv.n_pages;
        }
    } else if (threadIdx.x < CC_MAXR) {
        H->cnt[threadIdx.x] = sched->cnt[threadIdx.x];
        H->goff[threadIdx.x] = sched->goff[threadIdx.x];
        H->blob[threadIdx.x] = tab->rep[threadIdx.x].blob;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    int nmax = 0;
#pragma unroll
    for (int r = 0; r < CC_MAXR; ++r) nmax = max(nmax, (H->cnt[r] + CC_ROW_ALIGN - 1) / CC_ROW_ALIGN * CC_ROW_ALIGN);
    nmax = uniform(nmax);
    const uint32_t act_bytes_max = (uint32_t)planes * (uint32_t)nmax * 128u;   // nmax % 16 == 0 => multiple of 2 KiB
    const uint32_t stage_bytes = kWStage + act_bytes_max;
    uint8_t* stage0 = smem_raw + kHdrBytes;                 // barriers and row tables live in front of the ring
    int n_stages = (kGemmSmem - kHdrBytes) / (int)stage_bytes;
    if (n_stages > kMaxStages) n_stages = kMaxStages;
    // TMEM: accumulator (buf, j) at column buf * 256 + j * acc_cols; one buffer only when the two
    // accumulators of a super tile need more than 256 columns
    const uint32_t nbuf_log2 = nmax <= 128 ? 1u : 0u;
    const uint32_t acc_cols = nmax <= 128 ? 128u : 256u;

    const long long u_begin = cc_range_begin(G, blockIdx.x), u_end = cc_range_begin(G, blockIdx.x + 1);
    const uint32_t tmem_base = uniform(H->tmem_base);

    const int kb_begin = (int)(u_begin % G.KB);
    if (nmax > 0 && u_begin < u_end) {
        // Producer and MMA issuer: the whole warp walks the (warp-uniform) unit loop and one lane
        // issues; every per-unit quantity is carried incrementally (no division, no 64-bit
        // multiply inside the loops) -- the single issuing thread is the critical path of a
        // weight-streaming kernel.
        if (warp == 0) {
            // ===================== producer =====================
            // Weights do not depend on the previous kernel: the ring is filled with weight atoms
            // first (mode 0), then the kernel waits for its predecessor, adds the activation
            // slabs of those stages and carries on (mode 1), so the HBM stream restarts while
            // the small kernel between two GEMMs is still running.
            const uint64_t pol_w = policy_evict_first();   // weights: used once
            const uint64_t pol_a = policy_evict_last();    // activation slabs: re-read by every CTA, keep them in L2
            const size_t kb_stride = (size_t)(Mpad >> 3) * planes * 1024;   // bytes between k-blocks of the operand
            const long long per_rep = u_end - u_begin;
            int n_act = 0;
            for (int r = 0; r < CC_MAXR; ++r) n_act += uniform(H->cnt[r]) > 0;
            const long long total = per_rep * n_act;
            const int n_pre = total < n_stages ? (int)total : n_stages;
            auto run = [&](const int mode) {
                int stage = 0;
                uint32_t ph = 0;
                uint8_t* sW = stage0;
                long long idx = 0;
                for (int r = 0; r < CC_MAXR; ++r) {
                    const int cnt = uniform(H->cnt[r]);
                    if (cnt == 0) continue;
                    const uint32_t nb = (uint32_t)((cnt + 15) & ~15) * 128u * (uint32_t)planes;   // bytes of one slab
                    const uint32_t tx = kWStage + nb;
                    const uint8_t* wsrc = uniform(H->blob[r]) + G.w_off + (size_t)u_begin * kWStage;
                    const uint8_t* abase = act + (size_t)(uniform(H->goff[r]) >> 3) * planes * 1024;
                    const uint8_t* asrc = abase + (size_t)kb_begin * kb_stride;
                    int kb = kb_begin;
                    for (long long u = u_begin; u < u_end; ++u, ++idx) {
                        if (mode == 0 && idx >= n_pre) return;
                        const bool pre = idx < n_pre;            // stage already holds its weights
                        if (mode == 1 && !pre) mbar_wait(&H->empty[stage], ph ^ 1);
                        if (elect_one()) {
                            if (mode == 0 || !pre) {
                                mbar_expect_tx(&H->full[stage], tx);
                                bulk_g2s_hint(sW, wsrc, kWStage, &H->full[stage], pol_w);
                            }
                            if (mode == 1) bulk_g2s_hint(sW + kWStage, asrc, nb, &H->full[stage], pol_a);
                        }
                        wsrc += kWStage;
                        asrc += kb_stride;
                        if (++kb == G.KB) { kb = 0; asrc = abase; }
                        sW += stage_bytes;
                        if (++stage == n_stages) { stage = 0; ph ^= 1; sW = stage0; }
                    }
                }
            };
            run(0);
            pdl_wait();
            if (lane == 0) CC_TP(W, 2 + KIND, 1);
            __syncwarp();
            if (elect_one()) pdl_launch_dependents();
            run(1);
            if (lane == 0) CC_TP(W, 2 + KIND, 2);
            __syncwarp();
        } else if (warp == 1) {
            // ===================== MMA issuer =====================
            int stage = 0;
            uint32_t ph = 0;
            uint32_t pc = 0;   // super-tile pieces started so far
            const uint32_t a_hi = (uint32_t)(umma_desc_sw128(0) >> 32);
            const uint32_t b_hi = (uint32_t)(umma_desc_sw128(0, (uint32_t)planes * 1024u) >> 32);
            const uint32_t desc_lo0 = (uint32_t)umma_desc_sw128(smem_u32(stage0));
            const uint32_t dstage = stage_bytes >> 4, dact = kWStage >> 4;
            uint32_t da = desc_lo0;
            for (int r = 0; r < CC_MAXR; ++r) {
                const int cnt = uniform(H->cnt[r]);
                if (cnt == 0) continue;
                const uint32_t idesc = umma_idesc_m128((uint32_t)((cnt + 15) & ~15), D.fmt);
                int kb = kb_begin;
                bool first = true;
                for (long long u = u_begin; u < u_end; ++u) {
                    const bool last = (u == u_end - 1) || kb == G.KB - 1;
                    const uint32_t buf = pc & nbuf_log2;
                    if (first) {
                        mbar_wait(&H->tmem_empty[buf], ((pc >> nbuf_log2) & 1) ^ 1);
                        tc_fence_after();
                    }
                    mbar_wait(&H->full[stage], ph);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t db = da + dact;
#pragma unroll
                        for (int j = 0; j < CC_G; ++j) {
                            const uint32_t d_tmem = tmem_base + buf * 256 + (uint32_t)j * acc_cols;
                            const uint32_t daj = da + (uint32_t)j * (CC_A_TILE_BYTES >> 4);
#pragma unroll
                            for (int k = 0; k < CC_TILE_K / 16; ++k) {
                                umma_bf16_lo(d_tmem, daj + 2 * k, db + 2 * k, a_hi, b_hi, idesc, (first && k == 0) ? 0u : 1u);
                                if (planes == 2) umma_bf16_lo(d_tmem, daj + 2 * k, db + 64 + 2 * k, a_hi, b_hi, idesc, 1u);
                            }
                        }
                        umma_commit(&H->empty[stage]);
                        if (last) umma_commit(&H->tmem_full[buf]);
                    }
                    __syncwarp();
                    first = last;
                    if (last) ++pc;
                    if (++kb == G.KB) kb = 0;
                    da += dstage;
                    if (++stage == n_stages) { stage = 0; ph ^= 1; da = desc_lo0; }
                }
            }
        } else if (warp < 6) {
            // ===================== epilogue: TMEM -> fp32 partial pieces =====================
            const int q = warp & 3;                          // TMEM lane quarter this warp may read
            const int f = q * 32 + lane;                     // output feature within the tile
            uint32_t pc = 0;
            for (int r = 0; r < CC_MAXR; ++r) {
                const int cnt = H->cnt[r];
                if (cnt == 0) continue;
                const int n = (cnt + 15) & ~15;
                const int goff = H->goff[r];
                long long u = u_begin;
                while (u < u_end) {
                    const int st = (int)(u / G.KB);
                    long long u_next = (long long)(st + 1) * G.KB;
                    if (u_next > u_end) u_next = u_end;
                    const uint32_t buf = pc & nbuf_log2;
                    mbar_wait(&H->tmem_full[buf], (pc >> nbuf_log2) & 1);
                    tc_fence_after();
#pragma unroll
                    for (int j = 0; j < CC_G; ++j) {
                        float* dst = part + ((size_t)((blockIdx.x + st) * CC_G + j) * D.Mpart + goff) * 128 + f;
                        const uint32_t tcol = tmem_base + ((uint32_t)(q * 32) << 16) + buf * 256 + (uint32_t)j * acc_cols;
                        for (int c = 0; c < n; c += 16) {
                            uint32_t v[16];
                            tmem_ld_32x32b_x16(tcol + c, v);
                            tmem_ld_wait();
#pragma unroll
                            for (int i = 0; i < 16; ++i)
                                if (c + i < cnt) dst[(size_t)(c + i) * 128] = __uint_as_float(v[i]);
                        }
                    }
                    tc_fence_before();
                    __syncwarp();
                    if (lane == 0) mbar_arrive(&H->tmem_empty[buf]);
                    ++pc;
                    u = u_next;
                }
            }
        } else {
            // ===================== helper warps: per-row tables of the fused epilogue =====================
            // built while the weights stream; the rows' statistics come from the previous kernel
            pdl_wait();
            const int n_pos = sched->n_pos;
            for (int p = (int)threadIdx.x - 6 * 32; p < n_pos; p += kGemmThreads - 6 * 32) {
                const int b = W.perm[p];
                H->perm[p] = b;
                if (KIND == EPI_QKV) {
                    int pos = -1, page = -1;
                    if (b >= 0) {
                        pos = E.seq_lens[b] - 1;
                        page = E.kv.block_table[(size_t)b * D.max_blocks + pos / CC_PAGE];
                    }
                    H->aux[p] = pos;
                    H->page[p] = page;
                } else if (KIND == EPI_GU) {
                    float ss = 0.f;
                    if (b >= 0) {
                        const int nt = (D.d + 127) >> 7;
                        for (int t = 0; t < nt; ++t) ss += W.ssq[(size_t)t * Mpad + p];   // tile order: fixed
                    }
                    H->aux[p] = __float_as_int(b >= 0 ? rsqrtf(ss / (float)D.d + D.eps) / W.inv_in[p] : 0.f);
                } else if (KIND == EPI_O) {
                    H->aux[p] = __float_as_int(b >= 0 ? W.inv_in[p] : 0.f);
                }
            }
        }
    }
    // (the partial sums of this CTA become visible GPU-wide through thread 0's fence below: the block barrier
    // orders every warp's stores before it, and the fence is cumulative -- a fence in every thread cost each
    // warp a MEMBAR.ALL.GPU on the kernel's tail)
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<kTmemCols>(tmem_base);
    if (threadIdx.x == 0) CC_TP(W, 2 + KIND, 3);
    if (nmax == 0) {
        // No row runs this step.  The chain's ordering argument ("what was written two kernels back is visible") needs
        // every kernel to retire after its predecessor, so wait for it here as well.
        pdl_wait();
        return;
    }

    // ---- stream-K fixup: the CTAs c0..c1 whose ranges meet in a super tile split its rows ----------
    // Every reduction below adds pieces 0..m-1 in that order, whatever CTA does it and whatever the
    // replica split.  All CTAs of the grid are co-resident (one per SM, P <= SMs), and
    // each signals before it waits, so the waits are short and cannot deadlock.
    const int n_pos = uniform(sched->n_pos);
    const int st_first = (int)(u_begin / G.KB), st_last = (int)((u_end - 1) / G.KB);
    if (threadIdx.x == 0) {
        __threadfence();
        for (int st = st_first; st <= st_last; ++st) atomicAdd(&flags[st], 1);
    }
    for (int st = st_first; st <= st_last; ++st) {
        const int c0 = cc_range_of_unit(G, (long long)st * G.KB);
        const int c1 = cc_range_of_unit(G, (long long)(st + 1) * G.KB - 1);
        const int m = c1 - c0 + 1, k = (int)blockIdx.x - c0;
        if (threadIdx.x == 0) {
            uint32_t spins = 0;
            while (ld_acquire(&flags[st]) < m) {
                __nanosleep(40);
                if (++spins > (1u << 24)) __trap();
            }
        }
        __syncthreads();
        if (threadIdx.x == 0 && st == st_first) CC_TP(W, 2 + KIND, 4);
#ifdef CC_TRACE
        const unsigned long long t_pass = cc_gtime();
#endif
        // few contributors: several items per warp; many: one item, its pieces loaded together
        if (m <= 3) fixup_tile<KIND, 4, 3>(part, E, D, W, H, st, c0, m, k, n_pos, warp, lane);
        else if (m <= 8) fixup_tile<KIND, 2, 4>(part, E, D, W, H, st, c0, m, k, n_pos, warp, lane);
        else fixup_tile<KIND, 1, 8>(part, E, D, W, H, st, c0, m, k, n_pos, warp, lane);
#ifdef CC_TRACE
        __syncthreads();
        if (threadIdx.x == 0 && W.trace != nullptr) {           // duration of this CTA's fixup pass
            const unsigned long long dt = cc_gtime() - t_pass;
            const int slot = st == st_first ? 0 : 1;
            cc_trace_minmax(W.trace, 8 + KIND, slot, dt);
            atomicAdd(W.trace + ((size_t)(12 + KIND) * CC_TRACE_POINTS + slot) * 2 + 1, 1ull);
            atomicAdd(W.trace + ((size_t)(12 + KIND) * CC_TRACE_POINTS + 2 + slot) * 2 + 1, dt);
        }
#endif
    }
#ifdef CC_TRACE
    __syncthreads();
    if (threadIdx.x == 0) CC_TP(W, 2 + KIND, 5);
#endif
}


// ---------------------------------------------------------------------------------------------------------------
// k_gemm_cl -- the same projections for SMALL steps (at most kClRows grouped rows) as a CLUSTER split-K: one cluster of S CTAs per super tile (256 output features), CTA `rank` streams k-blocks
// [rank KB / S, (rank + 1) KB / S) of every active replica's blob into ONE pair of TMEM accumulators (group r at
// columns goff[r] ..), and the S partial sums are reduced through distributed shared memory instead of global
// memory: after the main loops every CTA scatters the columns (batch rows) CTA j owns into CTA j's ring memory
// (st.shared::cluster, slot = sender rank), a cluster barrier, and every CTA adds the S slots of its own columns in
// rank order and runs the fused epilogue on them.  No partial sums in global memory, no arrival flags, no fixup
// pass: the kernel's tail is one DSMEM exchange (~2 us) instead of the stream-K chain (~8 us: partial store, fence,
// counter, wait for the slowest of the m CTAs of a super tile, one or two fixup passes).  The k split and the sum
// order are functions of the layer shape only => bit-identical across replica counts; the host picks
// this kernel from the step's ROW COUNT only, so the choice cannot differ between replica counts either.
constexpr int kClRows = 192;                  // grouped rows (n_pos) the two accumulators and the exchange buffers are sized for
constexpr int kClMaxS = 8;
constexpr int kClMaxStages = 8;              // ring depth of the one-tile variant (24 KiB stages at batch 64; 12 measured slower)

__device__ __forceinline__ bool planes_out_one(const CcDims& D) { return D.pl[CC_OP_A] == 1; }

template <int KIND, int TILES>
__global__ void __launch_bounds__(kGemmThreads, 1)
k_gemm_cl(CcGemmGeo G, const uint8_t* __restrict__ act, CcEpi E, CcDims D, CcWork W, const CcLayerTable* __restrict__ tab, int S) {
    const int planes = D.pl[KIND];
    const CcSched* __restrict__ sched = W.sched;
    const int Mpad = D.Mpad;
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    GemmSmemHdr* H = reinterpret_cast<GemmSmemHdr*>(smem_raw);
    const int warp = uniform((int)(threadIdx.x >> 5)), lane = threadIdx.x & 31;
    const int rank = (int)cluster_ctarank();
    // TILES = 2: the cluster owns a super tile (two adjacent tiles, one 32 KiB copy per k-block); TILES = 1: ONE tile of
    // 128 output features (a 16 KiB atom per k-block, every other atom of its super tile): twice the clusters, half the
    // exchange, for the projections whose super tiles are too few to fill the GPU with co-resident clusters (O, down)
    const int unit = (int)blockIdx.x / S;                            // the cluster's super tile (TILES = 2) or tile (TILES = 1)
    const int st = TILES == 2 ? unit : unit / CC_G, tile0 = TILES == 2 ? unit * CC_G : unit;
    constexpr uint32_t kWBytes = (uint32_t)TILES * CC_A_TILE_BYTES;   // weight bytes per stage

    if (threadIdx.x == 0) CC_TP(W, 2 + KIND, 0);
    if (threadIdx.x == 0) {
        for (int i = 0; i < kClMaxStages; ++i) {
            mbar_init(&H->full[i], 1);
            mbar_init(&H->empty[i], 1);
        }
        mbar_init(&H->tmem_full[0], 1);
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc<kTmemCols>(&H->tmem_base);
    if (KIND == EPI_QKV) {                                           // starts before k_prologue has finished: counts the groups itself
        int* wcnt = H->aux;
        if (threadIdx.x < 256) {
            uint32_t err = 0;
            const int rep = cc_row_replica(E.assign, E.seq_lens, threadIdx.x, E.batch, D, tab->active_mask, err);
#pragma unroll
            for (int r = 0; r < CC_MAXR; ++r) {
                const uint32_t bal = __ballot_sync(0xffffffffu, rep == r);
                if (lane == 0) wcnt[warp * CC_MAXR + r] = __popc(bal);
            }
        }
        __syncthreads();
        if (threadIdx.x == 0) {
            int off = 0;
            for (int r = 0; r < CC_MAXR; ++r) {
                int c = 0;
                for (int w = 0; w < 8; ++w) c += wcnt[w * CC_MAXR + r];
                H->cnt[r] = c;
                H->goff[r] = off;
                off += (c + CC_ROW_ALIGN - 1) / CC_ROW_ALIGN * CC_ROW_ALIGN;
            }
        }
    } else if (threadIdx.x < CC_MAXR) {
        H->cnt[threadIdx.x] = sched->cnt[threadIdx.x];
        H->goff[threadIdx.x] = sched->goff[threadIdx.x];
    }
    if (threadIdx.x < CC_MAXR) {
        const CcReplicaRow rr = tab->rep[threadIdx.x];
        H->blob[threadIdx.x] = rr.blob;
        H->kpool[threadIdx.x] = rr.k_pool ? (__nv_bfloat16*)rr.k_pool : E.kv.k_pool;
        H->vpool[threadIdx.x] = rr.k_pool ? (__nv_bfloat16*)rr.v_pool : E.kv.v_pool;
        H->kvpages[threadIdx.x] = rr.k_pool ? rr.n_pages : E.kv.n_pages;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    int nmax = 0, n_pos = 0;
#pragma unroll
    for (int r = 0; r < CC_MAXR; ++r) {
        const int n = (H->cnt[r] + CC_ROW_ALIGN - 1) / CC_ROW_ALIGN * CC_ROW_ALIGN;
        nmax = max(nmax, n);
        n_pos = max(n_pos, n ? H->goff[r] + n : 0);
    }
    nmax = uniform(nmax);
    n_pos = uniform(n_pos);
    const uint32_t stage_bytes = kWBytes + (uint32_t)planes * (uint32_t)nmax * 128u;
    uint8_t* stage0 = smem_raw + kHdrBytes;
    int n_stages = (kGemmSmem - kHdrBytes) / (int)stage_bytes;
    if (n_stages > (TILES == 2 ? kMaxStages : kClMaxStages)) n_stages = TILES == 2 ? kMaxStages : kClMaxStages;
    const int kb0 = (int)((long long)rank * G.KB / S), kb1 = (int)((long long)(rank + 1) * G.KB / S);
    const uint32_t tmem_base = uniform(H->tmem_base);
    // columns (grouped rows) CTA j owns in the reduction: [j * cper, (j + 1) * cper)
    const int cper = ((n_pos + S - 1) / S + 7) & ~7;

    if (nmax > 0) {
        if (warp == 0) {
            // ===================== producer (as in k_gemm: weights first, then the dependency, then the slabs) =====
            const uint64_t pol_w = policy_evict_first(), pol_a = policy_evict_last();
            const size_t kb_stride = (size_t)(Mpad >> 3) * planes * 1024;
            int n_act = 0;
            for (int r = 0; r < CC_MAXR; ++r) n_act += uniform(H->cnt[r]) > 0;
            const int total = (kb1 - kb0) * n_act;
            const int n_pre = total < n_stages ? total : n_stages;
            auto run = [&](const int mode) {
                int stage = 0, idx = 0;
                uint32_t ph = 0;
                uint8_t* sW = stage0;
                for (int r = 0; r < CC_MAXR; ++r) {
                    const int cnt = uniform(H->cnt[r]);
                    if (cnt == 0) continue;
                    const uint32_t nb = (uint32_t)((cnt + 15) & ~15) * 128u * (uint32_t)planes;
                    const uint32_t tx = kWBytes + nb;
                    const uint8_t* wsrc = uniform(H->blob[r]) + G.w_off + ((size_t)st * G.KB + kb0) * kWStage +
                                          (TILES == 2 ? 0 : (size_t)(unit % CC_G) * CC_A_TILE_BYTES);
                    const uint8_t* asrc = act + (size_t)(uniform(H->goff[r]) >> 3) * planes * 1024 + (size_t)kb0 * kb_stride;
                    for (int kb = kb0; kb < kb1; ++kb, ++idx) {
                        if (mode == 0 && idx >= n_pre) return;
                        const bool pre = idx < n_pre;
                        if (mode == 1 && !pre) mbar_wait(&H->empty[stage], ph ^ 1);
                        if (elect_one()) {
                            if (mode == 0 || !pre) {
                                mbar_expect_tx(&H->full[stage], tx);
                                bulk_g2s_hint(sW, wsrc, kWBytes, &H->full[stage], pol_w);
                            }
                            if (mode == 1) bulk_g2s_hint(sW + kWBytes, asrc, nb, &H->full[stage], pol_a);
                        }
                        wsrc += kWStage;
                        asrc += kb_stride;
                        sW += stage_bytes;
                        if (++stage == n_stages) { stage = 0; ph ^= 1; sW = stage0; }
                    }
                }
            };
            run(0);
            // the ring is full and the predecessor still runs: the next stages of my range go to L2 meanwhile
            cc_prefetch_weights(G, H->blob, H->cnt, (int)blockIdx.x, (int)gridDim.x, n_pre, D.pf_self, lane);
            pdl_wait();
            if (lane == 0) CC_TP(W, 2 + KIND, 1);
            __syncwarp();
            if (elect_one()) pdl_launch_dependents();
            run(1);
            // my copies are issued; the exchange and the epilogue follow: the first weight stages of the NEXT projection's CTAs
            // go to L2 meanwhile (gate/up behind O, down behind gate/up)
            if (KIND == EPI_O) cc_prefetch_weights(D.gu, H->blob, H->cnt, (int)blockIdx.x, (int)gridDim.x, 0, D.pf_next, lane);
            if (KIND == EPI_GU) cc_prefetch_weights(D.dn, H->blob, H->cnt, (int)blockIdx.x, (int)gridDim.x, 0, D.pf_next, lane);
            if (lane == 0) CC_TP(W, 2 + KIND, 2);
            __syncwarp();
        } else if (warp == 1) {
            // ===================== MMA issuer: group r accumulates into columns goff[r] .. of the two tiles =====
            int stage = 0;
            uint32_t ph = 0;
            const uint32_t a_hi = (uint32_t)(umma_desc_sw128(0) >> 32);
            const uint32_t b_hi = (uint32_t)(umma_desc_sw128(0, (uint32_t)planes * 1024u) >> 32);
            const uint32_t desc_lo0 = (uint32_t)umma_desc_sw128(smem_u32(stage0));
            const uint32_t dstage = stage_bytes >> 4, dact = kWBytes >> 4;
            uint32_t da = desc_lo0;
            for (int r = 0; r < CC_MAXR; ++r) {
                const int cnt = uniform(H->cnt[r]);
                if (cnt == 0) continue;
                const uint32_t idesc = umma_idesc_m128((uint32_t)((cnt + 15) & ~15), D.fmt);
                const uint32_t col0 = (uint32_t)uniform(H->goff[r]);
                for (int kb = kb0; kb < kb1; ++kb) {
                    mbar_wait(&H->full[stage], ph);
                    tc_fence_after();
                    if (elect_one()) {
                        const uint32_t db = da + dact;
#pragma unroll
                        for (int j = 0; j < TILES; ++j) {
                            const uint32_t d_tmem = tmem_base + (uint32_t)j * 256 + col0;
                            const uint32_t daj = da + (uint32_t)j * (CC_A_TILE_BYTES >> 4);
#pragma unroll
                            for (int k = 0; k < CC_TILE_K / 16; ++k) {
                                umma_bf16_lo(d_tmem, daj + 2 * k, db + 2 * k, a_hi, b_hi, idesc, (kb == kb0 && k == 0) ? 0u : 1u);
                                if (planes == 2) umma_bf16_lo(d_tmem, daj + 2 * k, db + 64 + 2 * k, a_hi, b_hi, idesc, 1u);
                            }
                        }
                        umma_commit(&H->empty[stage]);
                    }
                    __syncwarp();
                    da += dstage;
                    if (++stage == n_stages) { stage = 0; ph ^= 1; da = desc_lo0; }
                }
            }
            if (elect_one()) umma_commit(&H->tmem_full[0]);
            __syncwarp();
        } else if (warp >= 6) {
            // ===================== helper warps: per-row tables of the fused epilogue =====================
            pdl_wait();
            for (int p = (int)threadIdx.x - 6 * 32; p < n_pos; p += kGemmThreads - 6 * 32) {
                const int b = W.perm[p];
                H->perm[p] = b;
                if (KIND == EPI_QKV) {
                    int pos = -1, page = -1;
                    if (b >= 0) {
                        pos = E.seq_lens[b] - 1;
                        page = E.kv.block_table[(size_t)b * D.max_blocks + pos / CC_PAGE];
                    }
                    H->aux[p] = pos;
                    H->page[p] = page;
                } else if (KIND == EPI_O) {
                    H->aux[p] = __float_as_int(b >= 0 ? W.inv_in[p] : 0.f);
                } else if (KIND == EPI_GU) {
                    float ss = 0.f;
                    if (b >= 0) {
                        const int nt = (D.d + 127) >> 7;
                        for (int t = 0; t < nt; ++t) ss += W.ssq[(size_t)t * Mpad + p];   // tile order: fixed
                    }
                    H->aux[p] = __float_as_int(b >= 0 ? rsqrtf(ss / (float)D.d + D.eps) / W.inv_in[p] : 0.f);
                }
            }
        }
        // the scatter warps wait for this CTA's accumulators here, so that "my main loop is over" reaches the barrier
        if (warp >= 2 && warp < 6) {
            mbar_wait(&H->tmem_full[0], 0);
            tc_fence_after();
        }
    }
    __syncthreads();
    if (threadIdx.x == 0) CC_TP(W, 2 + KIND, 3);
    if (nmax == 0) {                                                 // nothing runs this step (the same in every CTA of the cluster)
        pdl_wait();
        if (warp == 1) tmem_dealloc<kTmemCols>(tmem_base);
        return;
    }
    if (KIND == EPI_GU && S == 1 && D.fmt == CC_FMT_F16 && planes_out_one(D)) {
        // ---- gate/up alone on its super tile (no split-K, no exchange): SwiGLU straight from tensor memory ----
        // The generic tail below moves the fp32 accumulators through shared memory and then runs one warp per (column, tile)
        // item: 250 instructions per two items, four passes per warp at batch 64 = 4.5 us in which HBM idles and the down
        // projection waits.  Here the warps pair gate (even TMEM lane) with up (odd lane) by one shuffle,
        // apply the row scale and SiLU in registers, and drop the fp16 results into an image of the operand rows in the
        // (dead) ring -- [tile][column][128 B], 16-byte chunks swizzled as in a_act; then all threads copy the image out
        // in 16-byte chunks.
        uint8_t* img = stage0;
        const int kb_end = D.dn.KB;                                  // tiles at or beyond it are padding of the last super tile
        {
            // all sixteen warps (the producer, the issuer and the helpers are done): four per TMEM lane quarter share the
            // 8-column chunks
            const int q = warp & 3, grp = warp >> 2, odd = lane & 1;
            const int jo = q * 16 + (lane >> 1);                     // output (= down-projection k) index within the tile's 64
            tc_fence_after();
            for (int c0 = grp * 8; c0 < n_pos; c0 += 32) {
                uint32_t v[TILES][8];
#pragma unroll
                for (int j = 0; j < TILES; ++j)
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                                 : "=r"(v[j][0]), "=r"(v[j][1]), "=r"(v[j][2]), "=r"(v[j][3]), "=r"(v[j][4]), "=r"(v[j][5]), "=r"(v[j][6]),
                                   "=r"(v[j][7])
                                 : "r"(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)j * 256 + (uint32_t)c0)
                                 : "memory");
                tmem_ld_wait();
                // the even lane (gate) finishes columns c0 .. c0 + 3, the odd lane (up) columns c0 + 4 .. c0 + 7
#pragma unroll
                for (int i = 0; i < 4; ++i) {
                    const int col = c0 + 4 * odd + i;
                    const bool live = col < n_pos && H->perm[min(col, n_pos - 1)] >= 0;
                    const float inv = __int_as_float(H->aux[min(col, n_pos - 1)]);
                    uint8_t* dst = img + (size_t)col * 128 + (((jo >> 3) ^ (col & 7)) << 4) + (jo & 7) * 2;
#pragma unroll
                    for (int j = 0; j < TILES; ++j) {
                        const uint32_t mine = odd ? v[j][4 + i] : v[j][i];
                        const uint32_t send = odd ? v[j][i] : v[j][4 + i];
                        const uint32_t recv = __shfl_xor_sync(0xffffffffu, send, 1);
                        const float g0 = __uint_as_float(odd ? recv : mine) * inv, u0 = __uint_as_float(odd ? mine : recv) * inv;
                        // silu(g) u with the special-function unit's 2^x and 1/x (a few ulp from the IEEE division of the
                        // generic tail; g -> -inf gives -0, g -> +inf gives g)
                        float ex;
                        asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(ex) : "f"(g0 * -1.4426950408889634f));
                        float a = g0 * __frcp_rn(1.f + ex) * u0;
                        a = fminf(fmaxf(a, -65504.f), 65504.f);
                        if (live && tile0 + j < kb_end) *reinterpret_cast<__half*>(dst + (size_t)j * n_pos * 128) = __float2half_rn(a);
                    }
                }
            }
        }
        tc_fence_before();
        __syncthreads();
        if (warp == 1) tmem_dealloc<kTmemCols>(tmem_base);
        if (threadIdx.x == 0) CC_TP(W, 2 + KIND, 4);
        for (int id = (int)threadIdx.x; id < TILES * n_pos * 8; id += kGemmThreads) {
            const int j = id / (n_pos * 8), rem = id - j * n_pos * 8, col = rem >> 3, c = rem & 7;
            if (tile0 + j >= kb_end || H->perm[col] < 0) continue;
            const uint4 val = *reinterpret_cast<const uint4*>(img + ((size_t)j * n_pos + col) * 128 + c * 16);
            // physical chunk c of the row holds the values k = kb * 64 + (c ^ (col & 7)) * 8 ..
            *reinterpret_cast<uint4*>(W.a_act + act_chunk_off(col, (tile0 + j) * 64 + ((c ^ (col & 7)) << 3), D.Mpad, 1, 0)) = val;
        }
#ifdef CC_TRACE
        __syncthreads();
        if (threadIdx.x == 0) CC_TP(W, 2 + KIND, 5);
#endif
        return;
    }
    // The first items of this warp's epilogue are known already (my columns, the row tables): issue their global loads
    // (residual rows, gains, RoPE table, h1) now, so that their latency runs under the exchange.  (kNI = 4 items per warp
    // iteration measured 2.5 us SLOWER per step than 2; 1 the same as 2.)
    constexpr int kWarps = kGemmThreads / 32, kNI = 2;
    const int c_lo = rank * cper, c_hi = min(n_pos, c_lo + cper);
    const int n_items = max(0, c_hi - c_lo) * TILES;
    EpiPre pre[kNI];
    int pp[kNI], bb[kNI], tt[kNI];
    auto setup = [&](int it0) {
#pragma unroll
        for (int u = 0; u < kNI; ++u) {
            const int it = it0 + u, cl = it / TILES, j = it - cl * TILES;
            pp[u] = c_lo + cl;
            tt[u] = tile0 + j;
            bb[u] = it < n_items ? H->perm[pp[u]] : -1;
            if (bb[u] >= 0) epi_pre<KIND>(pre[u], E, D, W, SmemTab{H}, tt[u], pp[u], bb[u], lane);
        }
    };
    setup(warp * kNI);
    cluster_sync_all();                                              // every ring of the cluster is dead: it becomes the exchange buffer
    // exchange buffer in CTA j: [sender rank][tile 0 | 1][column of j's range][128 features] fp32
    const uint32_t slot_bytes = (uint32_t)TILES * (uint32_t)cper * 512u;
    if (warp >= 2 && warp < 14) {                                    // three warps per TMEM lane quarter share the chunks
        const int q = warp & 3, f = q * 32 + lane, grp = (warp - 2) >> 2;   // lane quarter; output feature within the tile
        const uint32_t my_buf = smem_u32(stage0) + (uint32_t)rank * slot_bytes;
        int chunk = 0;
        tc_fence_after();
        // owners in rotation starting behind this CTA, so that the S senders write to S different CTAs at any time
        for (int oo = 1; oo <= S; ++oo) {
            const int owner = (rank + oo) % S;
            const uint32_t dst_owner = mapa_u32(my_buf, (uint32_t)owner) + (uint32_t)f * 4u;
            for (int cl = 0; cl < cper; cl += 8) {                   // 8 columns of that owner
                const int c0 = owner * cper + cl;
                if (c0 >= n_pos) break;
                if (chunk++ % 3 != grp) continue;
                uint32_t v[TILES][8];
#pragma unroll
                for (int j = 0; j < TILES; ++j)
                    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0, %1, %2, %3, %4, %5, %6, %7}, [%8];"
                                 : "=r"(v[j][0]), "=r"(v[j][1]), "=r"(v[j][2]), "=r"(v[j][3]), "=r"(v[j][4]), "=r"(v[j][5]), "=r"(v[j][6]),
                                   "=r"(v[j][7])
                                 : "r"(tmem_base + ((uint32_t)(q * 32) << 16) + (uint32_t)j * 256 + (uint32_t)c0)
                                 : "memory");
                tmem_ld_wait();
                if (owner == rank) {                                 // my own columns: plain shared-memory stores
#pragma unroll
                    for (int j = 0; j < TILES; ++j)
#pragma unroll
                        for (int i = 0; i < 8; ++i)
                            asm volatile("st.shared.b32 [%0], %1;" ::"r"(my_buf + (uint32_t)f * 4u + ((uint32_t)j * (uint32_t)cper + (uint32_t)(cl + i)) * 512u),
                                         "r"(v[j][i])
                                         : "memory");
                } else {
#pragma unroll
                    for (int j = 0; j < TILES; ++j)
#pragma unroll
                        for (int i = 0; i < 8; ++i)
                            asm volatile("st.shared::cluster.b32 [%0], %1;" ::"r"(dst_owner + ((uint32_t)j * (uint32_t)cper + (uint32_t)(cl + i)) * 512u),
                                         "r"(v[j][i])
                                         : "memory");
                }
            }
        }
    }
    tc_fence_before();
    cluster_sync_all();                                              // all slots of my columns have landed (release / acquire at cluster scope)
    if (warp == 1) tmem_dealloc<kTmemCols>(tmem_base);
    if (threadIdx.x == 0) CC_TP(W, 2 + KIND, 4);
    // ---- my columns: add the S slots in rank order, fused epilogue; one warp per (column, tile) item ----
    {
        const float* buf = reinterpret_cast<const float*>(stage0);
        const size_t slot_f = slot_bytes / 4;
        for (int it0 = warp * kNI; it0 < n_items; it0 += kWarps * kNI) {
            if (it0 != warp * kNI) setup(it0);
            float4 acc[kNI];
#pragma unroll
            for (int u = 0; u < kNI; ++u) {
                const int it = it0 + u, cl = it / TILES, j = it - cl * TILES;
                acc[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (bb[u] >= 0) {
                    const float* src = buf + ((size_t)j * cper + cl) * 128 + 4 * lane;
                    for (int sdr = 0; sdr < S; ++sdr) {               // rank order: fixed
                        const float4 v = *reinterpret_cast<const float4*>(src + (size_t)sdr * slot_f);
                        acc[u].x += v.x; acc[u].y += v.y; acc[u].z += v.z; acc[u].w += v.w;
                    }
                }
            }
#pragma unroll
            for (int u = 0; u < kNI; ++u)
                if (bb[u] >= 0) epi_fin<KIND>(pre[u], E, D, W, SmemTab{H}, tt[u], pp[u], bb[u], acc[u], lane);
        }
    }
#ifdef CC_TRACE
    __syncthreads();
    if (threadIdx.x == 0) CC_TP(W, 2 + KIND, 5);
#endif
}

}  // namespace

// ---- cluster split-K variant (k_gemm_cl): the four projections of small steps --------------------------------------
typedef void (*ClKernel)(CcGemmGeo, const uint8_t*, CcEpi, CcDims, CcWork, const CcLayerTable*, int);
static ClKernel cl_kernel(int which, int tiles) {
    if (tiles == 2)
        return which == 0 ? (ClKernel)k_gemm_cl<EPI_QKV, 2> : which == 1 ? (ClKernel)k_gemm_cl<EPI_O, 2>
               : which == 2 ? (ClKernel)k_gemm_cl<EPI_GU, 2> : (ClKernel)k_gemm_cl<EPI_DN, 2>;
    return which == 0 ? (ClKernel)k_gemm_cl<EPI_QKV, 1> : which == 1 ? (ClKernel)k_gemm_cl<EPI_O, 1>
           : which == 2 ? (ClKernel)k_gemm_cl<EPI_GU, 1> : (ClKernel)k_gemm_cl<EPI_DN, 1>;
}

cudaError_t cc_gemm_configure() {
    cudaError_t e = cudaFuncSetAttribute(k_gemm<EPI_QKV>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_gemm<EPI_O>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_gemm<EPI_GU>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_gemm<EPI_DN>, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem);
    for (int which = 0; which < 4 && e == cudaSuccess; ++which)
        for (int tiles = 1; tiles <= 2 && e == cudaSuccess; ++tiles)
            e = cudaFuncSetAttribute((const void*)cl_kernel(which, tiles), cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem);
    return e;
}

static void cl_config(cudaLaunchConfig_t& cfg, cudaLaunchAttribute* attr, int n_clusters, int S, cudaStream_t st, bool pdl) {
    cfg = cudaLaunchConfig_t{};
    cfg.gridDim = dim3((unsigned)(n_clusters * S));
    cfg.blockDim = dim3(kGemmThreads);
    cfg.dynamicSmemBytes = kGemmSmem;
    cfg.stream = st;
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = (unsigned)S;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    attr[1].id = cudaLaunchAttributeProgrammaticStreamSerialization;
    attr[1].val.programmaticStreamSerializationAllowed = 1;
    cfg.attrs = attr;
    cfg.numAttrs = pdl ? 2 : 1;
}
// Cluster geometry of projection `which` for small steps: g.cl_tiles in {1, 2} tiles per cluster and the largest cluster
// size g.S <= 8 for which all clusters are co-resident (one wave) and every CTA gets at least one k-block -- whichever of
// the two puts more CTAs on the GPU (two tiles on a tie: one 32 KiB copy per k-block).  g.S = 0 keeps the projection on
// the stream-K kernel: no co-resident geometry, or one that would use fewer than 60 % of the CTAs stream-K would.  A
// function of the layer shape and the device.
void cc_gemm_cl_geometry(int which, CcGemmGeo& g, int n_sms) {
    g.S = 0;
    g.cl_tiles = 2;
    int best_ctas = 0;
    for (int tiles = 2; tiles >= 1; --tiles) {
        const int n_clusters = g.ST * CC_G / tiles;
        for (int S = 1; S <= kClMaxS; ++S) {
            if (S > g.KB || n_clusters * S > n_sms) continue;
            cudaLaunchConfig_t cfg;
            cudaLaunchAttribute attr[2];
            cl_config(cfg, attr, n_clusters, S, nullptr, false);
            int n = 0;
            if (cudaOccupancyMaxActiveClusters(&n, (void*)cl_kernel(which, tiles), &cfg) != cudaSuccess) {
                cudaGetLastError();
                continue;
            }
            if (n >= n_clusters && n_clusters * S > best_ctas) {
                best_ctas = n_clusters * S;
                g.S = S;
                g.cl_tiles = tiles;
            }
        }
    }
    if ((long long)best_ctas * 10 < (long long)g.P * 6) g.S = 0;
}
int cc_gemm_cl_max_rows() { return kClRows; }

cudaError_t cc_launch_gemm_cl(int which, const CcDims& D, const CcLayerTable* tab, const CcWork& W, const int* seq_lens,
                              const int* assign, int batch, const CcKv& kv, __nv_bfloat16* hidden, const CcLaunch& L) {
    CcEpi E{assign, batch, seq_lens, kv, hidden};
    const CcGemmGeo& g = which == 0 ? D.qkv : which == 1 ? D.o : which == 2 ? D.gu : D.dn;
    const uint8_t* act = which == 0 ? W.x_act : which == 1 ? W.o_act : which == 2 ? W.y_act : W.a_act;
    cudaLaunchConfig_t cfg;
    cudaLaunchAttribute attr[2];
    cl_config(cfg, attr, g.ST * CC_G / g.cl_tiles, g.S, L.st, L.pdl);
    return cudaLaunchKernelEx(&cfg, cl_kernel(which, g.cl_tiles), g, act, E, D, W, tab, g.S);
}

// which: 0 = QKV, 1 = O, 2 = gate/up, 3 = down
cudaError_t cc_launch_gemm(int which, const CcDims& D, const CcLayerTable* tab, const CcWork& W, const int* seq_lens,
                           const int* assign, int batch, const CcKv& kv, __nv_bfloat16* hidden, const CcLaunch& L) {
    const dim3 block(kGemmThreads);
    const size_t smem = (size_t)kGemmSmem;
    CcEpi E{assign, batch, seq_lens, kv, hidden};
    int* flags = W.flags + which * CC_FLAG_STRIDE;
    switch (which) {
        case 0: return cc_launch_kernel(k_gemm<EPI_QKV>, dim3(D.qkv.P), block, smem, L, D.qkv, W.x_act, W.qkv_part, flags, E, D, W, tab);
        case 1: return cc_launch_kernel(k_gemm<EPI_O>, dim3(D.o.P), block, smem, L, D.o, W.o_act, W.o_part, flags, E, D, W, tab);
        case 2: return cc_launch_kernel(k_gemm<EPI_GU>, dim3(D.gu.P), block, smem, L, D.gu, W.y_act, W.gu_part, flags, E, D, W, tab);
        default: return cc_launch_kernel(k_gemm<EPI_DN>, dim3(D.dn.P), block, smem, L, D.dn, W.a_act, W.d_part, flags, E, D, W, tab);
    }
}
