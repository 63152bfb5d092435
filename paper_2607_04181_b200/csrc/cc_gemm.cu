// cc_gemm.cu -- the weight-streaming projection GEMM of the replicated decoder layer (sm_100a).
//
// SURVEY.md 8(a) rows a2 (QKV), a6 (O), a8 (gate/up), a9 (down); replica indirection row a10.
// Decode is HBM-bound: every weight byte is read once per replica group, so the kernel is built
// around the weight stream, not around the MMA:
//   * swap-AB: a packed weight tile (128 output features x 64 k, a 16 KiB pre-swizzled image
//     made once at cc_create_layer) is the tcgen05 A operand (M = 128); the activations of one
//     replica group (n rows, n = multiple of 16, <= 256) are the B operand (N = n), held as two
//     bf16 planes hi + lo that are both multiplied into the same accumulator (cc_rowwise.cu).
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
//   * a tile's partial sums ("pieces") are added up in fixed order by the next kernel of the
//     chain, which also applies the fused epilogue (RoPE, residual + RMSNorm, SwiGLU, ...).
#include "cc_kernels.h"

namespace {

constexpr int kGemmThreads = 192;
constexpr int kMaxStages = 8;
constexpr int kGemmSmem = 225 * 1024;     // dynamic shared memory per CTA
constexpr int kTmemCols = 512;
constexpr uint32_t kWStage = CC_G * CC_A_TILE_BYTES;   // weight bytes per stage (32 KiB)

struct GemmSmemHdr {                      // lives at the start of dynamic smem
    uint64_t full[kMaxStages];
    uint64_t empty[kMaxStages];
    uint64_t tmem_full[2];
    uint64_t tmem_empty[2];
    uint32_t tmem_base;
    int cnt[CC_MAXR];
    int goff[CC_MAXR];
    const uint8_t* blob[CC_MAXR];
};

__global__ void __launch_bounds__(kGemmThreads, 1)
k_gemm(CcGemmGeo G, const uint8_t* __restrict__ act, int planes, float* __restrict__ part, int Mpad,
       const CcLayerTable* __restrict__ tab, const CcSched* __restrict__ sched) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    GemmSmemHdr* H = reinterpret_cast<GemmSmemHdr*>(smem_raw);
    const int warp = uniform((int)(threadIdx.x >> 5)), lane = threadIdx.x & 31;

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
    // The grouping (k_group) and the replica table were written at least two kernels back in the
    // chain; every kernel of the chain waits for its predecessor BEFORE it lets its successor
    // start, so both are complete and visible here although this kernel's own predecessor (the
    // producer of the activations) may still be running.
    if (threadIdx.x < CC_MAXR) {
        H->cnt[threadIdx.x] = sched->cnt[threadIdx.x];
        H->goff[threadIdx.x] = sched->goff[threadIdx.x];
        H->blob[threadIdx.x] = tab->rep[threadIdx.x].blob;
    }
    tc_fence_before();
    __syncthreads();
    tc_fence_after();

    const int nmax = uniform(sched->nmax);
    const uint32_t act_bytes_max = (uint32_t)planes * (uint32_t)nmax * 128u;   // nmax % 16 == 0 => multiple of 2 KiB
    const uint32_t stage_bytes = kWStage + act_bytes_max;
    uint8_t* stage0 = smem_raw + 1024;                      // header occupies the first KiB
    int n_stages = (kGemmSmem - 1024) / (int)stage_bytes;
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
            const uint64_t pol_w = policy_evict_first();
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
                            if (mode == 1) bulk_g2s(sW + kWStage, asrc, nb, &H->full[stage]);
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
            if (elect_one()) pdl_launch_dependents();
            run(1);
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
                const uint32_t idesc = umma_idesc_bf16_m128((uint32_t)((cnt + 15) & ~15));
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
        } else {
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
                        float* dst = part + ((size_t)((blockIdx.x + st) * CC_G + j) * Mpad + goff) * 128 + f;
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
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<kTmemCols>(tmem_base);
}

}  // namespace

cudaError_t cc_gemm_configure() {
    return cudaFuncSetAttribute(k_gemm, cudaFuncAttributeMaxDynamicSharedMemorySize, kGemmSmem);
}

cudaError_t cc_launch_gemm(int which, const CcDims& D, const CcLayerTable* tab, const CcWork& W, const CcLaunch& L) {
    const CcGemmGeo* G;
    const uint8_t* act;
    float* part;
    int planes = 2;   // hi + lo activation planes; the O projection's input needs one
    switch (which) {
        case 0: G = &D.qkv; act = W.x_act; part = W.qkv_part; break;
        case 1: G = &D.o; act = W.o_act; part = W.o_part; planes = 1; break;
        case 2: G = &D.gu; act = W.y_act; part = W.gu_part; break;
        default: G = &D.dn; act = W.a_act; part = W.d_part; break;
    }
    return cc_launch_kernel(k_gemm, dim3(G->P), dim3(kGemmThreads), (size_t)kGemmSmem, L, *G, act, planes, part, D.Mpad,
                            tab, W.sched);
}
