// cc_prefill.cu -- causal chunked-prefill attention over the paged KV cache on tcgen05 (sm_100a).
//
// SURVEY.md 8(f) NEXT-2 (kernel K8), BASELINE.json configs[3]; `l` = prompt length in prefill.  A prompt
// chunk is a run of rows of one step that share a request's block-table row at consecutive seq_lens (k_big_group
// finds them); token t of the chunk attends positions 0 .. its own, all K/V -- the chunk's own included -- being in
// the cache already (the QKV epilogue appended them).  Unlike the decode kernel, which streams a row's whole prefix
// for every row, this is a dense contraction with M = tokens x G >= 64, so it runs on the tensor pipe:
//   * work item = (chunk, query tile of T = 128 / G tokens, kv head): the G query heads of the T tokens are the 128
//     rows of the MMA (row m = token m / G, head m % G), so one K/V read serves the GQA group and T tokens;
//   * the kv axis is walked in tiles of 64 tokens (4 pages): a producer warp stages the head's K and V of each page
//     by TMA (boxes of 16 rows x 128 B, 128-byte swizzle, straight into the operand layout), ring of five stages;
//   * S = Q K^T (M 128, N 64, K 128) and O += P V (M 128, N 128, K 64) are tcgen05.mma into TMEM (three S
//     buffers: the scores run two tiles ahead of the products; O resident); K is the K-major B operand, V the MN-major one (no transpose anywhere);
//   * eight softmax warps, one query row per thread (TMEM lane = row) and two warps per lane quarter that share a tile's 64
//     columns (row maxima and sums meet through shared memory, one named barrier per pair and tile): tcgen05.ld of the
//     scores, causal mask on the diagonal tiles only, online softmax in log2 units against a reference maximum that
//     follows the running one only when that grew by more than 2^8 (then O is rescaled in TMEM); the probabilities
//     OVERWRITE the tile's scores in tensor memory (tcgen05.st, bf16 pairs) and are the A operand of the P V product
//     from there (no shared memory, no proxy fence), so the softmax of tile j + 1 runs while the product of tile j does;
//   * the Q rows of the next item are requested before the epilogue of the current one;
//   * q and the probabilities enter as bf16 hi + lo planes (two MMAs each) like in the decode kernel: the K/V are
//     bf16 by definition, and a single bf16 plane of q or p costs 2e-3 on the attention output;
//   * items are dealt round-robin in decreasing cost; every row is finished by one item in one fixed order, so the
//     result does not depend on the replica split or on timing.
#include "cc_kvmaps.h"

namespace {

constexpr int kSmWarps = 8;                  // softmax warps: two per TMEM lane quarter, each takes half of a tile's columns
constexpr int kPfThreads = (2 + kSmWarps) * 32;   // warp 0 producer, warp 1 MMA issuer, warps 2..9 softmax (TMEM lane quarter = warp % 4)
constexpr int kKvTile = 64;                  // kv tokens per tile (4 pages)
constexpr int kKvStages = 5;                 // what Q leaves of the 227 KiB (the probabilities live in TMEM)
constexpr int kQBytes = 2 * 2 * 128 * 128;   // Q: [hi | lo][half of Dh][128 rows][128 B]
constexpr int kKvStageBytes = 2 * 2 * kKvTile * 128;   // [K | V][half of Dh][64 tokens][128 B]
constexpr int kPfHdr = 3072;                 // barriers (1 KiB) + the softmax pairs' exchange of row maxima / sums (2 KiB)
constexpr int kPfSmem = kPfHdr + kQBytes + kKvStages * kKvStageBytes;
constexpr float kLazyLog2 = 8.f;             // O and l are rescaled only when a row maximum has grown by more than 2^8
constexpr int kSBufs = 3;                    // score / probability buffers: Q K^T runs two tiles ahead of P V
constexpr uint32_t kColS = 0, kColO = 192;   // TMEM columns: S buffers at 0, 64, 128, O at 192..319.  The probabilities of a tile
                                             // overwrite its scores: bf16 pairs, hi plane in columns 0..31 of the buffer, lo in 32..63

struct PfHdr {
    uint64_t kv_full[kKvStages], kv_empty[kKvStages];
    uint64_t s_full[kSBufs], p_full[kSBufs];      // [score buffer = kv tile % 3]
    uint64_t pv_done[2], q_ready;                 // pv_done: [kv tile parity]
    uint32_t tmem_base;
};

// K-major / MN-major shared-memory descriptors with an explicit leading byte offset (cc_common.cuh has the K-major one)
__device__ __forceinline__ uint64_t umma_desc_sw128_lbo(uint32_t smem_addr, uint32_t lbo_bytes, uint32_t sbo_bytes) {
    uint64_t d = 0;
    d |= (uint64_t)((smem_addr & 0x3FFFFu) >> 4);
    d |= (uint64_t)(lbo_bytes >> 4) << 16;
    d |= (uint64_t)(sbo_bytes >> 4) << 32;
    d |= (uint64_t)1 << 46;
    d |= (uint64_t)2 << 61;
    return d;
}
// bf16 x bf16 -> fp32, M = 128; b_mn: the B operand is MN-major (V: head dim contiguous, kv tokens are the K axis)
__device__ __forceinline__ uint32_t idesc_bf16(uint32_t n, bool b_mn) {
    return (1u << 4) | (1u << 7) | (1u << 10) | ((b_mn ? 1u : 0u) << 16) | ((n >> 3) << 17) | ((128u >> 4) << 24);
}
__device__ __forceinline__ void tmem_st_32x32b_x32(uint32_t taddr, const uint32_t (&r)[32]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x32.b32 [%0], "
        "{%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16, "
        "%17, %18, %19, %20, %21, %22, %23, %24, %25, %26, %27, %28, %29, %30, %31, %32};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
        "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15]), "r"(r[16]), "r"(r[17]), "r"(r[18]), "r"(r[19]), "r"(r[20]),
        "r"(r[21]), "r"(r[22]), "r"(r[23]), "r"(r[24]), "r"(r[25]), "r"(r[26]), "r"(r[27]), "r"(r[28]), "r"(r[29]), "r"(r[30]),
        "r"(r[31])
        : "memory");
}
// 2^x by the special-function unit alone (exp2f adds a range fix-up of three instructions per value; what it would fix --
// results below 2^-126 -- is zero against a row sum of at least 1 here)
__device__ __forceinline__ float ex2_ftz(float x) {
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}
__device__ __forceinline__ void tmem_st_wait() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tmem_st_32x32b_x16(uint32_t taddr, const uint32_t (&r)[16]) {
    asm volatile(
        "tcgen05.st.sync.aligned.32x32b.x16.b32 [%0], {%1, %2, %3, %4, %5, %6, %7, %8, %9, %10, %11, %12, %13, %14, %15, %16};" ::"r"(taddr),
        "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]), "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]), "r"(r[8]), "r"(r[9]), "r"(r[10]),
        "r"(r[11]), "r"(r[12]), "r"(r[13]), "r"(r[14]), "r"(r[15])
        : "memory");
}
// D += A B with the A operand in TENSOR MEMORY (lane = row, 32-bit column c = the bf16 pair k = 2c, 2c + 1 of the row: 8 columns
// per MMA of K = 16) and B through a shared-memory descriptor: no shared-memory read for A, no proxy fence for its writer.
__device__ __forceinline__ void umma_bf16_ts(uint32_t d_tmem, uint32_t a_tmem, uint32_t b_lo, uint32_t b_hi, uint32_t idesc,
                                             uint32_t accumulate) {
    asm volatile(
        "{\n\t.reg .pred p;\n\t.reg .b64 db;\n\t"
        "setp.ne.b32 p, %5, 0;\n\t"
        "mov.b64 db, {%2, %3};\n\t"
        "tcgen05.mma.cta_group::1.kind::f16 [%0], [%1], db, %4, p;\n\t}" ::"r"(d_tmem),
        "r"(a_tmem), "r"(b_lo), "r"(b_hi), "r"(idesc), "r"(accumulate)
        : "memory");
}

struct Item {                 // one (chunk, query tile, kv head)
    int row0;                 // original row of the tile's first token
    int n_tok;                // tokens of the tile (<= T)
    int bt_row;               // original row whose block-table row is used (the chunk's first row)
    int s_last;               // seq_len of the tile's last token = kv positions the tile attends
    int h;                    // kv head
    int n_tiles;              // kv tiles
};
__device__ __forceinline__ bool item_at(const CcWork& W, const CcDims& D, const int* __restrict__ seq_lens, int id, Item& it) {
    const int n = W.bs->n_items * D.Hkv;
    {   // rounds of gridDim.x items in decreasing cost, dealt forwards and backwards in turn: dealt forwards only, block 0
        // would get the dearest item of every round and the last block the cheapest (11 % apart at cfg4)
        const int grid = (int)gridDim.x, round = id / grid, idx = id - round * grid;
        if (round & 1) id = round * grid + (grid - 1 - idx);
    }
    if (id >= n) return false;
    const int k = id / D.Hkv, T = 128 / D.G;
    const int c = W.item_chunk[k], j = W.item_tile[k];
    const int r0 = W.chunk_row0[c], len = W.chunk_len[c];
    it.h = id - k * D.Hkv;
    it.bt_row = r0;
    it.row0 = r0 + j * T;
    it.n_tok = min(T, len - j * T);
    it.s_last = seq_lens[it.row0 + it.n_tok - 1];
    it.n_tiles = (it.s_last + kKvTile - 1) / kKvTile;
    return true;
}

__global__ void __launch_bounds__(kPfThreads, 1)
k_prefill_attn(const int* __restrict__ seq_lens, CcKv kv, CcDims D, CcWork W, const __grid_constant__ CcKvMaps maps) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    PfHdr* H = reinterpret_cast<PfHdr*>(smem_raw);
    uint8_t* sQ = smem_raw + kPfHdr;
    uint8_t* sKV = sQ + kQBytes;
    const int warp = uniform((int)(threadIdx.x >> 5)), lane = threadIdx.x & 31;
    const int G = D.G;

    if (threadIdx.x == 0) {
        for (int i = 0; i < kKvStages; ++i) {
            mbar_init(&H->kv_full[i], 1);
            mbar_init(&H->kv_empty[i], 1);
        }
        for (int i = 0; i < kSBufs; ++i) {
            mbar_init(&H->s_full[i], 1);
            mbar_init(&H->p_full[i], kSmWarps);
        }
        for (int i = 0; i < 2; ++i) mbar_init(&H->pv_done[i], 1);
        mbar_init(&H->q_ready, kSmWarps);
        fence_mbar_init();
    }
    if (warp == 1) tmem_alloc<512>(&H->tmem_base);
    tc_fence_before();
    __syncthreads();
    tc_fence_after();
    const uint32_t tmem_base = uniform(H->tmem_base);

    if (warp == 0) {
        // ===================== producer: the head's K and V of every page of the tile, by TMA =====================
        uint32_t g = 0;                                                // kv tiles issued so far (all items)
        Item it;
        for (int id = blockIdx.x; item_at(W, D, seq_lens, id, it); id += gridDim.x) {
            const int n_pages = (it.s_last + CC_PAGE - 1) / CC_PAGE;
            const int rep = replica_of_pos(W.sched->cnt, W.sched->goff, W.pos_of[it.row0]);   // whose KV partition the chunk lives in
            const CUtensorMap* tmK = &maps.k[rep];
            const CUtensorMap* tmV = &maps.v[rep];
            for (int j = 0; j < it.n_tiles; ++j, ++g) {
                const int stage = (int)(g % kKvStages);
                mbar_wait(&H->kv_empty[stage], ((g / kKvStages) & 1) ^ 1);
                const int pg0 = j * (kKvTile / CC_PAGE), in_tile = min(kKvTile / CC_PAGE, n_pages - pg0);
                int pid = 0;
                if (lane < in_tile) {
                    pid = kv.block_table[(size_t)it.bt_row * D.max_blocks + pg0 + lane];
                    if (pid < 0 || pid >= kv.n_pages_r[rep]) {
                        atomicOr(W.err, CC_DEVERR_BAD_PAGE);
                        pid = 0;
                    }
                }
                int pids[kKvTile / CC_PAGE];
#pragma unroll
                for (int i = 0; i < kKvTile / CC_PAGE; ++i) pids[i] = __shfl_sync(0xffffffffu, pid, i);
                if (elect_one()) {
                    const uint32_t bar = smem_u32(&H->kv_full[stage]);
                    const uint32_t dst0 = smem_u32(sKV) + (uint32_t)stage * kKvStageBytes;
                    mbar_expect_tx(&H->kv_full[stage], (uint32_t)in_tile * 4u * 2048u);
#pragma unroll
                    for (int i = 0; i < kKvTile / CC_PAGE; ++i) {
                        if (i < in_tile) {
                            const int row0 = (pids[i] * D.Hkv + it.h) * CC_PAGE;   // the pool as [pages * Hkv * 16 rows][Dh]
                            const uint32_t d = dst0 + (uint32_t)i * 2048u;
#pragma unroll
                            for (int hf = 0; hf < 2; ++hf) {
                                tma_load_2d(d + hf * 8192u, tmK, hf * 64, row0, bar);
                                tma_load_2d(d + 16384u + hf * 8192u, tmV, hf * 64, row0, bar);
                            }
                        }
                    }
                }
                __syncwarp();
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer =====================
        const uint32_t idesc_s = idesc_bf16(kKvTile, false), idesc_o = idesc_bf16(128, true);
        const uint32_t q_lo = (uint32_t)umma_desc_sw128(smem_u32(sQ)), k_hi32 = (uint32_t)(umma_desc_sw128(0) >> 32);
        const uint64_t v_d0 = umma_desc_sw128_lbo(smem_u32(sKV) + 16384u, 8192u, 1024u);
        const uint32_t v_hi32 = (uint32_t)(v_d0 >> 32);
        uint32_t g = 0, n_item = 0;                                    // g: kv tiles of the items before this one
        Item it;
        // The tensor pipe executes in issue order, and the order below is S(0) S(1) | PV(0) S(2) | PV(1) S(3) | ...: the scores of a
        // tile are ready two softmax periods before they are needed, and S(j + 2), which overwrites the buffer of P(j - 1), is
        // issued behind PV(j - 1) -- no "buffer free" barrier.
        auto issue_s = [&](uint32_t gt) {
            const int stage = (int)(gt % kKvStages);
            const uint32_t sb = gt % kSBufs;
            mbar_wait(&H->kv_full[stage], (gt / kKvStages) & 1);
            tc_fence_after();
            if (elect_one()) {
                const uint32_t k_lo = (uint32_t)umma_desc_sw128(smem_u32(sKV) + (uint32_t)stage * kKvStageBytes);
                const uint32_t d = tmem_base + kColS + sb * kKvTile;
#pragma unroll
                for (int ks = 0; ks < 8; ++ks) {
                    // Q: [plane][half][128 rows][128 B] -> half = ks / 4 at + 16 KiB, 32 B per step; K: halves 8 KiB apart
                    const uint32_t qa = q_lo + (uint32_t)(ks >> 2) * 1024 + 2 * (ks & 3);
                    const uint32_t kb = k_lo + (uint32_t)(ks >> 2) * 512 + 2 * (ks & 3);
                    umma_bf16_lo(d, qa, kb, k_hi32, k_hi32, idesc_s, ks == 0 ? 0u : 1u);
                    umma_bf16_lo(d, qa + 2048, kb, k_hi32, k_hi32, idesc_s, 1u);       // the lo plane of q, 32 KiB further
                }
                umma_commit(&H->s_full[sb]);
            }
            __syncwarp();
        };
        auto issue_pv = [&](uint32_t gt, bool first) {
            const int stage = (int)(gt % kKvStages);
            const uint32_t sb = gt % kSBufs;                           // the probabilities replaced the tile's scores
            mbar_wait(&H->p_full[sb], (gt / kSBufs) & 1);
            tc_fence_after();
            if (elect_one()) {
                const uint32_t v_lo = (uint32_t)v_d0 + (((uint32_t)stage * kKvStageBytes) >> 4);
                const uint32_t p_t = tmem_base + kColS + sb * kKvTile;   // hi pairs at + 0, lo pairs at + 32
#pragma unroll
                for (int ks = 0; ks < kKvTile / 16; ++ks) {
                    // A: P plane in TMEM (16 kv = 8 columns per step); B: V, MN-major, 16 kv rows = 2 KiB per step
                    umma_bf16_ts(tmem_base + kColO, p_t + 8 * ks, v_lo + ks * 128, v_hi32, idesc_o, (first && ks == 0) ? 0u : 1u);
                    umma_bf16_ts(tmem_base + kColO, p_t + 32 + 8 * ks, v_lo + ks * 128, v_hi32, idesc_o, 1u);
                }
                umma_commit(&H->pv_done[gt & 1]);
                umma_commit(&H->kv_empty[stage]);
            }
            __syncwarp();
        };
        for (int id = blockIdx.x; item_at(W, D, seq_lens, id, it); id += gridDim.x, ++n_item) {
            mbar_wait(&H->q_ready, n_item & 1);
            const uint32_t n = (uint32_t)it.n_tiles;
            issue_s(g);
            if (n > 1) issue_s(g + 1);
            for (uint32_t j = 0; j < n; ++j) {
                issue_pv(g + j, j == 0);
                if (j + 2 < n) issue_s(g + j + 2);
            }
            g += n;
        }
    } else {
        // ===================== softmax warps: one query row per thread, the tile's 64 columns shared by two warps =====================
        const int q4 = warp & 3;                                       // TMEM lane quarter of this warp (fixed by the hardware: warp % 4)
        const int half = (warp - 2) >> 2;                              // columns 32 half .. 32 half + 31 of every score tile, 64 half .. of O
        const int m = q4 * 32 + lane;                                  // row of the tile: token m / G, q head m % G
        const uint32_t lane_addr = tmem_base + ((uint32_t)(q4 * 32) << 16);
        float* xch = reinterpret_cast<float*>(smem_raw + 1024);        // [tile parity][half][128 rows]: the pair's row maxima (and row sums)
        uint32_t g = 0, n_pv = 0;
        Item it;
        // The sixteen Q rows this warp stages per item (q_rot, fp32, post-RoPE) are requested one item ahead: the loads of
        // item i + 1 are issued before the epilogue of item i and used after it (one row at a time they cost an item ~20 us,
        // in two batches after the epilogue still ~4 us during which the tensor pipe has nothing to do).  The rows of a
        // chunk are consecutive in their replica group (stable partition), so one table read gives all their positions.
        constexpr int kQR = 128 / kSmWarps;
        float4 xq[kQR];
        auto load_q = [&](const Item& t) {
            const int pos0 = W.pos_of[t.row0];
#pragma unroll
            for (int u = 0; u < kQR; ++u) {
                const int r = (warp - 2) + kSmWarps * u, tl = r / G, gq = r - tl * G;
                xq[u] = make_float4(0.f, 0.f, 0.f, 0.f);
                if (tl < t.n_tok)
                    xq[u] = *reinterpret_cast<const float4*>(W.q_rot + (size_t)min(pos0 + tl, D.Mpad - 1) * D.QD +
                                                             (size_t)(t.h * G + gq) * 128 + 4 * lane);
            }
        };
        Item nx;
        int id = blockIdx.x;
        bool have = item_at(W, D, seq_lens, id, it);
        if (have) load_q(it);
        for (; have; id += gridDim.x, it = nx) {
            // ---- Q of the item: x log2(e)/sqrt(Dh) -> bf16 hi + lo operand planes ----
#pragma unroll
            for (int u = 0; u < kQR; ++u) {
                const int r = (warp - 2) + kSmWarps * u;
                float4 v = xq[u];
                v.x *= D.qk_scale_log2; v.y *= D.qk_scale_log2; v.z *= D.qk_scale_log2; v.w *= D.qk_scale_log2;
                uint32_t h0, l0, h1, l1;
                split_hilo(v.x, v.y, h0, l0);
                split_hilo(v.z, v.w, h1, l1);
                // dims 4 lane .. 4 lane + 3: half = lane / 16, 16-byte chunk (lane % 16) / 2, byte (lane & 1) * 8 inside it
                const uint32_t off = (uint32_t)(lane >> 4) * 16384u + (uint32_t)(r >> 3) * 1024u + (uint32_t)(r & 7) * 128u +
                                     (uint32_t)((((lane & 15) >> 1) ^ (r & 7)) << 4) + (uint32_t)(lane & 1) * 8u;
                *reinterpret_cast<uint2*>(sQ + off) = make_uint2(h0, h1);
                *reinterpret_cast<uint2*>(sQ + 32768u + off) = make_uint2(l0, l1);
            }
            fence_proxy_async_smem();
            __syncwarp();
            if (lane == 0) mbar_arrive(&H->q_ready);
            const int tl = min(m / G, it.n_tok - 1);                   // padding rows take the last token's mask
            const int p_row = seq_lens[it.row0 + tl] - 1;              // kv positions 0 .. p_row are visible
            float m_run = -INFINITY, l_run = 0.f;                      // l_run: the sum over THIS warp's columns
            for (int j = 0; j < it.n_tiles; ++j, ++g) {
                const uint32_t sb = g % kSBufs;
                const int kv0 = j * kKvTile + half * 32;               // kv position of this warp's first column
                mbar_wait(&H->s_full[sb], (g / kSBufs) & 1);
                tc_fence_after();
                uint32_t sv[32];
                tmem_ld_32x32b_x32(lane_addr + kColS + sb * kKvTile + half * 32, sv);
                tmem_ld_wait();
                float mx = -INFINITY;
                const int lim = p_row - kv0;                           // columns 0 .. lim (of this warp's 32) are visible
                if (__all_sync(0xffffffffu, lim >= 31)) {              // not on the diagonal for this warp's rows: no mask
#pragma unroll
                    for (int i = 0; i < 32; ++i) mx = fmaxf(mx, __uint_as_float(sv[i]));
                } else {
#pragma unroll
                    for (int i = 0; i < 32; ++i) {
                        const float v = (i <= lim) ? __uint_as_float(sv[i]) : -INFINITY;
                        sv[i] = __float_as_uint(v);
                        mx = fmaxf(mx, v);
                    }
                }
                // the row maximum over both halves: through shared memory, one named barrier per pair of warps and tile
                float* xm = xch + (g & 1) * 256;
                xm[half * 128 + m] = mx;
                named_bar_sync(1 + q4, 64);
                mx = fmaxf(mx, xm[(half ^ 1) * 128 + m]);
                // Lazy rescale: the probabilities are taken against a reference m_run that follows the running maximum only
                // when that has grown by more than 2^kLazyLog2 in some row of the warp (p <= 2^8: harmless in fp32 / bf16
                // hi + lo).  Then O (this warp's half of the columns of its 32 TMEM lanes) and l are rescaled, which needs
                // every P V product issued so far to be complete; otherwise this tile's probabilities go into the other P
                // buffer while the previous product still runs.  Both warps of a pair see the same maxima, hence take the
                // same decision; it is a function of the data only.
                const float m_seen = fmaxf(m_run, mx);                 // finite from tile 0 on: position 0 is visible to every row
                float alpha = 1.f;
                if (j == 0) {
                    m_run = m_seen;                                    // first tile: O is overwritten, l_run = 0
                } else if (__any_sync(0xffffffffu, m_seen > m_run + kLazyLog2)) {
                    mbar_wait(&H->pv_done[(n_pv - 1) & 1], ((n_pv - 1) >> 1) & 1);   // O holds tiles 0 .. j-1
                    tc_fence_after();
                    alpha = exp2f(m_run - m_seen);
                    m_run = m_seen;
#pragma unroll 1
                    for (int c = half * 64; c < half * 64 + 64; c += 32) {
                        uint32_t ov[32];
                        tmem_ld_32x32b_x32(lane_addr + kColO + c, ov);
                        tmem_ld_wait();
#pragma unroll
                        for (int i = 0; i < 32; ++i) ov[i] = __float_as_uint(__uint_as_float(ov[i]) * alpha);
                        tmem_st_32x32b_x32(lane_addr + kColO + c, ov);
                    }
                    tmem_st_wait();
                }
                const float m_new = m_run;
                // the probabilities replace the tile's scores: both warps of the pair have theirs in registers (the barrier above)
                if (j == it.n_tiles - 1 && it.s_last < j * kKvTile + kKvTile) {
                    // ragged last tile: V rows past the last position hold other data (or nothing): p = 0 must meet 0
                    mbar_wait(&H->kv_full[g % kKvStages], (g / kKvStages) & 1);
                    uint8_t* sV = sKV + (size_t)(g % kKvStages) * kKvStageBytes + 16384;
                    const int first = it.s_last - j * kKvTile;
                    for (int q = (warp - 2) * 32 + lane; q < (kKvTile - first) * 16; q += kSmWarps * 32) {
                        const int r = first + (q >> 4), c = q & 15;    // row r, 16-byte chunk c of its 256 bytes
                        *reinterpret_cast<uint4*>(sV + (c >> 3) * 8192 + r * 128 + ((c & 7) << 4)) = make_uint4(0, 0, 0, 0);
                    }
                }
                float lsum = 0.f;
                uint32_t hi[16], lo[16];                               // this warp's 32 kv columns as bf16 pairs
#pragma unroll
                for (int i = 0; i < 16; ++i) {
                    const float p0 = ex2_ftz(__uint_as_float(sv[2 * i]) - m_new);
                    const float p1 = ex2_ftz(__uint_as_float(sv[2 * i + 1]) - m_new);
                    lsum += p0 + p1;
                    split_hilo(p0, p1, hi[i], lo[i]);
                }
                tmem_st_32x32b_x16(lane_addr + kColS + sb * kKvTile + half * 16, hi);
                tmem_st_32x32b_x16(lane_addr + kColS + sb * kKvTile + 32 + half * 16, lo);
                tmem_st_wait();
                l_run = l_run * alpha + lsum;
                if (j == it.n_tiles - 1 && it.s_last < j * kKvTile + kKvTile) fence_proxy_async_smem();   // the zeroed V rows
                tc_fence_before();
                __syncwarp();
                if (lane == 0) mbar_arrive(&H->p_full[sb]);
                ++n_pv;
            }
            have = item_at(W, D, seq_lens, id + (int)gridDim.x, nx);
            if (have) load_q(nx);                                      // in flight during the epilogue below
            // ---- the item's rows: O / l -> the O-projection operand; this warp writes its 64 columns ----
            {
                // the row sums of the two halves, added in half order; the parity buffer the last tile did not use
                float* xl = xch + (g & 1) * 256;
                xl[half * 128 + m] = l_run;
                named_bar_sync(1 + q4, 64);
                l_run = xl[m] + xl[128 + m];
            }
            mbar_wait(&H->pv_done[(n_pv - 1) & 1], ((n_pv - 1) >> 1) & 1);
            tc_fence_after();
            const int tlr = m / G, gq = m - tlr * G;
            const bool live = tlr < it.n_tok;
            const int pos = live ? W.pos_of[it.row0 + tlr] : 0;
            const float inv = 1.f / l_run;
#pragma unroll 1
            for (int c = half * 64; c < half * 64 + 64; c += 32) {
                uint32_t ov[32];
                tmem_ld_32x32b_x32(lane_addr + kColO + c, ov);
                tmem_ld_wait();
                if (live) {
#pragma unroll
                    for (int i = 0; i < 32; i += 8) {
                        float x[8];
#pragma unroll
                        for (int e = 0; e < 8; ++e) x[e] = __uint_as_float(ov[i + e]) * inv;
                        act_store<8>(W.o_act, D, D.pl[CC_OP_O], pos, (it.h * G + gq) * 128 + c + i, x);
                    }
                }
            }
            tc_fence_before();
        }
    }
    tc_fence_before();
    __syncthreads();
    if (warp == 1) tmem_dealloc<512>(tmem_base);
}

}  // namespace

cudaError_t cc_prefill_configure() {
    return cudaFuncSetAttribute(k_prefill_attn, cudaFuncAttributeMaxDynamicSharedMemorySize, kPfSmem);
}

cudaError_t cc_launch_prefill_attention(const int* seq_lens, const CcKv& kv, const CcDims& D, const CcWork& W, const CcLaunch& L) {
    if (D.Dh != 128) return cudaErrorInvalidValue;
    CcKvMaps maps;
    cudaError_t e = cc_make_kv_maps(&maps, kv, D.Hkv, D.Dh, CC_PAGE);
    if (e != cudaSuccess) return e;
    CcLaunch plain{L.st, L.n_sms, false};
    return cc_launch_kernel(k_prefill_attn, dim3(L.n_sms), dim3(kPfThreads), (size_t)kPfSmem, plain, seq_lens, kv, D, W, maps);
}
