// cc_big_gemm.cu -- the large-M projection GEMM of mixed prefill + decode steps (sm_100a).
//
// SURVEY.md 8(f) NEXT-2 / BASELINE.json configs[3]: a step of thousands of rows (prompt chunks + decode rows) is
// tensor-bound, not HBM-bound (2 * rows flop per weight byte), so this kernel is built around the tensor pipe:
//   * CTA pairs (clusters of 2, tcgen05 cta_group::2): one tile = 256 output features x 256 rows of one replica
//     group.  Swap-AB as in the decode kernel: the pre-packed weight atoms are the A operand -- the two atoms of a
//     super tile (cc_common.cuh) are the two M halves, CTA rank c streams atom c -- and the activations are the B
//     operand, N = 256 rows, 128 from each CTA's shared memory, so every operand byte is fetched once per pair.
//   * the whole K loop of a tile runs into one fp32 accumulator D[128 lanes][256 columns] per CTA in TMEM, double
//     buffered (512 columns): no split-K, no partial sums; the epilogue of tile i overlaps the main loop of tile i+1.
//   * warp 0 = producer (descriptor-free bulk copies into an mbarrier ring, weights from the replica table's blob),
//     warp 1 = MMA issuer in the leader CTA / arrival relay in its peer (the leader must know that the peer's stage
//     has landed), warps 4..11 = epilogue: TMEM -> registers -> a [32 rows][128 features] fp32 staging tile in shared
//     memory -> the SAME fused epilogues as the decode kernel (cc_epilogue.cuh: RoPE + KV append | residual + norm
//     statistics + operand | SwiGLU | residual + write-back in request order), one warp per row, lane = 4 features.
//   * persistent: pair p takes tiles p, p + pairs, ... of the list (replica group, super tile, row block) with the
//     row block fastest, so the pairs running together share a few weight super tiles and all row blocks in L2.
// Every output element is one fixed-order K sum whatever the replica split: bit-identical across replica counts.
#include "cc_epilogue.cuh"

namespace {

constexpr int kBigThreads = 384;              // warps: 0 producer, 1 MMA / relay, 2-3 idle, 4..11 epilogue
constexpr int kBigMaxStages = 6;
constexpr int kBigHdrBytes = 1024;
constexpr int kStagingBytes = 32 * 128 * 4;   // one [32 rows][128 features] fp32 tile
constexpr int kBigSmem = 226 * 1024;
constexpr int kBlockRows = 256;               // rows of a tile (UMMA N)

struct BigHdr {
    uint64_t full[kBigMaxStages];             // this CTA's stage has landed
    uint64_t peer_full[kBigMaxStages];        // leader only: the peer's stage has landed (relayed)
    uint64_t empty[kBigMaxStages];            // the pair's MMAs have consumed the stage (commit, multicast)
    uint64_t tmem_full[2];                    // accumulator buffer complete (commit, multicast)
    uint64_t tmem_empty[2];                   // leader only: both CTAs' epilogue warps have drained the buffer
    uint32_t tmem_base;
    int cnt[CC_MAXR], goff[CC_MAXR];
    const uint8_t* blob[CC_MAXR];
    __nv_bfloat16* kpool[CC_MAXR];            // the KV pools replica r's rows append to (its partition, else the call's pools)
    __nv_bfloat16* vpool[CC_MAXR];
    int kvpages[CC_MAXR];
};
static_assert(sizeof(BigHdr) <= kBigHdrBytes, "header does not fit");

// per-row tables of the fused epilogues, in global memory (k_big_group / k_big_rowstat wrote them)
struct GlobalTab {
    const int* aux_;
    const int* page_;
    const BigHdr* H;
    __device__ __forceinline__ int aux(int p) const { return aux_[p]; }
    __device__ __forceinline__ int page(int p) const { return page_[p]; }
    __device__ __forceinline__ const uint8_t* blob(int p) const { return H->blob[replica_of_pos(H->cnt, H->goff, p)]; }
    __device__ __forceinline__ __nv_bfloat16* k_pool(int p) const { return H->kpool[replica_of_pos(H->cnt, H->goff, p)]; }
    __device__ __forceinline__ __nv_bfloat16* v_pool(int p) const { return H->vpool[replica_of_pos(H->cnt, H->goff, p)]; }
    __device__ __forceinline__ int kv_pages(int p) const { return H->kvpages[replica_of_pos(H->cnt, H->goff, p)]; }
};

struct TileIter {                             // walks this pair's tiles: (replica group r, super tile st, row block rb)
    int r, st, rb, row0, rows;                // row0: first grouped row of the block; rows: live rows in it
};
// MMA N of a row block: its rows rounded up to 32 (each CTA of the pair stages half of them, a multiple of 16)
__device__ __forceinline__ int tile_n(int rows) { return (rows + 31) & ~31; }
__device__ __forceinline__ bool tile_at(const BigHdr* H, int ST, long long t, TileIter& it) {
#pragma unroll
    for (int r = 0; r < CC_MAXR; ++r) {
        const int cnt = H->cnt[r];
        if (cnt == 0) continue;
        const int RB = (cnt + kBlockRows - 1) / kBlockRows;
        const long long n = (long long)ST * RB;
        if (t < n) {
            it.r = r;
            it.st = (int)(t / RB);
            it.rb = (int)(t - (long long)it.st * RB);
            it.row0 = H->goff[r] + it.rb * kBlockRows;
            it.rows = min(kBlockRows, cnt - it.rb * kBlockRows);
            return true;
        }
        t -= n;
    }
    return false;
}

template <int KIND>
__global__ void __launch_bounds__(kBigThreads, 1)
k_big_gemm(CcGemmGeo G, const uint8_t* __restrict__ act, CcEpi E, CcDims D, CcWork W, const CcLayerTable* __restrict__ tab) {
    extern __shared__ __align__(1024) uint8_t smem_raw[];
    BigHdr* H = reinterpret_cast<BigHdr*>(smem_raw);
    const int warp = uniform((int)(threadIdx.x >> 5)), lane = threadIdx.x & 31;
    const uint32_t rank = cluster_ctarank();
    const int pair = blockIdx.x >> 1, n_pairs = gridDim.x >> 1;
    const int planes = D.pl[KIND];
    const uint32_t b_bytes = 128u * 128u * (uint32_t)planes;          // this CTA's rows of one k-block, at most 128
    const uint32_t stage_bytes = CC_A_TILE_BYTES + b_bytes;
    const int n_stages = planes == 1 ? 6 : 4;
    uint8_t* stage0 = smem_raw + kBigHdrBytes;
    float* staging = reinterpret_cast<float*>(stage0 + (size_t)n_stages * stage_bytes);   // two tiles, one per epilogue group

    if (threadIdx.x == 0) {
        for (int i = 0; i < kBigMaxStages; ++i) {
            mbar_init(&H->full[i], 1);
            mbar_init(&H->peer_full[i], 1);
            mbar_init(&H->empty[i], 1);
        }
        for (int i = 0; i < 2; ++i) {
            mbar_init(&H->tmem_full[i], 1);
            mbar_init(&H->tmem_empty[i], 16);                          // 8 epilogue warps in each CTA of the pair
        }
        fence_mbar_init();
    }
    if (threadIdx.x < CC_MAXR) {
        H->cnt[threadIdx.x] = W.sched->cnt[threadIdx.x];
        H->goff[threadIdx.x] = W.sched->goff[threadIdx.x];
        const CcReplicaRow rr = tab->rep[threadIdx.x];
        H->blob[threadIdx.x] = rr.blob;
        H->kpool[threadIdx.x] = rr.k_pool ? (__nv_bfloat16*)rr.k_pool : E.kv.k_pool;
        H->vpool[threadIdx.x] = rr.k_pool ? (__nv_bfloat16*)rr.v_pool : E.kv.v_pool;
        H->kvpages[threadIdx.x] = rr.k_pool ? rr.n_pages : E.kv.n_pages;
    }
    if (warp == 1) tmem_alloc_pair<512>(&H->tmem_base);
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                                                // both CTAs' barriers exist before any remote arrive
    tc_fence_after();
    const uint32_t tmem_base = uniform(H->tmem_base);
    const size_t kb_stride = (size_t)(D.Mpad >> 3) * planes * 1024;   // bytes between k-blocks of the operand

    if (warp == 0) {
        // ===================== producer (both CTAs) =====================
        // with the row block fastest, the pairs running together cover a few super tiles x every row block: the
        // activations are re-read by every wave (evict_last keeps them in L2); a weight super tile is read by the ~9
        // pairs of its row blocks at about the same time -- with evict_first it was gone before the last of them
        // came (measured: 2.7 GB of DRAM reads for 0.76 GB of operands), so weights take the default policy
        const uint64_t pol_a = policy_evict_last();
        int stage = 0;
        uint32_t ph = 0;
        TileIter it;
        for (long long t = pair; tile_at(H, G.ST, t, it); t += n_pairs) {
            const uint8_t* wsrc = uniform(H->blob[it.r]) + G.w_off + cc_atom_off(G.KB, it.st * CC_G + (int)rank, 0);
            // a ragged last row block of a replica group is an MMA of N = its rows rounded up to 32 (half from each CTA), not 256
            const int half = tile_n(it.rows) >> 1;
            const uint32_t bt_bytes = (uint32_t)half * 128u * (uint32_t)planes;
            const uint8_t* asrc = act + (size_t)((it.row0 + (int)rank * half) >> 3) * planes * 1024;
            for (int kb = 0; kb < G.KB; ++kb) {
                mbar_wait(&H->empty[stage], ph ^ 1);
                if (elect_one()) {
                    uint8_t* s = stage0 + (size_t)stage * stage_bytes;
                    mbar_expect_tx(&H->full[stage], CC_A_TILE_BYTES + bt_bytes);
                    bulk_g2s(s, wsrc, CC_A_TILE_BYTES, &H->full[stage]);
                    bulk_g2s_hint(s + CC_A_TILE_BYTES, asrc, bt_bytes, &H->full[stage], pol_a);
                }
                wsrc += (size_t)CC_G * CC_A_TILE_BYTES;
                asrc += kb_stride;
                if (++stage == n_stages) { stage = 0; ph ^= 1; }
            }
        }
    } else if (warp == 1 && rank == 1) {
        // ===================== relay (peer CTA): tell the leader that this CTA's stage has landed =====================
        int stage = 0;
        uint32_t ph = 0;
        TileIter it;
        for (long long t = pair; tile_at(H, G.ST, t, it); t += n_pairs) {
            for (int kb = 0; kb < G.KB; ++kb) {
                mbar_wait(&H->full[stage], ph);
                if (elect_one()) mbar_arrive_cluster(mapa_u32(smem_u32(&H->peer_full[stage]), 0));
                __syncwarp();
                if (++stage == n_stages) { stage = 0; ph ^= 1; }
            }
        }
    } else if (warp == 1) {
        // ===================== MMA issuer (leader CTA) =====================
        int stage = 0;
        uint32_t ph = 0, pc = 0;
        const uint32_t a_hi = (uint32_t)(umma_desc_sw128(0) >> 32);
        const uint32_t b_hi = (uint32_t)(umma_desc_sw128(0, (uint32_t)planes * 1024u) >> 32);
        const uint32_t desc_lo0 = (uint32_t)umma_desc_sw128(smem_u32(stage0));
        const uint32_t dstage = stage_bytes >> 4, dact = CC_A_TILE_BYTES >> 4;
        TileIter it;
        for (long long t = pair; tile_at(H, G.ST, t, it); t += n_pairs, ++pc) {
            const uint32_t buf = pc & 1;
            mbar_wait(&H->tmem_empty[buf], ((pc >> 1) & 1) ^ 1);
            tc_fence_after();
            const uint32_t d_tmem = tmem_base + buf * 256;
            const uint32_t idesc = umma_idesc_pair_m256((uint32_t)tile_n(it.rows), D.fmt);
            for (int kb = 0; kb < G.KB; ++kb) {
                mbar_wait(&H->full[stage], ph);
                mbar_wait(&H->peer_full[stage], ph);
                tc_fence_after();
                if (elect_one()) {
                    const uint32_t da = desc_lo0 + (uint32_t)stage * dstage, db = da + dact;
#pragma unroll
                    for (int k = 0; k < CC_TILE_K / 16; ++k) {
                        umma_pair_lo(d_tmem, da + 2 * k, db + 2 * k, a_hi, b_hi, idesc, (kb == 0 && k == 0) ? 0u : 1u);
                        if (planes == 2) umma_pair_lo(d_tmem, da + 2 * k, db + 64 + 2 * k, a_hi, b_hi, idesc, 1u);
                    }
                    umma_commit_pair(&H->empty[stage]);
                    if (kb == G.KB - 1) umma_commit_pair(&H->tmem_full[buf]);
                }
                __syncwarp();
                if (++stage == n_stages) { stage = 0; ph ^= 1; }
            }
        }
    } else if (warp >= 4) {
        // ===================== epilogue (both CTAs): TMEM -> staging tile -> fused epilogue, one warp per row ==========
        const int ew = warp - 4, grp = ew >> 2, q = ew & 3;            // group 0 takes the even 32-row chunks, group 1 the odd ones
        float* stg = staging + (size_t)grp * (kStagingBytes / 4);
        const GlobalTab T{KIND == EPI_QKV ? W.row_pos : KIND == EPI_O ? reinterpret_cast<const int*>(W.inv_in)
                                                                      : reinterpret_cast<const int*>(W.gu_scale),
                          W.row_page, H};
        const uint32_t empty_remote = mapa_u32(smem_u32(&H->tmem_empty[0]), 0);
        uint32_t pc = 0;
        TileIter it;
        for (long long t = pair; tile_at(H, G.ST, t, it); t += n_pairs, ++pc) {
            const uint32_t buf = pc & 1;
            mbar_wait(&H->tmem_full[buf], (pc >> 1) & 1);
            tc_fence_after();
            const int tile = it.st * CC_G + (int)rank;
            for (int c = grp * 32; c < it.rows; c += 64) {
                uint32_t v[32];
                tmem_ld_32x32b_x32(tmem_base + ((uint32_t)(q * 32) << 16) + buf * 256 + (uint32_t)c, v);
                tmem_ld_wait();
#pragma unroll
                for (int i = 0; i < 32; ++i) stg[i * 128 + q * 32 + lane] = __uint_as_float(v[i]);
                named_bar_sync(2 + grp, 128);
                // rows q*8 .. q*8+7 of the chunk: lane = features 4*lane .. 4*lane+3 of the tile
#pragma unroll
                for (int h = 0; h < 2; ++h) {
                    EpiPre pre[4];
                    int pp[4], bb[4];
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int i = q * 8 + h * 4 + u;
                        pp[u] = it.row0 + c + i;
                        bb[u] = (c + i < it.rows) ? W.perm[pp[u]] : -1;
                        if (bb[u] >= 0) epi_pre<KIND>(pre[u], E, D, W, T, tile, pp[u], bb[u], lane);
                    }
#pragma unroll
                    for (int u = 0; u < 4; ++u) {
                        const int i = q * 8 + h * 4 + u;
                        const float4 a = *reinterpret_cast<const float4*>(stg + i * 128 + 4 * lane);
                        if (bb[u] >= 0) epi_fin<KIND>(pre[u], E, D, W, T, tile, pp[u], bb[u], a, lane);   // warp-uniform branch
                    }
                }
                named_bar_sync(2 + grp, 128);                           // the staging tile may be rewritten
            }
            tc_fence_before();
            __syncwarp();
            if (lane == 0) mbar_arrive_cluster(empty_remote + buf * 8);
        }
    }
    tc_fence_before();
    __syncthreads();
    cluster_sync_all();                                                // the peer may still be reading this CTA's smem / TMEM
    if (warp == 1) tmem_dealloc_pair<512>(tmem_base);
}

}  // namespace

cudaError_t cc_big_gemm_configure() {
    cudaError_t e = cudaFuncSetAttribute(k_big_gemm<EPI_QKV>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBigSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_big_gemm<EPI_O>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBigSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_big_gemm<EPI_GU>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBigSmem);
    if (e == cudaSuccess) e = cudaFuncSetAttribute(k_big_gemm<EPI_DN>, cudaFuncAttributeMaxDynamicSharedMemorySize, kBigSmem);
    return e;
}

template <typename... KArgs, typename... Args>
static cudaError_t launch_pairs(void (*kern)(KArgs...), int n_pairs, cudaStream_t st, Args&&... args) {
    cudaLaunchConfig_t cfg = {};
    cfg.gridDim = dim3(2 * n_pairs);
    cfg.blockDim = dim3(kBigThreads);
    cfg.dynamicSmemBytes = kBigSmem;
    cfg.stream = st;
    cudaLaunchAttribute attr[1];
    attr[0].id = cudaLaunchAttributeClusterDimension;
    attr[0].val.clusterDim.x = 2;
    attr[0].val.clusterDim.y = 1;
    attr[0].val.clusterDim.z = 1;
    cfg.attrs = attr;
    cfg.numAttrs = 1;
    return cudaLaunchKernelEx(&cfg, kern, KArgs(args)...);
}

// which: 0 = QKV, 1 = O, 2 = gate/up, 3 = down
cudaError_t cc_launch_big_gemm(int which, const CcDims& D, const CcLayerTable* tab, const CcWork& W, const int* seq_lens,
                               const int* assign, int batch, const CcKv& kv, __nv_bfloat16* hidden, const CcLaunch& L) {
    CcEpi E{assign, batch, seq_lens, kv, hidden};
    const int n_pairs = L.n_sms / 2;
    switch (which) {
        case 0: return launch_pairs(k_big_gemm<EPI_QKV>, n_pairs, L.st, D.qkv, W.x_act, E, D, W, tab);
        case 1: return launch_pairs(k_big_gemm<EPI_O>, n_pairs, L.st, D.o, W.o_act, E, D, W, tab);
        case 2: return launch_pairs(k_big_gemm<EPI_GU>, n_pairs, L.st, D.gu, W.y_act, E, D, W, tab);
        default: return launch_pairs(k_big_gemm<EPI_DN>, n_pairs, L.st, D.dn, W.a_act, E, D, W, tab);
    }
}
