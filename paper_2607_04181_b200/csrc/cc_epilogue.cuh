// cc_epilogue.cuh -- the fused epilogues of the four projections, shared by the
// decode GEMM (cc_gemm.cu: stream-K fixup) and the large-M GEMM (cc_big_gemm.cu: straight from TMEM).
// One warp owns one item = (tile t of 128 output features, grouped row p); lane l holds the four summed output
// features t*128 + 4l .. 4l+3 of original row b.  Each epilogue is split into `pre` (every global load that does
// not depend on the sum) and `fin` (math + stores).  TAB supplies the per-row tables: aux(p), page(p), and
// what the row's replica owns: blob(p), k_pool(p), v_pool(p), kv_pages(p).
#pragma once
#include "cc_kernels.h"

enum { EPI_QKV = 0, EPI_O = 1, EPI_GU = 2, EPI_DN = 3 };
struct CcEpi {
    const int* assign;          // replica_assign and batch: the QKV GEMM counts the groups itself
    int batch;
    const int* seq_lens;
    CcKv kv;
    __nv_bfloat16* hidden;
};
struct EpiPre {
    float4 f0, f1;      // QKV: (cos, sin) x 4; down: h1
    uint2 u0, u1;       // O: hidden bits, g2 bits
};

template <int KIND, class TAB>
__device__ __forceinline__ void epi_pre(EpiPre& P, const CcEpi& E, const CcDims& D, const CcWork& W, const TAB& H,
                                        int t, int p, int b, int lane) {
    const int col = t * 128 + 4 * lane;
    if (KIND == EPI_QKV) {
        if (col < D.QD + D.KD) {
            const int half = D.Dh >> 1;
            const float4* cs = reinterpret_cast<const float4*>(W.rope_cs + (size_t)H.aux(p) * half + ((col % D.Dh) % half));
            P.f0 = cs[0];
            P.f1 = cs[1];
        }
    } else if (KIND == EPI_O) {
        if (col < D.d) {
            const uint8_t* blob = H.blob(p);
            P.u0 = *reinterpret_cast<const uint2*>(E.hidden + (size_t)b * D.d + col);
            P.u1 = *reinterpret_cast<const uint2*>(blob + D.off_g2 + (size_t)col * 2);
        }
    } else if (KIND == EPI_DN) {
        if (col < D.d) P.f0 = *reinterpret_cast<const float4*>(W.h1 + (size_t)p * D.d + col);
    }
}

template <int KIND, class TAB>
__device__ __forceinline__ void epi_fin(const EpiPre& P, const CcEpi& E, const CcDims& D, const CcWork& W,
                                        const TAB& H, int t, int p, int b, float4 a, int lane) {
    const int col = t * 128 + 4 * lane;
    if (KIND == EPI_QKV) {
        // a3 + a4: RoPE at position s-1 (rotate-half pairs (i, i + Dh/2), fp64-built cos/sin table), q kept
        // in fp32, bf16(k), bf16(v) stored into the page slot of position s-1 (PAPER.md:103 local append).
        const int hl = D.Dh >> 3;                                // lanes per half head: 16 (Dh 128) or 8 (Dh 64)
        float4 o;                                                // the partner half of the same head
        o.x = __shfl_xor_sync(0xffffffffu, a.x, hl); o.y = __shfl_xor_sync(0xffffffffu, a.y, hl);
        o.z = __shfl_xor_sync(0xffffffffu, a.z, hl); o.w = __shfl_xor_sync(0xffffffffu, a.w, hl);
        if (col >= D.QD + 2 * D.KD) return;                      // padding columns of the last tile
        const int pos = H.aux(p), i0 = col % D.Dh;
        if (col < D.QD + D.KD) {                                 // q or k: rotate
            const float sg = (lane & hl) ? 1.f : -1.f;           // first half: a cos - b sin; second: b cos + a sin
            a.x = a.x * P.f0.x + sg * o.x * P.f0.y; a.y = a.y * P.f0.z + sg * o.y * P.f0.w;
            a.z = a.z * P.f1.x + sg * o.z * P.f1.y; a.w = a.w * P.f1.z + sg * o.w * P.f1.w;
            if (col < D.QD) {
                *reinterpret_cast<float4*>(W.q_rot + (size_t)p * D.QD + col) = a;
                return;
            }
        }
        const int page = H.page(p);
        if (page < 0 || page >= H.kv_pages(p)) {
            if (lane == 0) atomicOr(W.err, CC_DEVERR_BAD_PAGE);
            return;
        }
        const bool is_k = col < D.QD + D.KD;
        const int hk = (col - D.QD - (is_k ? 0 : D.KD)) / D.Dh;
        __nv_bfloat16* dst = (is_k ? H.k_pool(p) : H.v_pool(p)) + (((size_t)page * D.Hkv + hk) * CC_PAGE + pos % CC_PAGE) * D.Dh + i0;
        *reinterpret_cast<uint2*>(dst) = make_uint2(pack_bf16(a.x, a.y), pack_bf16(a.z, a.w));
    } else if (KIND == EPI_O) {
        // a6 + first half of a7: h1 = h + O-projection (kept in fp32); sum of squares of this tile's 128
        // columns (the RMSNorm statistic; the 1/rms factor is applied by the gate/up epilogue, the GEMM
        // being linear in a per-row scale); operand y' = h1 * g2 * (1/rms of the INPUT row, known already).
        float ss = 0.f;
        if (col < D.d) {
            a.x += bf16lo(P.u0.x); a.y += bf16hi(P.u0.x); a.z += bf16lo(P.u0.y); a.w += bf16hi(P.u0.y);
            *reinterpret_cast<float4*>(W.h1 + (size_t)p * D.d + col) = a;
            ss = (a.x * a.x + a.y * a.y) + (a.z * a.z + a.w * a.w);
            const float sc = __int_as_float(H.aux(p));           // 1/rms of the input row: keeps y' of order 1 (fp16 range)
            const float y[4] = {a.x * bf16lo(P.u1.x) * sc, a.y * bf16hi(P.u1.x) * sc, a.z * bf16lo(P.u1.y) * sc, a.w * bf16hi(P.u1.y) * sc};
            act_store<4>(W.y_act, D, D.pl[CC_OP_Y], p, col, y);
        }
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) ss += __shfl_xor_sync(0xffffffffu, ss, o);
        if (lane == 0 && t < ((D.d + 127) >> 7)) W.ssq[(size_t)t * D.Mpad + p] = ss;   // not the zero padding tile of an odd tile count
    } else if (KIND == EPI_GU) {
        // second half of a7 + a8: scale by 1/rms of the row (over the factor the O epilogue put in), a_j = silu(gate_j) * up_j
        // with gate_j, up_j at interleaved columns 2j, 2j+1 -> operand of the down projection.
        const float inv = __int_as_float(H.aux(p));
        const float g0 = a.x * inv, u0 = a.y * inv, g1 = a.z * inv, u1 = a.w * inv;
        const int k = t * 64 + 2 * lane;                          // output index = K index of the down GEMM
        if (k >= D.dn.KB * CC_TILE_K) return;                     // padding tile of the last super tile
        const float av[2] = {g0 / (1.f + __expf(-g0)) * u0, g1 / (1.f + __expf(-g1)) * u1};
        act_store<2>(W.a_act, D, D.pl[CC_OP_A], p, k, av);
    } else {
        // a9: out[b] = bf16(h1 + down projection), written to row b = original request order.
        if (col >= D.d) return;
        *reinterpret_cast<uint2*>(E.hidden + (size_t)b * D.d + col) =
            make_uint2(pack_bf16(P.f0.x + a.x, P.f0.y + a.y), pack_bf16(P.f0.z + a.z, P.f0.w + a.w));
    }
}

