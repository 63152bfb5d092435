// cc_kernels.cu -- replica creation kernels (sm_100a):
//   k_copy     a11  vectorised replica copy (256-bit accesses, streaming hints)
//   k_publish  a12  replica-table flip
//   k_pack          one-time re-pack of [out][in] weights into tcgen05 operand tile images
#include "cc_kernels.h"

namespace {

// ---------------------------------------------------------------------------------------------
// a11: vectorised copy, 4 x 32 B in flight per thread, streaming cache hints.
// ---------------------------------------------------------------------------------------------
constexpr int kCopyThreads = 512;
constexpr int kCopyUnroll = 4;
struct alignas(32) u32x8 { uint32_t v[8]; };
// 256-bit global accesses (sm_100): streaming load that does not linger in L1/L2, plain store.
__device__ __forceinline__ u32x8 ld_stream32(const u32x8* p) {
    u32x8 r;
    asm volatile("ld.global.nc.L1::no_allocate.L2::evict_first.v8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r.v[0]), "=r"(r.v[1]), "=r"(r.v[2]), "=r"(r.v[3]), "=r"(r.v[4]), "=r"(r.v[5]), "=r"(r.v[6]),
                   "=r"(r.v[7])
                 : "l"(p));
    return r;
}
__device__ __forceinline__ void st_stream32(u32x8* p, const u32x8& r) {
    asm volatile("st.global.L1::no_allocate.v8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"l"(p), "r"(r.v[0]), "r"(r.v[1]),
                 "r"(r.v[2]), "r"(r.v[3]), "r"(r.v[4]), "r"(r.v[5]), "r"(r.v[6]), "r"(r.v[7])
                 : "memory");
}
// n32 = number of 32-byte words; the (< 32 byte) remainder is copied as 16-byte words by block 0.
__global__ void __launch_bounds__(kCopyThreads) k_copy(u32x8* __restrict__ dst, const u32x8* __restrict__ src, size_t n32,
                                                       int tail16) {
    // Chunks are independent: let the next chunk's kernel start while this one drains (programmatic
    // dependent launch on the side stream) ...
    pdl_launch_dependents();
    const size_t span = (size_t)kCopyThreads * kCopyUnroll;
    const size_t stride = (size_t)gridDim.x * span;
    size_t base = (size_t)blockIdx.x * span;
    for (; base + span <= n32; base += stride) {
        u32x8 v[kCopyUnroll];
#pragma unroll
        for (int j = 0; j < kCopyUnroll; ++j) v[j] = ld_stream32(src + base + threadIdx.x + (size_t)j * kCopyThreads);
#pragma unroll
        for (int j = 0; j < kCopyUnroll; ++j) st_stream32(dst + base + threadIdx.x + (size_t)j * kCopyThreads, v[j]);
    }
    if (base < n32) {   // ragged tail of this block's last span
        for (size_t i = base + threadIdx.x; i < n32 && i < base + span; i += kCopyThreads) st_stream32(dst + i, ld_stream32(src + i));
    }
    if (tail16 && blockIdx.x == 0 && threadIdx.x == 0)
        reinterpret_cast<uint4*>(dst + n32)[0] = reinterpret_cast<const uint4*>(src + n32)[0];
    // ... but do not retire before the previous chunk has: the event recorded after the last chunk
    // then covers every chunk of the replica.
    pdl_wait();
}

// KV page migration (NEXT-1): block (move i, pool) copies one page of all kv heads, 256-bit accesses.
__global__ void __launch_bounds__(256) k_page_copy(uint8_t* __restrict__ k_pool, uint8_t* __restrict__ v_pool, size_t page_bytes,
                                                   const int* __restrict__ src, const int* __restrict__ dst) {
    uint8_t* pool = blockIdx.y ? v_pool : k_pool;
    const u32x8* s = reinterpret_cast<const u32x8*>(pool + (size_t)src[blockIdx.x] * page_bytes);
    u32x8* d = reinterpret_cast<u32x8*>(pool + (size_t)dst[blockIdx.x] * page_bytes);
    const size_t n32 = page_bytes / 32;
    for (size_t i = threadIdx.x; i < n32; i += 4 * 256) {
        u32x8 v[4];
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (i + j * 256 < n32) v[j] = ld_stream32(s + i + j * 256);
#pragma unroll
        for (int j = 0; j < 4; ++j)
            if (i + j * 256 < n32) st_stream32(d + i + j * 256, v[j]);
    }
}

// a12: the flip.  One thread rewrites the layer's table row; ordering comes from the stream.
__global__ void k_publish(CcLayerTable* row, CcLayerTable value) {
    for (int r = 0; r < CC_MAXR; ++r) row->rep[r] = value.rep[r];
    __threadfence();
    row->active_mask = value.active_mask;
}

// One-time weight re-pack: [out][in] bf16 rows -> 16 KiB tile images (fp16 or bf16 elements: CcDims::fmt) (128 rows x 64 k, 128B swizzle),
// tile (t, kb) at cc_atom_off(k_blocks, t, kb): the CC_G tiles of a super tile are adjacent per k-block.
// Rows / k beyond the matrix are zero.
__global__ void __launch_bounds__(256) k_pack(uint8_t* __restrict__ dst, const __nv_bfloat16* __restrict__ src0,
                                              const __nv_bfloat16* __restrict__ src1,
                                              const __nv_bfloat16* __restrict__ src2, int rows0, int rows1, int rows2,
                                              int mode, int K, int n_tiles, int k_blocks, int fmt,
                                              uint32_t* __restrict__ overflow) {
    const size_t total = (size_t)n_tiles * k_blocks * (CC_A_TILE_BYTES / 16);
    for (size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x; idx < total; idx += (size_t)gridDim.x * blockDim.x) {
        const int c = idx & 7, i = (idx >> 3) & 127;
        const size_t tk = idx >> 10;
        const int kb = (int)(tk % k_blocks), t = (int)(tk / k_blocks);
        const int n = t * CC_TILE_N + i, k0 = kb * CC_TILE_K + c * 8;
        const __nv_bfloat16* row = nullptr;
        if (mode == 0) {
            if (n < rows0) row = src0 + (size_t)n * K;
            else if (n < rows0 + rows1) row = src1 + (size_t)(n - rows0) * K;
            else if (n < rows0 + rows1 + rows2) row = src2 + (size_t)(n - rows0 - rows1) * K;
        } else {
            const int j = n >> 1;
            if (j < rows0) row = ((n & 1) ? src1 : src0) + (size_t)j * K;
        }
        uint4 v = make_uint4(0, 0, 0, 0);
        if (row && k0 < K) v = *reinterpret_cast<const uint4*>(row + k0);   // K % 8 == 0
        if (fmt == CC_FMT_F16) {
            // bf16 -> fp16: exact for 2^-17 <= |w| <= 65504 (fp16 subnormals included), rounded to the 2^-24 grid below that
            uint32_t w[4] = {v.x, v.y, v.z, v.w};
            bool bad = false;
#pragma unroll
            for (int j = 0; j < 4; ++j) {
                const float a = bf16lo(w[j]), b = bf16hi(w[j]);
                bad |= !(fabsf(a) <= 65504.f) || !(fabsf(b) <= 65504.f);
                w[j] = pack_f16(a, b);
            }
            if (bad) atomicOr(overflow, 1u);
            v = make_uint4(w[0], w[1], w[2], w[3]);
        }
        *reinterpret_cast<uint4*>(dst + cc_atom_off(k_blocks, t, kb) + (size_t)i * 128 + ((c ^ (i & 7)) << 4)) = v;
    }
}

}  // namespace

cudaError_t cc_launch_copy(void* dst, const void* src, size_t bytes, int n_sms, cudaStream_t st) {
    if (bytes == 0) return cudaSuccess;
    if (((((uintptr_t)dst) | ((uintptr_t)src)) & 31) || (bytes & 15)) return cudaErrorInvalidValue;
    const size_t n32 = bytes / 32;
    const int tail16 = (bytes % 32) ? 1 : 0;
    const size_t span = (size_t)kCopyThreads * kCopyUnroll;
    size_t blocks = (n32 + span - 1) / span;
    if (blocks == 0) blocks = 1;
    const size_t cap = (size_t)n_sms * 4;   // 4 resident blocks of 512 threads per SM
    if (blocks > cap) blocks = cap;
    CcLaunch L{st, n_sms, true};
    return cc_launch_kernel(k_copy, dim3((unsigned)blocks), dim3(kCopyThreads), 0, L, reinterpret_cast<u32x8*>(dst),
                            reinterpret_cast<const u32x8*>(src), n32, tail16);
}
cudaError_t cc_launch_publish(CcLayerTable* row_dev, const CcLayerTable& value, cudaStream_t st) {
    k_publish<<<1, 1, 0, st>>>(row_dev, value);
    return cudaGetLastError();
}
cudaError_t cc_launch_pack(uint8_t* dst, const __nv_bfloat16* src0, const __nv_bfloat16* src1,
                           const __nv_bfloat16* src2, int rows0, int rows1, int rows2, int mode, int K, int n_tiles,
                           int k_blocks, int fmt, uint32_t* overflow_dev, cudaStream_t st) {
    k_pack<<<1184, 256, 0, st>>>(dst, src0, src1, src2, rows0, rows1, rows2, mode, K, n_tiles, k_blocks, fmt, overflow_dev);
    return cudaGetLastError();
}
cudaError_t cc_launch_page_copy(void* k_pool, void* v_pool, size_t page_bytes, const int* src, const int* dst, int n_moves,
                                cudaStream_t st) {
    if (n_moves <= 0) return cudaSuccess;
    k_page_copy<<<dim3((unsigned)n_moves, 2), 256, 0, st>>>((uint8_t*)k_pool, (uint8_t*)v_pool, page_bytes, src, dst);
    return cudaGetLastError();
}
