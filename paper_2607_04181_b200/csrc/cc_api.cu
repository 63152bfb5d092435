// cc_api.cu -- host side of libcocoscale: the C ABI of include/cocoscale.h (product code).
// Context, weight-slot allocator over donated ("reclaimed") HBM, replica state machine, device
// replica table, chunked side-stream replica copy, and the enqueue-only forward chain.
#include "../../include/cocoscale.h"
#include "cc_kernels.h"

#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <cstring>
#include <map>
#include <new>
#include <string>
#include <vector>

cudaError_t cc_gemm_configure();
cudaError_t cc_attn_configure();
cudaError_t cc_big_gemm_configure();
cudaError_t cc_prefill_configure();

namespace {

thread_local std::string g_err;

cc_status fail(cc_status st, const char* fmt, ...) {
    char buf[512];
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(buf, sizeof buf, fmt, ap);
    va_end(ap);
    g_err = buf;
    return st;
}
}  // namespace
// for the other translation units of the library (cc_noalloc.cu): what cc_last_error() returns on this thread
void cc_internal_set_error(const char* msg) { g_err = msg ? msg : ""; }
namespace {
#define CC_CUDA(expr)                                                                              \
    do {                                                                                           \
        cudaError_t e_ = (expr);                                                                   \
        if (e_ != cudaSuccess) return fail(CC_ERR_CUDA, "%s: %s", #expr, cudaGetErrorString(e_)); \
    } while (0)

constexpr uint64_t kSlotAlign = 1024;
inline uint64_t up(uint64_t x, uint64_t a) { return (x + a - 1) / a * a; }

}  // namespace

// ---- slot allocator (host only; also exported for CPU tests) ------------------------------------
// Address-ordered: donated ranges keyed by the base the caller passed, live allocations in one
// ordered map.  alloc = first fit inside each range, lowest address over all ranges.
struct cc_slotalloc {
    struct Range { uint64_t key, lo, hi; };
    std::vector<Range> ranges;
    std::map<uint64_t, uint64_t> live;   // addr -> size (rounded up to kSlotAlign)
};

extern "C" {

cc_slotalloc* cc_slotalloc_create(void) { return new (std::nothrow) cc_slotalloc(); }
void cc_slotalloc_destroy(cc_slotalloc* a) { delete a; }

cc_status cc_slotalloc_donate(cc_slotalloc* a, uint64_t base, uint64_t bytes) {
    if (!a) return fail(CC_ERR_INVALID, "null allocator");
    const uint64_t lo = up(base, kSlotAlign), hi = (base + bytes) / kSlotAlign * kSlotAlign;
    if (hi <= lo) return fail(CC_ERR_INVALID, "donated range is empty after trimming to %llu-byte boundaries",
                              (unsigned long long)kSlotAlign);
    for (const auto& r : a->ranges)
        if (r.key == base || (lo < r.hi && r.lo < hi)) return fail(CC_ERR_INVALID, "range overlaps a donated range");
    a->ranges.push_back({base, lo, hi});
    return CC_OK;
}

cc_status cc_slotalloc_reclaim(cc_slotalloc* a, uint64_t base) {
    if (!a) return fail(CC_ERR_INVALID, "null allocator");
    for (size_t i = 0; i < a->ranges.size(); ++i) {
        if (a->ranges[i].key != base) continue;
        const auto& r = a->ranges[i];
        auto it = a->live.lower_bound(r.lo);
        if (it != a->live.end() && it->first < r.hi) return fail(CC_ERR_BUSY, "range still holds a live slot");
        a->ranges.erase(a->ranges.begin() + i);
        return CC_OK;
    }
    return fail(CC_ERR_INVALID, "range was not donated");
}

cc_status cc_slotalloc_alloc(cc_slotalloc* a, uint64_t bytes, uint64_t* addr) {
    if (!a || !addr) return fail(CC_ERR_INVALID, "null argument");
    const uint64_t size = up(bytes ? bytes : 1, kSlotAlign);
    bool found = false;
    uint64_t best = 0;
    for (const auto& r : a->ranges) {
        uint64_t cur = r.lo;   // walk the gaps between live allocations of this range
        for (auto it = a->live.lower_bound(r.lo); it != a->live.end() && it->first < r.hi; ++it) {
            if (it->first >= cur + size) break;
            cur = it->first + it->second;
        }
        if (cur + size <= r.hi && (!found || cur < best)) {
            found = true;
            best = cur;
        }
    }
    if (!found) return fail(CC_ERR_NO_SLOT, "no donated range can hold %llu bytes", (unsigned long long)size);
    a->live[best] = size;
    *addr = best;
    return CC_OK;
}

cc_status cc_slotalloc_free(cc_slotalloc* a, uint64_t addr) {
    if (!a) return fail(CC_ERR_INVALID, "null allocator");
    if (!a->live.erase(addr)) return fail(CC_ERR_INVALID, "address is not a live slot");
    return CC_OK;
}

uint64_t cc_slotalloc_free_bytes(const cc_slotalloc* a) {
    if (!a) return 0;
    uint64_t tot = 0;
    for (const auto& r : a->ranges) tot += r.hi - r.lo;
    for (const auto& kv : a->live) tot -= kv.second;
    return tot;
}

const char* cc_last_error(void) { return g_err.c_str(); }
const char* cc_version(void) { return "cocoscale-b200 0.1 (sm_100a)"; }

}  // extern "C"

// ---- context ----------------------------------------------------------------------------------
namespace {
enum RepState { REP_EMPTY = 0, REP_COPYING = 1, REP_LIVE = 2, REP_RETIRING = 3 };
struct Replica {
    int state = REP_EMPTY;
    uint8_t* blob = nullptr;
    cudaEvent_t copied = nullptr;   // recorded on the side stream after the last chunk
    bool published = false;         // named in the device table row
};
struct Zombie {                     // a retired slot waiting for its last reader
    uint64_t addr;
    cudaEvent_t after_flip;
};
}  // namespace

struct cc_ctx {
    int device = 0, n_sms = 0;
    cudaStream_t side = nullptr;
    cc_slotalloc* slots = nullptr;
    CcLayerTable* table_dev = nullptr;   // [CC_MAX_LAYERS], fixed address for the life of the context
    uint32_t* err_dev = nullptr;
    unsigned long long* trace_dev = nullptr;   // CC_TRACE builds only
    size_t chunk = (size_t)32 << 20;
    bool row_used[CC_MAX_LAYERS] = {};
    int n_layers = 0;
    bool pdl = true;
    bool cluster_gemm = true;                  // small steps run QKV / O / down as cluster split-K (CC_CLUSTER_GEMM=0: stream-K everywhere)
    int operand_format = CC_OPERAND_AUTO;      // layers created from now on (cc_ctx_set_operand_format)
    // activation planes of the four GEMM operands (x, o, y, a) of an fp16 layer, per step: steps of at most
    // `planes_rows` rows take planes_small, larger ones planes_large (cc_ctx_set_operand_planes).
    // Both default to {2, 1, 1, 1}: the QKV input is the operand whose rounding shows (measured), and a second plane
    // of the others costs ring depth even where the tensor work is free (4 instead of 5 stages at batch 64: +4 us)
    int planes_rows = 64;
    int planes_small[4] = {2, 1, 1, 1};
    int planes_large[4] = {2, 1, 1, 1};
    // L2 weight prefetch of the small-step cluster GEMMs (CcDims::pf_next / pf_self; env CC_PREFETCH="next,self" for
    // experiments).  Measured at cfg2: 3 / 4 stages take 2-3 us off the step at every replica count; 6 / 8
    // gain nothing, 12 / 16 and more LOSE 5-10 us
    int pf_next = 3, pf_self = 4;
    std::vector<Zombie> zombies;
};

struct cc_layer {
    cc_ctx* ctx = nullptr;
    int row = -1;
    cc_layer_desc desc{};
    CcDims D{};
    CcWork W{};
    size_t blob_bytes = 0;
    uint8_t* blob0 = nullptr;
    uint8_t* work_base = nullptr;
    Replica rep[CC_MAX_REPLICAS];
    CcLayerTable host_row{};
    // staging for cc_forward_host
    __nv_bfloat16* st_hidden = nullptr;
    int* st_bt = nullptr;
    int* st_sl = nullptr;
    int* st_ra = nullptr;
    void* st_tbl_host = nullptr;         // pinned mirrors of [st_sl | st_ra | st_bt]: a ring of kTblRing, so that an enqueue-only
                                         // host step can fill the next one while the previous copy is still in flight
    size_t st_tbl_bytes = 0;
    cudaEvent_t st_tbl_done[4] = {};     // recorded after the copy out of mirror i
    unsigned st_tbl_next = 0;
    struct { void* k; void* v; int n; } kvp[CC_MAX_REPLICAS] = {};   // a replica's own KV partition (cc_layer_set_kv_partition)
    bool big = false;                    // created with max_batch > 256: steps of more than 256 rows take the large-M path
    int last_batch = 0;
    int last_pl[4] = {2, 2, 2, 2};       // plane counts of the last forward (cc_debug_tap reads the operands back)
};

namespace {

void reap_zombies(cc_ctx* ctx, bool block) {
    for (size_t i = 0; i < ctx->zombies.size();) {
        Zombie& z = ctx->zombies[i];
        cudaError_t e = block ? cudaEventSynchronize(z.after_flip) : cudaEventQuery(z.after_flip);
        if (e == cudaSuccess) {
            cc_slotalloc_free(ctx->slots, z.addr);
            cudaEventDestroy(z.after_flip);
            ctx->zombies.erase(ctx->zombies.begin() + i);
        } else {
            if (e != cudaErrorNotReady) cudaGetLastError();
            ++i;
        }
    }
}

cc_status set_device(cc_ctx* ctx) {
    CC_CUDA(cudaSetDevice(ctx->device));
    return CC_OK;
}

cc_status launch_chunked_copy(cc_ctx* ctx, void* dst, const void* src, size_t bytes, size_t chunk, cudaStream_t st) {
    if (chunk == 0) chunk = ctx->chunk;
    for (size_t off = 0; off < bytes; off += chunk) {
        const size_t n = bytes - off < chunk ? bytes - off : chunk;
        CC_CUDA(cc_launch_copy((uint8_t*)dst + off, (const uint8_t*)src + off, n, ctx->n_sms, st));
    }
    return CC_OK;
}

}  // namespace

extern "C" {

cc_status cc_ctx_create(int device, cc_ctx** out) {
    if (!out) return fail(CC_ERR_INVALID, "out is null");
    *out = nullptr;
    int n_dev = 0;
    if (cudaGetDeviceCount(&n_dev) != cudaSuccess || n_dev == 0) {
        cudaGetLastError();
        return fail(CC_ERR_CUDA, "no CUDA device (this library has no CPU fallback)");
    }
    if (device < 0 || device >= n_dev) return fail(CC_ERR_INVALID, "device %d out of range", device);
    cudaDeviceProp prop;
    CC_CUDA(cudaGetDeviceProperties(&prop, device));
    if (prop.major != 10) return fail(CC_ERR_CUDA, "device is sm_%d%d; this library is sm_100a only", prop.major, prop.minor);
    cc_ctx* ctx = new (std::nothrow) cc_ctx();
    if (!ctx) return fail(CC_ERR_INVALID, "out of host memory");
    ctx->device = device;
    ctx->n_sms = prop.multiProcessorCount;
    cudaError_t e = cudaSetDevice(device);
    if (e == cudaSuccess) e = cudaStreamCreateWithFlags(&ctx->side, cudaStreamNonBlocking);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->table_dev, sizeof(CcLayerTable) * CC_MAX_LAYERS);
    if (e == cudaSuccess) e = cudaMemset(ctx->table_dev, 0, sizeof(CcLayerTable) * CC_MAX_LAYERS);
    if (e == cudaSuccess) e = cudaMalloc(&ctx->err_dev, 256);
    if (e == cudaSuccess) e = cudaMemset(ctx->err_dev, 0, 256);
#ifdef CC_TRACE
    if (e == cudaSuccess) e = cudaMalloc(&ctx->trace_dev, sizeof(unsigned long long) * CC_TRACE_KERNELS * CC_TRACE_POINTS * 2);
#endif
    if (e == cudaSuccess) e = cc_gemm_configure();
    if (e == cudaSuccess) e = cc_attn_configure();
    if (e == cudaSuccess) e = cc_big_gemm_configure();
    if (e == cudaSuccess) e = cc_prefill_configure();
    if (e == cudaSuccess && !(ctx->slots = cc_slotalloc_create())) e = cudaErrorMemoryAllocation;
    if (e != cudaSuccess) {                       // nothing half-made is left behind
        if (ctx->side) cudaStreamDestroy(ctx->side);
        cudaFree(ctx->table_dev);
        cudaFree(ctx->err_dev);
        cudaFree(ctx->trace_dev);
        cc_slotalloc_destroy(ctx->slots);
        delete ctx;
        cudaGetLastError();
        return fail(CC_ERR_CUDA, "cc_ctx_create: %s", cudaGetErrorString(e));
    }
    const char* env = getenv("CC_PDL");
    if (env && env[0] == '0') ctx->pdl = false;
    env = getenv("CC_CLUSTER_GEMM");
    if (env && env[0] == '0') ctx->cluster_gemm = false;
    env = getenv("CC_PREFETCH");                // "next,self": weight stages prefetched into L2 across / inside the small-step GEMMs
    if (env) sscanf(env, "%d,%d", &ctx->pf_next, &ctx->pf_self);
    env = getenv("CC_PLANES");                  // "xoya,xoya[,rows]": planes of small and large steps, e.g. 2222,1212,64
    if (env && std::strlen(env) >= 9 && env[4] == ',') {
        bool ok = true;
        for (int i = 0; i < 4; ++i) ok &= (env[i] == '1' || env[i] == '2') && (env[5 + i] == '1' || env[5 + i] == '2');
        if (ok) {
            for (int i = 0; i < 4; ++i) { ctx->planes_small[i] = env[i] - '0'; ctx->planes_large[i] = env[5 + i] - '0'; }
            if (env[9] == ',') ctx->planes_rows = atoi(env + 10);
        }
    }
    env = getenv("CC_OPERAND_FORMAT");          // "f16" | "bf16x2": what cc_ctx_set_operand_format would set
    if (env && !std::strcmp(env, "f16")) ctx->operand_format = CC_OPERAND_F16;
    if (env && !std::strcmp(env, "bf16x2")) ctx->operand_format = CC_OPERAND_BF16X2;
    *out = ctx;
    return CC_OK;
}

cc_status cc_ctx_destroy(cc_ctx* ctx) {
    if (!ctx) return CC_OK;
    if (ctx->n_layers) return fail(CC_ERR_BUSY, "%d layer(s) still alive", ctx->n_layers);
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    reap_zombies(ctx, true);
    cudaStreamDestroy(ctx->side);
    cudaFree(ctx->table_dev);
    cudaFree(ctx->err_dev);
    cudaFree(ctx->trace_dev);
    cc_slotalloc_destroy(ctx->slots);
    delete ctx;
    return CC_OK;
}

cc_status cc_ctx_donate(cc_ctx* ctx, void* dev_base, size_t bytes) {
    if (!ctx || !dev_base) return fail(CC_ERR_INVALID, "null argument");
    return cc_slotalloc_donate(ctx->slots, (uint64_t)(uintptr_t)dev_base, bytes);
}

cc_status cc_ctx_reclaim(cc_ctx* ctx, void* dev_base) {
    if (!ctx) return fail(CC_ERR_INVALID, "null context");
    reap_zombies(ctx, false);
    cc_status st = cc_slotalloc_reclaim(ctx->slots, (uint64_t)(uintptr_t)dev_base);
    if (st == CC_ERR_BUSY && !ctx->zombies.empty()) {   // retired slots whose last reader is still running
        reap_zombies(ctx, true);
        st = cc_slotalloc_reclaim(ctx->slots, (uint64_t)(uintptr_t)dev_base);
    }
    return st;
}

cc_status cc_ctx_set_copy_chunk(cc_ctx* ctx, size_t chunk_bytes) {
    if (!ctx) return fail(CC_ERR_INVALID, "null context");
    if (chunk_bytes == 0 || chunk_bytes % ((size_t)1 << 20)) return fail(CC_ERR_INVALID, "chunk must be a multiple of 1 MiB");
    ctx->chunk = chunk_bytes;
    return CC_OK;
}

cc_status cc_ctx_set_pdl(cc_ctx* ctx, int enabled) {
    if (!ctx) return fail(CC_ERR_INVALID, "null context");
    ctx->pdl = enabled != 0;
    return CC_OK;
}

cc_status cc_ctx_set_operand_format(cc_ctx* ctx, int format) {
    if (!ctx) return fail(CC_ERR_INVALID, "null context");
    if (format != CC_OPERAND_AUTO && format != CC_OPERAND_F16 && format != CC_OPERAND_BF16X2)
        return fail(CC_ERR_INVALID, "unknown operand format %d", format);
    ctx->operand_format = format;
    return CC_OK;
}

cc_status cc_ctx_set_operand_planes(cc_ctx* ctx, int rows, const int* planes_upto_rows, const int* planes_above) {
    if (!ctx || !planes_upto_rows || !planes_above) return fail(CC_ERR_INVALID, "null argument");
    if (rows < 0) return fail(CC_ERR_INVALID, "rows must be >= 0");
    for (int i = 0; i < 4; ++i)
        if (planes_upto_rows[i] < 1 || planes_upto_rows[i] > 2 || planes_above[i] < 1 || planes_above[i] > 2)
            return fail(CC_ERR_INVALID, "plane counts must be 1 or 2");
    ctx->planes_rows = rows;
    for (int i = 0; i < 4; ++i) { ctx->planes_small[i] = planes_upto_rows[i]; ctx->planes_large[i] = planes_above[i]; }
    return CC_OK;
}

cc_status cc_poll_device_error(cc_ctx* ctx, uint32_t* bits) {
    if (!ctx || !bits) return fail(CC_ERR_INVALID, "null argument");
    CC_CUDA(cudaSetDevice(ctx->device));
    CC_CUDA(cudaDeviceSynchronize());
    CC_CUDA(cudaMemcpy(bits, ctx->err_dev, 4, cudaMemcpyDeviceToHost));
    CC_CUDA(cudaMemset(ctx->err_dev, 0, 4));
    return CC_OK;
}

cc_status cc_replica_copy(cc_ctx* ctx, void* dst_dev, const void* src_dev, size_t bytes, size_t chunk_bytes,
                          void* stream) {
    if (!ctx || !dst_dev || !src_dev) return fail(CC_ERR_INVALID, "null argument");
    if ((((uintptr_t)dst_dev | (uintptr_t)src_dev) & 31) || (bytes & 15))
        return fail(CC_ERR_INVALID, "pointers must be 32-byte aligned and the size a multiple of 16");
    if (set_device(ctx) != CC_OK) return CC_ERR_CUDA;
    return launch_chunked_copy(ctx, dst_dev, src_dev, bytes, chunk_bytes, (cudaStream_t)stream);
}

}  // extern "C"

// ---- layer lifecycle ----------------------------------------------------------------------------
namespace {

CcGemmGeo make_geo(int n_out, int k_in, int n_sms, size_t w_off) {
    CcGemmGeo g{};
    g.ST = (n_out + CC_G * CC_TILE_N - 1) / (CC_G * CC_TILE_N);
    g.KB = (k_in + CC_TILE_K - 1) / CC_TILE_K;
    const long long units = (long long)g.ST * g.KB;
    g.P = units < n_sms ? (int)units : n_sms;   // no empty range => every piece slot is written
    g.w_off = w_off;
    return g;
}
size_t geo_bytes(const CcGemmGeo& g) { return (size_t)g.ST * CC_G * g.KB * CC_A_TILE_BYTES; }

struct Carver {   // bump allocator over one cudaMalloc
    size_t off = 0;
    size_t take(size_t bytes, size_t align = 1024) {
        off = (off + align - 1) / align * align;
        const size_t r = off;
        off += bytes;
        return r;
    }
};

void destroy_layer_memory(cc_layer* L) {
    cudaFree(L->blob0);
    cudaFree(L->work_base);
    if (L->st_tbl_host) cudaFreeHost(L->st_tbl_host);
    for (auto& ev : L->st_tbl_done)
        if (ev) cudaEventDestroy(ev);
}

// cc_forward_host: the three per-step tables through the layer's pinned mirror, one host-to-device copy.
constexpr int kTblRing = 4;
cudaError_t stage_tables(cc_layer* L, const int32_t* bt, const int32_t* sl, const int32_t* ra, int batch, cudaStream_t st) {
    const size_t mb = (size_t)L->desc.max_batch, bb = (size_t)batch * L->desc.max_blocks_per_seq * 4;
    const int slot = (int)(L->st_tbl_next++ % kTblRing);
    cudaError_t e = cudaEventSynchronize(L->st_tbl_done[slot]);       // the copy that last read this mirror (no-op if none)
    if (e != cudaSuccess) return e;
    uint8_t* h = (uint8_t*)L->st_tbl_host + (size_t)slot * L->st_tbl_bytes;
    std::memcpy(h, sl, (size_t)batch * 4);
    std::memcpy(h + mb * 4, ra, (size_t)batch * 4);
    std::memcpy(h + mb * 8, bt, bb);
    e = cudaMemcpyAsync(L->st_sl, h, mb * 8 + bb, cudaMemcpyHostToDevice, st);
    if (e == cudaSuccess) e = cudaEventRecord(L->st_tbl_done[slot], st);
    return e;
}

}  // namespace

extern "C" {

cc_status cc_create_layer(cc_ctx* ctx, const cc_layer_desc* desc, const cc_layer_weights* w, cc_layer** out) {
    if (!ctx || !desc || !w || !out) return fail(CC_ERR_INVALID, "null argument");
    *out = nullptr;
    const cc_layer_desc& d = *desc;
    if (d.hidden <= 0 || d.hidden % 64 || d.hidden > cc_max_hidden())
        return fail(CC_ERR_INVALID, "hidden must be a positive multiple of 64, at most %d", cc_max_hidden());
    if (d.head_dim != 64 && d.head_dim != 128) return fail(CC_ERR_INVALID, "head_dim must be 64 or 128");
    if (d.n_kv_heads <= 0 || d.n_q_heads <= 0 || d.n_q_heads % d.n_kv_heads || d.n_q_heads / d.n_kv_heads > 8)
        return fail(CC_ERR_INVALID, "need n_q_heads %% n_kv_heads == 0 and a GQA group of at most 8");
    if (8 % d.n_kv_heads) return fail(CC_ERR_INVALID, "n_kv_heads must be 1, 2, 4 or 8 (one page of all kv heads is staged per TMA box)");
    if (d.ffn <= 0 || d.ffn % 8) return fail(CC_ERR_INVALID, "ffn must be a positive multiple of 8");
    if (d.page_size != CC_PAGE_SIZE) return fail(CC_ERR_INVALID, "page_size must be %d", CC_PAGE_SIZE);
    if (d.max_batch < 1 || d.max_batch > CC_BIG_MAX_ROWS) return fail(CC_ERR_INVALID, "max_batch must be in 1..%d", CC_BIG_MAX_ROWS);
    if (d.max_batch > 256 && d.head_dim != 128)
        return fail(CC_ERR_INVALID, "steps of more than 256 rows (mixed prefill + decode) need head_dim 128");
    if (d.max_blocks_per_seq < 1 || d.max_position < 1) return fail(CC_ERR_INVALID, "max_blocks_per_seq / max_position must be >= 1");
    if (!(d.rms_eps > 0.f) || !(d.rope_base > 1.f)) return fail(CC_ERR_INVALID, "bad rms_eps / rope_base");
    const void* ptrs[9] = {w->g1, w->wq, w->wk, w->wv, w->wo, w->g2, w->wgate, w->wup, w->wdown};
    for (const void* p : ptrs)
        if (!p || ((uintptr_t)p & 15)) return fail(CC_ERR_INVALID, "weight pointers must be non-null and 16-byte aligned");
    int row = -1;
    for (int i = 0; i < CC_MAX_LAYERS; ++i)
        if (!ctx->row_used[i]) { row = i; break; }
    if (row < 0) return fail(CC_ERR_INVALID, "context already holds %d layers", CC_MAX_LAYERS);
    CC_CUDA(cudaSetDevice(ctx->device));

    cc_layer* L = new (std::nothrow) cc_layer();
    if (!L) return fail(CC_ERR_INVALID, "out of host memory");
    L->ctx = ctx;
    L->row = row;
    L->desc = d;
    CcDims& D = L->D;
    D.d = d.hidden; D.Hq = d.n_q_heads; D.Hkv = d.n_kv_heads; D.Dh = d.head_dim; D.G = D.Hq / D.Hkv; D.F = d.ffn;
    D.QD = D.Hq * D.Dh; D.KD = D.Hkv * D.Dh;
    D.max_batch = d.max_batch; D.max_blocks = d.max_blocks_per_seq; D.max_position = d.max_position;
    D.Mpad = (d.max_batch + 15) / 16 * 16 + 16 * CC_MAXR;
    D.Mpart = D.Mpad < CC_MAX_MPAD ? D.Mpad : CC_MAX_MPAD;
    const bool big = d.max_batch > 256;                       // the layer also takes steps of more than 256 rows
    D.fmt = ctx->operand_format == CC_OPERAND_BF16X2 ? CC_FMT_BF16X2 : CC_FMT_F16;   // AUTO: fp16 unless a weight overflows it (below)
    for (int i = 0; i < 4; ++i) D.pl[i] = 2;                                           // per step: step_dims()
    D.pf_next = D.pf_self = 0;
    D.eps = d.rms_eps;
    D.qk_scale_log2 = (float)(1.4426950408889634 / std::sqrt((double)D.Dh));
    // blob layout: [QKV tiles][O tiles][gate/up tiles][down tiles][g1][g2]
    Carver blob;
    D.qkv = make_geo(D.QD + 2 * D.KD, D.d, ctx->n_sms, 0);
    D.qkv.w_off = blob.take(geo_bytes(D.qkv));
    D.o = make_geo(D.d, D.QD, ctx->n_sms, 0);
    D.o.w_off = blob.take(geo_bytes(D.o));
    D.gu = make_geo(2 * D.F, D.d, ctx->n_sms, 0);
    D.gu.w_off = blob.take(geo_bytes(D.gu));
    D.dn = make_geo(D.d, D.F, ctx->n_sms, 0);
    D.dn.w_off = blob.take(geo_bytes(D.dn));
    D.off_g1 = blob.take((size_t)D.d * 2);
    D.off_g2 = blob.take((size_t)D.d * 2);
    L->blob_bytes = blob.take(0);
    if (ctx->cluster_gemm) {
        cc_gemm_cl_geometry(0, D.qkv, ctx->n_sms);
        cc_gemm_cl_geometry(1, D.o, ctx->n_sms);
        cc_gemm_cl_geometry(2, D.gu, ctx->n_sms);
        cc_gemm_cl_geometry(3, D.dn, ctx->n_sms);
    }
    if (D.qkv.ST > CC_FLAG_STRIDE || D.o.ST > CC_FLAG_STRIDE || D.gu.ST > CC_FLAG_STRIDE || D.dn.ST > CC_FLAG_STRIDE ||
        D.Mpart > CC_MAX_MPAD) {
        delete L;
        return fail(CC_ERR_INVALID, "shape exceeds the stream-K bookkeeping limits (%d super tiles, %d rows)", CC_FLAG_STRIDE, CC_MAX_MPAD);
    }

    // workspace
    CcWork& W = L->W;
    Carver ws;
    const size_t Mp = (size_t)D.Mpad;
    const size_t o_sched = ws.take(sizeof(CcSched));
    const size_t o_perm = ws.take(Mp * 4);
    const size_t o_pgpre = ws.take((size_t)((d.max_batch > CC_BIG_MAX_DEC ? d.max_batch : CC_BIG_MAX_DEC) + 1) * 4);
    const size_t o_posof = ws.take((size_t)d.max_batch * 4);
    const size_t o_fwr = ws.take((size_t)d.max_batch * 4);
    // operands: sized for two planes (the plane count is a per-step choice); a large step's last row block reads up
    // to 256 rows past the last group, so the buffers carry that much slack behind them
    const size_t slack = big ? (size_t)2 * 256 * 128 : 0;
    const size_t o_x = ws.take((size_t)2 * D.qkv.KB * Mp * 128 + slack);
    const size_t o_o = ws.take((size_t)2 * D.o.KB * Mp * 128 + slack);
    const size_t o_y = ws.take((size_t)2 * D.gu.KB * Mp * 128 + slack);
    const size_t o_a = ws.take((size_t)2 * D.dn.KB * Mp * 128 + slack);
    const size_t o_invin = ws.take(Mp * 4);
    const size_t o_bs = ws.take(sizeof(CcBigSched));
    const size_t o_rpos = ws.take(big ? Mp * 4 : 0), o_rpage = ws.take(big ? Mp * 4 : 0), o_gus = ws.take(big ? Mp * 4 : 0);
    const size_t o_dec = ws.take((size_t)(CC_BIG_MAX_DEC + 1) * 4);
    const size_t o_cr0 = ws.take((size_t)CC_BIG_MAX_CHUNKS * 4), o_clen = ws.take((size_t)CC_BIG_MAX_CHUNKS * 4);
    const size_t o_ic = ws.take((size_t)CC_BIG_MAX_ITEMS * 4), o_it = ws.take((size_t)CC_BIG_MAX_ITEMS * 4);
    auto part_bytes = [&](const CcGemmGeo& g) { return (size_t)(g.P + g.ST) * CC_G * D.Mpart * 128 * 4; };
    const size_t o_pq = ws.take(part_bytes(D.qkv));
    const size_t o_po = ws.take(part_bytes(D.o));
    const size_t o_pg = ws.take(part_bytes(D.gu));
    const size_t o_pd = ws.take(part_bytes(D.dn));
    const size_t o_qrot = ws.take(Mp * D.QD * 4);
    const size_t o_h1 = ws.take(Mp * D.d * 4);
    const size_t o_ssq = ws.take((size_t)((D.d + 127) / 128) * Mp * 4);
    const size_t o_flags = ws.take((size_t)4 * CC_FLAG_STRIDE * 4);
    const size_t o_acnt = ws.take(Mp * D.Hkv * 4);
    const size_t n_slots = (size_t)d.max_batch + ctx->n_sms;          // attention pieces: one per (row, CTA) overlap
    const size_t o_atto = ws.take(n_slots * D.Hq * D.Dh * 4);
    const size_t o_attml = ws.take(n_slots * D.Hq * sizeof(float2));
    const size_t o_rope = ws.take((size_t)d.max_position * (D.Dh / 2) * sizeof(float2));
    const size_t o_sth = ws.take((size_t)d.max_batch * D.d * 2);
    // cc_forward_host's tables as one region [seq_lens | replica_assign | block table]: one copy from a pinned mirror
    const size_t tbl_bytes = (size_t)d.max_batch * 8 + (size_t)d.max_batch * d.max_blocks_per_seq * 4;
    const size_t o_tbl = ws.take(tbl_bytes);
    const size_t ws_bytes = ws.take(0);

    cudaError_t e = cudaMalloc(&L->blob0, L->blob_bytes);
    if (e == cudaSuccess) e = cudaMalloc(&L->work_base, ws_bytes);
    L->st_tbl_bytes = (tbl_bytes + 255) / 256 * 256;
    if (e == cudaSuccess) e = cudaHostAlloc(&L->st_tbl_host, L->st_tbl_bytes * kTblRing, cudaHostAllocDefault);
    for (int i = 0; i < kTblRing && e == cudaSuccess; ++i) e = cudaEventCreateWithFlags(&L->st_tbl_done[i], cudaEventDisableTiming);
    if (e == cudaSuccess) e = cudaMemset(L->work_base, 0, ws_bytes);
    if (e == cudaSuccess) e = cudaMemset(L->blob0, 0, L->blob_bytes);
    if (e != cudaSuccess) {
        const size_t blob_bytes = L->blob_bytes;
        destroy_layer_memory(L);
        delete L;
        cudaGetLastError();
        return fail(CC_ERR_CUDA, "device allocation of %zu + %zu bytes failed: %s", blob_bytes, ws_bytes, cudaGetErrorString(e));
    }
    uint8_t* wb = L->work_base;
    W.sched = (CcSched*)(wb + o_sched); W.perm = (int*)(wb + o_perm); W.pg_prefix = (int*)(wb + o_pgpre); W.pos_of = (int*)(wb + o_posof);
    W.first_wr = (int*)(wb + o_fwr);
    W.x_act = wb + o_x; W.o_act = wb + o_o; W.y_act = wb + o_y; W.a_act = wb + o_a;
    W.qkv_part = (float*)(wb + o_pq); W.o_part = (float*)(wb + o_po); W.gu_part = (float*)(wb + o_pg);
    W.d_part = (float*)(wb + o_pd);
    W.q_rot = (float*)(wb + o_qrot); W.h1 = (float*)(wb + o_h1);
    W.ssq = (float*)(wb + o_ssq); W.flags = (int*)(wb + o_flags);
    W.inv_in = (float*)(wb + o_invin);
    W.bs = (CcBigSched*)(wb + o_bs);
    W.row_pos = (int*)(wb + o_rpos); W.row_page = (int*)(wb + o_rpage); W.gu_scale = (float*)(wb + o_gus);
    W.dec_rows = (int*)(wb + o_dec); W.chunk_row0 = (int*)(wb + o_cr0); W.chunk_len = (int*)(wb + o_clen);
    W.item_chunk = (int*)(wb + o_ic); W.item_tile = (int*)(wb + o_it);
    L->big = big;
    W.attn_cnt = (int*)(wb + o_acnt);
    W.att_o = (float*)(wb + o_atto); W.att_ml = (float2*)(wb + o_attml);
    W.rope_cs = (const float2*)(wb + o_rope);
    W.err = ctx->err_dev;
    W.trace = ctx->trace_dev;
    L->st_hidden = (__nv_bfloat16*)(wb + o_sth);
    L->st_sl = (int*)(wb + o_tbl); L->st_ra = L->st_sl + d.max_batch; L->st_bt = L->st_ra + d.max_batch;

    // RoPE table in fp64 on the host: angle = p * base^(-2i/Dh)  (rotate-half pairing, reading 4)
    {
        const int half = D.Dh / 2;
        std::vector<float2> tab((size_t)d.max_position * half);
        for (int i = 0; i < half; ++i) {
            const double inv_freq = std::pow((double)d.rope_base, -2.0 * i / D.Dh);
            for (int p = 0; p < d.max_position; ++p) {
                const double th = (double)p * inv_freq;
                tab[(size_t)p * half + i] = make_float2((float)std::cos(th), (float)std::sin(th));
            }
        }
        e = cudaMemcpy(wb + o_rope, tab.data(), tab.size() * sizeof(float2), cudaMemcpyHostToDevice);
    }
    // one-time re-pack of the nine tensors into the blob (tcgen05 operand tile images + gains).  fp16 images unless a
    // weight does not fit fp16 (then, in AUTO, the layer falls back to bf16 images and two activation planes).
    typedef const __nv_bfloat16* bp;
    uint32_t* ovf = ctx->err_dev + 16;
    for (int attempt = 0; attempt < 2 && e == cudaSuccess; ++attempt) {
        e = cudaMemset(ovf, 0, 4);
        if (e == cudaSuccess)
            e = cc_launch_pack(L->blob0 + D.qkv.w_off, (bp)w->wq, (bp)w->wk, (bp)w->wv, D.QD, D.KD, D.KD, 0, D.d, D.qkv.ST * CC_G,
                               D.qkv.KB, D.fmt, ovf, 0);
        if (e == cudaSuccess)
            e = cc_launch_pack(L->blob0 + D.o.w_off, (bp)w->wo, nullptr, nullptr, D.d, 0, 0, 0, D.QD, D.o.ST * CC_G, D.o.KB, D.fmt, ovf, 0);
        if (e == cudaSuccess)
            e = cc_launch_pack(L->blob0 + D.gu.w_off, (bp)w->wgate, (bp)w->wup, nullptr, D.F, D.F, 0, 1, D.d, D.gu.ST * CC_G,
                               D.gu.KB, D.fmt, ovf, 0);
        if (e == cudaSuccess)
            e = cc_launch_pack(L->blob0 + D.dn.w_off, (bp)w->wdown, nullptr, nullptr, D.d, 0, 0, 0, D.F, D.dn.ST * CC_G, D.dn.KB, D.fmt, ovf, 0);
        uint32_t overflow = 0;
        if (e == cudaSuccess) e = cudaMemcpy(&overflow, ovf, 4, cudaMemcpyDeviceToHost);
        if (e != cudaSuccess || !overflow || D.fmt != CC_FMT_F16) break;
        if (ctx->operand_format == CC_OPERAND_F16) {
            destroy_layer_memory(L);
            delete L;
            return fail(CC_ERR_INVALID, "a weight does not fit fp16 (|w| > 65504 or not finite) and the context demands CC_OPERAND_F16");
        }
        D.fmt = CC_FMT_BF16X2;
    }
    if (e == cudaSuccess) e = cudaMemcpy(L->blob0 + D.off_g1, w->g1, (size_t)D.d * 2, cudaMemcpyDeviceToDevice);
    if (e == cudaSuccess) e = cudaMemcpy(L->blob0 + D.off_g2, w->g2, (size_t)D.d * 2, cudaMemcpyDeviceToDevice);
    L->rep[0].state = REP_LIVE;
    L->rep[0].blob = L->blob0;
    L->rep[0].published = true;
    L->host_row = CcLayerTable{};
    L->host_row.rep[0].blob = L->blob0;
    L->host_row.active_mask = 1u;
    if (e == cudaSuccess)
        e = cudaMemcpy(ctx->table_dev + row, &L->host_row, sizeof(CcLayerTable), cudaMemcpyHostToDevice);
    if (e == cudaSuccess) e = cudaDeviceSynchronize();
    if (e != cudaSuccess) {
        destroy_layer_memory(L);
        delete L;
        cudaGetLastError();
        return fail(CC_ERR_CUDA, "cc_create_layer: %s", cudaGetErrorString(e));
    }
    ctx->row_used[row] = true;
    ctx->n_layers++;
    *out = L;
    return CC_OK;
}

cc_status cc_destroy_layer(cc_layer* L) {
    if (!L) return CC_OK;
    cc_ctx* ctx = L->ctx;
    cudaSetDevice(ctx->device);
    cudaDeviceSynchronize();
    for (int r = 1; r < CC_MAX_REPLICAS; ++r) {
        if (L->rep[r].state != REP_EMPTY) cc_slotalloc_free(ctx->slots, (uint64_t)(uintptr_t)L->rep[r].blob);
        if (L->rep[r].copied) cudaEventDestroy(L->rep[r].copied);
    }
    reap_zombies(ctx, true);
    CcLayerTable zero{};
    cudaMemcpy(ctx->table_dev + L->row, &zero, sizeof zero, cudaMemcpyHostToDevice);
    destroy_layer_memory(L);
    ctx->row_used[L->row] = false;
    ctx->n_layers--;
    delete L;
    return CC_OK;
}

cc_status cc_layer_operand_format(const cc_layer* L, int* format) {
    if (!L || !format) return fail(CC_ERR_INVALID, "null argument");
    *format = L->D.fmt == CC_FMT_F16 ? CC_OPERAND_F16 : CC_OPERAND_BF16X2;
    return CC_OK;
}

cc_status cc_layer_blob_bytes(const cc_layer* L, size_t* bytes) {
    if (!L || !bytes) return fail(CC_ERR_INVALID, "null argument");
    *bytes = L->blob_bytes;
    return CC_OK;
}

}  // extern "C"

// ---- scaling: create / publish / retire replicas ------------------
extern "C" {

cc_status cc_scale_layer(cc_layer* L, int n_replicas) {
    if (!L) return fail(CC_ERR_INVALID, "null layer");
    if (n_replicas < 1 || n_replicas > CC_MAX_REPLICAS) return fail(CC_ERR_INVALID, "n_replicas must be in 1..%d", CC_MAX_REPLICAS);
    cc_ctx* ctx = L->ctx;
    CC_CUDA(cudaSetDevice(ctx->device));
    reap_zombies(ctx, false);
    int cur = 0;
    for (int r = 0; r < CC_MAX_REPLICAS; ++r) cur += (L->rep[r].state == REP_LIVE || L->rep[r].state == REP_COPYING);
    if (n_replicas > cur) {
        // take every slot first so that a failure changes nothing
        int want = n_replicas - cur, got = 0, idx[CC_MAX_REPLICAS];
        uint64_t addr[CC_MAX_REPLICAS];
        for (int r = 1; r < CC_MAX_REPLICAS && got < want; ++r) {
            if (L->rep[r].state != REP_EMPTY) continue;
            if (cc_slotalloc_alloc(ctx->slots, L->blob_bytes, &addr[got]) != CC_OK) break;
            idx[got++] = r;
        }
        if (got < want) {
            for (int i = 0; i < got; ++i) cc_slotalloc_free(ctx->slots, addr[i]);
            return fail(CC_ERR_NO_SLOT, "no free slot of %zu bytes for replica %d of this layer (free: %llu bytes)",
                        L->blob_bytes, cur + got, (unsigned long long)cc_slotalloc_free_bytes(ctx->slots));
        }
        for (int i = 0; i < got; ++i) {
            Replica& R = L->rep[idx[i]];
            cudaError_t e = cudaSuccess;
            if (!R.copied) e = cudaEventCreateWithFlags(&R.copied, cudaEventDisableTiming);
            cc_status st = CC_OK;
            if (e == cudaSuccess) st = launch_chunked_copy(ctx, (void*)(uintptr_t)addr[i], L->blob0, L->blob_bytes, 0, ctx->side);
            if (e == cudaSuccess && st == CC_OK) e = cudaEventRecord(R.copied, ctx->side);
            if (e != cudaSuccess || st != CC_OK) {
                // roll back: the slots of this and the later replicas go back to the allocator once the side stream
                // has drained (a chunk of the failed copy may still be writing); replicas already enqueued stay
                cudaStreamSynchronize(ctx->side);
                cudaGetLastError();
                for (int j = i; j < got; ++j) cc_slotalloc_free(ctx->slots, addr[j]);
                return st != CC_OK ? st : fail(CC_ERR_CUDA, "cc_scale_layer: %s", cudaGetErrorString(e));
            }
            R.blob = (uint8_t*)(uintptr_t)addr[i];
            R.state = REP_COPYING;
            R.published = false;
        }
    } else if (n_replicas < cur) {
        int drop = cur - n_replicas;
        for (int r = CC_MAX_REPLICAS - 1; r >= 1 && drop > 0; --r) {
            if (L->rep[r].state == REP_LIVE || L->rep[r].state == REP_COPYING) {
                L->rep[r].state = REP_RETIRING;
                --drop;
            }
        }
    }
    return CC_OK;
}

cc_status cc_release_replica(cc_layer* L, int replica) {
    if (!L) return fail(CC_ERR_INVALID, "null layer");
    if (replica < 0 || replica >= CC_MAX_REPLICAS) return fail(CC_ERR_INVALID, "replica index out of range");
    if (replica == 0) return fail(CC_ERR_STATE, "replica 0 (the layer itself) cannot be released");
    if (L->rep[replica].state != REP_LIVE) return fail(CC_ERR_STATE, "replica %d is not live", replica);
    L->rep[replica].state = REP_RETIRING;
    return CC_OK;
}

cc_status cc_commit(cc_layer* L, void* stream) {
    if (!L) return fail(CC_ERR_INVALID, "null layer");
    cc_ctx* ctx = L->ctx;
    cudaStream_t st = (cudaStream_t)stream;
    CC_CUDA(cudaSetDevice(ctx->device));
    reap_zombies(ctx, false);
    bool pending = false;
    for (int r = 1; r < CC_MAX_REPLICAS; ++r) pending |= (L->rep[r].state == REP_COPYING || L->rep[r].state == REP_RETIRING);
    if (!pending) return CC_OK;
    std::vector<uint64_t> retired;
    for (int r = 1; r < CC_MAX_REPLICAS; ++r) {
        Replica& R = L->rep[r];
        if (R.state == REP_COPYING) {
            CC_CUDA(cudaStreamWaitEvent(st, R.copied, 0));    // two-phase publish: visible only once copied
            R.state = REP_LIVE;
            R.published = true;
        } else if (R.state == REP_RETIRING) {
            CC_CUDA(cudaStreamWaitEvent(st, R.copied, 0));    // a retired copy may still be in flight
            retired.push_back((uint64_t)(uintptr_t)R.blob);
            R.state = REP_EMPTY;
            R.published = false;
            R.blob = nullptr;
        }
    }
    CcLayerTable row{};
    for (int r = 0; r < CC_MAX_REPLICAS; ++r) {
        if (L->rep[r].state == REP_LIVE) {
            row.rep[r].blob = L->rep[r].blob;
            row.active_mask |= 1u << r;
        }
        row.rep[r].k_pool = L->kvp[r].k;
        row.rep[r].v_pool = L->kvp[r].v;
        row.rep[r].n_pages = L->kvp[r].n;
    }
    L->host_row = row;
    CC_CUDA(cc_launch_publish(ctx->table_dev + L->row, row, st));
    for (uint64_t a : retired) {
        Zombie z{a, nullptr};
        CC_CUDA(cudaEventCreateWithFlags(&z.after_flip, cudaEventDisableTiming));
        CC_CUDA(cudaEventRecord(z.after_flip, st));           // everything enqueued before the flip has run
        ctx->zombies.push_back(z);
    }
    return CC_OK;
}

cc_status cc_layer_set_kv_partition(cc_layer* L, int replica, void* k_pool_dev, void* v_pool_dev, int32_t n_pages, void* stream) {
    if (!L) return fail(CC_ERR_INVALID, "null layer");
    if (replica < 0 || replica >= CC_MAX_REPLICAS) return fail(CC_ERR_INVALID, "replica index out of range");
    if ((k_pool_dev == nullptr) != (v_pool_dev == nullptr)) return fail(CC_ERR_INVALID, "give both pools or neither");
    if (k_pool_dev && (n_pages < 1 || (((uintptr_t)k_pool_dev | (uintptr_t)v_pool_dev) & 15)))
        return fail(CC_ERR_INVALID, "a partition needs n_pages >= 1 and 16-byte aligned pools");
    cc_ctx* ctx = L->ctx;
    CC_CUDA(cudaSetDevice(ctx->device));
    L->kvp[replica].k = k_pool_dev;
    L->kvp[replica].v = v_pool_dev;
    L->kvp[replica].n = k_pool_dev ? n_pages : 0;
    L->host_row.rep[replica].k_pool = L->kvp[replica].k;
    L->host_row.rep[replica].v_pool = L->kvp[replica].v;
    L->host_row.rep[replica].n_pages = L->kvp[replica].n;
    CC_CUDA(cc_launch_publish(ctx->table_dev + L->row, L->host_row, (cudaStream_t)stream));
    return CC_OK;
}

cc_status cc_query(cc_layer* L, int* n_active, int* n_pending) {
    if (!L) return fail(CC_ERR_INVALID, "null layer");
    int a = 0, p = 0;
    for (int r = 0; r < CC_MAX_REPLICAS; ++r) {
        a += (L->host_row.active_mask >> r) & 1u;
        p += (L->rep[r].state == REP_COPYING);
    }
    if (n_active) *n_active = a;
    if (n_pending) *n_pending = p;
    return CC_OK;
}

cc_status cc_active_replicas(cc_layer* L, uint32_t* mask) {
    if (!L || !mask) return fail(CC_ERR_INVALID, "null argument");
    *mask = L->host_row.active_mask;
    return CC_OK;
}

cc_status cc_replica_blob(cc_layer* L, int replica, const void** blob_dev, size_t* bytes) {
    if (!L || !blob_dev || !bytes) return fail(CC_ERR_INVALID, "null argument");
    if (replica < 0 || replica >= CC_MAX_REPLICAS) return fail(CC_ERR_INVALID, "replica index out of range");
    if (L->rep[replica].state == REP_EMPTY) return fail(CC_ERR_STATE, "replica %d holds no slot", replica);
    *blob_dev = L->rep[replica].blob;
    *bytes = L->blob_bytes;
    return CC_OK;
}

}  // extern "C"

// ---- the hot path -------------------------------------------------------------------------------
namespace {
constexpr int kForwardLaunches = 6;

// Device-visible alias of a pinned, mapped host buffer (null when `p` is anything else).
void* mapped_host(const void* p) {
    cudaPointerAttributes a;
    if (cudaPointerGetAttributes(&a, p) != cudaSuccess) { cudaGetLastError(); return nullptr; }
    return a.type == cudaMemoryTypeHost && !((uintptr_t)a.devicePointer & 15) ? a.devicePointer : nullptr;
}

// The KV pools of one forward: the call's pools, and per replica its own partition where it has one.
CcKv make_kv(const cc_layer* L, void* k_pool, void* v_pool, const int* block_table, int n_pages) {
    CcKv k{};
    k.k_pool = (__nv_bfloat16*)k_pool;
    k.v_pool = (__nv_bfloat16*)v_pool;
    k.block_table = block_table;
    k.n_pages = n_pages;
    for (int r = 0; r < CC_MAX_REPLICAS; ++r) {
        const bool own = L->kvp[r].k != nullptr;
        k.k_pool_r[r] = own ? L->kvp[r].k : k_pool;
        k.v_pool_r[r] = own ? L->kvp[r].v : v_pool;
        k.n_pages_r[r] = own ? L->kvp[r].n : n_pages;
    }
    return k;
}

// Geometry of one step: the layer's, with the activation plane counts of a step of `batch` rows.
CcDims step_dims(cc_layer* L, int batch) {
    CcDims D = L->D;
    const cc_ctx* ctx = L->ctx;
    for (int i = 0; i < 4; ++i)
        D.pl[i] = D.fmt == CC_FMT_BF16X2 ? 2 : (batch <= ctx->planes_rows ? ctx->planes_small[i] : ctx->planes_large[i]);
    for (int i = 0; i < 4; ++i) L->last_pl[i] = D.pl[i];
    // the row tables of the small-step kernels and of the decode attention hold at most 256 rows: a small step of a
    // large layer sees 256, a large step's attention walks its (at most CC_BIG_MAX_DEC) decode rows
    if (D.max_batch > 256) D.max_batch = 256;
    return D;
}


// A step of more than 256 rows (prompt chunks + decode rows): plain stream order, no PDL.
cudaError_t enqueue_big(cc_layer* L, __nv_bfloat16* hidden, const CcKv& kv, const int* seq_lens, const int* assign, int batch,
                        cudaStream_t st, cudaEvent_t* ev) {
    cc_ctx* ctx = L->ctx;
    CcDims D = step_dims(L, batch);
    const CcWork& W = L->W;
    const CcLayerTable* tab = ctx->table_dev + L->row;
    CcLaunch Ln{st, ctx->n_sms, false};
    cudaError_t e = cudaSuccess;
    for (int stage = 0; stage < 9 && e == cudaSuccess; ++stage) {
        if (ev && (e = cudaEventRecord(ev[stage], st)) != cudaSuccess) break;
        switch (stage) {
            case 0: e = cc_launch_big_group(assign, seq_lens, kv.block_table, batch, D, tab, W, st); break;
            case 1: e = cc_launch_big_norm(hidden, batch, D, tab, W, st); break;
            case 2: e = cc_launch_big_gemm(0, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln); break;
            case 3: e = cc_launch_attention(seq_lens, kv, D, tab, W, Ln, W.dec_rows); break;
            case 4: e = cc_launch_prefill_attention(seq_lens, kv, D, W, Ln); break;
            case 5: e = cc_launch_big_gemm(1, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln); break;
            case 6: e = cc_launch_big_rowstat(D, W, st); break;
            case 7: e = cc_launch_big_gemm(2, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln); break;
            default: e = cc_launch_big_gemm(3, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln); break;
        }
    }
    if (ev && e == cudaSuccess) e = cudaEventRecord(ev[9], st);
    return e;
}

cudaError_t enqueue_forward(cc_layer* L, __nv_bfloat16* hidden, const CcKv& kv, const int* seq_lens, const int* assign,
                            int batch, cudaStream_t st, cudaEvent_t* ev = nullptr, __nv_bfloat16* hidden_host_alias = nullptr) {
    if (batch > 256) return enqueue_big(L, hidden, kv, seq_lens, assign, batch, st, ev);
    cc_ctx* ctx = L->ctx;
    CcDims D = step_dims(L, batch);
    const CcWork& W = L->W;
    const CcLayerTable* tab = ctx->table_dev + L->row;
    CcLaunch Ln{st, ctx->n_sms, ctx->pdl && ev == nullptr};
    cudaError_t e = cudaSuccess;
    // a0 grouping + a1 norm | a2 QKV (+ a3 RoPE, a4 append) | a5 attention (+ chunk merge) |
    // a6 O (+ residual, a7 statistics) | a8 gate/up (+ a7 scale, SwiGLU) | a9 down (+ residual, request order)
    // hidden_host_alias (cc_forward_host with a pinned buffer): the prologue reads the rows over PCIe and leaves a
    // device copy in `hidden` (the O epilogue's residual); the last epilogue writes the result rows straight into the
    // caller's host buffer.  The same bytes cross PCIe as with two copies, without the copies' fixed cost.
    CcStageOut so;
    __nv_bfloat16 *h_in = hidden, *h_out = hidden;
    if (hidden_host_alias) {
        so.hidden = hidden;
        h_in = h_out = hidden_host_alias;
    }
    // the three short projections of a SMALL step run as cluster split-K (k_gemm_cl): decided by the row count alone --
    // the worst-case grouped size of `batch` rows over CC_MAX_REPLICAS groups -- so it cannot differ between replica counts
    const bool cl = (batch + 15) / 16 * 16 + 16 * (CC_MAX_REPLICAS - 1) <= cc_gemm_cl_max_rows();
    D.pf_next = cl ? ctx->pf_next : 0;
    D.pf_self = cl ? ctx->pf_self : 0;
    for (int stage = 0; stage < kForwardLaunches && e == cudaSuccess; ++stage) {
        if (ev && (e = cudaEventRecord(ev[stage], st)) != cudaSuccess) break;
        switch (stage) {
            case 0: e = cc_launch_prologue(assign, seq_lens, kv.block_table, batch, h_in, D, tab, W, Ln, so); break;
            case 1: e = (cl && D.qkv.S) ? cc_launch_gemm_cl(0, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln)
                                       : cc_launch_gemm(0, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln); break;
            case 2: e = cc_launch_attention(seq_lens, kv, D, tab, W, Ln); break;
            case 3: e = (cl && D.o.S) ? cc_launch_gemm_cl(1, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln)
                                     : cc_launch_gemm(1, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln); break;
            case 4: e = (cl && D.gu.S) ? cc_launch_gemm_cl(2, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln)
                                      : cc_launch_gemm(2, D, tab, W, seq_lens, assign, batch, kv, hidden, Ln); break;
            default: e = (cl && D.dn.S) ? cc_launch_gemm_cl(3, D, tab, W, seq_lens, assign, batch, kv, h_out, Ln)
                                        : cc_launch_gemm(3, D, tab, W, seq_lens, assign, batch, kv, h_out, Ln); break;
        }
    }
    if (ev && e == cudaSuccess) e = cudaEventRecord(ev[kForwardLaunches], st);
    return e;
}
}  // namespace

extern "C" {

cc_status cc_forward(cc_layer* L, void* hidden_dev, const cc_kv_pages* kv, const int32_t* seq_lens_dev,
                     const int32_t* replica_assign_dev, int batch, void* stream) {
    if (!L || !hidden_dev || !kv || !seq_lens_dev || !replica_assign_dev) return fail(CC_ERR_INVALID, "null argument");
    if (batch < 1 || batch > L->desc.max_batch) return fail(CC_ERR_INVALID, "batch %d outside 1..max_batch=%d", batch, L->desc.max_batch);
    if (!kv->k_pool || !kv->v_pool || !kv->block_table || kv->n_pages < 1) return fail(CC_ERR_INVALID, "bad cc_kv_pages");
    if (((uintptr_t)hidden_dev | (uintptr_t)kv->k_pool | (uintptr_t)kv->v_pool) & 15)
        return fail(CC_ERR_INVALID, "hidden and KV pools must be 16-byte aligned");
    const CcKv k = make_kv(L, kv->k_pool, kv->v_pool, kv->block_table, kv->n_pages);
    cudaError_t e = enqueue_forward(L, (__nv_bfloat16*)hidden_dev, k, seq_lens_dev, replica_assign_dev, batch,
                                    (cudaStream_t)stream);
    if (e != cudaSuccess) return fail(CC_ERR_CUDA, "cc_forward launch: %s", cudaGetErrorString(e));
    L->last_batch = batch;
    return CC_OK;
}

static cc_status forward_host_impl(cc_layer* L, void* hidden_host, void* k_pool_dev, void* v_pool_dev, int32_t n_pages,
                                   const int32_t* block_table_host, const int32_t* seq_lens_host,
                                   const int32_t* replica_assign_host, int batch, void* stream, bool sync) {
    if (!L || !hidden_host || !block_table_host || !seq_lens_host || !replica_assign_host)
        return fail(CC_ERR_INVALID, "null argument");
    if (batch < 1 || batch > L->desc.max_batch) return fail(CC_ERR_INVALID, "batch %d outside 1..max_batch=%d", batch, L->desc.max_batch);
    cudaStream_t st = (cudaStream_t)stream;
    CC_CUDA(cudaSetDevice(L->ctx->device));
    const size_t hb = (size_t)batch * L->D.d * 2;
    // Pinned hidden buffer: the kernels read and write it in place (measured: 280 us per cfg2 step against 300 us
    // with the two 512 KB copies; reading the three small tables in place as well costs more than their copies).
    if (void* alias = batch <= 256 ? mapped_host(hidden_host) : nullptr) {
        if (!k_pool_dev || !v_pool_dev || n_pages < 1) return fail(CC_ERR_INVALID, "bad KV pool arguments");
        if (((uintptr_t)k_pool_dev | (uintptr_t)v_pool_dev) & 15) return fail(CC_ERR_INVALID, "KV pools must be 16-byte aligned");
        CC_CUDA(stage_tables(L, block_table_host, seq_lens_host, replica_assign_host, batch, st));
        const CcKv k = make_kv(L, k_pool_dev, v_pool_dev, L->st_bt, n_pages);
        cudaError_t e = enqueue_forward(L, L->st_hidden, k, L->st_sl, L->st_ra, batch, st, nullptr, (__nv_bfloat16*)alias);
        if (e != cudaSuccess) return fail(CC_ERR_CUDA, "cc_forward_host launch: %s", cudaGetErrorString(e));
        L->last_batch = batch;
        if (sync) CC_CUDA(cudaStreamSynchronize(st));
        return CC_OK;
    }
    if (!sync) return fail(CC_ERR_INVALID, "cc_forward_host_async needs a pinned (page-locked, mapped) hidden buffer and a step of at most 256 rows");
    CC_CUDA(cudaMemcpyAsync(L->st_hidden, hidden_host, hb, cudaMemcpyHostToDevice, st));
    CC_CUDA(stage_tables(L, block_table_host, seq_lens_host, replica_assign_host, batch, st));
    cc_kv_pages kv{k_pool_dev, v_pool_dev, L->st_bt, n_pages};
    cc_status s = cc_forward(L, L->st_hidden, &kv, L->st_sl, L->st_ra, batch, stream);
    if (s != CC_OK) return s;
    CC_CUDA(cudaMemcpyAsync(hidden_host, L->st_hidden, hb, cudaMemcpyDeviceToHost, st));
    CC_CUDA(cudaStreamSynchronize(st));
    return CC_OK;
}

cc_status cc_forward_host(cc_layer* L, void* hidden_host, void* k_pool_dev, void* v_pool_dev, int32_t n_pages,
                          const int32_t* block_table_host, const int32_t* seq_lens_host,
                          const int32_t* replica_assign_host, int batch, void* stream) {
    return forward_host_impl(L, hidden_host, k_pool_dev, v_pool_dev, n_pages, block_table_host, seq_lens_host, replica_assign_host,
                             batch, stream, true);
}

cc_status cc_forward_host_async(cc_layer* L, void* hidden_host, void* k_pool_dev, void* v_pool_dev, int32_t n_pages,
                                const int32_t* block_table_host, const int32_t* seq_lens_host,
                                const int32_t* replica_assign_host, int batch, void* stream) {
    return forward_host_impl(L, hidden_host, k_pool_dev, v_pool_dev, n_pages, block_table_host, seq_lens_host, replica_assign_host,
                             batch, stream, false);
}

cc_status cc_forward_profiled(cc_layer* L, void* hidden_dev, const cc_kv_pages* kv, const int32_t* seq_lens_dev,
                              const int32_t* replica_assign_dev, int batch, void* stream, float* stage_ms_host) {
    if (!L || !hidden_dev || !kv || !seq_lens_dev || !replica_assign_dev || !stage_ms_host)
        return fail(CC_ERR_INVALID, "null argument");
    if (batch < 1 || batch > L->desc.max_batch) return fail(CC_ERR_INVALID, "batch %d outside 1..max_batch=%d", batch, L->desc.max_batch);
    CC_CUDA(cudaSetDevice(L->ctx->device));
    cudaEvent_t ev[CC_MAX_PROFILE_STAGES + 1];
    for (auto& x : ev) CC_CUDA(cudaEventCreate(&x));
    const int n_stages = batch > 256 ? 9 : kForwardLaunches;
    for (int i = 0; i < CC_MAX_PROFILE_STAGES; ++i) stage_ms_host[i] = 0.f;
    const CcKv k = make_kv(L, kv->k_pool, kv->v_pool, kv->block_table, kv->n_pages);
    // a pinned host `hidden`: the stages of cc_forward_host's in-place path (the rows are staged for the residual)
    void* alias = batch <= 256 ? mapped_host(hidden_dev) : nullptr;
    cudaError_t e = enqueue_forward(L, alias ? L->st_hidden : (__nv_bfloat16*)hidden_dev, k, seq_lens_dev, replica_assign_dev,
                                    batch, (cudaStream_t)stream, ev, (__nv_bfloat16*)alias);
    if (e == cudaSuccess) e = cudaStreamSynchronize((cudaStream_t)stream);
    for (int i = 0; i < n_stages && e == cudaSuccess; ++i) e = cudaEventElapsedTime(&stage_ms_host[i], ev[i], ev[i + 1]);
    for (auto& x : ev) cudaEventDestroy(x);
    if (e != cudaSuccess) return fail(CC_ERR_CUDA, "cc_forward_profiled: %s", cudaGetErrorString(e));
    return CC_OK;
}

cc_status cc_layer_gemm_grids(const cc_layer* L, int* ctas, int* cluster) {
    if (!L || !ctas || !cluster) return fail(CC_ERR_INVALID, "null argument");
    const CcGemmGeo* g[4] = {&L->D.qkv, &L->D.o, &L->D.gu, &L->D.dn};
    for (int i = 0; i < 4; ++i) {
        cluster[i] = g[i]->S;
        ctas[i] = g[i]->S ? g[i]->ST * CC_G / g[i]->cl_tiles * g[i]->S : g[i]->P;
    }
    return CC_OK;
}

cc_status cc_forward_launch_count(const cc_layer* L, int* n) {
    if (!L || !n) return fail(CC_ERR_INVALID, "null argument");
    *n = kForwardLaunches;
    return CC_OK;
}

// ---- KV partition per replica: planner (host) + page migration (device) ---------------------------------
cc_status cc_kv_plan_migration(const int32_t* bt, const int32_t* seq_lens, const int32_t* assign, int batch, int max_blocks,
                               int n_pages, int n_replicas, int32_t* new_bt, int32_t* src, int32_t* dst, int* n_moves) {
    if (!bt || !seq_lens || !assign || !new_bt || !src || !dst || !n_moves) return fail(CC_ERR_INVALID, "null argument");
    if (batch < 1 || max_blocks < 1 || n_pages < 1 || n_replicas < 1 || n_replicas > CC_MAX_REPLICAS || n_pages < n_replicas)
        return fail(CC_ERR_INVALID, "bad sizes");
    const int psz = n_pages / n_replicas;
    std::vector<char> used((size_t)n_pages, 0);
    for (int b = 0; b < batch; ++b) {
        const int need = seq_lens[b] > 0 ? (seq_lens[b] + CC_PAGE_SIZE - 1) / CC_PAGE_SIZE : 0;
        if (need > max_blocks) return fail(CC_ERR_INVALID, "row %d needs %d pages, table has %d", b, need, max_blocks);
        if (need && (assign[b] < 0 || assign[b] >= n_replicas)) return fail(CC_ERR_INVALID, "row %d: replica %d out of range", b, assign[b]);
        for (int j = 0; j < need; ++j) {
            const int pg = bt[(size_t)b * max_blocks + j];
            if (pg < 0 || pg >= n_pages) return fail(CC_ERR_INVALID, "row %d page %d: id %d out of range", b, j, pg);
            if (used[pg]) return fail(CC_ERR_INVALID, "page %d is referenced twice", pg);
            used[pg] = 1;
        }
    }
    std::memcpy(new_bt, bt, (size_t)batch * max_blocks * sizeof(int32_t));
    int cursor[CC_MAX_REPLICAS];                               // lowest candidate of each partition
    for (int r = 0; r < n_replicas; ++r) cursor[r] = r * psz;
    int n = 0;
    for (int b = 0; b < batch; ++b) {
        const int need = seq_lens[b] > 0 ? (seq_lens[b] + CC_PAGE_SIZE - 1) / CC_PAGE_SIZE : 0;
        if (!need) continue;
        const int r = assign[b], lo = r * psz, hi = lo + psz;
        for (int j = 0; j < need; ++j) {
            const int pg = bt[(size_t)b * max_blocks + j];
            if (pg >= lo && pg < hi) continue;
            while (cursor[r] < hi && used[cursor[r]]) ++cursor[r];
            if (cursor[r] >= hi) return fail(CC_ERR_NO_SLOT, "partition %d has no free page left for row %d", r, b);
            used[cursor[r]] = 1;                               // sources stay "used": never a destination of this plan
            src[n] = pg;
            dst[n] = cursor[r];
            new_bt[(size_t)b * max_blocks + j] = cursor[r];
            ++n;
        }
    }
    *n_moves = n;
    return CC_OK;
}

// Catch-up plan of a pre-copy migration: pages that cannot have been written since the first plan keep their
// planned place; the rest (the tail page of then, pages added since) is planned again from the table the decode
// steps kept using.
cc_status cc_kv_plan_catchup(const int32_t* bt_now, const int32_t* seq_planned, const int32_t* seq_now, const int32_t* planned_bt,
                             const int32_t* assign, int batch, int max_blocks, int n_pages, int n_replicas, int32_t* final_bt,
                             int32_t* src, int32_t* dst, int* n_moves) {
    if (!bt_now || !seq_planned || !seq_now || !planned_bt || !final_bt) return fail(CC_ERR_INVALID, "null argument");
    if (batch < 1 || max_blocks < 1) return fail(CC_ERR_INVALID, "bad sizes");
    std::vector<int32_t> hybrid(bt_now, bt_now + (size_t)batch * max_blocks);
    for (int b = 0; b < batch; ++b) {
        if (seq_now[b] <= 0) continue;                         // the row finished meanwhile: nothing to keep
        if (seq_now[b] < seq_planned[b]) return fail(CC_ERR_INVALID, "row %d shrank from %d to %d tokens during the migration", b, seq_planned[b], seq_now[b]);
        // a step with seq_len s writes position s - 1: whether the step of seq_planned had run or not when the plan
        // was made, only positions >= seq_planned - 1 can have been written since -- pages below that are clean
        const int clean = seq_planned[b] > 0 ? (seq_planned[b] - 1) / CC_PAGE_SIZE : 0;
        for (int j = 0; j < clean && j < max_blocks; ++j) hybrid[(size_t)b * max_blocks + j] = planned_bt[(size_t)b * max_blocks + j];
    }
    return cc_kv_plan_migration(hybrid.data(), seq_now, assign, batch, max_blocks, n_pages, n_replicas, final_bt, src, dst, n_moves);
}

cc_status cc_kv_migrate(cc_ctx* ctx, void* k_pool_dev, void* v_pool_dev, size_t page_bytes, const int32_t* src_dev,
                        const int32_t* dst_dev, int n_moves, void* stream) {
    if (!ctx || !k_pool_dev || !v_pool_dev) return fail(CC_ERR_INVALID, "null argument");
    if (n_moves < 0 || (n_moves > 0 && (!src_dev || !dst_dev))) return fail(CC_ERR_INVALID, "bad move list");
    if (page_bytes == 0 || page_bytes % 32 || (((uintptr_t)k_pool_dev | (uintptr_t)v_pool_dev) & 31))
        return fail(CC_ERR_INVALID, "page_bytes must be a multiple of 32 and the pools 32-byte aligned");
    CC_CUDA(cudaSetDevice(ctx->device));
    CC_CUDA(cc_launch_page_copy(k_pool_dev, v_pool_dev, page_bytes, src_dev, dst_dev, n_moves, (cudaStream_t)stream));
    return CC_OK;
}

// ---- %globaltimer trace of a tracing build --------------------------------------------------------
cc_status cc_debug_trace(cc_ctx* ctx, uint64_t* out_host, int reset) {
    if (!ctx) return fail(CC_ERR_INVALID, "null argument");
#ifdef CC_TRACE
    constexpr size_t n = (size_t)CC_TRACE_KERNELS * CC_TRACE_POINTS * 2;
    CC_CUDA(cudaSetDevice(ctx->device));
    CC_CUDA(cudaDeviceSynchronize());
    if (out_host) CC_CUDA(cudaMemcpy(out_host, ctx->trace_dev, n * 8, cudaMemcpyDeviceToHost));
    if (reset) {
        std::vector<unsigned long long> h(n);
        for (size_t i = 0; i < n; ++i) h[i] = (i & 1) ? 0ull : ~0ull;         // [min, max] pairs
        CC_CUDA(cudaMemcpy(ctx->trace_dev, h.data(), n * 8, cudaMemcpyHostToDevice));
    }
    return CC_OK;
#else
    (void)out_host; (void)reset;
    return fail(CC_ERR_STATE, "this library was built without CC_TRACE (python -m paper_2607_04181_b200.build --trace)");
#endif
}

// ---- stage taps (tests only) ----------------------------------------------------------------------
cc_status cc_debug_tap(cc_layer* L, cc_tap which, float* out_host, int batch) {
    if (!L || !out_host) return fail(CC_ERR_INVALID, "null argument");
    if (batch < 1 || batch > L->desc.max_batch) return fail(CC_ERR_INVALID, "bad batch");
    const CcDims& D = L->D;
    const void* src;
    int kind, dim, planes = 1;
    switch (which) {
        case CC_TAP_X: src = L->W.x_act; kind = 2; dim = D.d; planes = L->last_pl[0]; break;
        case CC_TAP_Q: src = L->W.q_rot; kind = 1; dim = D.QD; break;
        case CC_TAP_O: src = L->W.o_act; kind = 2; dim = D.QD; planes = L->last_pl[1]; break;
        case CC_TAP_H1: src = L->W.h1; kind = 1; dim = D.d; break;
        case CC_TAP_Y: src = L->W.y_act; kind = 3; dim = D.d; planes = L->last_pl[2]; break;
        case CC_TAP_A: src = L->W.a_act; kind = 2; dim = D.F; planes = L->last_pl[3]; break;
        default: return fail(CC_ERR_INVALID, "unknown tap");
    }
    CC_CUDA(cudaSetDevice(L->ctx->device));
    CC_CUDA(cudaDeviceSynchronize());
    float* tmp = nullptr;
    const size_t bytes = (size_t)batch * dim * 4;
    CC_CUDA(cudaMalloc(&tmp, bytes));
    cudaError_t e = cudaMemset(tmp, 0, bytes);
    if (e == cudaSuccess) e = cc_launch_tap(src, kind, planes, dim, D, L->W, tmp, batch, 0);
    if (e == cudaSuccess) e = cudaMemcpy(out_host, tmp, bytes, cudaMemcpyDeviceToHost);
    cudaFree(tmp);
    if (e != cudaSuccess) return fail(CC_ERR_CUDA, "cc_debug_tap: %s", cudaGetErrorString(e));
    return CC_OK;
}

cc_status cc_debug_grouping(cc_layer* L, int32_t* perm_host, int32_t* counts_host, int32_t* n_pos) {
    if (!L || !perm_host || !counts_host || !n_pos) return fail(CC_ERR_INVALID, "null argument");
    CC_CUDA(cudaSetDevice(L->ctx->device));
    CC_CUDA(cudaDeviceSynchronize());
    CcSched s;
    CC_CUDA(cudaMemcpy(&s, L->W.sched, sizeof s, cudaMemcpyDeviceToHost));
    CC_CUDA(cudaMemcpy(perm_host, L->W.perm, (size_t)L->D.Mpad * 4, cudaMemcpyDeviceToHost));
    for (int r = 0; r < CC_MAX_REPLICAS; ++r) counts_host[r] = s.cnt[r];
    *n_pos = s.n_pos;
    return CC_OK;
}

}  // extern "C"
