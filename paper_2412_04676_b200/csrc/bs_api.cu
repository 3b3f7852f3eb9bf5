// bs_api.cu — the C ABI of include/bs.h: argument checks, workspace layout, launches.  No data-path work
// happens on the host; every step of the path runs in the kernels of bs_scan.cu / bs_move*.cu.
#include <string.h>

#include "bs_internal.cuh"

namespace bs {

static thread_local int g_last_cuda_error = 0;

int cuda_fail(cudaError_t e)
{
    g_last_cuda_error = (int)e;
    cudaGetLastError();  // a non-sticky error must not resurface in the cudaGetLastError() behind a later, unrelated launch
    return BS_ERR_CUDA;
}

int device_sm_count(int* out)
{
    static thread_local int cached_dev = -1, cached_sms = 0;
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    if (dev != cached_dev) {
        int sms = 0;
        e = cudaDeviceGetAttribute(&sms, cudaDevAttrMultiProcessorCount, dev);
        if (e != cudaSuccess) return cuda_fail(e);
        cached_dev = dev;
        cached_sms = sms;
    }
    *out = cached_sms;
    return BS_OK;
}

static bool aligned(const void* p, uintptr_t a) { return ((uintptr_t)p & (a - 1)) == 0; }

int check_set(const bs_set_desc* s)
{
    if (s == nullptr) return BS_ERR_ARG;
    if (s->n_qn != 2 || (s->dtype & BS_DTYPE_MASK) > (uint32_t)BS_C128 || (s->dtype & ~(BS_DTYPE_MASK | BS_ALIGN8 | BS_RANK4)) != 0 ||
        (s->dtype & (BS_ALIGN8 | BS_RANK4)) == (BS_ALIGN8 | BS_RANK4))
        return BS_ERR_UNSUPPORTED;
    if (s->n_tensors && (s->tensors == nullptr || !aligned(s->tensors, 16))) return BS_ERR_ARG;
    // a BS_RANK4 set's qn / dim rows are 32 / 16 bytes and the kernels move them as 16-byte words (bs_move_common.cuh)
    const uintptr_t qa = (s->dtype & BS_RANK4) ? 16 : 8, da = (s->dtype & BS_RANK4) ? 16 : 4;
    if (s->n_blocks && (s->qn == nullptr || !aligned(s->qn, qa))) return BS_ERR_ARG;
    if (s->n_blocks && (s->dim == nullptr || !aligned(s->dim, da))) return BS_ERR_ARG;
    if (s->n_blocks && (s->addr == nullptr || !aligned(s->addr, 8))) return BS_ERR_ARG;
    return BS_OK;
}

int check_opts(const bs_opts& o)
{
    if (o.variant != BS_VARIANT_LDG && o.variant != BS_VARIANT_TMA) return BS_ERR_ARG;
    if (o.ctas_per_sm > 32) return BS_ERR_ARG;
    // the named switches (bs.h): garbage in them is refused, not interpreted
    if (o.fuse > 2u || (o.tune & ~BS_TUNE_KNOWN_BITS) != 0) return BS_ERR_ARG;
    if (o.variant == BS_VARIANT_TMA && o.tile_bytes == 0 && o.stages == 0 && o.warps == 0) return BS_OK;  // presets
    // the LDG variant works on whole granules; a TMA tile is any multiple of 1 KiB (the block range of a tile is looked up
    // by the granules it touches)
    if (o.tile_bytes == 0 || o.tile_bytes % (o.variant == BS_VARIANT_TMA ? 1024u : kGranule) != 0 || o.tile_bytes > 65536 ||
        (o.variant == BS_VARIANT_TMA && o.tile_bytes < 4096))
        return BS_ERR_ARG;
    if (o.variant == BS_VARIANT_TMA &&
        (o.stages < 3 || o.stages > 8 || o.warps < 1 || o.warps > 16 ||
         (uint64_t)o.warps * ((uint64_t)o.stages * o.tile_bytes + kMetaBytesPerWarp) > 224u * 1024u))
        return BS_ERR_ARG;
    return BS_OK;
}

static ScanParams serialize_scan_params(const bs_set_desc* set, const WsLayout& L, uint64_t capacity, uint64_t expect_total,
                                        bs_result* d_result)
{
    ScanParams sp;
    memset(&sp, 0, sizeof(sp));
    sp.ws = L;
    sp.result = d_result;
    sp.capacity = capacity;
    sp.expect_total = expect_total;
    sp.tensors = set->tensors;
    sp.dim = set->dim;
    sp.addr = set->addr;
    sp.T = set->n_tensors;
    sp.B = set->n_blocks;
    sp.dtype = set->dtype;
    return sp;
}

// S1/S2/S4: run the size / offset pass for `set`
int run_serialize_scan(const bs_set_desc* set, const WsLayout& L, uint64_t capacity, uint64_t expect_total,
                       bs_result* d_result, int sms, cudaStream_t stream)
{
    const cudaError_t e = launch_scan(false, serialize_scan_params(set, L, capacity, expect_total, d_result), sms, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

static MoveParams pack_params(const bs_set_desc* set, const WsLayout& L, void* d_dst, uint64_t lo, uint64_t hi, const bs_opts& o,
                              uint32_t flags = 0)
{
    MoveParams mp;
    memset(&mp, 0, sizeof(mp));
    mp.ws = L;
    mp.tensors = set->tensors;
    mp.qn = set->qn;
    mp.dim = set->dim;
    mp.addr = set->addr;
    mp.stream = (unsigned char*)d_dst;
    mp.lo = lo;
    mp.hi = hi;
    mp.tile_bytes = o.tile_bytes;
    mp.tune = o.tune;
    mp.pace = o.pace;
    mp.flags = flags;
    mp.rank4 = set->dtype & BS_RANK4;
    return mp;
}

int run_pack_range(const bs_set_desc* set, const WsLayout& L, void* d_dst, uint64_t lo, uint64_t hi,
                   const bs_opts& o, int sms, cudaStream_t stream, uint32_t flags)
{
    const cudaError_t e = launch_move(false, pack_params(set, L, d_dst, lo, hi, o, flags), o, sms, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

// One launch or two?  bs_opts.fuse: 0 = by size, 1 = always separate launches, 2 = always one fused launch.  By size:
// the fused kernel runs the pass on one CTA per SM, so sets of more work items than that leave the pass to its own,
// wider launch (whose ~5 us are then < 1 % of the call).
static bool use_fused(const bs_opts& o, uint64_t T, uint64_t B, int sms)
{
    if (o.variant != BS_VARIANT_TMA || o.fuse == 1u) return false;
    if (o.fuse == 2u) return true;
    const uint64_t nt = (B + kScanTile - 1) / kScanTile, ntt = (T + kScanTile - 1) / kScanTile;
    return (nt > ntt ? nt : ntt) <= (uint64_t)sms;
}

static ScanParams deserialize_scan_params(const void* d_header, const void* d_payload, uint64_t nbytes, const bs_set_desc* out,
                                          void* d_pool, uint64_t pool_bytes, uint32_t flags, const WsLayout& L, bs_result* d_result)
{
    ScanParams sp;
    memset(&sp, 0, sizeof(sp));
    sp.ws = L;
    sp.result = d_result;
    sp.T = out->n_tensors;
    sp.B = out->n_blocks;
    sp.header = (const unsigned char*)d_header;
    sp.payload = (const unsigned char*)d_payload;
    sp.nbytes = nbytes;
    sp.pool_base = (uint64_t)(uintptr_t)d_pool;
    sp.pool_bytes = pool_bytes;
    sp.out_dim = out->dim;
    sp.out_addr = out->addr;
    sp.flags = flags;
    sp.dtype = out->dtype & BS_RANK4;  // the shape of the out arrays (three or four legs per block)
    return sp;
}

int run_deserialize_scan(const void* d_header, const void* d_payload, uint64_t nbytes, const bs_set_desc* out,
                         void* d_pool, uint64_t pool_bytes, uint32_t flags, const WsLayout& L, bs_result* d_result,
                         int sms, cudaStream_t stream)
{
    const cudaError_t e = launch_scan(true, deserialize_scan_params(d_header, d_payload, nbytes, out, d_pool, pool_bytes, flags, L, d_result),
                                      sms, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

static MoveParams unpack_params(const bs_set_desc* out, const WsLayout& L, const void* d_src, const void* d_header, uint64_t lo,
                                uint64_t hi, uint32_t flags, const bs_opts& o)
{
    MoveParams mp;
    memset(&mp, 0, sizeof(mp));
    mp.ws = L;
    mp.tensors = out->tensors;
    mp.qn = out->qn;
    mp.dim = out->dim;
    mp.addr = out->addr;
    mp.stream = (unsigned char*)const_cast<void*>(d_src);
    mp.header = (const unsigned char*)d_header;
    mp.lo = lo;
    mp.hi = hi;
    mp.tile_bytes = o.tile_bytes;
    mp.tune = o.tune;
    mp.pace = o.pace;
    mp.flags = flags;
    mp.rank4 = out->dtype & BS_RANK4;
    return mp;
}

int run_unpack_range(const bs_set_desc* out, const WsLayout& L, const void* d_src, const void* d_header,
                     uint64_t lo, uint64_t hi, uint32_t flags, const bs_opts& o, int sms, cudaStream_t stream)
{
    const cudaError_t e = launch_move(true, unpack_params(out, L, d_src, d_header, lo, hi, flags, o), o, sms, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

// the whole stream <-> package slots in one launch each (bs.h "packages"; PkgMap in bs_internal.cuh)
int run_pack_packages(const bs_set_desc* set, const WsLayout& L, const PkgMap& pm, const bs_opts& o, int sms, cudaStream_t stream)
{
    return run_pack_packages_range(set, L, pm, 0, UINT64_MAX, o, sms, stream);
}

// stream bytes [lo, hi) (whole packages of the cut) -> their slots
int run_pack_packages_range(const bs_set_desc* set, const WsLayout& L, const PkgMap& pm, uint64_t lo, uint64_t hi, const bs_opts& o,
                            int sms, cudaStream_t stream)
{
    MoveParams mp;
    memset(&mp, 0, sizeof(mp));
    mp.ws = L;
    mp.tensors = set->tensors;
    mp.qn = set->qn;
    mp.dim = set->dim;
    mp.addr = set->addr;
    mp.lo = lo;
    mp.hi = hi;
    mp.tile_bytes = o.tile_bytes;
    mp.tune = o.tune;
    mp.pace = o.pace;
    mp.pkg = pm;
    mp.rank4 = set->dtype & BS_RANK4;
    cudaError_t e = launch_move(false, mp, o, sms, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

// payload only: the header region was gathered and parsed before (header = nullptr: no descriptor rebuild here)
int run_unpack_packages(const bs_set_desc* out, const WsLayout& L, const PkgMap& pm, uint64_t header_bytes, uint32_t flags,
                        const bs_opts& o, int sms, cudaStream_t stream)
{
    (void)header_bytes;
    return run_unpack_packages_range(out, L, pm, 0, UINT64_MAX, flags, o, sms, stream);
}

// payload bytes of the stream range [lo, hi) (whole packages of the cut) out of their slots
int run_unpack_packages_range(const bs_set_desc* out, const WsLayout& L, const PkgMap& pm, uint64_t lo, uint64_t hi, uint32_t flags,
                              const bs_opts& o, int sms, cudaStream_t stream)
{
    MoveParams mp;
    memset(&mp, 0, sizeof(mp));
    mp.ws = L;
    mp.tensors = out->tensors;
    mp.qn = out->qn;
    mp.dim = out->dim;
    mp.addr = out->addr;
    mp.lo = lo;
    mp.hi = hi;
    mp.tile_bytes = o.tile_bytes;
    mp.tune = o.tune;
    mp.pace = o.pace;
    mp.flags = flags;
    mp.pkg = pm;
    mp.rank4 = out->dtype & BS_RANK4;
    cudaError_t e = launch_move(true, mp, o, sms, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

}  // namespace bs

using namespace bs;

extern "C" {

uint32_t bs_version(void) { return BS_VERSION; }

const char* bs_strerror(int code)
{
    switch (code) {
        case BS_OK: return "ok";
        case BS_PENDING: return "pending";
        case BS_ERR_ARG: return "invalid argument or descriptor";
        case BS_ERR_CAPACITY: return "capacity too small";
        case BS_ERR_CORRUPT: return "corrupt stream header";
        case BS_ERR_UNSUPPORTED: return "unsupported rank, dtype or label count";
        case BS_ERR_CUDA: return "CUDA runtime error";
        case BS_ERR_IO: return "file IO error in the storage tier";
        default: return "unknown error";
    }
}

int bs_last_cuda_error(void) { return g_last_cuda_error; }

uint64_t bs_header_bytes(uint64_t n_tensors, uint64_t n_blocks)
{
    return align_up(kFixedHeader + kTensorRec * n_tensors + kBlockRec * n_blocks, kHeaderAlign);
}

uint64_t bs_header_bytes_rank4(uint64_t n_tensors, uint64_t n_blocks) { return header_bytes_of(n_tensors, n_blocks, BS_RANK4); }

uint64_t bs_workspace_bytes(uint32_t n_tensors, uint32_t n_blocks, uint64_t stream_capacity)
{
    (void)n_tensors;
    return ws_fixed_bytes(n_blocks) + align_up(4 * (stream_capacity / kGranule + 4), 256);
}

int bs_stream_info(const void* h, bs_stream_info_t* out)
{
    if (h == nullptr || out == nullptr) return BS_ERR_ARG;
    const unsigned char* s = (const unsigned char*)h;
    uint32_t w[8];
    uint64_t q[4];
    memcpy(w, s, 32);
    memcpy(q, s + 32, 32);
    if (memcmp(s, "BSPARSE1", 8) != 0) return BS_ERR_CORRUPT;
    const bool v3 = w[2] == 3u;  // wire format v3: four legs per block record
    if ((w[2] != 1u && !v3) || w[3] != 0x01020304u || w[4] > (uint32_t)BS_C128 || w[5] != 2u || w[6] != (v3 ? 4u : 3u) ||
        (w[7] != 16u && !(w[7] == 8u && !v3)))
        return BS_ERR_CORRUPT;
    if (q[0] >= (1ull << 32) || q[1] >= (1ull << 32)) return BS_ERR_CORRUPT;
    if (q[2] != header_bytes_of(q[0], q[1], v3 ? BS_RANK4 : 0u)) return BS_ERR_CORRUPT;
    out->max_rank = w[6];
    out->n_tensors = q[0];
    out->n_blocks = q[1];
    out->header_bytes = q[2];
    out->payload_bytes = q[3];
    out->total_bytes = q[2] + q[3];
    out->dtype = w[4];
    out->align = w[7];
    return BS_OK;
}

int bs_serialized_size(const bs_set_desc* set, void* d_ws, uint64_t ws_bytes, uint64_t* header_bytes,
                       uint64_t* total_bytes, cudaStream_t stream)
{
    int rc = check_set(set);
    if (rc) return rc;
    if (header_bytes == nullptr || total_bytes == nullptr) return BS_ERR_ARG;
    WsLayout L;
    if (!ws_layout(d_ws, ws_bytes, set->n_blocks, &L)) return d_ws && aligned(d_ws, 256) ? BS_ERR_CAPACITY : BS_ERR_ARG;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    if ((rc = run_serialize_scan(set, L, UINT64_MAX, 0, nullptr, sms, stream))) return rc;
    WsHead h;
    cudaError_t e = cudaMemcpyAsync(&h, L.head, sizeof(h), cudaMemcpyDeviceToHost, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return cuda_fail(e);
    *header_bytes = h.header_bytes;
    *total_bytes = h.header_bytes + h.payload_bytes;
    // a workspace too small for the tile index is not an error for a size query
    if (h.status == BS_ERR_CAPACITY) return BS_OK;
    return h.status;
}

int bs_serialize_range(const bs_set_desc* set, void* d_dst, uint64_t lo, uint64_t hi, int run_scan, void* d_ws,
                       uint64_t ws_bytes, bs_result* d_result, const bs_opts* opts, cudaStream_t stream)
{
    int rc = check_set(set);
    if (rc) return rc;
    if (d_dst == nullptr || !aligned(d_dst, 16) || (lo & 15) || (hi & 15) || lo > hi) return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    if ((rc = check_opts(o))) return rc;
    if ((set->dtype & BS_ALIGN8) && o.variant != BS_VARIANT_TMA) return BS_ERR_UNSUPPORTED;  // the LDG variant moves 16-byte units
    WsLayout L;
    if (!ws_layout(d_ws, ws_bytes, set->n_blocks, &L)) return d_ws && aligned(d_ws, 256) ? BS_ERR_CAPACITY : BS_ERR_ARG;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    if (run_scan && (rc = run_serialize_scan(set, L, UINT64_MAX, 0, d_result, sms, stream))) return rc;
    return run_pack_range(set, L, d_dst, lo, hi, o, sms, stream);
}

int bs_serialize(const bs_set_desc* set, void* d_stream, uint64_t capacity, void* d_ws, uint64_t ws_bytes,
                 bs_result* d_result, const bs_opts* opts, cudaStream_t stream)
{
    int rc = check_set(set);
    if (rc) return rc;
    if (d_stream == nullptr || !aligned(d_stream, 16)) return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    if ((rc = check_opts(o))) return rc;
    if ((set->dtype & BS_ALIGN8) && o.variant != BS_VARIANT_TMA) return BS_ERR_UNSUPPORTED;  // the LDG variant moves 16-byte units
    WsLayout L;
    if (!ws_layout(d_ws, ws_bytes, set->n_blocks, &L)) return d_ws && aligned(d_ws, 256) ? BS_ERR_CAPACITY : BS_ERR_ARG;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    // the range is the whole stream: the pass refuses a total beyond `capacity`, the movement clips to the total
    constexpr uint64_t kAll = ~15ull;
    if (use_fused(o, set->n_tensors, set->n_blocks, sms)) {  // the pass and the pack in ONE launch
        const cudaError_t e = launch_fused_tma(false, serialize_scan_params(set, L, capacity, 0, d_result),
                                               pack_params(set, L, d_stream, 0, kAll, o), o, capacity, sms, stream);
        return e == cudaSuccess ? BS_OK : cuda_fail(e);
    }
    if ((rc = run_serialize_scan(set, L, capacity, 0, d_result, sms, stream))) return rc;
    return run_pack_range(set, L, d_stream, 0, kAll, o, sms, stream);
}

int bs_deserialize(const void* d_stream, uint64_t nbytes, bs_set_desc* out, void* d_pool, uint64_t pool_bytes,
                   uint32_t flags, void* d_ws, uint64_t ws_bytes, bs_result* d_result, const bs_opts* opts,
                   cudaStream_t stream)
{
    int rc = check_set(out);
    if (rc) return rc;
    if (d_stream == nullptr || !aligned(d_stream, 16)) return BS_ERR_ARG;
    if (flags != BS_LAYOUT_POOL && flags != BS_SCATTER_TO_ADDR) return BS_ERR_ARG;
    if (flags == BS_LAYOUT_POOL && pool_bytes && (d_pool == nullptr || !aligned(d_pool, 256))) return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    if ((rc = check_opts(o))) return rc;
    WsLayout L;
    if (!ws_layout(d_ws, ws_bytes, out->n_blocks, &L)) return d_ws && aligned(d_ws, 256) ? BS_ERR_CAPACITY : BS_ERR_ARG;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    const unsigned char* s = (const unsigned char*)d_stream;
    // an align-8 stream cannot go through the LDG variant (16-byte units): its parse pass then refuses it
    const uint32_t pflags = flags | (o.variant != BS_VARIANT_TMA ? kFlagNoAlign8 : 0u);
    constexpr uint64_t kAll = ~15ull;  // the parse pass proves header_bytes + payload_bytes == nbytes; the movement clips to it
    // the payload is only dereferenced (pad-zero check) after the fixed header proved header_bytes + P == nbytes
    if (use_fused(o, out->n_tensors, out->n_blocks, sms)) {  // parse / validate and unpack in ONE launch
        const cudaError_t e = launch_fused_tma(true, deserialize_scan_params(s, s, nbytes, out, d_pool, pool_bytes, pflags, L, d_result),
                                               unpack_params(out, L, s, s, 0, kAll, flags, o), o, nbytes, sms, stream);
        return e == cudaSuccess ? BS_OK : cuda_fail(e);
    }
    if ((rc = run_deserialize_scan(s, s, nbytes, out, d_pool, pool_bytes, pflags, L, d_result, sms, stream))) return rc;
    return run_unpack_range(out, L, s, s, 0, kAll, flags, o, sms, stream);
}

int bs_deserialize_range(const void* d_src, uint64_t lo, uint64_t hi, const void* d_header, bs_set_desc* out, uint32_t flags,
                         void* d_ws, uint64_t ws_bytes, const bs_opts* opts, cudaStream_t stream)
{
    int rc = check_set(out);
    if (rc) return rc;
    if (d_src == nullptr || !aligned(d_src, 16) || (lo & 15) || (hi & 15) || lo > hi) return BS_ERR_ARG;
    if (d_header != nullptr && !aligned(d_header, 16)) return BS_ERR_ARG;
    if (flags != BS_LAYOUT_POOL && flags != BS_SCATTER_TO_ADDR) return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    if ((rc = check_opts(o))) return rc;
    WsLayout L;
    if (!ws_layout(d_ws, ws_bytes, out->n_blocks, &L)) return d_ws && aligned(d_ws, 256) ? BS_ERR_CAPACITY : BS_ERR_ARG;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    return run_unpack_range(out, L, d_src, d_header, lo, hi, flags, o, sms, stream);
}

}  // extern "C"
