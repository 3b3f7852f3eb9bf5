// bs_pkg.cu — self-contained packages (PAPER §III.B.3; include/bs.h "packages").
//
// A package is a 64-byte header + a range of the wire-format-v1 stream; the header "pinpoints the location of the
// component within the original, whole object" (L124), so packages can be "mixed with other packages and received
// back without the need to keep track of their order".  Nothing new moves the data: a package's bytes are a byte range
// [lo, hi) of the stream, which is exactly what the tile-partitioned pack / unpack kernels take (a range of tiles), so
//   emit   = scan | per package: pkg_header_kernel (64 bytes: where am I, which block do I start in) + pack [lo,hi)
//   unpack = gather the header-region packages | parse/validate scan | pkg_check_kernel (every package against the
//            offset table) | descriptor rebuild | per payload package, in the order the slots lie: unpack [lo,hi)
// and when the size limit is a multiple of the work tile (16 KiB by default) no tile straddles a package, so the move
// kernels take a PkgMap (stream byte -> slot address, bs_internal.cuh) and the whole set costs a fixed number of
// launches however many packages the limit makes:
//   emit   = scan | pkg_headers_kernel (all headers) | pack (whole stream -> slots)
//   unpack = pkg_index_kernel | pkg_gather_header_kernel | scan | pkg_check_kernel | rebuild | unpack (slots -> blocks)
// The host reads package headers only to plan these launches (which slot holds which range); see bs.h for who checks
// what.
#include <string.h>

#include <algorithm>
#include <vector>

#include "bs_pkg.cuh"

namespace bs {

namespace {

// the block holding payload byte x (x < P): the largest i in [0,B) with off_i <= x
__device__ __forceinline__ uint32_t block_of_byte(const Blk* __restrict__ blk, uint32_t B, uint64_t x)
{
    uint32_t lo = 0, hi = B;  // invariant: off[lo] <= x (off[0] = 0), answer in [lo, hi)
    while (hi - lo > 1) {
        const uint32_t mid = lo + ((hi - lo) >> 1);
        if (blk[mid].off <= x) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ void pkg_fail(WsHead* head, bs_result* result, int code)
{
    atomicCAS(&head->status, 0, code);
    if (result != nullptr) result->status = head->status;
}

// the 64-byte header of package k -> dst
// poison (engine path): on a deferred error the slot's header is blanked, so a stale package never reaches the host as valid
__device__ __forceinline__ void pkg_write_header(const WsLayout& ws, uint64_t cap, uint64_t stream_id, uint64_t k,
                                                 uint64_t expect_count, unsigned char* dst, bs_result* result, bool poison)
{
    WsHead* head = ws.head;
    if (head->status != 0) {  // deferred error: nothing is written
        if (poison)
            for (int z = 0; z < 4; ++z) reinterpret_cast<uint4*>(dst)[z] = make_uint4(0, 0, 0, 0);
        return;
    }
    const uint64_t hb = head->header_bytes, total = hb + head->payload_bytes;
    const uint32_t B = head->n_blocks;
    const uint64_t count = pkg_count(hb, total, cap);
    uint64_t lo = 0, hi = 0;
    if (count != expect_count || !pkg_range(hb, total, cap, k, &lo, &hi)) {
        pkg_fail(head, result, BS_ERR_ARG);
        return;
    }
    uint32_t first_block = BS_PKG_NO_BLOCK;
    uint64_t intra = 0;
    if (lo >= hb) {
        first_block = block_of_byte(ws.blk, B, lo - hb);
        intra = lo - hb - ws.blk[first_block].off;
    }
    uint4* o = reinterpret_cast<uint4*>(dst);
    o[0] = make_uint4(0x4b505342u, 0x31303047u, 1u, (uint32_t)k);  // "BSPKG001", version, index
    o[1] = make_uint4((uint32_t)count, first_block, (uint32_t)stream_id, (uint32_t)(stream_id >> 32));
    o[2] = make_uint4((uint32_t)total, (uint32_t)(total >> 32), (uint32_t)lo, (uint32_t)(lo >> 32));
    const uint64_t nb = hi - lo;
    o[3] = make_uint4((uint32_t)nb, (uint32_t)(nb >> 32), (uint32_t)intra, (uint32_t)(intra >> 32));
    if (k == 0 && result != nullptr) result->reserved[3] = (uint32_t)count;
}

// one thread: package k -> dst
__global__ void pkg_header_kernel(WsLayout ws, uint64_t cap, uint64_t stream_id, uint64_t k, uint64_t expect_count,
                                  unsigned char* dst, bs_result* result, bool poison)
{
    if (threadIdx.x != 0 || blockIdx.x != 0) return;
    pkg_write_header(ws, cap, stream_id, k, expect_count, dst, result, poison);
}

// one thread per package: every header of the cut -> its slot (slot_of: device table index -> slot, or identity)
__global__ void pkg_headers_kernel(WsLayout ws, uint64_t cap, uint64_t stream_id, uint64_t first, uint64_t n, uint64_t count,
                                   unsigned char* base, uint64_t slot_bytes, const uint32_t* slot_of, bs_result* result, bool poison)
{
    const uint64_t i = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const uint64_t k = first + i;  // packages [first, first + n) of the cut; without a table they lie in slots 0 .. n-1
    const uint64_t slot = slot_of ? (uint64_t)slot_of[k] : i;
    pkg_write_header(ws, cap, stream_id, k, count, base + slot * slot_bytes, result, poison);
}

// one thread per slot: slot_of[index] = slot for the packages of this stream (the host plan proved the indices unique)
__global__ void pkg_index_kernel(const unsigned char* base, uint64_t stride, uint64_t n_slots, uint64_t stream_id,
                                 uint32_t* slot_of, uint64_t count)
{
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_slots) return;
    const uint4* h = reinterpret_cast<const uint4*>(base + s * stride);
    const uint4 a = h[0], b = h[1];
    if (a.x != 0x4b505342u || a.y != 0x31303047u || (((uint64_t)b.w << 32) | b.z) != stream_id) return;
    if (a.w < count) slot_of[a.w] = (uint32_t)s;
}

// the header region [0, hb), stored continuously (L126): 16-byte units out of the header-region packages
__global__ void pkg_gather_header_kernel(const unsigned char* base, uint64_t slot_bytes, const uint32_t* slot_of,
                                         uint64_t cap, uint64_t hb, unsigned char* dst)
{
    const uint64_t n = hb / 16;
    for (uint64_t u = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x; u < n; u += (uint64_t)gridDim.x * blockDim.x) {
        const uint64_t s = u * 16, k = s / cap;
        const uint4 v = *reinterpret_cast<const uint4*>(base + (uint64_t)slot_of[k] * slot_bytes + BS_PKG_HEADER + (s - k * cap));
        *reinterpret_cast<uint4*>(dst + s) = v;
    }
}

// one thread per slot: the package header at base + s*stride against the parsed stream (after the DESER scan)
__global__ void pkg_check_kernel(WsLayout ws, const unsigned char* base, uint64_t stride, uint64_t n_slots,
                                 uint64_t stream_id, bs_result* result)
{
    const uint64_t s = (uint64_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (s >= n_slots) return;
    WsHead* head = ws.head;
    if (head->status != 0) return;
    const uint4* h = reinterpret_cast<const uint4*>(base + s * stride);
    const uint4 a = h[0], b = h[1], c = h[2], d = h[3];
    if (a.x != 0x4b505342u || a.y != 0x31303047u) return;                 // foreign slot
    if ((((uint64_t)b.w << 32) | b.z) != stream_id) return;               // another serialization call's package
    const uint64_t hb = head->header_bytes, total = hb + head->payload_bytes;
    const uint32_t B = head->n_blocks;
    const uint64_t p_total = ((uint64_t)c.y << 32) | c.x, lo = ((uint64_t)c.w << 32) | c.z;
    const uint64_t nb = ((uint64_t)d.y << 32) | d.x, intra = ((uint64_t)d.w << 32) | d.z;
    const uint32_t first_block = b.y;
    bool ok = a.z == 1u && p_total == total && nb != 0 && lo <= total && nb <= total - lo;
    if (ok) {
        if (lo < hb) {
            ok = lo + nb <= hb && first_block == BS_PKG_NO_BLOCK && intra == 0;
        } else if (B == 0) {
            ok = false;
        } else {
            const uint32_t i = block_of_byte(ws.blk, B, lo - hb);
            ok = first_block == i && intra == lo - hb - ws.blk[i].off;
        }
    }
    if (!ok) pkg_fail(head, result, BS_ERR_CORRUPT);
}

// bytes per work tile of the move kernels for these options (the TMA presets use 16 KiB tiles)
uint32_t work_tile_bytes(const bs_opts& o) { return o.tile_bytes ? o.tile_bytes : kGranule; }

uint32_t rd32(const unsigned char* p) { uint32_t v; memcpy(&v, p, 4); return v; }
uint64_t rd64(const unsigned char* p) { uint64_t v; memcpy(&v, p, 8); return v; }

}  // namespace

cudaError_t launch_pkg_header(const WsLayout& L, uint64_t cap, uint64_t stream_id, uint64_t k, uint64_t expect_count,
                              void* d_dst, bs_result* d_result, cudaStream_t stream, bool poison)
{
    pkg_header_kernel<<<1, 32, 0, stream>>>(L, cap, stream_id, k, expect_count, (unsigned char*)d_dst, d_result, poison);
    return cudaGetLastError();
}

cudaError_t launch_pkg_headers(const WsLayout& L, uint64_t cap, uint64_t stream_id, uint64_t first, uint64_t n, uint64_t count,
                               void* d_base, uint64_t slot_bytes, const uint32_t* d_slot_of, bs_result* d_result, cudaStream_t stream,
                               bool poison)
{
    if (n == 0) return cudaSuccess;
    pkg_headers_kernel<<<(unsigned)((n + 127) / 128), 128, 0, stream>>>(L, cap, stream_id, first, n, count, (unsigned char*)d_base,
                                                                         slot_bytes, d_slot_of, d_result, poison);
    return cudaGetLastError();
}

cudaError_t launch_pkg_check(const WsLayout& L, const void* d_hdrs, uint64_t stride, uint64_t n_slots, uint64_t stream_id,
                             bs_result* d_result, cudaStream_t stream)
{
    if (n_slots == 0) return cudaSuccess;
    const unsigned threads = 128;
    const unsigned grid = (unsigned)((n_slots + threads - 1) / threads);
    pkg_check_kernel<<<grid, threads, 0, stream>>>(L, (const unsigned char*)d_hdrs, stride, n_slots, stream_id, d_result);
    return cudaGetLastError();
}

// Host: read n_slots package headers (h_hdrs + s*stride) and lay out the copies.  Checks what the plan relies on.
int pkg_plan(const unsigned char* h_hdrs, uint64_t stride, uint64_t n_slots, uint64_t slot_bytes, uint64_t stream_id,
             PkgPlan* plan)
{
    plan->items.clear();
    plan->total = 0;
    plan->hb = 0;
    plan->n_header = 0;
    uint64_t count = 0;
    for (uint64_t s = 0; s < n_slots; ++s) {
        const unsigned char* h = h_hdrs + s * stride;
        if (memcmp(h, "BSPKG001", 8) != 0 || rd64(h + 24) != stream_id) continue;  // foreign slot
        if (rd32(h + 8) != 1u) return BS_ERR_CORRUPT;
        PkgItem it;
        it.slot = s;
        it.index = rd32(h + 12);
        it.first_block = rd32(h + 20);
        it.lo = rd64(h + 40);
        it.nbytes = rd64(h + 48);
        if (plan->items.empty()) {
            count = rd32(h + 16);
            plan->total = rd64(h + 32);
        } else if (rd32(h + 16) != count || rd64(h + 32) != plan->total) {
            return BS_ERR_CORRUPT;
        }
        plan->items.push_back(it);
    }
    if (plan->items.empty() || plan->items.size() != count) return BS_ERR_CORRUPT;
    std::sort(plan->items.begin(), plan->items.end(), [](const PkgItem& a, const PkgItem& b) { return a.index < b.index; });
    uint64_t next = 0;
    bool in_header = true;
    for (uint64_t k = 0; k < count; ++k) {
        const PkgItem& it = plan->items[k];
        if (it.index != k) return BS_ERR_CORRUPT;  // a duplicate or a hole
        if (it.lo != next || it.nbytes == 0 || it.nbytes > plan->total - it.lo || (it.lo & 15) || (it.nbytes & 7)) return BS_ERR_CORRUPT;  // (the last package of an align-8 stream ends 8 off the grid)
        if (it.nbytes > slot_bytes - BS_PKG_HEADER) return BS_ERR_CORRUPT;
        const bool hdr = it.first_block == BS_PKG_NO_BLOCK;
        if (hdr && !in_header) return BS_ERR_CORRUPT;  // header-region packages are a prefix in index order
        if (hdr) { plan->hb = it.lo + it.nbytes; ++plan->n_header; }
        else in_header = false;
        next = it.lo + it.nbytes;
    }
    if (next != plan->total || plan->hb < kFixedHeader) return BS_ERR_CORRUPT;
    return BS_OK;
}

// The size limit `cap` whose cut (bs.h) these packages are, if it is a multiple of `tile`; 0 if they are cut otherwise.
uint64_t plan_uniform_cap(const PkgPlan& plan, uint32_t tile)
{
    const uint64_t n = plan.items.size(), nh = plan.n_header;
    uint64_t cap;
    if (nh > 1) cap = plan.items[0].nbytes;
    else if (n - nh > 1) cap = plan.items[nh].nbytes;
    else cap = align_up(std::max(plan.hb, plan.total - plan.hb), 65536);  // one package per region: any limit this large
    if (cap == 0 || cap % tile != 0 || pkg_count(plan.hb, plan.total, cap) != n) return 0;
    for (uint64_t k = 0; k < n; ++k) {
        uint64_t lo = 0, hi = 0;
        if (!pkg_range(plan.hb, plan.total, cap, k, &lo, &hi) || lo != plan.items[k].lo || hi - lo != plan.items[k].nbytes) return 0;
    }
    return cap;
}

}  // namespace bs

using namespace bs;

#define CK(call)                                          \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) return cuda_fail(e__);    \
    } while (0)

static bool aligned16(const void* p) { return ((uintptr_t)p & 15) == 0; }

extern "C" {

uint64_t bs_package_count(uint64_t header_bytes, uint64_t total_bytes, uint64_t cap)
{
    return pkg_count(header_bytes, total_bytes, cap);
}

int bs_package_range(uint64_t header_bytes, uint64_t total_bytes, uint64_t cap, uint64_t index, uint64_t* lo, uint64_t* hi)
{
    if (lo == nullptr || hi == nullptr) return BS_ERR_ARG;
    return pkg_range(header_bytes, total_bytes, cap, index, lo, hi) ? BS_OK : BS_ERR_ARG;
}

uint64_t bs_package_workspace_bytes(uint32_t n_tensors, uint32_t n_blocks, uint64_t stream_capacity)
{
    // v1 workspace | slot table of the one-launch path (limits >= 16 KiB: at most one entry per 16 KiB) | header region
    const uint64_t hb = header_bytes_of(n_tensors, n_blocks, BS_RANK4);  // room for 64-byte block records (wire format v3)
    return bs_workspace_bytes(n_tensors, n_blocks, stream_capacity) + align_up(4 * (stream_capacity / kGranule + hb / kGranule + 4), 256) +
           256 + align_up(hb, 256);
}

int bs_package_emit(const bs_set_desc* set, uint64_t total_bytes, uint64_t cap, uint64_t stream_id, void* d_slots,
                    uint64_t slot_bytes, uint64_t n_slots, const uint32_t* h_slot_of, void* d_ws, uint64_t ws_bytes,
                    bs_result* d_result, const bs_opts* opts, cudaStream_t stream)
{
    if (set == nullptr) return BS_ERR_ARG;
    { const int rc0 = check_set(set); if (rc0) return rc0; }
    if (d_slots == nullptr || !aligned16(d_slots) || cap == 0 || (cap & 15) || (slot_bytes & 15) ||
        slot_bytes < BS_PKG_HEADER + cap)
        return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    int rc;
    if ((rc = check_opts(o))) return rc;
    if ((set->dtype & BS_ALIGN8) && o.variant != BS_VARIANT_TMA) return BS_ERR_UNSUPPORTED;  // the LDG variant moves 16-byte units
    WsLayout L;
    if (!ws_layout(d_ws, ws_bytes, set->n_blocks, &L)) return d_ws && ((uintptr_t)d_ws & 255) == 0 ? BS_ERR_CAPACITY : BS_ERR_ARG;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    const uint64_t hb = header_bytes_of(set->n_tensors, set->n_blocks, set->dtype);
    if (total_bytes == 0) {
        uint64_t hb2 = 0;
        if ((rc = bs_serialized_size(set, d_ws, ws_bytes, &hb2, &total_bytes, stream))) return rc;
    }
    const uint64_t count = pkg_count(hb, total_bytes, cap);
    if (count == 0 || count >= (1ull << 32)) return BS_ERR_ARG;
    if (count > n_slots) return BS_ERR_CAPACITY;
    if (h_slot_of != nullptr) {  // a permutation into [0, n_slots)
        std::vector<bool> used((size_t)n_slots, false);
        for (uint64_t k = 0; k < count; ++k) {
            if (h_slot_of[k] >= n_slots || used[h_slot_of[k]]) return BS_ERR_ARG;
            used[h_slot_of[k]] = true;
        }
    }
    if ((rc = run_serialize_scan(set, L, UINT64_MAX, total_bytes, d_result, sms, stream))) return rc;
    if (cap % work_tile_bytes(o) == 0) {
        // every work tile lies inside one package: ONE launch writes all package headers, ONE moves the whole stream
        // into the slots, however many packages the size limit makes
        uint32_t* d_tab = nullptr;
        bool tab_owned = false;
        if (h_slot_of != nullptr) {  // the slot table: the tail of a bs_package_workspace_bytes workspace, else a stream-ordered allocation
            const uint64_t tab = align_up(count * sizeof(uint32_t), 256);
            if (ws_bytes >= bs_workspace_bytes(set->n_tensors, set->n_blocks, total_bytes) + tab) {
                d_tab = (uint32_t*)((unsigned char*)d_ws + ((ws_bytes - tab) & ~255ull));
            } else {
                CK(cudaMallocAsync((void**)&d_tab, count * sizeof(uint32_t), stream));
                tab_owned = true;
            }
            CK(cudaMemcpyAsync(d_tab, h_slot_of, count * sizeof(uint32_t), cudaMemcpyHostToDevice, stream));
        }
        CK(launch_pkg_headers(L, cap, stream_id, 0, count, count, d_slots, slot_bytes, d_tab, d_result, stream));
        PkgMap pm;
        pm.cap = cap; pm.slot_bytes = slot_bytes; pm.base = (unsigned char*)d_slots; pm.slot_of = d_tab; pm.k_base = 0;
        rc = run_pack_packages(set, L, pm, o, sms, stream);
        if (tab_owned) CK(cudaFreeAsync(d_tab, stream));
        return rc;
    }
    for (uint64_t k = 0; k < count; ++k) {  // any other limit: package by package
        uint64_t lo = 0, hi = 0;
        pkg_range(hb, total_bytes, cap, k, &lo, &hi);
        unsigned char* slot = (unsigned char*)d_slots + (h_slot_of ? (uint64_t)h_slot_of[k] : k) * slot_bytes;
        CK(launch_pkg_header(L, cap, stream_id, k, count, slot, d_result, stream));
        if ((rc = run_pack_range(set, L, slot + BS_PKG_HEADER, lo, hi, o, sms, stream))) return rc;
    }
    return BS_OK;
}

int bs_package_unpack(const void* d_slots, uint64_t slot_bytes, uint64_t n_slots, uint64_t stream_id, bs_set_desc* out,
                      void* d_pool, uint64_t pool_bytes, uint32_t flags, void* d_ws, uint64_t ws_bytes, bs_result* d_result,
                      const bs_opts* opts, cudaStream_t stream)
{
    if (out == nullptr) return BS_ERR_ARG;
    { const int rc0 = check_set(out); if (rc0) return rc0; }
    if (d_slots == nullptr || !aligned16(d_slots) || (slot_bytes & 15) || slot_bytes < BS_PKG_HEADER + 16 || n_slots == 0)
        return BS_ERR_ARG;
    if (flags != BS_LAYOUT_POOL && flags != BS_SCATTER_TO_ADDR) return BS_ERR_ARG;
    if (flags == BS_LAYOUT_POOL && pool_bytes && (d_pool == nullptr || ((uintptr_t)d_pool & 255))) return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    int rc;
    if ((rc = check_opts(o))) return rc;
    // workspace := v1 workspace | room for the assembled header region
    const uint64_t hdr_cap = align_up(header_bytes_of(out->n_tensors, out->n_blocks, out->dtype), 256);
    if (d_ws == nullptr || ((uintptr_t)d_ws & 255)) return BS_ERR_ARG;
    if (ws_bytes < hdr_cap) return BS_ERR_CAPACITY;
    const uint64_t w1 = (ws_bytes - hdr_cap) & ~255ull;
    WsLayout L;
    if (!ws_layout(d_ws, w1, out->n_blocks, &L)) return BS_ERR_CAPACITY;
    unsigned char* d_header = (unsigned char*)d_ws + w1;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;

    std::vector<unsigned char> hdrs((size_t)n_slots * BS_PKG_HEADER);
    CK(cudaMemcpy2DAsync(hdrs.data(), BS_PKG_HEADER, d_slots, slot_bytes, BS_PKG_HEADER, n_slots, cudaMemcpyDeviceToHost, stream));
    CK(cudaStreamSynchronize(stream));
    PkgPlan plan;
    if ((rc = pkg_plan(hdrs.data(), BS_PKG_HEADER, n_slots, slot_bytes, stream_id, &plan))) return rc;
    if (plan.hb > hdr_cap) return BS_ERR_CAPACITY;

    const unsigned char* slots = (const unsigned char*)d_slots;
    const uint64_t cut = plan_uniform_cap(plan, work_tile_bytes(o));
    if (cut != 0) {
        // the packages are the cut of one size limit whose tiles never straddle a package: the slot table is built on
        // the device, the header region gathered, and ONE launch unpacks every payload package wherever it lies
        const uint64_t count = plan.items.size();
        uint32_t* d_tab = nullptr;
        bool tab_owned = false;
        const uint64_t tab = align_up(count * sizeof(uint32_t), 256);
        if (w1 >= bs_workspace_bytes(out->n_tensors, out->n_blocks, plan.total) + tab) {  // bs_package_workspace_bytes has room
            const uint64_t w2 = (w1 - tab) & ~255ull;  // the v1 part shrinks, the table sits between it and the header scratch
            if (!ws_layout(d_ws, w2, out->n_blocks, &L)) return BS_ERR_CAPACITY;
            d_tab = (uint32_t*)((unsigned char*)d_ws + w2);
        } else {
            CK(cudaMallocAsync((void**)&d_tab, count * sizeof(uint32_t), stream));
            tab_owned = true;
        }
        pkg_index_kernel<<<(unsigned)((n_slots + 127) / 128), 128, 0, stream>>>(slots, slot_bytes, n_slots, stream_id, d_tab, count);
        CK(cudaGetLastError());
        {
            const uint64_t units = plan.hb / 16;
            unsigned grid = (unsigned)std::min<uint64_t>((units + 255) / 256, (uint64_t)sms * 8);
            pkg_gather_header_kernel<<<grid ? grid : 1, 256, 0, stream>>>(slots, slot_bytes, d_tab, cut, plan.hb, d_header);
            CK(cudaGetLastError());
        }
        if ((rc = run_deserialize_scan(d_header, nullptr, plan.total, out, d_pool, pool_bytes,
                                       flags | (o.variant != BS_VARIANT_TMA ? kFlagNoAlign8 : 0u), L, d_result, sms, stream))) return rc;
        CK(launch_pkg_check(L, d_slots, slot_bytes, n_slots, stream_id, d_result, stream));
        if ((rc = run_unpack_range(out, L, d_header, d_header, 0, 0, flags, o, sms, stream))) return rc;  // descriptor rebuild
        PkgMap pm;
        pm.cap = cut; pm.slot_bytes = slot_bytes; pm.base = const_cast<unsigned char*>(slots); pm.slot_of = d_tab; pm.k_base = 0;
        if ((rc = run_unpack_packages(out, L, pm, plan.hb, flags | kFlagCheckPad, o, sms, stream))) return rc;
        if (d_result != nullptr)
            CK(cudaMemcpyAsync(&d_result->status, &L.head->status, sizeof(int32_t), cudaMemcpyDeviceToDevice, stream));
        if (tab_owned) CK(cudaFreeAsync(d_tab, stream));
        return BS_OK;
    }
    for (uint32_t k = 0; k < plan.n_header; ++k) {  // the header region, stored continuously (L126)
        const PkgItem& it = plan.items[k];
        CK(cudaMemcpyAsync(d_header + it.lo, slots + it.slot * slot_bytes + BS_PKG_HEADER, it.nbytes, cudaMemcpyDeviceToDevice, stream));
    }
    if ((rc = run_deserialize_scan(d_header, nullptr, plan.total, out, d_pool, pool_bytes,
                                       flags | (o.variant != BS_VARIANT_TMA ? kFlagNoAlign8 : 0u), L, d_result, sms, stream))) return rc;
    CK(launch_pkg_check(L, d_slots, slot_bytes, n_slots, stream_id, d_result, stream));
    if ((rc = run_unpack_range(out, L, d_header, d_header, 0, 0, flags, o, sms, stream))) return rc;  // descriptor rebuild
    std::vector<PkgItem> by_slot(plan.items.begin() + plan.n_header, plan.items.end());
    std::sort(by_slot.begin(), by_slot.end(), [](const PkgItem& a, const PkgItem& b) { return a.slot < b.slot; });
    for (const PkgItem& it : by_slot) {  // every payload package on its own, in the order the slots lie
        if ((rc = run_unpack_range(out, L, slots + it.slot * slot_bytes + BS_PKG_HEADER, nullptr, it.lo, it.lo + it.nbytes,
                                   flags | kFlagCheckPad, o, sms, stream)))
            return rc;
    }
    if (d_result != nullptr)  // the pad check of the unpack kernels can still flip the status
        CK(cudaMemcpyAsync(&d_result->status, &L.head->status, sizeof(int32_t), cudaMemcpyDeviceToDevice, stream));
    return BS_OK;
}

// ---- layered sets: packages of a wire-format-v2 stream ------------------------------------------------------------------
// The package kernels only look at the flat block table blk[] and the sizes in WsHead, which the layered plan builds exactly
// as the v1 scan does, so they are shared; only the plan and the header generator / parser behind the move kernels differ.
uint64_t bs_layered_package_workspace_bytes(uint32_t n_structs, uint32_t n_struct_blocks, uint32_t n_layers, uint64_t n_addr,
                                            uint64_t stream_capacity)
{
    return bs_layered_workspace_bytes(n_structs, n_struct_blocks, n_layers, n_addr, stream_capacity) + 256 +
           align_up(bs_layered_header_bytes(n_structs, n_layers, n_struct_blocks), 256);
}

int bs_layered_package_emit(const bs_layered_desc* set, uint64_t total_bytes, uint64_t cap, uint64_t stream_id, void* d_slots,
                            uint64_t slot_bytes, uint64_t n_slots, const uint32_t* h_slot_of, void* d_ws, uint64_t ws_bytes,
                            bs_result* d_result, const bs_opts* opts, cudaStream_t stream)
{
    if (set == nullptr) return BS_ERR_ARG;
    { const int rc0 = check_layered_desc(set); if (rc0) return rc0; }
    if (d_slots == nullptr || !aligned16(d_slots) || cap == 0 || (cap & 15) || (slot_bytes & 15) ||
        slot_bytes < BS_PKG_HEADER + cap)
        return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    int rc;
    if ((rc = check_opts(o))) return rc;
    if (d_ws == nullptr || ((uintptr_t)d_ws & 255)) return BS_ERR_ARG;
    WsLayout L;
    if (!layered_ws(d_ws, ws_bytes, set->n_struct_blocks, set->n_layers, set->n_addr, &L)) return BS_ERR_CAPACITY;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    const uint64_t hb = bs_layered_header_bytes(set->n_structs, set->n_layers, set->n_struct_blocks);
    if (total_bytes == 0) {
        uint64_t hb2 = 0;
        if ((rc = bs_layered_serialized_size(set, d_ws, ws_bytes, &hb2, &total_bytes, stream))) return rc;
    }
    const uint64_t count = pkg_count(hb, total_bytes, cap);
    if (count == 0 || count >= (1ull << 32)) return BS_ERR_ARG;
    if (count > n_slots) return BS_ERR_CAPACITY;
    if (h_slot_of != nullptr) {
        std::vector<bool> used((size_t)n_slots, false);
        for (uint64_t k = 0; k < count; ++k) {
            if (h_slot_of[k] >= n_slots || used[h_slot_of[k]]) return BS_ERR_ARG;
            used[h_slot_of[k]] = true;
        }
    }
    if ((rc = run_layered_serialize_plan(set, d_ws, ws_bytes, UINT64_MAX, total_bytes, d_result, sms, stream))) return rc;
    if (cap % work_tile_bytes(o) == 0) {  // the fixed-launch-count path, as bs_package_emit
        uint32_t* d_tab = nullptr;
        if (h_slot_of != nullptr) {
            CK(cudaMallocAsync((void**)&d_tab, count * sizeof(uint32_t), stream));
            CK(cudaMemcpyAsync(d_tab, h_slot_of, count * sizeof(uint32_t), cudaMemcpyHostToDevice, stream));
        }
        CK(launch_pkg_headers(L, cap, stream_id, 0, count, count, d_slots, slot_bytes, d_tab, d_result, stream));
        PkgMap pm;
        pm.cap = cap; pm.slot_bytes = slot_bytes; pm.base = (unsigned char*)d_slots; pm.slot_of = d_tab; pm.k_base = 0;
        rc = run_layered_pack_range(set, d_ws, ws_bytes, nullptr, 0, UINT64_MAX, o, sms, stream, &pm);
        if (d_tab) CK(cudaFreeAsync(d_tab, stream));
        return rc;
    }
    for (uint64_t k = 0; k < count; ++k) {
        uint64_t lo = 0, hi = 0;
        pkg_range(hb, total_bytes, cap, k, &lo, &hi);
        unsigned char* slot = (unsigned char*)d_slots + (h_slot_of ? (uint64_t)h_slot_of[k] : k) * slot_bytes;
        CK(launch_pkg_header(L, cap, stream_id, k, count, slot, d_result, stream));
        if ((rc = run_layered_pack_range(set, d_ws, ws_bytes, slot + BS_PKG_HEADER, lo, hi, o, sms, stream, nullptr))) return rc;
    }
    return BS_OK;
}

int bs_layered_package_unpack(const void* d_slots, uint64_t slot_bytes, uint64_t n_slots, uint64_t stream_id, bs_layered_desc* out,
                              void* d_pool, uint64_t pool_bytes, uint32_t flags, void* d_ws, uint64_t ws_bytes, bs_result* d_result,
                              const bs_opts* opts, cudaStream_t stream)
{
    if (out == nullptr) return BS_ERR_ARG;
    { const int rc0 = check_layered_desc(out); if (rc0) return rc0; }
    if (d_slots == nullptr || !aligned16(d_slots) || (slot_bytes & 15) || slot_bytes < BS_PKG_HEADER + 16 || n_slots == 0)
        return BS_ERR_ARG;
    if (flags != BS_LAYOUT_POOL && flags != BS_SCATTER_TO_ADDR) return BS_ERR_ARG;
    if (flags == BS_LAYOUT_POOL && pool_bytes && (d_pool == nullptr || ((uintptr_t)d_pool & 255))) return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    int rc;
    if ((rc = check_opts(o))) return rc;
    // workspace := layered workspace | room for the assembled header region
    const uint64_t hdr_cap = align_up(bs_layered_header_bytes(out->n_structs, out->n_layers, out->n_struct_blocks), 256);
    if (d_ws == nullptr || ((uintptr_t)d_ws & 255)) return BS_ERR_ARG;
    if (ws_bytes < hdr_cap) return BS_ERR_CAPACITY;
    const uint64_t w1 = (ws_bytes - hdr_cap) & ~255ull;
    WsLayout L;
    if (!layered_ws(d_ws, w1, out->n_struct_blocks, out->n_layers, out->n_addr, &L)) return BS_ERR_CAPACITY;
    unsigned char* d_header = (unsigned char*)d_ws + w1;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    std::vector<unsigned char> hdrs((size_t)n_slots * BS_PKG_HEADER);
    CK(cudaMemcpy2DAsync(hdrs.data(), BS_PKG_HEADER, d_slots, slot_bytes, BS_PKG_HEADER, n_slots, cudaMemcpyDeviceToHost, stream));
    CK(cudaStreamSynchronize(stream));
    PkgPlan plan;
    if ((rc = pkg_plan(hdrs.data(), BS_PKG_HEADER, n_slots, slot_bytes, stream_id, &plan))) return rc;
    if (plan.hb > hdr_cap) return BS_ERR_CAPACITY;
    const unsigned char* slots = (const unsigned char*)d_slots;
    for (uint32_t k = 0; k < plan.n_header; ++k) {  // the header region, stored continuously (L126)
        const PkgItem& it = plan.items[k];
        CK(cudaMemcpyAsync(d_header + it.lo, slots + it.slot * slot_bytes + BS_PKG_HEADER, it.nbytes, cudaMemcpyDeviceToDevice, stream));
    }
    if ((rc = run_layered_deserialize_plan(d_header, nullptr, plan.total, out, d_pool, pool_bytes, flags, d_ws, w1, d_result, sms, stream)))
        return rc;
    CK(launch_pkg_check(L, d_slots, slot_bytes, n_slots, stream_id, d_result, stream));
    if ((rc = run_layered_unpack_range(out, d_ws, w1, d_header, d_header, 0, 0, flags, o, sms, stream, nullptr))) return rc;  // rebuild
    const uint64_t cut = plan_uniform_cap(plan, work_tile_bytes(o));
    if (cut != 0) {  // one launch for every payload package, wherever it lies
        const uint64_t count = plan.items.size();
        uint32_t* d_tab = nullptr;
        CK(cudaMallocAsync((void**)&d_tab, count * sizeof(uint32_t), stream));
        pkg_index_kernel<<<(unsigned)((n_slots + 127) / 128), 128, 0, stream>>>(slots, slot_bytes, n_slots, stream_id, d_tab, count);
        CK(cudaGetLastError());
        PkgMap pm;
        pm.cap = cut; pm.slot_bytes = slot_bytes; pm.base = const_cast<unsigned char*>(slots); pm.slot_of = d_tab; pm.k_base = 0;
        rc = run_layered_unpack_range(out, d_ws, w1, nullptr, nullptr, 0, UINT64_MAX, flags | kFlagCheckPad, o, sms, stream, &pm);
        CK(cudaFreeAsync(d_tab, stream));
        if (rc) return rc;
    } else {
        std::vector<PkgItem> by_slot(plan.items.begin() + plan.n_header, plan.items.end());
        std::sort(by_slot.begin(), by_slot.end(), [](const PkgItem& a, const PkgItem& b) { return a.slot < b.slot; });
        for (const PkgItem& it : by_slot)
            if ((rc = run_layered_unpack_range(out, d_ws, w1, slots + it.slot * slot_bytes + BS_PKG_HEADER, nullptr, it.lo,
                                               it.lo + it.nbytes, flags | kFlagCheckPad, o, sms, stream, nullptr)))
                return rc;
    }
    if (d_result != nullptr)
        CK(cudaMemcpyAsync(&d_result->status, &L.head->status, sizeof(int32_t), cudaMemcpyDeviceToDevice, stream));
    return BS_OK;
}

}  // extern "C"
