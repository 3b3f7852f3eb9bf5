// bs_engine.cu — asynchronous offload / prefetch engine: steps S8, S9 of SURVEY §8(a).
//
// PAPER L89 (Fig 4(b)): "serialization of data in small segments based on the size of a preallocated buffer
// and saving each segment ... immediately"; L90/L132: "a single CPU thread takes care of saving the serialized
// data while the remaining CPU threads ... proceed with subsequent computational tasks"; L134: the load runs
// "in parallel of the renormalization step"; L138: "checkpoints to make sure that required data ... are already
// available".  On a B200 the "single thread" is a pair of high-priority side streams and the copy engine:
//     kernel stream : scan | pack(chunk 0) | pack(chunk 1) | ...          (waits for staging buffer k%S to drain)
//     copy   stream :        D2H(chunk 0)  | D2H(chunk 1)  | ...          (waits for pack(chunk k))
// with S = n_staging (2: double buffering) staging buffers of chunk_bytes (256 MiB).  The producer / consumer
// stream is never blocked on the host; the ticket's event is the checkpoint.  Device memory held by the engine
// is S*chunk_bytes + O(max_blocks) — the "small additional memory" of L89/L94, not the +30-50 % of L92/L166.
// Bound: the PCIe link (one direction per call); the pack / unpack kernels are ~50x faster than the DMA.
#include <new>
#include <string.h>


#include <algorithm>
#include <mutex>
#include <vector>

#include "bs_engine.cuh"

using namespace bs;


// Pinned result words of the tickets come from a process-wide slab: cudaHostAlloc / cudaFreeHost synchronise the
// device, and a ticket created while another lane's transfer is running must not wait for it.
namespace {
constexpr size_t kResultSlab = 1024;
std::mutex g_slab_mutex;
bs_result* g_slab = nullptr;
std::vector<bs_result*> g_slab_free;

cudaError_t result_slot_get(bs_result** out)
{
    std::lock_guard<std::mutex> lock(g_slab_mutex);
    if (g_slab == nullptr) {
        cudaError_t e = cudaHostAlloc((void**)&g_slab, kResultSlab * sizeof(bs_result), cudaHostAllocDefault);
        if (e != cudaSuccess) return e;
        for (size_t i = kResultSlab; i-- > 0;) g_slab_free.push_back(g_slab + i);
    }
    if (g_slab_free.empty()) return cudaHostAlloc((void**)out, sizeof(bs_result), cudaHostAllocDefault);  // > 1024 live tickets
    *out = g_slab_free.back();
    g_slab_free.pop_back();
    return cudaSuccess;
}

void result_slot_put(bs_result* r)
{
    std::lock_guard<std::mutex> lock(g_slab_mutex);
    if (g_slab != nullptr && r >= g_slab && r < g_slab + kResultSlab) g_slab_free.push_back(r);
    else cudaFreeHost(r);
}
}  // namespace

// The deferred outcome reaches the ticket's pinned result word by plain stores of a one-thread kernel (pinned host
// memory is device-addressable), not by a copy-engine transfer: a 64-byte cudaMemcpyAsync would queue behind the
// bulk DMA chunks of the OTHER lane that go in the same direction and stall this lane's kernel stream for milliseconds.
__global__ void post_result_kernel(bs_result* h_dst, const bs_result* d_src)
{
    const bs_result r = *d_src;
    volatile bs_result* o = h_dst;
    o->total_bytes = r.total_bytes; o->header_bytes = r.header_bytes; o->payload_bytes = r.payload_bytes;
    o->pool_bytes = r.pool_bytes; o->n_tensors = r.n_tensors; o->n_blocks = r.n_blocks;
    for (int i = 0; i < 5; ++i) o->reserved[i] = r.reserved[i];
    __threadfence_system();
    o->status = r.status;
    __threadfence_system();
}
__global__ void post_status_kernel(bs_result* h_dst, const int32_t* d_status)
{
    volatile bs_result* o = h_dst;
    o->status = *d_status;
    __threadfence_system();
}
static cudaError_t post_result(bs_result* h_dst, const bs_result* d_src, cudaStream_t stream)
{
    post_result_kernel<<<1, 1, 0, stream>>>(h_dst, d_src);
    return cudaGetLastError();
}
static cudaError_t post_status(bs_result* h_dst, const int32_t* d_status, cudaStream_t stream)
{
    post_status_kernel<<<1, 1, 0, stream>>>(h_dst, d_status);
    return cudaGetLastError();
}

static int ticket_create(bs_ticket** out)
{
    bs_ticket* t = new (std::nothrow) bs_ticket;
    if (!t) return BS_ERR_ARG;
    memset(t, 0, sizeof(*t));
    cudaError_t e;
    if ((e = cudaEventCreate(&t->t_begin)) != cudaSuccess || (e = cudaEventCreate(&t->dma_begin)) != cudaSuccess ||
        (e = cudaEventCreate(&t->dma_end)) != cudaSuccess || (e = cudaEventCreate(&t->done)) != cudaSuccess ||
        (e = result_slot_get(&t->h_result)) != cudaSuccess) {
        delete t;
        return cuda_fail(e);
    }
    memset(t->h_result, 0, sizeof(bs_result));
    t->h_result->status = BS_PENDING;
    *out = t;
    return BS_OK;
}

// A call that fails halfway (a CUDA error while enqueueing) must not leak its ticket, and must not free it under work that
// is already enqueued and will still write the ticket's result word: drain the engine's streams, then destroy.
struct TicketGuard {
    bs_engine* e;
    bs_ticket* t;
    ~TicketGuard()
    {
        if (t == nullptr) return;
        cudaStreamSynchronize(e->kstream);
        cudaStreamSynchronize(e->cstream);
        bs_ticket_destroy(t);
    }
    bs_ticket* release() { bs_ticket* r = t; t = nullptr; return r; }
};

// serialise engine calls: everything already enqueued on either side stream precedes the new call on both
static int engine_fence(bs_engine* e)
{
    CK(cudaEventRecord(e->ev_fence_k, e->kstream));
    CK(cudaEventRecord(e->ev_fence_c, e->cstream));
    CK(cudaStreamWaitEvent(e->cstream, e->ev_fence_k, 0));
    CK(cudaStreamWaitEvent(e->kstream, e->ev_fence_c, 0));
    return BS_OK;
}

extern "C" {

int bs_engine_create(bs_engine** out, const bs_engine_cfg* cfg)
{
    if (out == nullptr || cfg == nullptr) return BS_ERR_ARG;
    bs_engine* e = new (std::nothrow) bs_engine;
    if (!e) return BS_ERR_ARG;
    memset(e, 0, sizeof(*e));
    e->cfg = *cfg;
    if (e->cfg.chunk_bytes == 0) e->cfg.chunk_bytes = 256ull << 20;
    if (e->cfg.n_staging == 0) e->cfg.n_staging = 2;
    if (e->cfg.chunk_bytes % 65536 != 0 || e->cfg.n_staging > kMaxStaging || e->cfg.n_staging < 1) { delete e; return BS_ERR_ARG; }
    resolve_opts(&cfg->opts, &e->opts);
    int rc = check_opts(e->opts);  // a shape the kernels cannot run must not wait for the first call to show
    if (rc == BS_OK) rc = device_sm_count(&e->sms);
    if (rc) { delete e; return rc; }
    int lo_prio = 0, hi_prio = 0;
    cudaError_t ce = cudaDeviceGetStreamPriorityRange(&lo_prio, &hi_prio);
    if (ce == cudaSuccess) ce = cudaStreamCreateWithPriority(&e->kstream, cudaStreamNonBlocking, hi_prio);
    if (ce == cudaSuccess) ce = cudaStreamCreateWithPriority(&e->cstream, cudaStreamNonBlocking, hi_prio);
    for (uint32_t b = 0; ce == cudaSuccess && b < e->cfg.n_staging; ++b) {
        ce = cudaMalloc((void**)&e->staging[b], e->cfg.chunk_bytes);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e->ev_k[b], cudaEventDisableTiming);
        if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e->ev_c[b], cudaEventDisableTiming);
    }
    if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e->ev_fence_k, cudaEventDisableTiming);
    if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e->ev_fence_c, cudaEventDisableTiming);
    if (ce == cudaSuccess) ce = cudaEventCreateWithFlags(&e->ev_dep, cudaEventDisableTiming);
    e->ws_bytes = bs_workspace_bytes(e->cfg.max_tensors, e->cfg.max_blocks, e->cfg.max_stream_bytes);
    e->header_cap = header_bytes_of(e->cfg.max_tensors, e->cfg.max_blocks, BS_RANK4);  // room for 64-byte block records (wire format v3)
    {   // layered sets (wire format v2): C, T <= max_tensors; Bs, B <= max_blocks
        const uint64_t w2 = bs_layered_workspace_bytes(e->cfg.max_tensors, e->cfg.max_blocks, e->cfg.max_tensors,
                                                       e->cfg.max_blocks, e->cfg.max_stream_bytes);
        const uint64_t h2 = bs_layered_header_bytes(e->cfg.max_tensors, e->cfg.max_tensors, e->cfg.max_blocks);
        if (w2 > e->ws_bytes) e->ws_bytes = w2;
        if (h2 > e->header_cap) e->header_cap = h2;
    }
    if (ce == cudaSuccess) ce = cudaMalloc(&e->ws, e->ws_bytes);
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&e->header_buf, e->header_cap);
    if (ce == cudaSuccess) ce = cudaMalloc((void**)&e->d_result, sizeof(bs_result));
    if (ce != cudaSuccess) {
        bs_engine_destroy(e);
        return cuda_fail(ce);
    }
    *out = e;
    return BS_OK;
}

int bs_engine_destroy(bs_engine* e)
{
    if (e == nullptr) return BS_ERR_ARG;
    if (e->kstream) cudaStreamSynchronize(e->kstream);
    if (e->cstream) cudaStreamSynchronize(e->cstream);
    for (uint32_t b = 0; b < kMaxStaging; ++b) {
        if (e->staging[b]) cudaFree(e->staging[b]);
        if (e->ev_k[b]) cudaEventDestroy(e->ev_k[b]);
        if (e->ev_c[b]) cudaEventDestroy(e->ev_c[b]);
    }
    if (e->ev_fence_k) cudaEventDestroy(e->ev_fence_k);
    if (e->ev_fence_c) cudaEventDestroy(e->ev_fence_c);
    if (e->ev_dep) cudaEventDestroy(e->ev_dep);
    if (e->ws) cudaFree(e->ws);
    if (e->header_buf) cudaFree(e->header_buf);
    if (e->pkg_tab) cudaFree(e->pkg_tab);
    if (e->d_result) cudaFree(e->d_result);
    if (e->kstream) cudaStreamDestroy(e->kstream);
    if (e->cstream) cudaStreamDestroy(e->cstream);
    delete e;
    return BS_OK;
}

}  // extern "C"

// one body for both wire formats: exactly one of set / lset is non-null
int bs_engine_offload_impl(bs_engine* e, const bs_set_desc* set, const bs_layered_desc* lset, uint64_t total_bytes,
                        void* h_pinned, uint64_t h_capacity, cudaStream_t producer, bs_ticket** ticket)
{
    if (e == nullptr || (set == nullptr && lset == nullptr) || h_pinned == nullptr || ticket == nullptr) return BS_ERR_ARG;
    WsLayout L;
    int rc = set ? check_set(set) : check_layered_desc(lset);  // as the direct calls: a descriptor no loader accepts is refused here
    if (rc) return rc;
    if (set && (set->dtype & BS_ALIGN8) && e->opts.variant != BS_VARIANT_TMA) return BS_ERR_UNSUPPORTED;
    if (set) {
        if (set->n_blocks > e->cfg.max_blocks || set->n_tensors > e->cfg.max_tensors) return BS_ERR_CAPACITY;
        if (!ws_layout(e->ws, e->ws_bytes, set->n_blocks, &L)) return BS_ERR_CAPACITY;
    } else {
        if (lset->n_structs > e->cfg.max_tensors || lset->n_layers > e->cfg.max_tensors ||
            lset->n_struct_blocks > e->cfg.max_blocks || lset->n_addr > e->cfg.max_blocks)
            return BS_ERR_CAPACITY;
    }
    if (total_bytes == 0) {  // size prediction on the producer stream (synchronises it)
        uint64_t hb = 0;
        // the workspace may still be in use by the kernels of an earlier call: the query runs behind them
        CK(cudaEventRecord(e->ev_fence_k, e->kstream));
        CK(cudaStreamWaitEvent(producer, e->ev_fence_k, 0));
        rc = set ? bs_serialized_size(set, e->ws, e->ws_bytes, &hb, &total_bytes, producer)
                 : bs_layered_serialized_size(lset, e->ws, e->ws_bytes, &hb, &total_bytes, producer);
        if (rc) return rc;
    }
    if (total_bytes > h_capacity || total_bytes > e->cfg.max_stream_bytes) return BS_ERR_CAPACITY;
    if (total_bytes & 7) return BS_ERR_ARG;  // (a multiple of 16, or of 8 for an align-8 stream)
    bs_ticket* t = nullptr;
    if ((rc = ticket_create(&t))) return rc;
    TicketGuard guard{e, t};
    const uint64_t C = e->cfg.chunk_bytes;
    const uint32_t S = e->cfg.n_staging;
    t->bytes = total_bytes;
    t->n_chunks = (uint32_t)((total_bytes + C - 1) / C);

    if ((rc = engine_fence(e))) return rc;
    CK(cudaEventRecord(e->ev_dep, producer));          // the data is ready after everything enqueued so far
    CK(cudaStreamWaitEvent(e->kstream, e->ev_dep, 0));
    CK(cudaEventRecord(t->t_begin, e->kstream));
    rc = set ? run_serialize_scan(set, L, UINT64_MAX, total_bytes, e->d_result, e->sms, e->kstream)
             : run_layered_serialize_plan(lset, e->ws, e->ws_bytes, UINT64_MAX, total_bytes, e->d_result, e->sms, e->kstream);
    if (rc) return rc;
    CK(post_result(t->h_result, e->d_result, e->kstream));
    for (uint32_t k = 0; k < t->n_chunks; ++k) {
        const uint32_t b = k % S;
        const uint64_t lo = (uint64_t)k * C, hi = (lo + C < total_bytes) ? lo + C : total_bytes;
        if (k >= S) CK(cudaStreamWaitEvent(e->kstream, e->ev_c[b], 0));  // staging[b] drained by DMA k-S
        rc = set ? run_pack_range(set, L, e->staging[b], lo, hi, e->opts, e->sms, e->kstream, kFlagPoisonOnError)
                 : run_layered_pack_range(lset, e->ws, e->ws_bytes, e->staging[b], lo, hi, e->opts, e->sms, e->kstream, nullptr,
                                          kFlagPoisonOnError);
        if (rc) return rc;
        CK(cudaEventRecord(e->ev_k[b], e->kstream));
        CK(cudaStreamWaitEvent(e->cstream, e->ev_k[b], 0));
        if (k == 0) CK(cudaEventRecord(t->dma_begin, e->cstream));
        CK(cudaMemcpyAsync((unsigned char*)h_pinned + lo, e->staging[b], hi - lo, cudaMemcpyDeviceToHost, e->cstream));
        CK(cudaEventRecord(e->ev_c[b], e->cstream));
    }
    if (t->n_chunks == 0) CK(cudaEventRecord(t->dma_begin, e->cstream));
    CK(cudaEventRecord(t->dma_end, e->cstream));
    CK(cudaEventRecord(t->done, e->cstream));  // after the last DMA, which is after every kernel-stream step
    *ticket = guard.release();
    return BS_OK;
}

// `known` (v1 only): the counts of a stream that is still on its way to h_pinned (queue: a load submitted behind the save
// of the same key); otherwise the fixed header is read from host RAM.  Either way the device validates what arrives.
int bs_engine_prefetch_impl(bs_engine* e, const void* h_pinned, uint64_t nbytes, bs_set_desc* out, bs_layered_desc* lout,
                         void* d_pool, uint64_t pool_bytes, uint32_t flags, cudaStream_t consumer, bs_ticket** ticket,
                         const bs_stream_info_t* known, const bs_layered_stream_info_t* known_l)
{
    if (e == nullptr || h_pinned == nullptr || (out == nullptr && lout == nullptr) || ticket == nullptr) return BS_ERR_ARG;
    if (flags != BS_LAYOUT_POOL && flags != BS_SCATTER_TO_ADDR) return BS_ERR_ARG;
    int rc = out ? check_set(out) : check_layered_desc(lout);
    if (rc) return rc;
    if (flags == BS_LAYOUT_POOL && pool_bytes && (d_pool == nullptr || ((uintptr_t)d_pool & 255))) return BS_ERR_ARG;
    if (nbytes < kFixedHeader) return BS_ERR_CORRUPT;
    bs_stream_info_t info;
    WsLayout L;
    if (out) {
        if (known) info = *known;
        else if ((rc = bs_stream_info(h_pinned, &info))) return rc;  // the stream is in host RAM: its counts cost nothing to read
        if (info.total_bytes != nbytes) return BS_ERR_CORRUPT;
        if ((info.max_rank == 4) != ((out->dtype & BS_RANK4) != 0)) return BS_ERR_ARG;  // the out arrays have the other shape
        if (info.n_blocks > e->cfg.max_blocks || info.n_tensors > e->cfg.max_tensors || info.header_bytes > e->header_cap ||
            nbytes > e->cfg.max_stream_bytes)
            return BS_ERR_CAPACITY;
        if (info.n_blocks > out->n_blocks || info.n_tensors > out->n_tensors) return BS_ERR_CAPACITY;
        if (!ws_layout(e->ws, e->ws_bytes, out->n_blocks, &L)) return BS_ERR_CAPACITY;
    } else {
        bs_layered_stream_info_t li;
        if (known_l) li = *known_l;
        else if ((rc = bs_layered_stream_info(h_pinned, &li))) return rc;
        if (li.total_bytes != nbytes) return BS_ERR_CORRUPT;
        if (li.n_structs > e->cfg.max_tensors || li.n_layers > e->cfg.max_tensors || li.n_struct_blocks > e->cfg.max_blocks ||
            lout->n_addr > e->cfg.max_blocks || li.header_bytes > e->header_cap || nbytes > e->cfg.max_stream_bytes)
            return BS_ERR_CAPACITY;
        if (li.n_structs > lout->n_structs || li.n_layers > lout->n_layers || li.n_struct_blocks > lout->n_struct_blocks)
            return BS_ERR_CAPACITY;
        if (bs_layered_workspace_bytes(lout->n_structs, lout->n_struct_blocks, lout->n_layers, lout->n_addr, nbytes) > e->ws_bytes)
            return BS_ERR_CAPACITY;
        info.header_bytes = li.header_bytes;
        info.payload_bytes = li.payload_bytes;
    }
    bs_ticket* t = nullptr;
    if ((rc = ticket_create(&t))) return rc;
    TicketGuard guard{e, t};
    t->is_prefetch = true;
    const uint64_t C = e->cfg.chunk_bytes;
    const uint32_t S = e->cfg.n_staging;
    const uint64_t hb = info.header_bytes;
    t->bytes = nbytes;
    t->n_chunks = (uint32_t)((info.payload_bytes + C - 1) / C);

    if ((rc = engine_fence(e))) return rc;
    CK(cudaEventRecord(e->ev_dep, consumer));  // destinations may still be in use by work already enqueued
    CK(cudaStreamWaitEvent(e->cstream, e->ev_dep, 0));
    CK(cudaStreamWaitEvent(e->kstream, e->ev_dep, 0));
    CK(cudaEventRecord(t->t_begin, e->cstream));
    CK(cudaEventRecord(t->dma_begin, e->cstream));
    // header first: validate + offset table + descriptor rebuild, while the payload chunks stream in
    CK(cudaMemcpyAsync(e->header_buf, h_pinned, hb, cudaMemcpyHostToDevice, e->cstream));
    CK(cudaEventRecord(e->ev_fence_c, e->cstream));
    CK(cudaStreamWaitEvent(e->kstream, e->ev_fence_c, 0));
    rc = out ? run_deserialize_scan(e->header_buf, nullptr, nbytes, out, d_pool, pool_bytes,
                                    flags | (e->opts.variant != BS_VARIANT_TMA ? kFlagNoAlign8 : 0u), L, e->d_result, e->sms, e->kstream)
             : run_layered_deserialize_plan(e->header_buf, nullptr, nbytes, lout, d_pool, pool_bytes, flags, e->ws, e->ws_bytes,
                                            e->d_result, e->sms, e->kstream);
    if (rc) return rc;
    CK(post_result(t->h_result, e->d_result, e->kstream));
    rc = out ? run_unpack_range(out, L, e->header_buf, e->header_buf, 0, 0, flags, e->opts, e->sms, e->kstream)
             : run_layered_unpack_range(lout, e->ws, e->ws_bytes, e->header_buf, e->header_buf, 0, 0, flags, e->opts, e->sms,
                                        e->kstream);
    if (rc) return rc;
    for (uint32_t k = 0; k < t->n_chunks; ++k) {
        const uint32_t b = k % S;
        const uint64_t lo = hb + (uint64_t)k * C, hi = (lo + C < nbytes) ? lo + C : nbytes;
        if (k >= S) CK(cudaStreamWaitEvent(e->cstream, e->ev_k[b], 0));  // staging[b] consumed by unpack k-S
        CK(cudaMemcpyAsync(e->staging[b], (const unsigned char*)h_pinned + lo, hi - lo, cudaMemcpyHostToDevice, e->cstream));
        CK(cudaEventRecord(e->ev_c[b], e->cstream));
        CK(cudaStreamWaitEvent(e->kstream, e->ev_c[b], 0));
        rc = out ? run_unpack_range(out, L, e->staging[b], nullptr, lo, hi, flags | kFlagCheckPad, e->opts, e->sms, e->kstream)
                 : run_layered_unpack_range(lout, e->ws, e->ws_bytes, e->staging[b], nullptr, lo, hi, flags | kFlagCheckPad,
                                            e->opts, e->sms, e->kstream);
        if (rc) return rc;
        CK(cudaEventRecord(e->ev_k[b], e->kstream));
    }
    CK(cudaEventRecord(t->dma_end, e->cstream));
    // final status (the pad check of the unpack kernels can still flip it) and the checkpoint event
    CK(post_status(t->h_result, &((WsHead*)e->ws)->status, e->kstream));
    CK(cudaEventRecord(t->done, e->kstream));
    CK(cudaStreamWaitEvent(consumer, t->done, 0));
    *ticket = guard.release();
    return BS_OK;
}

extern "C" {

int bs_offload_async(bs_engine* e, const bs_set_desc* set, uint64_t total_bytes, void* h_pinned, uint64_t h_capacity,
                     cudaStream_t producer, bs_ticket** ticket)
{
    if (set == nullptr) return BS_ERR_ARG;
    return bs_engine_offload_impl(e, set, nullptr, total_bytes, h_pinned, h_capacity, producer, ticket);
}

int bs_offload_layered_async(bs_engine* e, const bs_layered_desc* set, uint64_t total_bytes, void* h_pinned,
                             uint64_t h_capacity, cudaStream_t producer, bs_ticket** ticket)
{
    if (set == nullptr) return BS_ERR_ARG;
    return bs_engine_offload_impl(e, nullptr, set, total_bytes, h_pinned, h_capacity, producer, ticket);
}

int bs_prefetch_async(bs_engine* e, const void* h_pinned, uint64_t nbytes, bs_set_desc* out, void* d_pool,
                      uint64_t pool_bytes, uint32_t flags, cudaStream_t consumer, bs_ticket** ticket)
{
    if (out == nullptr) return BS_ERR_ARG;
    return bs_engine_prefetch_impl(e, h_pinned, nbytes, out, nullptr, d_pool, pool_bytes, flags, consumer, ticket);
}

int bs_prefetch_layered_async(bs_engine* e, const void* h_pinned, uint64_t nbytes, bs_layered_desc* out, void* d_pool,
                              uint64_t pool_bytes, uint32_t flags, cudaStream_t consumer, bs_ticket** ticket)
{
    if (out == nullptr) return BS_ERR_ARG;
    return bs_engine_prefetch_impl(e, h_pinned, nbytes, nullptr, out, d_pool, pool_bytes, flags, consumer, ticket);
}

// ---- self-contained packages through the engine (bs.h "packages") ------------------------------------
// one body for both wire formats: exactly one of set / lset is non-null
static int offload_packages_impl(bs_engine* e, const bs_set_desc* set, const bs_layered_desc* lset, uint64_t total_bytes, uint64_t cap,
                                 uint64_t stream_id, void* h_slots, uint64_t slot_bytes, uint64_t n_slots, const uint32_t* h_slot_of,
                                 cudaStream_t producer, bs_ticket** ticket)
{
    if (e == nullptr || (set == nullptr && lset == nullptr) || h_slots == nullptr || ticket == nullptr) return BS_ERR_ARG;
    if (cap == 0 || (cap & 15) || (slot_bytes & 15) || slot_bytes < BS_PKG_HEADER + cap) return BS_ERR_ARG;
    if (cap + BS_PKG_HEADER > e->cfg.chunk_bytes) return BS_ERR_CAPACITY;
    WsLayout L;
    uint64_t hb;
    int rc = set ? check_set(set) : check_layered_desc(lset);
    if (rc) return rc;
    if (set && (set->dtype & BS_ALIGN8) && e->opts.variant != BS_VARIANT_TMA) return BS_ERR_UNSUPPORTED;
    if (set) {
        if (set->n_blocks > e->cfg.max_blocks || set->n_tensors > e->cfg.max_tensors) return BS_ERR_CAPACITY;
        if (!ws_layout(e->ws, e->ws_bytes, set->n_blocks, &L)) return BS_ERR_CAPACITY;
        hb = header_bytes_of(set->n_tensors, set->n_blocks, set->dtype);
    } else {
        if (lset->n_structs > e->cfg.max_tensors || lset->n_layers > e->cfg.max_tensors ||
            lset->n_struct_blocks > e->cfg.max_blocks || lset->n_addr > e->cfg.max_blocks)
            return BS_ERR_CAPACITY;
        if (!layered_ws(e->ws, e->ws_bytes, lset->n_struct_blocks, lset->n_layers, lset->n_addr, &L)) return BS_ERR_CAPACITY;
        hb = bs_layered_header_bytes(lset->n_structs, lset->n_layers, lset->n_struct_blocks);
    }
    if (total_bytes == 0) {
        CK(cudaEventRecord(e->ev_fence_k, e->kstream));  // the workspace may still be in use by an earlier call
        CK(cudaStreamWaitEvent(producer, e->ev_fence_k, 0));
        rc = set ? bs_serialized_size(set, e->ws, e->ws_bytes, &hb, &total_bytes, producer)
                 : bs_layered_serialized_size(lset, e->ws, e->ws_bytes, &hb, &total_bytes, producer);
        if (rc) return rc;
    }
    if (total_bytes > e->cfg.max_stream_bytes) return BS_ERR_CAPACITY;
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
    bs_ticket* t = nullptr;
    if ((rc = ticket_create(&t))) return rc;
    TicketGuard guard{e, t};
    const uint32_t S = e->cfg.n_staging;
    t->bytes = total_bytes + count * BS_PKG_HEADER;
    t->n_chunks = (uint32_t)count;

    if ((rc = engine_fence(e))) return rc;
    CK(cudaEventRecord(e->ev_dep, producer));
    CK(cudaStreamWaitEvent(e->kstream, e->ev_dep, 0));
    CK(cudaEventRecord(t->t_begin, e->kstream));
    rc = set ? run_serialize_scan(set, L, UINT64_MAX, total_bytes, e->d_result, e->sms, e->kstream)
             : run_layered_serialize_plan(lset, e->ws, e->ws_bytes, UINT64_MAX, total_bytes, e->d_result, e->sms, e->kstream);
    if (rc) return rc;
    // A staging buffer takes a BATCH of packages laid out as slots, and the batch leaves in ONE DMA, when the slots are
    // exactly header + limit long and the batch's host slots are consecutive; a short package (the last one of the header
    // region / of the payload) ends its batch, so no byte behind a short package is written on the host.
    const bool can_batch = slot_bytes == BS_PKG_HEADER + cap;
    // no work tile straddles a package when the limit is a multiple of the tile (bs_pkg.cu): then the move kernel takes a
    // package map and a whole batch costs two launches
    const bool one_launch = can_batch && cap % (e->opts.tile_bytes ? e->opts.tile_bytes : kGranule) == 0;
    const uint64_t per_buf = can_batch ? std::max<uint64_t>(1, e->cfg.chunk_bytes / slot_bytes) : 1;
    auto slot_of = [&](uint64_t k) { return h_slot_of ? (uint64_t)h_slot_of[k] : k; };
    uint64_t batch = 0;
    for (uint64_t k = 0; k < count; ++batch) {
        const uint32_t b = (uint32_t)(batch % S);
        if (batch >= S) CK(cudaStreamWaitEvent(e->kstream, e->ev_c[b], 0));  // staging[b] drained by the DMA of batch - S
        uint64_t m = 0, last_bytes = 0, lo0 = 0, hi1 = 0;
        const uint64_t k0 = k;
        for (; k < count && m < per_buf; ++k, ++m) {
            if (m > 0 && slot_of(k) != slot_of(k - 1) + 1) break;  // the host slots of a batch are consecutive
            uint64_t lo = 0, hi = 0;
            pkg_range(hb, total_bytes, cap, k, &lo, &hi);
            if (m == 0) lo0 = lo;
            hi1 = hi;
            if (!one_launch) {
                unsigned char* dst = e->staging[b] + m * slot_bytes;
                CK(launch_pkg_header(L, cap, stream_id, k, count, dst, e->d_result, e->kstream, true));
                rc = set ? run_pack_range(set, L, dst + BS_PKG_HEADER, lo, hi, e->opts, e->sms, e->kstream)
                         : run_layered_pack_range(lset, e->ws, e->ws_bytes, dst + BS_PKG_HEADER, lo, hi, e->opts, e->sms, e->kstream);
                if (rc) return rc;
            }
            last_bytes = hi - lo;
            if (last_bytes != cap) { ++k; ++m; break; }  // a short package ends its batch
        }
        if (one_launch) {  // the batch's headers in one launch, its stream range [lo0, hi1) in one more
            CK(launch_pkg_headers(L, cap, stream_id, k0, m, count, e->staging[b], slot_bytes, nullptr, e->d_result, e->kstream, true));
            PkgMap pm;
            pm.cap = cap; pm.slot_bytes = slot_bytes; pm.base = e->staging[b]; pm.slot_of = nullptr; pm.k_base = k0;
            rc = set ? run_pack_packages_range(set, L, pm, lo0, hi1, e->opts, e->sms, e->kstream)
                     : run_layered_pack_range(lset, e->ws, e->ws_bytes, nullptr, lo0, hi1, e->opts, e->sms, e->kstream, &pm);
            if (rc) return rc;
        }
        if (k0 == 0) CK(post_result(t->h_result, e->d_result, e->kstream));
        CK(cudaEventRecord(e->ev_k[b], e->kstream));
        CK(cudaStreamWaitEvent(e->cstream, e->ev_k[b], 0));
        if (k0 == 0) CK(cudaEventRecord(t->dma_begin, e->cstream));
        CK(cudaMemcpyAsync((unsigned char*)h_slots + slot_of(k0) * slot_bytes, e->staging[b],
                           (m - 1) * slot_bytes + BS_PKG_HEADER + last_bytes, cudaMemcpyDeviceToHost, e->cstream));
        CK(cudaEventRecord(e->ev_c[b], e->cstream));
    }
    CK(cudaEventRecord(t->dma_end, e->cstream));
    CK(cudaEventRecord(t->done, e->cstream));
    *ticket = guard.release();
    return BS_OK;
}

static int prefetch_packages_impl(bs_engine* e, const void* h_slots, uint64_t slot_bytes, uint64_t n_slots, uint64_t stream_id,
                                  bs_set_desc* out, bs_layered_desc* lout, void* d_pool, uint64_t pool_bytes, uint32_t flags,
                                  cudaStream_t consumer, bs_ticket** ticket)
{
    if (e == nullptr || h_slots == nullptr || (out == nullptr && lout == nullptr) || ticket == nullptr || n_slots == 0) return BS_ERR_ARG;
    if ((slot_bytes & 15) || slot_bytes < BS_PKG_HEADER + 16) return BS_ERR_ARG;
    if (flags != BS_LAYOUT_POOL && flags != BS_SCATTER_TO_ADDR) return BS_ERR_ARG;
    int rc = out ? check_set(out) : check_layered_desc(lout);
    if (rc) return rc;
    if (flags == BS_LAYOUT_POOL && pool_bytes && (d_pool == nullptr || ((uintptr_t)d_pool & 255))) return BS_ERR_ARG;
    const unsigned char* slots = (const unsigned char*)h_slots;
    PkgPlan plan;  // the packages are in host RAM: their headers cost nothing to read
    if ((rc = pkg_plan(slots, slot_bytes, n_slots, slot_bytes, stream_id, &plan))) return rc;
    if (plan.hb > e->header_cap || plan.total > e->cfg.max_stream_bytes) return BS_ERR_CAPACITY;
    WsLayout L;
    if (out) {
        if (out->n_blocks > e->cfg.max_blocks || out->n_tensors > e->cfg.max_tensors) return BS_ERR_CAPACITY;
        if (!ws_layout(e->ws, e->ws_bytes, out->n_blocks, &L)) return BS_ERR_CAPACITY;
    } else {
        if (lout->n_structs > e->cfg.max_tensors || lout->n_layers > e->cfg.max_tensors ||
            lout->n_struct_blocks > e->cfg.max_blocks || lout->n_addr > e->cfg.max_blocks)
            return BS_ERR_CAPACITY;
        if (!layered_ws(e->ws, e->ws_bytes, lout->n_struct_blocks, lout->n_layers, lout->n_addr, &L)) return BS_ERR_CAPACITY;
    }
    for (const PkgItem& it : plan.items)
        if (it.nbytes > e->cfg.chunk_bytes) return BS_ERR_CAPACITY;
    if (n_slots > e->pkg_tab_slots) {  // a call-time allocation, only when a call brings more slots than any before
        CK(cudaStreamSynchronize(e->kstream));
        if (e->pkg_tab) cudaFree(e->pkg_tab);
        e->pkg_tab = nullptr;
        e->pkg_tab_slots = 0;
        CK(cudaMalloc((void**)&e->pkg_tab, n_slots * BS_PKG_HEADER));
        e->pkg_tab_slots = n_slots;
    }
    bs_ticket* t = nullptr;
    if ((rc = ticket_create(&t))) return rc;
    TicketGuard guard{e, t};
    t->is_prefetch = true;
    const uint32_t S = e->cfg.n_staging;
    t->bytes = plan.total + plan.items.size() * BS_PKG_HEADER;
    t->n_chunks = (uint32_t)plan.items.size();

    if ((rc = engine_fence(e))) return rc;
    CK(cudaEventRecord(e->ev_dep, consumer));
    CK(cudaStreamWaitEvent(e->cstream, e->ev_dep, 0));
    CK(cudaStreamWaitEvent(e->kstream, e->ev_dep, 0));
    CK(cudaEventRecord(t->t_begin, e->cstream));
    CK(cudaEventRecord(t->dma_begin, e->cstream));
    // the package headers and the header region first: validate + offset table + descriptor rebuild
    CK(cudaMemcpy2DAsync(e->pkg_tab, BS_PKG_HEADER, slots, slot_bytes, BS_PKG_HEADER, n_slots, cudaMemcpyHostToDevice, e->cstream));
    for (uint32_t k = 0; k < plan.n_header; ++k) {
        const PkgItem& it = plan.items[k];
        CK(cudaMemcpyAsync(e->header_buf + it.lo, slots + it.slot * slot_bytes + BS_PKG_HEADER, it.nbytes, cudaMemcpyHostToDevice,
                           e->cstream));
    }
    CK(cudaEventRecord(e->ev_fence_c, e->cstream));
    CK(cudaStreamWaitEvent(e->kstream, e->ev_fence_c, 0));
    rc = out ? run_deserialize_scan(e->header_buf, nullptr, plan.total, out, d_pool, pool_bytes,
                                    flags | (e->opts.variant != BS_VARIANT_TMA ? kFlagNoAlign8 : 0u), L, e->d_result, e->sms, e->kstream)
             : run_layered_deserialize_plan(e->header_buf, nullptr, plan.total, lout, d_pool, pool_bytes, flags, e->ws, e->ws_bytes,
                                            e->d_result, e->sms, e->kstream);
    if (rc) return rc;
    CK(launch_pkg_check(L, e->pkg_tab, BS_PKG_HEADER, n_slots, stream_id, e->d_result, e->kstream));
    CK(post_result(t->h_result, e->d_result, e->kstream));
    rc = out ? run_unpack_range(out, L, e->header_buf, e->header_buf, 0, 0, flags, e->opts, e->sms, e->kstream)
             : run_layered_unpack_range(lout, e->ws, e->ws_bytes, e->header_buf, e->header_buf, 0, 0, flags, e->opts, e->sms, e->kstream);
    if (rc) return rc;
    std::vector<PkgItem> by_slot(plan.items.begin() + plan.n_header, plan.items.end());
    std::sort(by_slot.begin(), by_slot.end(), [](const PkgItem& a, const PkgItem& b) { return a.slot < b.slot; });
    // arrival order: each payload package is unpacked on its own; runs of consecutive slots that fit a staging buffer
    // come over in ONE DMA (what lies behind a short package inside the run is read and ignored)
    const uint64_t per_buf = std::max<uint64_t>(1, e->cfg.chunk_bytes / slot_bytes);
    const uint64_t cut = plan_uniform_cap(plan, e->opts.tile_bytes ? e->opts.tile_bytes : kGranule);  // the presets work on 16 KiB granules
    uint64_t batch = 0;
    for (size_t i = 0; i < by_slot.size(); ++batch) {
        const uint32_t b = (uint32_t)(batch % S);
        size_t n = 1;
        while (i + n < by_slot.size() && n < per_buf && by_slot[i + n].slot == by_slot[i + n - 1].slot + 1) ++n;
        if (batch >= S) CK(cudaStreamWaitEvent(e->cstream, e->ev_k[b], 0));  // staging[b] consumed by the unpacks of batch - S
        const uint64_t bytes = n == 1 ? by_slot[i].nbytes : (n - 1) * slot_bytes + BS_PKG_HEADER + by_slot[i + n - 1].nbytes;
        const unsigned char* src = slots + by_slot[i].slot * slot_bytes + (n == 1 ? BS_PKG_HEADER : 0);
        CK(cudaMemcpyAsync(e->staging[b], src, bytes, cudaMemcpyHostToDevice, e->cstream));
        CK(cudaEventRecord(e->ev_c[b], e->cstream));
        CK(cudaStreamWaitEvent(e->kstream, e->ev_c[b], 0));
        bool in_order = cut != 0 && n > 1;  // consecutive packages of the cut in consecutive slots: one launch for the batch
        for (size_t j = 1; in_order && j < n; ++j) in_order = by_slot[i + j].index == by_slot[i + j - 1].index + 1;
        if (in_order) {
            PkgMap pm;
            pm.cap = cut; pm.slot_bytes = slot_bytes; pm.base = e->staging[b]; pm.slot_of = nullptr; pm.k_base = by_slot[i].index;
            const uint64_t blo = by_slot[i].lo, bhi = by_slot[i + n - 1].lo + by_slot[i + n - 1].nbytes;
            rc = out ? run_unpack_packages_range(out, L, pm, blo, bhi, flags | kFlagCheckPad, e->opts, e->sms, e->kstream)
                     : run_layered_unpack_range(lout, e->ws, e->ws_bytes, nullptr, nullptr, blo, bhi, flags | kFlagCheckPad, e->opts,
                                                e->sms, e->kstream, &pm);
            if (rc) return rc;
        } else {
            for (size_t j = 0; j < n; ++j) {
                const PkgItem& it = by_slot[i + j];
                const unsigned char* d = e->staging[b] + (n == 1 ? 0 : j * slot_bytes + BS_PKG_HEADER);
                rc = out ? run_unpack_range(out, L, d, nullptr, it.lo, it.lo + it.nbytes, flags | kFlagCheckPad, e->opts, e->sms, e->kstream)
                         : run_layered_unpack_range(lout, e->ws, e->ws_bytes, d, nullptr, it.lo, it.lo + it.nbytes, flags | kFlagCheckPad,
                                                    e->opts, e->sms, e->kstream);
                if (rc) return rc;
            }
        }
        CK(cudaEventRecord(e->ev_k[b], e->kstream));
        i += n;
    }
    CK(cudaEventRecord(t->dma_end, e->cstream));
    CK(post_status(t->h_result, &((WsHead*)e->ws)->status, e->kstream));
    CK(cudaEventRecord(t->done, e->kstream));
    CK(cudaStreamWaitEvent(consumer, t->done, 0));
    *ticket = guard.release();
    return BS_OK;
}

int bs_offload_packages_async(bs_engine* e, const bs_set_desc* set, uint64_t total_bytes, uint64_t cap, uint64_t stream_id,
                              void* h_slots, uint64_t slot_bytes, uint64_t n_slots, const uint32_t* h_slot_of,
                              cudaStream_t producer, bs_ticket** ticket)
{
    if (set == nullptr) return BS_ERR_ARG;
    return offload_packages_impl(e, set, nullptr, total_bytes, cap, stream_id, h_slots, slot_bytes, n_slots, h_slot_of, producer, ticket);
}

int bs_offload_layered_packages_async(bs_engine* e, const bs_layered_desc* set, uint64_t total_bytes, uint64_t cap,
                                      uint64_t stream_id, void* h_slots, uint64_t slot_bytes, uint64_t n_slots,
                                      const uint32_t* h_slot_of, cudaStream_t producer, bs_ticket** ticket)
{
    if (set == nullptr) return BS_ERR_ARG;
    return offload_packages_impl(e, nullptr, set, total_bytes, cap, stream_id, h_slots, slot_bytes, n_slots, h_slot_of, producer, ticket);
}

int bs_prefetch_packages_async(bs_engine* e, const void* h_slots, uint64_t slot_bytes, uint64_t n_slots, uint64_t stream_id,
                               bs_set_desc* out, void* d_pool, uint64_t pool_bytes, uint32_t flags, cudaStream_t consumer,
                               bs_ticket** ticket)
{
    if (out == nullptr) return BS_ERR_ARG;
    return prefetch_packages_impl(e, h_slots, slot_bytes, n_slots, stream_id, out, nullptr, d_pool, pool_bytes, flags, consumer, ticket);
}

int bs_prefetch_layered_packages_async(bs_engine* e, const void* h_slots, uint64_t slot_bytes, uint64_t n_slots, uint64_t stream_id,
                                       bs_layered_desc* out, void* d_pool, uint64_t pool_bytes, uint32_t flags,
                                       cudaStream_t consumer, bs_ticket** ticket)
{
    if (out == nullptr) return BS_ERR_ARG;
    return prefetch_packages_impl(e, h_slots, slot_bytes, n_slots, stream_id, nullptr, out, d_pool, pool_bytes, flags, consumer, ticket);
}

int bs_ticket_query(const bs_ticket* t)
{
    if (t == nullptr) return BS_ERR_ARG;
    cudaError_t e = cudaEventQuery(t->done);
    if (e == cudaErrorNotReady) return BS_PENDING;
    if (e != cudaSuccess) return cuda_fail(e);
    return t->h_result->status;
}

int bs_ticket_wait(bs_ticket* t, bs_ticket_stats* stats)
{
    if (t == nullptr) return BS_ERR_ARG;
    CK(cudaEventSynchronize(t->done));
    if (stats) {
        stats->bytes = t->bytes;
        stats->n_chunks = t->n_chunks;
        stats->status = t->h_result->status;
        stats->dma_ms = 0.f;
        stats->total_ms = 0.f;
        CK(cudaEventSynchronize(t->dma_end));
        CK(cudaEventElapsedTime(&stats->dma_ms, t->dma_begin, t->dma_end));
        CK(cudaEventElapsedTime(&stats->total_ms, t->t_begin, t->done));
    }
    return t->h_result->status;
}

int bs_ticket_stream_wait(const bs_ticket* t, cudaStream_t stream)
{
    if (t == nullptr) return BS_ERR_ARG;
    CK(cudaStreamWaitEvent(stream, t->done, 0));
    return BS_OK;
}

int bs_ticket_destroy(bs_ticket* t)
{
    if (t == nullptr) return BS_ERR_ARG;
    cudaEventSynchronize(t->done);
    cudaEventDestroy(t->t_begin);
    cudaEventDestroy(t->dma_begin);
    cudaEventDestroy(t->dma_end);
    cudaEventDestroy(t->done);
    result_slot_put(t->h_result);
    delete t;
    return BS_OK;
}

}  // extern "C"
