// bs_queue.cu — the save / load queue with checkpoints and the storage tier below
// pinned host RAM (NEXT-4), on top of two engines (bs_engine.cu).  See include/bs.h "queue".
#include <new>
#include <string.h>

#include <fcntl.h>
#include <sys/stat.h>
#include <unistd.h>

#include <algorithm>
#include <chrono>
#include <condition_variable>
#include <deque>
#include <memory>
#include <mutex>
#include <string>
#include <thread>
#include <unordered_map>
#include <vector>

#include "bs_engine.cuh"

using namespace bs;

extern "C" {

// ==== save / load queue with checkpoints (bs.h "queue") ===============================================
// Two engines (one per PCIe direction) + a key table.  Ordering between the lanes is by CUDA events only.
// one job of the queue's host IO thread (the storage tier; bs.h)
struct IoJob {
    bool spill = true;             // else fill
    std::string path;
    unsigned char* h = nullptr;
    uint64_t nbytes = 0;
    cudaEvent_t after = nullptr;   // spill: recorded behind the save's last DMA; the thread waits for it
    const bs_ticket* save = nullptr;  // spill: the save whose stream is written out (alive while the job is pending: whatever
                                      // retires a key's save ticket waits for the key's storage job first)
    int status = BS_OK;
    uint64_t bytes = 0;
    double seconds = 0.0;
    bool done = false;             // under IoThread::m
    bool counted = false;
};
struct IoThread {
    std::thread th;
    std::mutex m;
    std::condition_variable cv, cv_done;
    std::deque<std::shared_ptr<IoJob>> jobs;
    bool stop = false;
    int device = 0;
};

struct bs_queue {
    struct Entry {
        std::shared_ptr<IoJob> io;  // last storage job of the key
        bs_ticket* save = nullptr;  // last save / last load of the key (each lane is in order, so the last one covers all)
        bs_ticket* load = nullptr;
        const void* h = nullptr;
        uint64_t nbytes = 0;
        bs_stream_info_t info;
        bs_layered_stream_info_t linfo;
        bool adopted = false;
        bool layered = false;  // the stored stream is wire format v2
        bool fill_pending = false;  // `io` is a fill whose outcome (and wire format) no load has looked at yet
    };
    bs_engine* lane_save = nullptr;
    bs_engine* lane_load = nullptr;
    std::unordered_map<uint64_t, Entry> keys;
    std::vector<bs_ticket*> retired;  // replaced tickets, destroyed once complete
    bs_queue_stats st;
    IoThread* io = nullptr;
};

// ---- the host IO thread ------------------------------------------------------------------------------------------
static void io_run(IoJob& j)
{
    constexpr size_t kPiece = 64u << 20;
    if (j.after) cudaEventSynchronize(j.after);  // the stream has landed in the host buffer
    if (j.spill && j.save != nullptr && j.save->h_result->status != BS_OK) {  // the save failed: the buffer holds no stream
        j.status = j.save->h_result->status;
        return;
    }
    const auto t0 = std::chrono::steady_clock::now();
    const int fd = j.spill ? open(j.path.c_str(), O_WRONLY | O_CREAT | O_TRUNC, 0644) : open(j.path.c_str(), O_RDONLY);
    if (fd < 0) { j.status = BS_ERR_IO; return; }
    uint64_t pos = 0;
    while (pos < j.nbytes) {
        const size_t want = (size_t)std::min<uint64_t>(kPiece, j.nbytes - pos);
        const ssize_t got = j.spill ? write(fd, j.h + pos, want) : read(fd, j.h + pos, want);
        if (got <= 0) { j.status = BS_ERR_IO; break; }
        pos += (uint64_t)got;
    }
    if (close(fd) != 0 && j.spill) j.status = BS_ERR_IO;
    j.bytes = pos;
    j.seconds = std::chrono::duration<double>(std::chrono::steady_clock::now() - t0).count();
}

static void io_loop(IoThread* t)
{
    cudaSetDevice(t->device);
    for (;;) {
        std::shared_ptr<IoJob> j;
        {
            std::unique_lock<std::mutex> lk(t->m);
            t->cv.wait(lk, [&] { return t->stop || !t->jobs.empty(); });
            if (t->jobs.empty()) return;  // stop requested and nothing left
            j = t->jobs.front();
            t->jobs.pop_front();
        }
        io_run(*j);
        {
            std::lock_guard<std::mutex> lk(t->m);
            j->done = true;
        }
        t->cv_done.notify_all();
    }
}

static int io_submit(bs_queue* q, const std::shared_ptr<IoJob>& j)
{
    if (q->io == nullptr) {
        IoThread* t = new (std::nothrow) IoThread;
        if (!t) return BS_ERR_ARG;
        if (cudaGetDevice(&t->device) != cudaSuccess) { delete t; return BS_ERR_CUDA; }
        t->th = std::thread(io_loop, t);
        q->io = t;
    }
    {
        std::lock_guard<std::mutex> lk(q->io->m);
        q->io->jobs.push_back(j);
    }
    q->io->cv.notify_one();
    return BS_OK;
}

static void io_wait(bs_queue* q, const std::shared_ptr<IoJob>& j)  // host-blocking; accounts the job once
{
    if (!j || q->io == nullptr) return;
    {
        std::unique_lock<std::mutex> lk(q->io->m);
        q->io->cv_done.wait(lk, [&] { return j->done; });
    }
    if (!j->counted) {
        j->counted = true;
        if (j->after) { cudaEventDestroy(j->after); j->after = nullptr; }
        if (j->status == BS_OK) (j->spill ? q->st.bytes_spilled : q->st.bytes_filled) += j->bytes;
    }
}

static void io_shutdown(bs_queue* q)
{
    if (q->io == nullptr) return;
    {
        std::lock_guard<std::mutex> lk(q->io->m);
        q->io->stop = true;
    }
    q->io->cv.notify_all();
    q->io->th.join();
    delete q->io;
    q->io = nullptr;
}

static uint64_t engine_device_bytes(const bs_engine* e)
{
    return (uint64_t)e->cfg.n_staging * e->cfg.chunk_bytes + e->ws_bytes + e->header_cap + sizeof(bs_result);
}

static int engine_wait_ticket(bs_engine* e, const bs_ticket* t)  // everything the engine does next waits for t
{
    CK(cudaStreamWaitEvent(e->kstream, t->done, 0));
    CK(cudaStreamWaitEvent(e->cstream, t->done, 0));
    return BS_OK;
}

static bool ticket_complete(const bs_ticket* t) { return cudaEventQuery(t->done) != cudaErrorNotReady; }

static void queue_reap(bs_queue* q, bool block)
{
    size_t w = 0;
    for (bs_ticket* t : q->retired) {
        if (block || ticket_complete(t)) bs_ticket_destroy(t);
        else q->retired[w++] = t;
    }
    q->retired.resize(w);
}

static void queue_retire(bs_queue* q, bs_ticket*& t)
{
    if (t) q->retired.push_back(t);
    t = nullptr;
}

static void queue_count_in_flight(bs_queue* q)
{
    uint32_t n = 0;
    for (auto& kv : q->keys) {
        if (kv.second.save && !ticket_complete(kv.second.save)) ++n;
        if (kv.second.load && !ticket_complete(kv.second.load)) ++n;
    }
    for (bs_ticket* t : q->retired)
        if (!ticket_complete(t)) ++n;
    q->st.in_flight = n;
    if (n > q->st.max_in_flight) q->st.max_in_flight = n;
}

static void queue_account_host(bs_queue* q)
{
    uint64_t live = 0;
    for (auto& kv : q->keys) live += kv.second.nbytes;
    q->st.host_bytes_live = live;
    q->st.keys_live = q->keys.size();
    if (live > q->st.host_bytes_peak) q->st.host_bytes_peak = live;
}

int bs_queue_create(bs_queue** out, const bs_engine_cfg* lane_cfg)
{
    if (out == nullptr || lane_cfg == nullptr) return BS_ERR_ARG;
    bs_queue* q = new (std::nothrow) bs_queue;
    if (!q) return BS_ERR_ARG;
    memset(&q->st, 0, sizeof(q->st));
    int rc = bs_engine_create(&q->lane_save, lane_cfg);
    if (rc == BS_OK) rc = bs_engine_create(&q->lane_load, lane_cfg);
    if (rc != BS_OK) {
        if (q->lane_save) bs_engine_destroy(q->lane_save);
        delete q;
        return rc;
    }
    q->st.device_bytes = engine_device_bytes(q->lane_save) + engine_device_bytes(q->lane_load);
    *out = q;
    return BS_OK;
}

int bs_queue_drain(bs_queue* q)
{
    if (q == nullptr) return BS_ERR_ARG;
    CK(cudaStreamSynchronize(q->lane_save->kstream));
    CK(cudaStreamSynchronize(q->lane_save->cstream));
    CK(cudaStreamSynchronize(q->lane_load->kstream));
    CK(cudaStreamSynchronize(q->lane_load->cstream));
    queue_reap(q, true);
    queue_count_in_flight(q);
    return BS_OK;
}

int bs_queue_destroy(bs_queue* q)
{
    if (q == nullptr) return BS_ERR_ARG;
    bs_queue_drain(q);
    for (auto& kv : q->keys) io_wait(q, kv.second.io);
    io_shutdown(q);
    for (auto& kv : q->keys) {
        if (kv.second.save) bs_ticket_destroy(kv.second.save);
        if (kv.second.load) bs_ticket_destroy(kv.second.load);
    }
    bs_engine_destroy(q->lane_save);
    bs_engine_destroy(q->lane_load);
    delete q;
    return BS_OK;
}

static int queue_save_impl(bs_queue* q, uint64_t key, const bs_set_desc* set, const bs_layered_desc* lset, uint64_t total_bytes,
                           void* h_pinned, uint64_t h_capacity, cudaStream_t producer)
{
    if (q == nullptr || (set == nullptr && lset == nullptr) || h_pinned == nullptr) return BS_ERR_ARG;
    queue_reap(q, false);
    int rc;
    auto it = q->keys.find(key);
    if (it != q->keys.end()) io_wait(q, it->second.io);  // a storage job may still be reading / filling the key's buffer
    // the host buffer may still be read by a load of this key (or, for a new buffer under the same key, nothing to wait for)
    if (it != q->keys.end() && it->second.load && !ticket_complete(it->second.load))
        if ((rc = engine_wait_ticket(q->lane_save, it->second.load))) return rc;
    bs_ticket* t = nullptr;
    if ((rc = bs_engine_offload_impl(q->lane_save, set, lset, total_bytes, h_pinned, h_capacity, producer, &t))) return rc;
    total_bytes = t->bytes;  // the size prediction, if the call made it
    bs_queue::Entry& en = q->keys[key];
    en.io.reset();  // the key's storage job (waited for above) described the stream this save replaces
    en.fill_pending = false;
    queue_retire(q, en.save);
    en.save = t;
    en.h = h_pinned;
    en.nbytes = total_bytes;
    en.adopted = false;
    en.layered = lset != nullptr;
    if (set) {
        en.info.n_tensors = set->n_tensors;
        en.info.n_blocks = set->n_blocks;
        en.info.header_bytes = header_bytes_of(set->n_tensors, set->n_blocks, set->dtype);
        en.info.max_rank = legs_of(set->dtype);
        en.info.align = (set->dtype & BS_ALIGN8) ? 8 : 16;
        en.info.payload_bytes = total_bytes - en.info.header_bytes;
        en.info.total_bytes = total_bytes;
        en.info.dtype = set->dtype & BS_DTYPE_MASK;
    } else {
        en.linfo.n_structs = lset->n_structs;
        en.linfo.n_struct_blocks = lset->n_struct_blocks;
        en.linfo.n_layers = lset->n_layers;
        en.linfo.header_bytes = bs_layered_header_bytes(lset->n_structs, lset->n_layers, lset->n_struct_blocks);
        en.linfo.payload_bytes = total_bytes - en.linfo.header_bytes;
        en.linfo.total_bytes = total_bytes;
    }
    q->st.saves += 1;
    q->st.bytes_saved += total_bytes;
    queue_account_host(q);
    queue_count_in_flight(q);
    return BS_OK;
}

int bs_queue_save(bs_queue* q, uint64_t key, const bs_set_desc* set, uint64_t total_bytes, void* h_pinned, uint64_t h_capacity,
                  cudaStream_t producer)
{
    if (set == nullptr) return BS_ERR_ARG;
    return queue_save_impl(q, key, set, nullptr, total_bytes, h_pinned, h_capacity, producer);
}

int bs_queue_save_layered(bs_queue* q, uint64_t key, const bs_layered_desc* set, uint64_t total_bytes, void* h_pinned,
                          uint64_t h_capacity, cudaStream_t producer)
{
    if (set == nullptr) return BS_ERR_ARG;
    return queue_save_impl(q, key, nullptr, set, total_bytes, h_pinned, h_capacity, producer);
}

int bs_queue_adopt(bs_queue* q, uint64_t key, const void* h_pinned, uint64_t nbytes)
{
    if (q == nullptr || h_pinned == nullptr || nbytes < kFixedHeader) return BS_ERR_ARG;
    queue_reap(q, false);
    auto it = q->keys.find(key);
    if (it != q->keys.end()) {  // the old buffer's operations are not ours to order against the new one: finish them
        io_wait(q, it->second.io);
        int rc = bs_queue_wait(q, key, nullptr, nullptr);
        (void)rc;
        queue_retire(q, it->second.save);
        queue_retire(q, it->second.load);
    }
    bs_queue::Entry& en = q->keys[key];
    en.io.reset();
    en.fill_pending = false;
    en.h = h_pinned;
    en.nbytes = nbytes;
    en.adopted = true;
    uint32_t version = 0;
    memcpy(&version, (const unsigned char*)h_pinned + 8, 4);  // the stream is complete and in host RAM
    en.layered = version == 2u;
    queue_account_host(q);
    return BS_OK;
}

static int queue_load_impl(bs_queue* q, uint64_t key, bs_set_desc* out, bs_layered_desc* lout, void* d_pool, uint64_t pool_bytes,
                           uint32_t flags, cudaStream_t consumer)
{
    if (q == nullptr || (out == nullptr && lout == nullptr)) return BS_ERR_ARG;
    queue_reap(q, false);
    auto it = q->keys.find(key);
    if (it == q->keys.end()) return BS_ERR_ARG;
    bs_queue::Entry& en = it->second;
    if (en.fill_pending) {  // the stream is still being read from its file: the host waits ("fetching", L132)
        io_wait(q, en.io);
        if (en.io->status != BS_OK) return BS_ERR_IO;  // stays pending: every load fails until a save / adopt / fill replaces it
        uint32_t version = 0;
        memcpy(&version, (const unsigned char*)en.h + 8, 4);
        en.layered = version == 2u;  // settled once, from the complete file
        en.fill_pending = false;
    }
    if (en.layered != (lout != nullptr)) return BS_ERR_ARG;  // the key holds a stream of the other wire format
    int rc;
    if (en.save && !ticket_complete(en.save))  // the stream is still on its way to the host buffer
        if ((rc = engine_wait_ticket(q->lane_load, en.save))) return rc;
    bs_ticket* t = nullptr;
    rc = bs_engine_prefetch_impl(q->lane_load, en.h, en.nbytes, out, lout, d_pool, pool_bytes, flags, consumer, &t,
                       (en.adopted || en.layered) ? nullptr : &en.info, (en.adopted || !en.layered) ? nullptr : &en.linfo);
    if (rc) return rc;
    queue_retire(q, en.load);
    en.load = t;
    q->st.loads += 1;
    q->st.bytes_loaded += en.nbytes;
    queue_count_in_flight(q);
    return BS_OK;
}

int bs_queue_load(bs_queue* q, uint64_t key, bs_set_desc* out, void* d_pool, uint64_t pool_bytes, uint32_t flags,
                  cudaStream_t consumer)
{
    if (out == nullptr) return BS_ERR_ARG;
    return queue_load_impl(q, key, out, nullptr, d_pool, pool_bytes, flags, consumer);
}

int bs_queue_load_layered(bs_queue* q, uint64_t key, bs_layered_desc* out, void* d_pool, uint64_t pool_bytes, uint32_t flags,
                          cudaStream_t consumer)
{
    if (out == nullptr) return BS_ERR_ARG;
    return queue_load_impl(q, key, nullptr, out, d_pool, pool_bytes, flags, consumer);
}

int bs_queue_checkpoint(bs_queue* q, uint64_t key, cudaStream_t stream)
{
    if (q == nullptr) return BS_ERR_ARG;
    auto it = q->keys.find(key);
    if (it == q->keys.end()) return BS_ERR_ARG;
    if (it->second.save) CK(cudaStreamWaitEvent(stream, it->second.save->done, 0));
    if (it->second.load) CK(cudaStreamWaitEvent(stream, it->second.load->done, 0));
    return BS_OK;
}

int bs_queue_wait(bs_queue* q, uint64_t key, bs_ticket_stats* save_stats, bs_ticket_stats* load_stats)
{
    if (q == nullptr) return BS_ERR_ARG;
    auto it = q->keys.find(key);
    if (it == q->keys.end()) return BS_ERR_ARG;
    if (save_stats) memset(save_stats, 0, sizeof(*save_stats));
    if (load_stats) memset(load_stats, 0, sizeof(*load_stats));
    int rc_s = it->second.save ? bs_ticket_wait(it->second.save, save_stats) : BS_OK;
    int rc_l = it->second.load ? bs_ticket_wait(it->second.load, load_stats) : BS_OK;
    queue_count_in_flight(q);
    return rc_s != BS_OK ? rc_s : rc_l;
}

int bs_queue_query(bs_queue* q, uint64_t key)
{
    if (q == nullptr) return BS_ERR_ARG;
    auto it = q->keys.find(key);
    if (it == q->keys.end()) return BS_ERR_ARG;
    int rc_s = it->second.save ? bs_ticket_query(it->second.save) : BS_OK;
    int rc_l = it->second.load ? bs_ticket_query(it->second.load) : BS_OK;
    if (rc_s < 0) return rc_s;
    if (rc_l < 0) return rc_l;
    return (rc_s == BS_PENDING || rc_l == BS_PENDING) ? BS_PENDING : BS_OK;
}

int bs_queue_forget(bs_queue* q, uint64_t key)
{
    if (q == nullptr) return BS_ERR_ARG;
    auto it = q->keys.find(key);
    if (it == q->keys.end()) return BS_ERR_ARG;
    io_wait(q, it->second.io);
    if (it->second.save) bs_ticket_destroy(it->second.save);  // waits for completion
    if (it->second.load) bs_ticket_destroy(it->second.load);
    q->keys.erase(it);
    queue_account_host(q);
    queue_count_in_flight(q);
    return BS_OK;
}

int bs_queue_spill(bs_queue* q, uint64_t key, const char* path)
{
    if (q == nullptr || path == nullptr) return BS_ERR_ARG;
    auto it = q->keys.find(key);
    if (it == q->keys.end()) return BS_ERR_ARG;
    bs_queue::Entry& en = it->second;
    io_wait(q, en.io);
    if (en.fill_pending) {  // a stream that never arrived from its file cannot be written out again
        if (en.io->status != BS_OK) return BS_ERR_IO;
        uint32_t version = 0;
        memcpy(&version, (const unsigned char*)en.h + 8, 4);
        en.layered = version == 2u;
        en.fill_pending = false;
    }
    auto j = std::make_shared<IoJob>();
    j->spill = true;
    j->path = path;
    j->h = (unsigned char*)const_cast<void*>(en.h);
    j->nbytes = en.nbytes;
    if (en.save) {  // behind the save's last DMA (the save lane is in order)
        CK(cudaEventCreateWithFlags(&j->after, cudaEventDisableTiming));
        CK(cudaEventRecord(j->after, q->lane_save->cstream));
        j->save = en.save;
    }
    int rc = io_submit(q, j);
    if (rc) return rc;
    en.io = j;
    return BS_OK;
}

int bs_queue_fill(bs_queue* q, uint64_t key, const char* path, void* h_pinned, uint64_t h_capacity)
{
    if (q == nullptr || path == nullptr || h_pinned == nullptr) return BS_ERR_ARG;
    struct stat sb;
    if (stat(path, &sb) != 0) return BS_ERR_IO;
    if ((uint64_t)sb.st_size > h_capacity) return BS_ERR_CAPACITY;
    if ((uint64_t)sb.st_size < kFixedHeader) return BS_ERR_CORRUPT;
    auto it = q->keys.find(key);
    if (it != q->keys.end()) {  // as bs_queue_adopt: finish what still uses the old buffer
        io_wait(q, it->second.io);
        bs_queue_wait(q, key, nullptr, nullptr);
        queue_retire(q, it->second.save);
        queue_retire(q, it->second.load);
    }
    auto j = std::make_shared<IoJob>();
    j->spill = false;
    j->path = path;
    j->h = (unsigned char*)h_pinned;
    j->nbytes = (uint64_t)sb.st_size;
    int rc = io_submit(q, j);
    if (rc) return rc;
    bs_queue::Entry& en = q->keys[key];
    en.h = h_pinned;
    en.nbytes = (uint64_t)sb.st_size;
    en.adopted = true;
    en.layered = false;  // settled from the version word once the file is in
    en.io = j;
    en.fill_pending = true;
    queue_account_host(q);
    return BS_OK;
}

int bs_queue_io_wait(bs_queue* q, uint64_t key, uint64_t* bytes, double* seconds)
{
    if (q == nullptr) return BS_ERR_ARG;
    auto it = q->keys.find(key);
    if (it == q->keys.end()) return BS_ERR_ARG;
    if (bytes) *bytes = 0;
    if (seconds) *seconds = 0.0;
    if (!it->second.io) return BS_OK;
    io_wait(q, it->second.io);
    if (bytes) *bytes = it->second.io->bytes;
    if (seconds) *seconds = it->second.io->seconds;
    return it->second.io->status;
}

int bs_queue_get_stats(bs_queue* q, bs_queue_stats* out)
{
    if (q == nullptr || out == nullptr) return BS_ERR_ARG;
    queue_reap(q, false);
    queue_count_in_flight(q);
    *out = q->st;
    return BS_OK;
}

}  // extern "C"
