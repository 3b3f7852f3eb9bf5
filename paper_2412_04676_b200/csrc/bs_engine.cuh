// bs_engine.cuh — what the engine (bs_engine.cu) shares with the queue built on top of it (bs_queue.cu).  Not part of the
// C ABI.
#pragma once
#include "bs_pkg.cuh"

namespace bs {
int cuda_fail(cudaError_t e);
constexpr uint32_t kMaxStaging = 8;
}  // namespace bs

struct bs_engine {
    bs_engine_cfg cfg;
    bs_opts opts;
    int sms;
    cudaStream_t kstream, cstream;
    unsigned char* staging[bs::kMaxStaging];
    cudaEvent_t ev_k[bs::kMaxStaging];  // kernel finished with staging[b]
    cudaEvent_t ev_c[bs::kMaxStaging];  // DMA finished with staging[b]
    cudaEvent_t ev_fence_k, ev_fence_c, ev_dep;
    void* ws;
    uint64_t ws_bytes;
    unsigned char* header_buf;
    uint64_t header_cap;
    bs_result* d_result;
    unsigned char* pkg_tab;  // device copy of the package headers of a bs_prefetch_packages_async call (grown on demand)
    uint64_t pkg_tab_slots;
};

struct bs_ticket {
    cudaEvent_t t_begin, dma_begin, dma_end, done;
    bs_result* h_result;  // pinned
    uint64_t bytes;
    uint32_t n_chunks;
    int immediate;  // status known at submit time (no device work was enqueued)
    bool is_prefetch;
};

#define CK(call)                                          \
    do {                                                  \
        cudaError_t e__ = (call);                         \
        if (e__ != cudaSuccess) return cuda_fail(e__);    \
    } while (0)

// one body for both wire formats and both directions (bs_engine.cu); hidden from the library's export table
__attribute__((visibility("hidden"))) int bs_engine_offload_impl(bs_engine* e, const bs_set_desc* set, const bs_layered_desc* lset,
                                                                 uint64_t total_bytes, void* h_pinned, uint64_t h_capacity,
                                                                 cudaStream_t producer, bs_ticket** ticket);
// `known` / `known_l`: the counts of a stream that is still on its way to h_pinned (a queue load submitted behind the save
// of the same key); otherwise the fixed header is read from host RAM.  Either way the device validates what arrives.
__attribute__((visibility("hidden"))) int bs_engine_prefetch_impl(bs_engine* e, const void* h_pinned, uint64_t nbytes, bs_set_desc* out,
                                                                  bs_layered_desc* lout, void* d_pool, uint64_t pool_bytes,
                                                                  uint32_t flags, cudaStream_t consumer, bs_ticket** ticket,
                                                                  const bs_stream_info_t* known = nullptr,
                                                                  const bs_layered_stream_info_t* known_l = nullptr);
