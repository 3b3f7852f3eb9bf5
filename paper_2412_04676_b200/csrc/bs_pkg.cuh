// bs_pkg.cuh — self-contained packages: the cut and the host-side plan (shared by bs_pkg.cu and bs_engine.cu).
#pragma once
#include <vector>

#include "bs_internal.cuh"

namespace bs {

// The cut (bs.h "packages"): header region and payload are cut separately into pieces of `cap` bytes.
__host__ __device__ inline uint64_t pkg_count(uint64_t hb, uint64_t total, uint64_t cap)
{
    if (cap == 0 || (cap & 15) || hb > total) return 0;
    return (hb + cap - 1) / cap + (total - hb + cap - 1) / cap;
}

__host__ __device__ inline bool pkg_range(uint64_t hb, uint64_t total, uint64_t cap, uint64_t k, uint64_t* lo, uint64_t* hi)
{
    if (k >= pkg_count(hb, total, cap)) return false;
    const uint64_t nh = (hb + cap - 1) / cap;
    const uint64_t base = k < nh ? k * cap : hb + (k - nh) * cap;
    const uint64_t end = k < nh ? hb : total;
    *lo = base;
    *hi = base + cap < end ? base + cap : end;
    return true;
}

struct PkgItem {
    uint64_t slot, lo, nbytes;
    uint32_t index, first_block;
};
struct PkgPlan {
    std::vector<PkgItem> items;  // in index order; the first n_header lie in the header region
    uint64_t total, hb;
    uint32_t n_header;
};

int pkg_plan(const unsigned char* h_hdrs, uint64_t stride, uint64_t n_slots, uint64_t slot_bytes, uint64_t stream_id,
             PkgPlan* plan);
// the size limit whose cut (bs.h) the planned packages are, if it is a multiple of `tile`; 0 if they are cut otherwise
uint64_t plan_uniform_cap(const PkgPlan& plan, uint32_t tile);
cudaError_t launch_pkg_header(const WsLayout& L, uint64_t cap, uint64_t stream_id, uint64_t k, uint64_t expect_count,
                              void* d_dst, bs_result* d_result, cudaStream_t stream, bool poison_on_error = false);
cudaError_t launch_pkg_headers(const WsLayout& L, uint64_t cap, uint64_t stream_id, uint64_t first, uint64_t n, uint64_t count,
                               void* d_base, uint64_t slot_bytes, const uint32_t* d_slot_of, bs_result* d_result, cudaStream_t stream,
                               bool poison_on_error = false);
cudaError_t launch_pkg_check(const WsLayout& L, const void* d_hdrs, uint64_t stride, uint64_t n_slots, uint64_t stream_id,
                             bs_result* d_result, cudaStream_t stream);

}  // namespace bs
