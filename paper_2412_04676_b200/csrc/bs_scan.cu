// bs_scan.cu — the size / offset pass on its own: steps S1, S2, S4 (serialize) and S6 (deserialize) of SURVEY §8(a) as ONE
// kernel launch (the pass itself is bs_scan_phase.cuh; the fused kernels of bs_move_tma.cu run the same code in front of
// the data movement).  Used where the pass and the movement are separate calls: bs_serialized_size, the range calls, the
// engine (one pass, then one pack / unpack launch per 256 MiB chunk), packages, and sets too large for the fused kernels.
#include <atomic>
#include <chrono>
#include <random>

#include "bs_scan_phase.cuh"

namespace bs {

namespace {

template <bool DESER>
__global__ void __launch_bounds__(kScanThreads, 4) scan_kernel(const ScanParams p)
{
    __shared__ scan::Shared sm;
    const scan::Shape s = scan::shape_of<DESER>(p);
    scan::run<DESER>(p, s, p.tag, sm, false);
}

}  // namespace

// A fresh 40-bit epoch for every call (bs_scan_phase.cuh), shifted into the tag position; never 0.  The counter starts at
// a random value so that words left in device memory by another process cannot carry a tag this process will use soon.
uint64_t next_epoch_tag()
{
    static std::atomic<uint64_t> counter{[] {
        std::random_device rd;
        const uint64_t t = (uint64_t)std::chrono::steady_clock::now().time_since_epoch().count();
        return ((uint64_t)rd() << 20) ^ ((uint64_t)rd() << 3) ^ t;
    }()};
    uint64_t e;
    do {
        e = counter.fetch_add(1, std::memory_order_relaxed) & ((1ull << 40) - 1);
    } while (e == 0);
    return e << 24;
}

// While `stream` is being captured into a CUDA graph every replay would reuse the epoch baked into the launch, so the
// call clears head + scan state in front of the kernel instead (one memset node); otherwise nothing needs clearing.
cudaError_t prepare_scan_state(const WsLayout& L, cudaStream_t stream)
{
    cudaStreamCaptureStatus cs = cudaStreamCaptureStatusNone;
    cudaError_t e = cudaStreamIsCapturing(stream, &cs);
    if (e != cudaSuccess) return e;
    if (cs == cudaStreamCaptureStatusNone) return cudaSuccess;
    return cudaMemsetAsync(L.head, 0, L.zero_bytes, stream);
}

cudaError_t launch_scan(bool deser, const ScanParams& p, int sm_count, cudaStream_t stream)
{
    cudaError_t e = prepare_scan_state(p.ws, stream);
    if (e != cudaSuccess) return e;
    ScanParams q = p;
    q.tag = next_epoch_tag();
    // grid: enough CTAs to cover the items, at most a few per SM (items are claimed dynamically)
    const uint64_t want = scan::host_items(p.T, p.B);
    const uint64_t cap = (uint64_t)sm_count * 4;
    const unsigned grid = (unsigned)(want < cap ? want : cap);
    if (deser) scan_kernel<true><<<grid, kScanThreads, 0, stream>>>(q);
    else scan_kernel<false><<<grid, kScanThreads, 0, stream>>>(q);
    return cudaGetLastError();
}

}  // namespace bs
