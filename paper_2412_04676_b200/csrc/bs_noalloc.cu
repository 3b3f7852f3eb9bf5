// bs_noalloc.cu — bs_serialize_noalloc (bs.h): bs_serialize for callers that have no device memory to give as a workspace
// and may not ask the CUDA allocator for any.
//
// Who that is.  The solver this library serves sizes its block pool to what the device has left (the memory peaks of
// PAPER L132-136 are why scratch data is offloaded at all), so at the moment a set must be saved a cudaMalloc of even
// a megabyte can fail; and a plug-in that runs inside such a host program is usually forbidden to allocate behind the
// back of the host's pool.  A cudaMalloc / cudaFree also synchronises the whole device, which would stall the side
// streams an offload is hidden behind.  Such callers still own the blocks, the stream buffer and the result word — what
// they lack is the pass's scratch (offset table, scan state, work counters: bs_workspace_bytes).
//
// What this file does about it.  The scratch is a file-scope device array, reserved once per GPU when the library's
// module is loaded there and held until the process exits.  The kernels are the ones bs_serialize launches; only the
// workspace pointer differs.  On the host the array's NAME is a stand-in symbol, not a device address — handing
// `g_scratch` itself to a kernel would fault (or, on a system where the GPU can reach host memory, quietly use the wrong
// bytes) — so the first call on each device asks the runtime for the real address with cudaGetSymbolAddress, with that
// device current, and caches it per device.
#include <atomic>

#include "bs_internal.cuh"

namespace bs {
namespace {

// 1.5 MiB: room for BS_NOALLOC_MAX_BLOCKS blocks and a stream of BS_NOALLOC_MAX_STREAM_BYTES (about 1.25 MiB is used
// at the limits; scratch_for_device checks that against bs_workspace_bytes, tests/test_zz_no_alloc.py pins it too).
constexpr uint64_t kScratchBytes = 1536u * 1024u;
static __device__ __align__(256) unsigned char g_scratch[kScratchBytes];

constexpr int kMaxDevices = 64;
std::atomic<void*> g_scratch_addr[kMaxDevices];  // device address of g_scratch on device d, once looked up

// Device address of the array on the CURRENT device.  The look-up runs once per device; two threads racing through
// it both get the same answer from the runtime, so the cache needs no lock.
int scratch_for_device(void** out)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e);
    if (dev < 0 || dev >= kMaxDevices) return BS_ERR_UNSUPPORTED;
    void* p = g_scratch_addr[dev].load(std::memory_order_acquire);
    if (p == nullptr) {
        e = cudaGetSymbolAddress(&p, g_scratch);
        if (e != cudaSuccess) return cuda_fail(e);
        if (p == nullptr || ((uintptr_t)p & 255) != 0) return BS_ERR_CUDA;
        if (bs_workspace_bytes(0, BS_NOALLOC_MAX_BLOCKS, BS_NOALLOC_MAX_STREAM_BYTES) > kScratchBytes) return BS_ERR_CAPACITY;
        g_scratch_addr[dev].store(p, std::memory_order_release);
    }
    *out = p;
    return BS_OK;
}

}  // namespace
}  // namespace bs

using namespace bs;

extern "C" {

uint64_t bs_noalloc_scratch_bytes(void) { return kScratchBytes; }

int bs_serialize_noalloc(const bs_set_desc* set, void* d_stream, uint64_t capacity, bs_result* d_result, const bs_opts* opts,
                         cudaStream_t stream)
{
    // the limits first, before anything touches the device: a set the fixed scratch cannot serve is refused as such
    // instead of surfacing later as a deferred BS_ERR_CAPACITY the caller would read as "stream buffer too small"
    int rc = check_set(set);
    if (rc) return rc;
    if (set->n_blocks > BS_NOALLOC_MAX_BLOCKS || capacity > BS_NOALLOC_MAX_STREAM_BYTES) return BS_ERR_CAPACITY;
    void* ws = nullptr;
    if ((rc = scratch_for_device(&ws))) return rc;
    // nothing to clear: every word of the workspace the kernels synchronise on carries the call's epoch tag, so what the
    // previous call left in the array reads as "not written yet" (bs_internal.cuh; the garbage-workspace tests)
    return bs_serialize(set, d_stream, capacity, ws, kScratchBytes, d_result, opts, stream);
}

}  // extern "C"
