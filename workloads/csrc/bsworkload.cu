// bsworkload.cu — HARNESS code, not the product: (1) the device twin of workloads/values.py (seeded input
// generation, exact in fp64 so host and device agree bit for bit), (2) the stand-in DMRG contraction of
// SURVEY §8(a) S10 / §8(d) "Config 5 protocol": batched fp64 block GEMMs on sector shapes that keep the compute
// stream busy while the offload engine runs.  Holds none of the serializer's arithmetic.
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>

namespace {

__device__ __forceinline__ double value_at(uint64_t seed, uint64_t block, uint64_t e)
{
    uint64_t ctr = (block << 32) | e;
    uint64_t z = seed + (ctr + 1ull) * 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    z ^= z >> 31;
    return __ull2double_rn(z >> 11) * 0x1.0p-52 - 1.0;
}

__global__ void __launch_bounds__(256) fill_kernel(const uint64_t* __restrict__ addr, const uint64_t* __restrict__ nelems,
                                                   uint64_t first_block, uint64_t n_blocks, uint64_t seed)
{
    for (uint64_t b = blockIdx.x; b < n_blocks; b += gridDim.x) {
        double* dst = reinterpret_cast<double*>(addr[b]);
        const uint64_t n = nelems[b];
        for (uint64_t e = threadIdx.x; e < n; e += blockDim.x) dst[e] = value_at(seed, first_block + b, e);
    }
}

// C_i (m x n) = A_i (m x k) * B_i (k x n), row-major, one CTA per item, 32x32 output tiles, 16-deep k slices
struct GemmItem {
    uint64_t a, b, c;
    uint32_t m, n, k, pad;
};

__global__ void __launch_bounds__(256) contract_kernel(const GemmItem* __restrict__ items, uint32_t n_items)
{
    __shared__ double sa[32][17];
    __shared__ double sb[16][33];
    const int tx = threadIdx.x & 15, ty = threadIdx.x >> 4;
    for (uint32_t it = blockIdx.x; it < n_items; it += gridDim.x) {
        const GemmItem g = items[it];
        const double* A = reinterpret_cast<const double*>(g.a);
        const double* Bm = reinterpret_cast<const double*>(g.b);
        double* Cm = reinterpret_cast<double*>(g.c);
        for (uint32_t i0 = 0; i0 < g.m; i0 += 32) {
            for (uint32_t j0 = 0; j0 < g.n; j0 += 32) {
                double acc[2][2] = {{0, 0}, {0, 0}};
                for (uint32_t k0 = 0; k0 < g.k; k0 += 16) {
                    for (int r = threadIdx.x; r < 32 * 16; r += 256) {
                        int ii = r / 16, kk = r % 16;
                        sa[ii][kk] = (i0 + ii < g.m && k0 + kk < g.k) ? A[(uint64_t)(i0 + ii) * g.k + k0 + kk] : 0.0;
                        int k2 = r / 32, jj = r % 32;
                        sb[k2][jj] = (k0 + k2 < g.k && j0 + jj < g.n) ? Bm[(uint64_t)(k0 + k2) * g.n + j0 + jj] : 0.0;
                    }
                    __syncthreads();
#pragma unroll
                    for (int kk = 0; kk < 16; ++kk) {
                        double a0 = sa[ty][kk], a1 = sa[ty + 16][kk];
                        double b0 = sb[kk][tx], b1 = sb[kk][tx + 16];
                        acc[0][0] += a0 * b0; acc[0][1] += a0 * b1;
                        acc[1][0] += a1 * b0; acc[1][1] += a1 * b1;
                    }
                    __syncthreads();
                }
                for (int di = 0; di < 2; ++di)
                    for (int dj = 0; dj < 2; ++dj) {
                        uint32_t i = i0 + ty + 16 * di, j = j0 + tx + 16 * dj;
                        if (i < g.m && j < g.n) Cm[(uint64_t)i * g.n + j] = acc[di][dj];
                    }
            }
        }
    }
}

}  // namespace

extern "C" {

// values of blocks [first_block, first_block + n_blocks): d_addr[b] / d_nelems[b] for b in [0, n_blocks)
int wl_fill_blocks(const uint64_t* d_addr, const uint64_t* d_nelems, uint64_t first_block, uint64_t n_blocks,
                   uint64_t seed, cudaStream_t stream)
{
    if (n_blocks == 0) return 0;
    unsigned grid = (unsigned)(n_blocks < 148ull * 16 ? n_blocks : 148ull * 16);
    fill_kernel<<<grid, 256, 0, stream>>>(d_addr, d_nelems, first_block, n_blocks, seed);
    return (int)cudaGetLastError();
}

// stand-in contraction: d_items = array of {a, b, c, m, n, k, pad} (32 bytes each)
int wl_contract(const void* d_items, uint32_t n_items, uint32_t grid, cudaStream_t stream)
{
    if (n_items == 0) return 0;
    if (grid == 0) grid = 148 * 8;
    contract_kernel<<<grid, 256, 0, stream>>>(reinterpret_cast<const GemmItem*>(d_items), n_items);
    return (int)cudaGetLastError();
}

// Library comparator for the pack step (context only): one cudaMemcpyAsync (device to device) per block over
// the same block list; h_dsts / h_srcs / h_sizes are HOST arrays of n entries.  Returns the first cudaError_t.
int wl_memcpy_each(void** h_dsts, void** h_srcs, size_t* h_sizes, uint64_t n, cudaStream_t stream)
{
    for (uint64_t i = 0; i < n; ++i) {
        cudaError_t e = cudaMemcpyAsync(h_dsts[i], h_srcs[i], h_sizes[i], cudaMemcpyDeviceToDevice, stream);
        if (e != cudaSuccess) return (int)e;
    }
    return 0;
}

}  // extern "C"
