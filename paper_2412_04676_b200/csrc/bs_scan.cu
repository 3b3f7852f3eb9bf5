// bs_scan.cu — the size / offset pass: steps S1, S2, S4 (serialize) and S6 (deserialize) of SURVEY §8(a).
//
// "low cost and exact prediction of post-serialization data size before the actual
// serialization takes place ... let the main thread map the output buffer".  In the paper one CPU thread
// does this; here it is ONE kernel launch: a single-pass chained (decoupled look-back) exclusive scan of
// the stored block sizes over all B blocks, which at the same time
//   - validates the descriptor (serialize) or every header field (deserialize: SURVEY §8(c) list),
//   - writes the blk[] table {payload offset, block address} = the "pointer structure" of L90-92,
//   - writes tile_first[] (which block holds the first byte of every 16 KiB payload granule) = the work
//     partition the data-movement kernel uses to give every CTA an exact, disjoint stream interval,
//   - reports header / payload / total bytes and the deferred status in bs_result.
// Roofline: HBM-bound, ~12+8 B read and 16 B written per block (serialize) — <1 % of the payload traffic.
#include "bs_internal.cuh"

namespace bs {

namespace {

constexpr uint64_t kFlagAgg = 1ull << 62;
constexpr uint64_t kFlagPrefix = 2ull << 62;
constexpr uint64_t kValMask = (1ull << 62) - 1;
constexpr uint32_t kInlineBoundaries = 4;

__device__ __forceinline__ uint64_t ld_acquire_u64(const uint64_t* p)
{
    uint64_t v;
    asm volatile("ld.acquire.gpu.global.u64 %0, [%1];" : "=l"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void st_release_u64(uint64_t* p, uint64_t v)
{
    asm volatile("st.release.gpu.global.u64 [%0], %1;" ::"l"(p), "l"(v) : "memory");
}
__device__ __forceinline__ void set_status(WsHead* h, int code)
{
    if (code != 0) atomicCAS(&h->status, 0, code);
}
__device__ __forceinline__ uint64_t warp_incl_scan(uint64_t v, uint32_t lane)
{
#pragma unroll
    for (int d = 1; d < 32; d <<= 1) {
        uint64_t o = __shfl_up_sync(0xffffffffu, v, d);
        if (lane >= (uint32_t)d) v += o;
    }
    return v;
}
__device__ __forceinline__ uint64_t warp_sum(uint64_t v)
{
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) v += __shfl_xor_sync(0xffffffffu, v, d);
    return v;
}

struct TensorHead {
    uint32_t rank, first, n, reserved;
};

template <bool DESER>
__device__ __forceinline__ TensorHead load_tensor(const ScanParams& p, uint64_t t)
{
    TensorHead h;
    if (DESER) {
        const uint4* r = reinterpret_cast<const uint4*>(p.header + kFixedHeader + kTensorRec * t);
        uint4 a = __ldg(r), b = __ldg(r + 1);
        h.rank = a.x; h.first = a.y; h.n = a.z; h.reserved = b.w;
    } else {
        const uint4* r = reinterpret_cast<const uint4*>(p.tensors + t);
        uint4 a = __ldg(r), b = __ldg(r + 1);
        h.rank = a.x; h.first = a.y; h.n = a.z; h.reserved = b.w;
    }
    return h;
}

template <bool DESER>
__global__ void __launch_bounds__(kScanThreads) scan_kernel(const ScanParams p)
{
    __shared__ uint32_t s_tile;
    __shared__ uint64_t s_warp_sum[kScanThreads / 32];
    __shared__ uint64_t s_tile_prefix;
    __shared__ uint64_t s_tile_total;
    __shared__ uint32_t s_big_n;
    __shared__ uint32_t s_big_idx[kScanTile];
    __shared__ uint32_t s_big_cnt[kScanTile];
    __shared__ uint64_t s_big_g0[kScanTile];

    WsHead* head = p.ws.head;
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int kErrBad = DESER ? BS_ERR_CORRUPT : BS_ERR_ARG;
    constexpr int kErrRank = DESER ? BS_ERR_CORRUPT : BS_ERR_UNSUPPORTED;

    // ---- counts; deserialize: the fixed header (SURVEY §8(c) checks, in order) ------------------------
    uint64_t T = p.T, B = p.B, hb = 0, P_hdr = 0;
    uint32_t dtype = p.dtype;
    bool ok = true;
    if (DESER) {
        int code = 0;
        T = B = 0;
        if (p.nbytes < kFixedHeader) {
            code = BS_ERR_CORRUPT;
        } else {
            const uint4* f = reinterpret_cast<const uint4*>(p.header);
            uint4 w0 = __ldg(f), w1 = __ldg(f + 1), w2 = __ldg(f + 2), w3 = __ldg(f + 3);
            uint64_t hT = (uint64_t)w2.x | ((uint64_t)w2.y << 32), hB = (uint64_t)w2.z | ((uint64_t)w2.w << 32);
            uint64_t hH = (uint64_t)w3.x | ((uint64_t)w3.y << 32), hP = (uint64_t)w3.z | ((uint64_t)w3.w << 32);
            if (w0.x != 0x41505342u || w0.y != 0x31455352u)      code = BS_ERR_CORRUPT;  // "BSPARSE1"
            else if (w0.z != 1u)                                  code = BS_ERR_CORRUPT;  // version
            else if (w0.w != 0x01020304u)                         code = BS_ERR_CORRUPT;  // endian_tag
            else if (w1.x > (uint32_t)BS_C128)                    code = BS_ERR_CORRUPT;  // dtype
            else if (w1.y != 2u)                                  code = BS_ERR_CORRUPT;  // n_qn
            else if (w1.z != 3u)                                  code = BS_ERR_CORRUPT;  // max_rank
            else if (w1.w != 16u)                                 code = BS_ERR_CORRUPT;  // align
            else if (hT >= (1ull << 32) || hB >= (1ull << 32))   code = BS_ERR_CORRUPT;
            else if (hH != align_up(kFixedHeader + kTensorRec * hT + kBlockRec * hB, kHeaderAlign)) code = BS_ERR_CORRUPT;
            else if (hH > p.nbytes || hP != p.nbytes - hH)        code = BS_ERR_CORRUPT;
            else if (hT > p.T || hB > p.B)                        code = BS_ERR_CAPACITY;  // out arrays too small
            else { T = hT; B = hB; hb = hH; P_hdr = hP; dtype = w1.x; }
            if (code == BS_ERR_CAPACITY) { /* report the counts so the caller can size its arrays */
                if (blockIdx.x == 0 && tid == 0) { head->n_tensors = (uint32_t)hT; head->n_blocks = (uint32_t)hB; }
            }
        }
        if (code != 0) {
            ok = false;
            if (blockIdx.x == 0 && tid == 0) set_status(head, code);
        }
    } else {
        hb = align_up(kFixedHeader + kTensorRec * T + kBlockRec * B, kHeaderAlign);
    }

    // ---- tensor records partition the block table in order (D5, D8) ------------------------------------
    if (ok) {
        for (uint64_t t = (uint64_t)blockIdx.x * kScanThreads + tid; t < T; t += (uint64_t)gridDim.x * kScanThreads) {
            TensorHead h = load_tensor<DESER>(p, t);
            uint64_t prev_end = 0;
            if (t > 0) {
                TensorHead q = load_tensor<DESER>(p, t - 1);
                prev_end = (uint64_t)q.first + q.n;
            }
            int code = 0;
            if (h.rank != 2 && h.rank != 3) code = kErrRank;
            else if (h.first != prev_end) code = kErrBad;
            else if (t == T - 1 && (uint64_t)h.first + h.n != B) code = kErrBad;
            else if (DESER && h.reserved != 0) code = kErrBad;
            set_status(head, code);
        }
        if (T == 0 && B != 0 && blockIdx.x == 0 && tid == 0) set_status(head, kErrBad);
        if (DESER && blockIdx.x == 0) {  // header slack must be zero
            uint64_t used = kFixedHeader + kTensorRec * T + kBlockRec * B;
            uint64_t z = used + 16ull * tid;
            if (z < hb) {
                uint4 w = __ldg(reinterpret_cast<const uint4*>(p.header + z));
                if ((w.x | w.y | w.z | w.w) != 0) set_status(head, BS_ERR_CORRUPT);
            }
        }
    }

    const uint64_t esize = elem_bytes(dtype);
    // ---- single-pass scan over tiles of kScanTile blocks -----------------------------------------------
    const uint64_t n_tiles = ok ? (B + kScanTile - 1) / kScanTile + (B == 0 ? 1 : 0) : 0;
    const unsigned char* brec = DESER ? p.header + kFixedHeader + kTensorRec * T : nullptr;
    for (;;) {
        __syncthreads();
        if (tid == 0) { s_tile = atomicAdd(&head->scan_ticket, 1u); s_big_n = 0; }
        __syncthreads();
        const uint64_t tile = s_tile;
        if (tile >= n_tiles) break;

        uint64_t val[kScanItems];      // what is scanned: stored size (SER) / pool slot size (DESER)
        uint64_t stored[kScanItems];   // align16(nbytes)
        uint64_t aux[kScanItems];      // SER: block address; DESER: payload offset from the record
        uint64_t dsta[kScanItems];     // DESER scatter: destination address
        uint32_t oddf[kScanItems];
        int err = 0;
        uint64_t tsum = 0;
#pragma unroll
        for (uint32_t k = 0; k < kScanItems; ++k) {
            const uint64_t i = tile * kScanTile + (uint64_t)tid * kScanItems + k;
            const bool valid = i < B;
            uint32_t d0 = 1, d1 = 1, d2 = 0;
            uint64_t a = 0, offset = 0;
            uint32_t owner = 0;
            int32_t q4 = 0, q5 = 0, q2 = 0, q3 = 0;
            if (valid) {
                if (DESER) {
                    const uint4* r = reinterpret_cast<const uint4*>(brec + kBlockRec * i);
                    uint4 r0 = __ldg(r), r1 = __ldg(r + 1), r2 = __ldg(r + 2);
                    q2 = (int32_t)r0.z; q3 = (int32_t)r0.w; q4 = (int32_t)r1.x; q5 = (int32_t)r1.y;
                    d0 = r1.z; d1 = r1.w; d2 = r2.x; owner = r2.y;
                    offset = (uint64_t)r2.z | ((uint64_t)r2.w << 32);
                } else {
                    d0 = __ldg(p.dim + 3 * i); d1 = __ldg(p.dim + 3 * i + 1); d2 = __ldg(p.dim + 3 * i + 2);
                    a = __ldg(reinterpret_cast<const unsigned long long*>(p.addr + i));
                }
            }
            // S1: nbytes = e * prod(dim) in u64 (D13), e = element size of the dtype; stored = align16(nbytes) (D3)
            uint64_t n01 = (uint64_t)d0 * d1;
            uint64_t n = n01 * d2;
            if (valid && (__umul64hi(n01, (uint64_t)d2) != 0 || n >= (1ull << 57))) { err = kErrBad; n = 0; }
            const uint64_t nbytes = n * esize;
            const uint64_t st = (nbytes + 15) & ~15ull;
            stored[k] = st;
            oddf[k] = (uint32_t)(st - nbytes) >> 2;  // pad code: 0..3 words of zero pad
            dsta[k] = 0;
            if (DESER) {
                aux[k] = offset;
                val[k] = valid ? align_up(nbytes, kPoolAlign) : 0;
                if (valid) {
                    // owner = the tensor whose block range holds i; unused legs: dim 1, labels 0
                    if (owner >= T) err = BS_ERR_CORRUPT;
                    else {
                        TensorHead h = load_tensor<true>(p, owner);
                        if (i < h.first || i >= (uint64_t)h.first + h.n) err = BS_ERR_CORRUPT;
                        if (h.rank == 2 && (d2 != 1 || q4 != 0 || q5 != 0)) err = BS_ERR_CORRUPT;
                        (void)q2; (void)q3;
                    }
                    // offsets = exclusive prefix sum of stored sizes, checked link by link, inside [0, P]
                    uint64_t next = P_hdr;
                    if (i + 1 < B) next = __ldg(reinterpret_cast<const unsigned long long*>(brec + kBlockRec * (i + 1) + 40));
                    if (i == 0 && offset != 0) err = BS_ERR_CORRUPT;
                    if (offset > P_hdr || st > P_hdr - offset || offset + st != next) err = BS_ERR_CORRUPT;
                    else if (st != nbytes && p.payload != nullptr) {  // pad bytes are zero: the last 16-byte unit of the block
                        const uint4 u = __ldg(reinterpret_cast<const uint4*>(p.payload + hb + offset + st - 16));
                        const uint32_t data_words = 4u - ((uint32_t)(st - nbytes) >> 2);
                        const uint32_t w[4] = {u.x, u.y, u.z, u.w};
                        uint32_t pad = 0;
#pragma unroll
                        for (uint32_t q = 0; q < 4; ++q) pad |= (q >= data_words) ? w[q] : 0u;
                        if (pad != 0) err = BS_ERR_CORRUPT;
                    }
                    if (p.flags == BS_SCATTER_TO_ADDR) {
                        if (__ldg(p.out_dim + 3 * i) != d0 || __ldg(p.out_dim + 3 * i + 1) != d1 ||
                            __ldg(p.out_dim + 3 * i + 2) != d2) { if (!err) err = BS_ERR_ARG; }
                        uint64_t da = __ldg(reinterpret_cast<const unsigned long long*>(p.out_addr + i));
                        if (da & 7) { if (!err) err = BS_ERR_ARG; }
                        dsta[k] = da;
                    }
                }
            } else {
                aux[k] = a;
                val[k] = valid ? st : 0;
                if (valid && (a & 7)) err = BS_ERR_ARG;  // D16
            }
            tsum += val[k];
        }
        if (err) set_status(head, err);

        // block-wide exclusive scan of tsum
        const uint64_t incl = warp_incl_scan(tsum, lane);
        if (lane == 31) s_warp_sum[warp] = incl;
        __syncthreads();
        if (warp == 0) {
            uint64_t ws = (lane < kScanThreads / 32) ? s_warp_sum[lane] : 0;
            const uint64_t agg = warp_sum(ws);
            uint64_t excl = 0;
            if (tile == 0) {
                if (lane == 0) st_release_u64(p.ws.scan_state, kFlagPrefix | agg);
            } else {
                if (lane == 0) st_release_u64(p.ws.scan_state + tile, kFlagAgg | agg);
                int64_t look = (int64_t)tile - 1;
                for (;;) {
                    const int64_t idx = look - (int64_t)lane;
                    uint64_t w = (idx >= 0) ? ld_acquire_u64(p.ws.scan_state + idx) : kFlagPrefix;
                    while (__any_sync(0xffffffffu, (w >> 62) == 0)) {
                        if ((w >> 62) == 0) w = ld_acquire_u64(p.ws.scan_state + idx);
                    }
                    const uint32_t is_prefix = __ballot_sync(0xffffffffu, (w >> 62) == 2);
                    const uint32_t first = is_prefix ? (uint32_t)__ffs((int)is_prefix) - 1u : 32u;
                    excl += warp_sum(lane <= first ? (w & kValMask) : 0ull);
                    if (is_prefix) break;
                    look -= 32;
                }
                if (lane == 0) st_release_u64(p.ws.scan_state + tile, kFlagPrefix | ((excl + agg) & kValMask));
            }
            if (lane == 0) { s_tile_prefix = excl; s_tile_total = agg; }
        }
        __syncthreads();
        uint64_t run = s_tile_prefix + (incl - tsum);
        for (uint32_t w = 0; w < warp; ++w) run += s_warp_sum[w];

        // blk[] table and tile_first[] boundaries
#pragma unroll
        for (uint32_t k = 0; k < kScanItems; ++k) {
            const uint64_t i = tile * kScanTile + (uint64_t)tid * kScanItems + k;
            if (i < B) {
                uint64_t off, address;
                if (DESER) {
                    off = aux[k];
                    address = (p.flags == BS_SCATTER_TO_ADDR) ? dsta[k] : p.pool_base + run;
                } else {
                    off = run;
                    address = aux[k];
                }
                Blk e;
                e.off = off;
                e.addr = (address & ~7ull) | oddf[k];
                p.ws.blk[i] = e;
                // granule boundaries g*kGranule inside [off, off + stored)
                const uint64_t g0 = (off + kGranule - 1) / kGranule;
                const uint64_t g1 = (off + stored[k] + kGranule - 1) / kGranule;
                if (g1 > g0) {
                    if (g1 - g0 <= kInlineBoundaries) {
                        for (uint64_t g = g0; g < g1; ++g)
                            if (g < p.ws.n_granules_cap) p.ws.tile_first[g] = (uint32_t)i;
                    } else {
                        uint32_t slot = atomicAdd(&s_big_n, 1u);
                        s_big_idx[slot] = (uint32_t)i;
                        s_big_g0[slot] = g0;
                        uint64_t cnt = g1 - g0;
                        s_big_cnt[slot] = cnt > 0xffffffffull ? 0xffffffffu : (uint32_t)cnt;
                    }
                }
            }
            run += val[k];
        }
        __syncthreads();
        // large blocks: one warp per block fills its boundaries; huge ones (> 2048 granules) take the whole CTA
        for (uint32_t s = warp; s < s_big_n; s += kScanThreads / 32) {
            const uint64_t g0 = s_big_g0[s];
            const uint32_t cnt = s_big_cnt[s], idx = s_big_idx[s];
            if (cnt > 2048) continue;
            for (uint64_t j = lane; j < cnt; j += 32)
                if (g0 + j < p.ws.n_granules_cap) p.ws.tile_first[g0 + j] = idx;
        }
        for (uint32_t s = 0; s < s_big_n; ++s) {
            const uint64_t g0 = s_big_g0[s];
            const uint32_t cnt = s_big_cnt[s], idx = s_big_idx[s];
            if (cnt <= 2048) continue;
            for (uint64_t j = tid; j < cnt; j += kScanThreads)
                if (g0 + j < p.ws.n_granules_cap) p.ws.tile_first[g0 + j] = idx;
        }
        if (tile == n_tiles - 1 && tid == 0) {  // the owner of the last tile knows the total
            const uint64_t total = s_tile_prefix + s_tile_total;
            if (DESER) head->pool_bytes = total; else head->payload_bytes = total;
        }
    }

    // ---- last CTA out: final checks, sentinel, result -----------------------------------------------------
    __shared__ uint32_t s_last;
    __syncthreads();
    if (tid == 0) {
        __threadfence();
        s_last = (atomicAdd(&head->ctas_done, 1u) == gridDim.x - 1) ? 1u : 0u;
    }
    __syncthreads();
    if (s_last && tid == 0) {
        __threadfence();
        volatile WsHead* vh = head;
        int status = vh->status;
        uint64_t P = DESER ? P_hdr : vh->payload_bytes;
        uint64_t pool = DESER ? vh->pool_bytes : 0;
        if (!ok) { P = 0; pool = 0; }
        const uint64_t total = hb + P;
        const uint64_t ng = (P + kGranule - 1) / kGranule;
        if (status == 0) {
            if (!DESER && total > p.capacity) status = BS_ERR_CAPACITY;
            else if (!DESER && p.expect_total != 0 && total != p.expect_total) status = BS_ERR_ARG;
            else if (ng + 1 > p.ws.n_granules_cap) status = BS_ERR_CAPACITY;
            else if (DESER && p.flags == BS_LAYOUT_POOL && pool > p.pool_bytes) status = BS_ERR_CAPACITY;
        }
        if (ok) {
            Blk e; e.off = P; e.addr = 0;
            p.ws.blk[B] = e;
            if (ng < p.ws.n_granules_cap) p.ws.tile_first[ng] = (uint32_t)B;
            vh->n_tensors = (uint32_t)T;
            vh->n_blocks = (uint32_t)B;
        }
        vh->header_bytes = hb;
        vh->dtype = dtype;
        vh->payload_bytes = P;
        vh->pool_bytes = pool;
        vh->n_granules = ng;
        vh->status = status;
        if (p.result != nullptr) {
            bs_result r;
            r.total_bytes = total; r.header_bytes = hb; r.payload_bytes = P; r.pool_bytes = pool;
            r.status = status; r.n_tensors = vh->n_tensors; r.n_blocks = vh->n_blocks;
            for (int z = 0; z < 5; ++z) r.reserved[z] = 0;
            r.reserved[2] = dtype;
            *p.result = r;
        }
        __threadfence();
    }
}

}  // namespace

cudaError_t launch_scan(bool deser, const ScanParams& p, int sm_count, cudaStream_t stream)
{
    // grid: enough CTAs to cover the tiles, at most a few per SM (tiles are claimed dynamically)
    uint64_t n_tiles = ((uint64_t)p.B + kScanTile - 1) / kScanTile + 1;
    uint64_t n_ttiles = ((uint64_t)p.T + kScanThreads - 1) / kScanThreads;
    uint64_t want = n_tiles > n_ttiles ? n_tiles : n_ttiles;
    uint64_t cap = (uint64_t)sm_count * 4;
    unsigned grid = (unsigned)(want < cap ? want : cap);
    if (grid == 0) grid = 1;
    if (deser) scan_kernel<true><<<grid, kScanThreads, 0, stream>>>(p);
    else scan_kernel<false><<<grid, kScanThreads, 0, stream>>>(p);
    return cudaGetLastError();
}

}  // namespace bs
