// bs_move.cu — the data-movement kernels: steps S3 + S5 (header write + pack) and S7 (descriptor rebuild +
// unpack / scatter) of SURVEY §8(a).
//
// once the output buffer is mapped, "all threads serialize in parallel and in complete
// independence. Yet, together they produce a single, continuos stream of bytes".  Here the unit of
// independence is a TILE of the stream (tile_bytes, a multiple of the 16 KiB granule): tile k of the payload is
// stream bytes [header_bytes + k*tile_bytes, +tile_bytes), whatever blocks happen to lie in it.  A persistent
// grid of CTAs walks the tiles; tile_first[] says which block the tile starts in, blk[] gives every block's
// {payload offset, device address}.  So the work per CTA is uniform no matter how skewed the block sizes are
// (0.5 KiB .. 1 MiB in the paper-shaped sets), the stream side of every access is perfectly contiguous, and a
// byte range [lo,hi) of the stream (one 256 MiB offload segment, PAPER Fig 4(b)) is just a range of tiles.
//
// Roofline: pure data movement — 1 byte read + 1 byte written per stream byte, HBM-bound.
//
// Variant LDG (this file, variant 1): every thread moves 16-byte units with vector loads / stores
// (ld.global.cs.v4 / st.global.cs.v4), UPT units in flight per thread.
// Variant TMA (bs_move_tma.cu, variant 2): cp.async.bulk global<->shared staging.
#include <string.h>

#include "bs_move_common.cuh"

namespace bs {

namespace {

constexpr uint32_t kThreads = 256;

__device__ __forceinline__ uint4 ld_stream16(const void* p) { return __ldcs(reinterpret_cast<const uint4*>(p)); }
__device__ __forceinline__ uint2 ld_stream8(const void* p) { return __ldcs(reinterpret_cast<const uint2*>(p)); }
__device__ __forceinline__ void st_stream16(void* p, uint4 v) { __stcs(reinterpret_cast<uint4*>(p), v); }
__device__ __forceinline__ void st_stream8(void* p, uint2 v) { __stcs(reinterpret_cast<uint2*>(p), v); }

// largest j in [jlo, jhi] with blk[j].off <= s   (zero-size blocks share an offset with their successor: the
// last of such a run is the one that owns byte s)
__device__ __forceinline__ uint32_t find_block(const Blk* __restrict__ blk, uint32_t jlo, uint32_t jhi, uint64_t s)
{
    while (jlo < jhi) {
        const uint32_t mid = jlo + ((jhi - jlo + 1) >> 1);
        if (__ldg(reinterpret_cast<const unsigned long long*>(&blk[mid].off)) <= s) jlo = mid; else jhi = mid - 1;
    }
    return jlo;
}

template <bool UNPACK, int UPT>
__global__ void __launch_bounds__(kThreads) move_kernel(const MoveParams p)
{
    const WsHead* head = p.ws.head;
    if (head->status != 0) {  // deferred error: nothing is written (the engine has a stale header blanked, see kFlagPoisonOnError)
        if (!UNPACK) poison_on_error(p);
        return;
    }
    if (head->dtype & BS_ALIGN8) {
        // tables of an unpadded stream (a range call behind a pass that ran for the TMA variant): this variant moves 16-byte
        // units and would scatter blocks that sit 8 off that grid wrongly.  Nothing is written; the workspace says why.
        // (Every CTA has read status == 0 above or returns here all the same: the store cannot change another CTA's path.)
        if (blockIdx.x == 0 && threadIdx.x == 0) const_cast<WsHead*>(head)->status = BS_ERR_UNSUPPORTED;
        return;
    }
    const uint32_t T = head->n_tensors, B = head->n_blocks;
    const uint64_t hb = head->header_bytes, P = head->payload_bytes, total = hb + P;
    const uint64_t ng = head->n_granules;
    const uint64_t lo = p.lo, hi = p.hi < total ? p.hi : total;
    const uint32_t tid = threadIdx.x;
    constexpr uint64_t kTileUnits = (uint64_t)kThreads * UPT;
    constexpr uint64_t kTileBytes = kTileUnits * 16;

    // ---- header tiles ----
    uint64_t nh = 0;
    if (UNPACK) {
        if (p.header != nullptr) nh = (n_rebuild_records(p, head) + kTileUnits - 1) / kTileUnits;
    } else if (lo < hb && lo < hi) {
        nh = ((hi < hb ? hi : hb) - lo + kTileBytes - 1) / kTileBytes;
    }
    // ---- payload tiles: tile k = payload bytes [k*kTileBytes, (k+1)*kTileBytes) ----
    uint64_t plo = 0, phi = 0, k0 = 0, np = 0;
    if (hi > hb && hi > lo && B != 0) {  // no block, no payload tile (the scan rejects a payload without blocks)
        plo = (lo > hb ? lo : hb) - hb;
        phi = hi - hb;
        k0 = plo / kTileBytes;
        np = (phi + kTileBytes - 1) / kTileBytes - k0;
    }
    const Blk* __restrict__ blk = p.ws.blk;

    for (uint64_t w = blockIdx.x; w < nh + np; w += gridDim.x) {
        if (w >= np) {
            const uint64_t h = w - np;
            if (UNPACK) {
#pragma unroll
                for (int k = 0; k < UPT; ++k) rebuild_record_any(p, head, h * kTileUnits + (uint64_t)k * kThreads + tid);
            } else {
                const uint64_t hend = hi < hb ? hi : hb;
#pragma unroll
                for (int k = 0; k < UPT; ++k) {
                    const uint64_t s = lo + (h * kTileUnits + (uint64_t)k * kThreads + tid) * 16;
                    if (s < hend) st_stream16(stream_at(p, hb, s), header_unit_any(p, s >> 4, T, B, hb, P));
                }
            }
            continue;
        }
        const uint64_t tile = k0 + w;
        const uint64_t tbase = tile * kTileBytes;
        const uint64_t g0 = tbase / kGranule;
        uint64_t g1 = (tbase + kTileBytes) / kGranule;
        if (g1 > ng) g1 = ng;
        const uint32_t jlo = __ldg(p.ws.tile_first + g0);
        uint32_t jhi = __ldg(p.ws.tile_first + g1);  // tile_first[ng] == B
        if (jhi >= B) jhi = B - 1;

        const uint64_t tfirst = tbase > plo ? tbase : plo;  // first payload byte of the tile inside [lo, hi)
        unsigned char* const tile_ptr = stream_at(p, hb, hb + tfirst) - (tfirst - tbase);  // where payload byte tbase would lie
        uint64_t src[UPT];   // pack: block address of the unit; unpack: destination address
        uint32_t kind[UPT];  // 0 skip, 1 full 16 B aligned, 2 full 16 B as 2x8, 4 / 8 / 12: tail unit of that many data bytes (+ zero pad)
        uint64_t soff[UPT];
#pragma unroll
        for (int k = 0; k < UPT; ++k) {
            const uint64_t s = tbase + ((uint64_t)k * kThreads + tid) * 16;  // payload offset of the unit
            soff[k] = s;
            kind[k] = 0;
            src[k] = 0;
            if (s >= plo && s < phi) {
                const uint32_t j = find_block(blk, jlo, jhi, s);
                const Blk e = blk[j];
                const uint64_t next = __ldg(reinterpret_cast<const unsigned long long*>(&blk[j + 1].off));
                const uint64_t intra = s - e.off;
                const uint64_t nbytes = (next - e.off) - (e.addr & 3ull) * 4;
                const uint64_t a = (e.addr & ~7ull) + intra;
                src[k] = a;
                kind[k] = (intra + 16 <= nbytes) ? ((a & 15ull) ? 2u : 1u) : (uint32_t)(nbytes - intra);
            }
        }
        if (!UNPACK) {
            uint4 v[UPT];
#pragma unroll
            for (int k = 0; k < UPT; ++k) {
                v[k] = make_uint4(0, 0, 0, 0);
                if (kind[k] == 1) v[k] = ld_stream16(reinterpret_cast<const void*>(src[k]));
                else if (kind[k] == 2) {
                    uint2 a = ld_stream8(reinterpret_cast<const void*>(src[k]));
                    uint2 b = ld_stream8(reinterpret_cast<const void*>(src[k] + 8));
                    v[k] = make_uint4(a.x, a.y, b.x, b.y);
                } else if (kind[k] == 8) {
                    uint2 a = ld_stream8(reinterpret_cast<const void*>(src[k]));
                    v[k] = make_uint4(a.x, a.y, 0u, 0u);  // 8 data bytes + 8 zero pad bytes (D3)
                } else if (kind[k] != 0) {                // f32 blocks: 4 or 12 data bytes
                    const uint32_t* w = reinterpret_cast<const uint32_t*>(src[k]);
                    v[k].x = __ldcs(w);
                    if (kind[k] == 12) { v[k].y = __ldcs(w + 1); v[k].z = __ldcs(w + 2); }
                }
            }
#pragma unroll
            for (int k = 0; k < UPT; ++k)
                if (kind[k]) st_stream16(tile_ptr + (soff[k] - tbase), v[k]);
        } else {
            uint4 v[UPT];
#pragma unroll
            for (int k = 0; k < UPT; ++k)
                if (kind[k]) v[k] = ld_stream16(tile_ptr + (soff[k] - tbase));
#pragma unroll
            for (int k = 0; k < UPT; ++k) {
                if (kind[k] == 1) st_stream16(reinterpret_cast<void*>(src[k]), v[k]);
                else if (kind[k] == 2) {
                    st_stream8(reinterpret_cast<void*>(src[k]), make_uint2(v[k].x, v[k].y));
                    st_stream8(reinterpret_cast<void*>(src[k] + 8), make_uint2(v[k].z, v[k].w));
                } else if (kind[k] == 8) {
                    st_stream8(reinterpret_cast<void*>(src[k]), make_uint2(v[k].x, v[k].y));
                    if ((p.flags & kFlagCheckPad) && (v[k].z | v[k].w) != 0)
                        atomicCAS(const_cast<int*>(&head->status), 0, BS_ERR_CORRUPT);
                } else if (kind[k] != 0) {                // f32 blocks: 4 or 12 data bytes
                    uint32_t* w = reinterpret_cast<uint32_t*>(src[k]);
                    __stcs(w, v[k].x);
                    if (kind[k] == 12) { __stcs(w + 1, v[k].y); __stcs(w + 2, v[k].z); }
                    const uint32_t z = kind[k] == 12 ? v[k].w : (v[k].y | v[k].z | v[k].w);
                    if ((p.flags & kFlagCheckPad) && z != 0) atomicCAS(const_cast<int*>(&head->status), 0, BS_ERR_CORRUPT);
                }
            }
        }
    }
}

// persistent grid: exactly one wave of resident CTAs (SM count x occupancy), tiles dealt round-robin
template <bool UNPACK, int UPT>
cudaError_t launch_ldg_upt(const MoveParams& p, const bs_opts& o, int sm_count, cudaStream_t stream)
{
    static int occ = 0;  // per kernel instantiation
    if (occ == 0) {
        int n = 0;
        cudaError_t e = cudaOccupancyMaxActiveBlocksPerMultiprocessor(&n, move_kernel<UNPACK, UPT>, (int)kThreads, 0);
        if (e != cudaSuccess) return e;
        occ = n > 0 ? n : 1;
    }
    unsigned per_sm = (unsigned)occ;
    if (o.ctas_per_sm && o.ctas_per_sm < per_sm) per_sm = o.ctas_per_sm;
    move_kernel<UNPACK, UPT><<<(unsigned)sm_count * per_sm, kThreads, 0, stream>>>(p);
    return cudaGetLastError();
}

template <bool UNPACK>
cudaError_t launch_ldg(const MoveParams& p, const bs_opts& o, int sm_count, cudaStream_t stream)
{
    switch (o.tile_bytes) {
        case 16384: return launch_ldg_upt<UNPACK, 4>(p, o, sm_count, stream);
        case 32768: return launch_ldg_upt<UNPACK, 8>(p, o, sm_count, stream);
        case 49152: return launch_ldg_upt<UNPACK, 12>(p, o, sm_count, stream);
        case 65536: return launch_ldg_upt<UNPACK, 16>(p, o, sm_count, stream);
        default: return cudaErrorInvalidValue;
    }
}

}  // namespace

void resolve_opts(const bs_opts* in, bs_opts* out)
{
    bs_opts o;
    memset(&o, 0, sizeof(o));
    if (in) o = *in;
    if (o.variant == BS_VARIANT_DEFAULT) o.variant = BS_VARIANT_TMA;
    if (o.variant == BS_VARIANT_TMA) {
        // tile_bytes == stages == warps == 0 stays 0: launch_move_tma uses its per-direction preset
        if (o.tile_bytes || o.stages || o.warps) {
            if (o.tile_bytes == 0) o.tile_bytes = 16384;
            if (o.stages == 0) o.stages = 3;
            if (o.warps == 0) {  // ~96 KiB of loads in flight per SM
                o.warps = (96u * 1024u) / ((o.stages - 1) * o.tile_bytes);
                while (o.warps > 1 && (uint64_t)o.warps * ((uint64_t)o.stages * o.tile_bytes + kMetaBytesPerWarp) > 216u * 1024u) --o.warps;
                o.warps = o.warps < 1 ? 1 : (o.warps > 16 ? 16 : o.warps);
            }
        }
    } else {
        if (o.tile_bytes == 0) o.tile_bytes = 16384;
    }
    *out = o;
}

cudaError_t launch_move(bool unpack, const MoveParams& p, const bs_opts& opts, int sm_count, cudaStream_t stream)
{
    if (opts.variant == BS_VARIANT_TMA) return launch_move_tma(unpack, p, opts, sm_count, stream);
    return unpack ? launch_ldg<true>(p, opts, sm_count, stream) : launch_ldg<false>(p, opts, sm_count, stream);
}

}  // namespace bs
