// bs_scan_phase.cuh — the size / offset pass as a device-side phase: steps S1, S2, S4 (serialize) and S6 (deserialize)
// of SURVEY §8(a).  Used by scan_kernel (bs_scan.cu: the pass alone) and by the fused kernels of bs_move_tma.cu (the
// pass and the data movement in ONE launch).
//
// "low cost and exact prediction of post-serialization data size before the actual serialization takes
// place ... let the main thread map the output buffer".  In the paper one CPU thread does this; here it is a
// single-pass chained (decoupled look-back) exclusive scan of the stored block sizes over all B blocks, which at the
// same time
//   - validates the descriptor (serialize) or every header field (deserialize: SURVEY §8(c) list),
//   - writes the blk[] table {payload offset, block address} = the "pointer structure" of L90-92,
//   - writes tile_first[] (which block holds the first byte of every 16 KiB payload granule) = the work partition
//     the data-movement code uses to give every worker an exact, disjoint stream interval,
//   - reports header / payload / total bytes and the deferred status in bs_result.
//
// Work is cut into ITEMS (item i = scan tile i of 1024 blocks + slice i of 1024 tensor records) that CTAs claim in
// order from one ticket; the CTA that completes the last item finalises (totals, capacity checks, sentinel, result).
// An item only ever waits (look-back) for items claimed before it, which are being executed
// by resident CTAs: forward progress needs no co-residency of the grid.
//
// No word the pass synchronises on needs clearing beforehand — the workspace may be uninitialised memory:
//   - every scan-state entry, the first-error word and the `ready` word carry the call's 40-bit EPOCH tag (a process-wide
//     counter handed out on the host); a word with another tag is "not written yet" whatever it holds;
//   - the three counters (items handed out, items completed, CTAs out of the item loop) carry a fixed IDLE tag and are
//     put back to {tag, 0} by the last CTA out of every launch, so a launch normally pays one atomic per count; a counter
//     that does not carry the tag (first use of the workspace) is re-based by whoever touches it first.
// (While a CUDA graph is being captured the host cannot hand out a fresh epoch per replay; the call then clears head +
// state in front of the kernel, as round 1 always did.)
//
// A set of at most 1024 blocks and 1024 tensors is ONE item: a fused kernel then runs it REPLICATED — every CTA computes
// the whole (tiny) table itself, identical values, and nobody waits for anybody; only CTA 0 writes head and result.
// Roofline: HBM-bound, ~20 B read and 16 B written per block — < 1 % of the payload traffic.
#pragma once
#include "bs_internal.cuh"

namespace bs {
namespace scan {

constexpr uint64_t kFlagAgg = 1ull << 62;
constexpr uint64_t kFlagPrefix = 2ull << 62;
constexpr uint64_t kValMask = (1ull << 62) - 1;
constexpr uint32_t kInlineBoundaries = 4;
constexpr uint64_t kCountMask = (1ull << 24) - 1;  // tagged words: [63:24] tag, [23:0] count / code
constexpr uint64_t kIdleTag = 0xB5C0DE5EEDull << 24;  // the counters' tag between launches

// what the data-movement code needs to know about the set once the pass is complete
struct HeadView {
    int32_t status;
    uint32_t T, B, dtype;  // dtype: element type | BS_ALIGN8
    uint64_t hb, P, ng;
};

struct __align__(16) Shared {
    uint64_t warp_sum[kScanItems * (kScanThreads / 32)];   // [row][warp]: sums in block order
    uint64_t warp_excl[kScanItems * (kScanThreads / 32)];  // their exclusive prefix inside the tile
    uint64_t tile_prefix, tile_total;
    uint64_t tot_payload, tot_pool;  // replicated mode: the totals stay in the CTA
    uint32_t item, big_n, last;
    int32_t err;                     // first error seen by this CTA
    HeadView out;                    // replicated mode / the finalising CTA: the outcome
    uint32_t big_idx[kScanTile];
    uint32_t big_cnt[kScanTile];
    uint64_t big_g0[kScanTile];
};

// the pass is run by threads 0 .. kScanThreads-1 of a CTA (a fused kernel may have more)
__device__ __forceinline__ void bar() { asm volatile("bar.sync 1, %0;" ::"n"(kScanThreads) : "memory"); }

__device__ __forceinline__ void ld_state(const ScanState* p, uint64_t* word, uint64_t* tag)
{
    asm volatile("ld.acquire.gpu.global.v2.u64 {%0, %1}, [%2];" : "=l"(*word), "=l"(*tag) : "l"(p) : "memory");
}
__device__ __forceinline__ void st_state(ScanState* p, uint64_t word, uint64_t tag)
{
    asm volatile("st.release.gpu.global.v2.u64 [%0], {%1, %2};" ::"l"(p), "l"(word), "l"(tag) : "memory");
}
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

// count before the increment, within the epoch of `tag`.  A word of another epoch (stale or never written) is re-based
// to {tag, 1} by whoever gets there first; increments that landed on the stale word are lost on purpose (nobody takes
// a number from them).  One atomic when the word is current; one add + one or two CAS on the first touch of a call.
__device__ __forceinline__ uint32_t tagged_inc(uint64_t* w, uint64_t tag)
{
    unsigned long long* a = reinterpret_cast<unsigned long long*>(w);
    unsigned long long old = atomicAdd(a, 1ull);
    if ((old & ~kCountMask) == tag) return (uint32_t)(old & kCountMask);
    unsigned long long cur = old + 1ull;
    for (;;) {
        if ((cur & ~kCountMask) == tag) {
            old = atomicAdd(a, 1ull);
            return (uint32_t)(old & kCountMask);
        }
        const unsigned long long prev = atomicCAS(a, cur, tag | 1ull);
        if (prev == cur) return 0u;
        cur = prev;
    }
}
__device__ __forceinline__ void post_err(WsHead* h, uint64_t tag, int code)  // first error of the epoch wins
{
    if (code == 0) return;
    unsigned long long* a = reinterpret_cast<unsigned long long*>(&h->ep_err);
    const unsigned long long want = tag | (unsigned long long)(uint32_t)(-code);
    unsigned long long cur = *reinterpret_cast<volatile unsigned long long*>(a);
    for (;;) {
        if ((cur & ~kCountMask) == tag && (cur & kCountMask) != 0) return;
        const unsigned long long prev = atomicCAS(a, cur, want);
        if (prev == cur) return;
        cur = prev;
    }
}
__device__ __forceinline__ int read_err(const WsHead* h, uint64_t tag)
{
    const uint64_t v = *reinterpret_cast<const volatile uint64_t*>(&h->ep_err);
    return ((v & ~kCountMask) == tag) ? -(int)(v & kCountMask) : 0;
}
__device__ __forceinline__ void cta_err(Shared& sm, int code)
{
    if (code != 0) atomicCAS(&sm.err, 0, code);
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
    const uint4* r = DESER ? reinterpret_cast<const uint4*>(p.header + kFixedHeader + kTensorRec * t)
                           : reinterpret_cast<const uint4*>(p.tensors + t);
    const uint4 a = __ldg(r), b = __ldg(r + 1);
    TensorHead h;
    h.rank = a.x; h.first = a.y; h.n = a.z; h.reserved = b.w;
    return h;
}

// uniform over the grid: derived from the call's arguments / the fixed header alone
struct Shape {
    uint64_t T, B, hb, P_hdr;
    uint64_t rep_T, rep_B;  // deserialize, out arrays too small: the stream's counts, reported so the caller can size them
    uint32_t dtype;         // element type (bs.h BS_F64 ..), without flags
    uint32_t align;         // 16, or 8 (BS_ALIGN8: stored sizes are rounded to 8 only, DESIGN.md §18 reading D19)
    uint32_t legs, rec;     // legs per block and bytes per block record: 3 / 48 (wire format v1), 4 / 64 (v3, BS_RANK4; D20)
    int code;               // != 0: the fixed header was rejected
    uint32_t n_tiles, n_items;
};

template <bool DESER>
__device__ __forceinline__ Shape shape_of(const ScanParams& p)
{
    Shape s;
    s.T = p.T; s.B = p.B; s.hb = 0; s.P_hdr = 0; s.rep_T = 0; s.rep_B = 0; s.code = 0;
    s.dtype = p.dtype & BS_DTYPE_MASK;
    s.align = (p.dtype & BS_ALIGN8) ? 8u : 16u;
    s.legs = legs_of(p.dtype);
    s.rec = block_rec_bytes(p.dtype);
    if (DESER) {  // the fixed header (SURVEY §8(c) checks, in order)
        s.T = s.B = 0;
        if (p.nbytes < kFixedHeader) {
            s.code = BS_ERR_CORRUPT;
        } else {
            const uint4* f = reinterpret_cast<const uint4*>(p.header);
            const uint4 w0 = __ldg(f), w1 = __ldg(f + 1), w2 = __ldg(f + 2), w3 = __ldg(f + 3);
            const uint64_t hT = (uint64_t)w2.x | ((uint64_t)w2.y << 32), hB = (uint64_t)w2.z | ((uint64_t)w2.w << 32);
            const uint64_t hH = (uint64_t)w3.x | ((uint64_t)w3.y << 32), hP = (uint64_t)w3.z | ((uint64_t)w3.w << 32);
            if (w0.x != 0x41505342u || w0.y != 0x31455352u)      s.code = BS_ERR_CORRUPT;  // "BSPARSE1"
            else if (w0.z != 1u && w0.z != 3u)                    s.code = BS_ERR_CORRUPT;  // version: 1, or 3 (four legs)
            else if (w0.w != 0x01020304u)                         s.code = BS_ERR_CORRUPT;  // endian_tag
            else if (w1.x > (uint32_t)BS_C128)                    s.code = BS_ERR_CORRUPT;  // dtype
            else if (w1.y != 2u)                                  s.code = BS_ERR_CORRUPT;  // n_qn
            else if (w1.z != (w0.z == 3u ? 4u : 3u))              s.code = BS_ERR_CORRUPT;  // max_rank
            else if (w1.w != 16u && !(w1.w == 8u && w0.z == 1u))  s.code = BS_ERR_CORRUPT;  // align (8: wire format v1 only)
            else if ((w0.z == 3u) != (s.legs == 4u))              s.code = BS_ERR_ARG;      // the out arrays have the other shape
            else if (w1.w == 8u && (p.flags & kFlagNoAlign8))     s.code = BS_ERR_UNSUPPORTED;  // the LDG variant moves 16-byte units
            else if (hT >= (1ull << 32) || hB >= (1ull << 32))   s.code = BS_ERR_CORRUPT;
            else if (hH != align_up(kFixedHeader + kTensorRec * hT + (uint64_t)s.rec * hB, kHeaderAlign)) s.code = BS_ERR_CORRUPT;
            else if (hH > p.nbytes || hP != p.nbytes - hH)        s.code = BS_ERR_CORRUPT;
            else if (hT > p.T || hB > p.B) { s.code = BS_ERR_CAPACITY; s.rep_T = hT; s.rep_B = hB; }  // out arrays too small
            else { s.T = hT; s.B = hB; s.hb = hH; s.P_hdr = hP; s.dtype = w1.x; s.align = w1.w; }
        }
    } else {
        s.hb = align_up(kFixedHeader + kTensorRec * s.T + (uint64_t)s.rec * s.B, kHeaderAlign);
    }
    const uint64_t nt = (s.B + kScanTile - 1) / kScanTile, ntt = (s.T + kScanTile - 1) / kScanTile;
    s.n_tiles = s.code ? 0u : (uint32_t)(nt ? nt : 1);
    s.n_items = s.code ? 1u : (uint32_t)(nt > ntt ? (nt ? nt : 1) : (ntt ? ntt : 1));  // a rejected header still needs its result written
    return s;
}

// number of items of a call, from the host's view (an upper bound for deserialize, where the counts are capacities)
inline uint32_t host_items(uint64_t T, uint64_t B)
{
    const uint64_t nt = (B + kScanTile - 1) / kScanTile, ntt = (T + kScanTile - 1) / kScanTile;
    const uint64_t n = nt > ntt ? nt : ntt;
    return (uint32_t)(n ? n : 1);
}

// ---- slice `item` of the tensor records: they partition the block table in order (D5, D8) ------------------------------
template <bool DESER>
__device__ __forceinline__ void tensor_slice(const ScanParams& p, const Shape& s, uint32_t item, Shared& sm)
{
    constexpr int kErrBad = DESER ? BS_ERR_CORRUPT : BS_ERR_ARG;
    constexpr int kErrRank = DESER ? BS_ERR_CORRUPT : BS_ERR_UNSUPPORTED;
    const uint32_t tid = threadIdx.x;
    int code = 0;
#pragma unroll
    for (uint32_t k = 0; k < kScanItems; ++k) {
        const uint64_t t = (uint64_t)item * kScanTile + (uint64_t)k * kScanThreads + tid;
        if (t < s.T) {
            const TensorHead h = load_tensor<DESER>(p, t);
            uint64_t prev_end = 0;
            if (t > 0) {
                const TensorHead q = load_tensor<DESER>(p, t - 1);
                prev_end = (uint64_t)q.first + q.n;
            }
            if (h.rank < 2 || h.rank > s.legs) code = kErrRank;
            else if (h.first != prev_end) code = kErrBad;
            else if (t == s.T - 1 && (uint64_t)h.first + h.n != s.B) code = kErrBad;
            else if (DESER && h.reserved != 0) code = kErrBad;
        }
    }
    if (item == 0) {
        if (s.T == 0 && s.B != 0 && tid == 0) code = kErrBad;
        if (DESER) {  // header slack must be zero
            const uint64_t used = kFixedHeader + kTensorRec * s.T + (uint64_t)s.rec * s.B;
            const uint64_t z = used + 16ull * tid;
            if (z < s.hb) {
                const uint4 w = __ldg(reinterpret_cast<const uint4*>(p.header + z));
                if ((w.x | w.y | w.z | w.w) != 0) code = BS_ERR_CORRUPT;
            }
        }
    }
    cta_err(sm, code);
}

// ---- scan tile `tile` of the block table.  REPL: the tile is the whole table and the CTA is on its own (no chain) --------
template <bool DESER, bool REPL>
__device__ __forceinline__ void block_tile(const ScanParams& p, const Shape& s, uint64_t tile, uint64_t tag, Shared& sm)
{
    const uint32_t tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    constexpr int kErrBad = DESER ? BS_ERR_CORRUPT : BS_ERR_ARG;
    const uint64_t T = s.T, B = s.B, hb = s.hb, P_hdr = s.P_hdr;
    const uint64_t esize = elem_bytes(s.dtype);
    const uint64_t amask = s.align - 1;  // S1: stored = align_up(nbytes, align), align = 16 (D3) or 8 (D19)
    const unsigned char* brec = DESER ? p.header + kFixedHeader + kTensorRec * T : nullptr;

    uint64_t val[kScanItems];      // what is scanned: stored size (SER) / pool slot size (DESER)
    uint64_t stored[kScanItems];   // align16(nbytes)
    uint64_t aux[kScanItems];      // SER: block address; DESER: payload offset from the record
    uint64_t dsta[kScanItems];     // DESER scatter: destination address
    uint32_t oddf[kScanItems];
    int err = 0;
#pragma unroll
    for (uint32_t k = 0; k < kScanItems; ++k) {
        const uint64_t i = tile * kScanTile + (uint64_t)k * kScanThreads + tid;  // row k of the tile: consecutive lanes, consecutive blocks
        const bool valid = i < B;
        uint32_t d0 = 1, d1 = 1, d2 = 0, d3 = 1;
        uint64_t a = 0, offset = 0;
        uint32_t owner = 0;
        uint32_t unused3 = 0, unused4 = 0;  // DESER: what must be {dim 1, labels 0} on leg 3 / leg 4 if the tensor does not use it
        if (valid) {
            if (DESER) {
                const uint4* r = reinterpret_cast<const uint4*>(brec + (uint64_t)s.rec * i);
                if (s.legs == 3) {  // i32 qn[3][2]; u32 dim[3]; u32 tensor; u64 offset
                    const uint4 r1 = __ldg(r + 1), r2 = __ldg(r + 2);
                    d0 = r1.z; d1 = r1.w; d2 = r2.x; owner = r2.y;
                    offset = (uint64_t)r2.z | ((uint64_t)r2.w << 32);
                    unused3 = (d2 ^ 1u) | r1.x | r1.y;
                } else {            // i32 qn[4][2]; u32 dim[4]; u32 tensor; u32 reserved; u64 offset
                    const uint4 r1 = __ldg(r + 1), r2 = __ldg(r + 2), r3 = __ldg(r + 3);
                    d0 = r2.x; d1 = r2.y; d2 = r2.z; d3 = r2.w; owner = r3.x;
                    offset = (uint64_t)r3.z | ((uint64_t)r3.w << 32);
                    unused3 = (d2 ^ 1u) | r1.x | r1.y;
                    unused4 = (d3 ^ 1u) | r1.z | r1.w;
                    if (r3.y != 0) err = BS_ERR_CORRUPT;  // reserved
                }
            } else {
                const uint32_t* d = p.dim + (uint64_t)s.legs * i;
                d0 = __ldg(d); d1 = __ldg(d + 1); d2 = __ldg(d + 2);
                if (s.legs == 4) d3 = __ldg(d + 3);
                a = __ldg(reinterpret_cast<const unsigned long long*>(p.addr + i));
            }
        }
        // S1: nbytes = e * prod(dim) in u64 (D13), e = element size of the dtype; stored = align_up(nbytes, align) (D3, D19)
        const uint64_t n01 = (uint64_t)d0 * d1, n23 = (uint64_t)d2 * d3;
        uint64_t n = n01 * n23;
        if (valid && (__umul64hi(n01, n23) != 0 || n >= (1ull << 57))) { err = kErrBad; n = 0; }
        const uint64_t nbytes = n * esize;
        const uint64_t st = (nbytes + amask) & ~amask;
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
                    const TensorHead h = load_tensor<true>(p, owner);
                    if (i < h.first || i >= (uint64_t)h.first + h.n) err = BS_ERR_CORRUPT;
                    if ((h.rank < 3 && unused3 != 0) || (h.rank < 4 && unused4 != 0)) err = BS_ERR_CORRUPT;
                }
                // offsets = exclusive prefix sum of stored sizes, checked link by link, inside [0, P]
                uint64_t next = P_hdr;
                if (i + 1 < B) next = __ldg(reinterpret_cast<const unsigned long long*>(brec + (uint64_t)s.rec * (i + 2) - 8));
                if (i == 0 && offset != 0) err = BS_ERR_CORRUPT;
                if (offset > P_hdr || st > P_hdr - offset || offset + st != next) err = BS_ERR_CORRUPT;
                else if (st != nbytes && p.payload != nullptr) {  // pad bytes are zero: the 1..3 words behind the block's data
                    const uint32_t* w = reinterpret_cast<const uint32_t*>(p.payload + hb + offset + nbytes);
                    uint32_t pad = 0;
                    for (uint32_t q = 0; q < (uint32_t)(st - nbytes) >> 2; ++q) pad |= __ldg(w + q);
                    if (pad != 0) err = BS_ERR_CORRUPT;
                }
                if ((p.flags & 1u) == BS_SCATTER_TO_ADDR) {
                    const uint32_t* od = p.out_dim + (uint64_t)s.legs * i;
                    if (__ldg(od) != d0 || __ldg(od + 1) != d1 || __ldg(od + 2) != d2 || (s.legs == 4 && __ldg(od + 3) != d3)) {
                        if (!err) err = BS_ERR_ARG;
                    }
                    const uint64_t da = __ldg(reinterpret_cast<const unsigned long long*>(p.out_addr + i));
                    if (da & 7) { if (!err) err = BS_ERR_ARG; }
                    dsta[k] = da;
                }
            }
        } else {
            aux[k] = a;
            val[k] = valid ? st : 0;
            if (valid && (a & 7)) err = BS_ERR_ARG;  // D16
        }
    }
    cta_err(sm, err);

    // block-wide exclusive scan in block order — row 0 of all threads, then row 1, ... (a thread's blocks lie kScanThreads
    // apart so that a warp's loads and table stores touch consecutive addresses) — chained to the earlier tiles
    static_assert(kScanItems * (kScanThreads / 32) == 32, "one warp scans the (row, warp) sums");
    uint64_t incl[kScanItems];
#pragma unroll
    for (uint32_t k = 0; k < kScanItems; ++k) {
        incl[k] = warp_incl_scan(val[k], lane);
        if (lane == 31) sm.warp_sum[k * (kScanThreads / 32) + warp] = incl[k];
    }
    if (tid == 0) sm.big_n = 0;
    bar();
    if (warp == 0) {
        const uint64_t ws = sm.warp_sum[lane];                 // lane = row * 8 + warp: block order
        const uint64_t ws_incl = warp_incl_scan(ws, lane);
        const uint64_t agg = __shfl_sync(0xffffffffu, ws_incl, 31);
        sm.warp_excl[lane] = ws_incl - ws;
        uint64_t excl = 0;
        if (!REPL) {
            if (tile == 0) {
                if (lane == 0) st_state(p.ws.scan_state, kFlagPrefix | agg, tag);
            } else {
                if (lane == 0) st_state(p.ws.scan_state + tile, kFlagAgg | agg, tag);
                int64_t look = (int64_t)tile - 1;
                for (;;) {
                    const int64_t idx = look - (int64_t)lane;
                    uint64_t w = kFlagPrefix, wt = tag;  // lanes in front of tile 0: an empty prefix
                    if (idx >= 0) ld_state(p.ws.scan_state + idx, &w, &wt);
                    while (__any_sync(0xffffffffu, wt != tag || (w >> 62) == 0)) {
                        if (wt != tag || (w >> 62) == 0) ld_state(p.ws.scan_state + idx, &w, &wt);
                    }
                    const uint32_t is_prefix = __ballot_sync(0xffffffffu, (w >> 62) == 2);
                    const uint32_t first = is_prefix ? (uint32_t)__ffs((int)is_prefix) - 1u : 32u;
                    excl += warp_sum(lane <= first ? (w & kValMask) : 0ull);
                    if (is_prefix) break;
                    look -= 32;
                }
                if (lane == 0) st_state(p.ws.scan_state + tile, kFlagPrefix | ((excl + agg) & kValMask), tag);
            }
        }
        if (lane == 0) { sm.tile_prefix = excl; sm.tile_total = agg; }
    }
    bar();

    // blk[] table and tile_first[] boundaries
#pragma unroll
    for (uint32_t k = 0; k < kScanItems; ++k) {
        const uint64_t i = tile * kScanTile + (uint64_t)k * kScanThreads + tid;
        const uint64_t run = sm.tile_prefix + sm.warp_excl[k * (kScanThreads / 32) + warp] + (incl[k] - val[k]);
        if (i < B) {
            uint64_t off, address;
            if (DESER) {
                off = aux[k];
                address = ((p.flags & 1u) == BS_SCATTER_TO_ADDR) ? dsta[k] : p.pool_base + run;
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
                    const uint32_t slot = atomicAdd(&sm.big_n, 1u);
                    sm.big_idx[slot] = (uint32_t)i;
                    sm.big_g0[slot] = g0;
                    const uint64_t cnt = g1 - g0;
                    sm.big_cnt[slot] = cnt > 0xffffffffull ? 0xffffffffu : (uint32_t)cnt;
                }
            }
        }
    }
    bar();
    // large blocks: one warp per block fills its boundaries; huge ones (> 2048 granules) take all the scan threads
    const uint32_t big_n = sm.big_n;
    for (uint32_t q = warp; q < big_n; q += kScanThreads / 32) {
        const uint64_t g0 = sm.big_g0[q];
        const uint32_t cnt = sm.big_cnt[q], idx = sm.big_idx[q];
        if (cnt > 2048) continue;
        for (uint64_t j = lane; j < cnt; j += 32)
            if (g0 + j < p.ws.n_granules_cap) p.ws.tile_first[g0 + j] = idx;
    }
    for (uint32_t q = 0; q < big_n; ++q) {
        const uint64_t g0 = sm.big_g0[q];
        const uint32_t cnt = sm.big_cnt[q], idx = sm.big_idx[q];
        if (cnt <= 2048) continue;
        for (uint64_t j = tid; j < cnt; j += kScanThreads)
            if (g0 + j < p.ws.n_granules_cap) p.ws.tile_first[g0 + j] = idx;
    }
    if (tile == s.n_tiles - 1 && tid == 0) {  // the owner of the last tile knows the total
        const uint64_t total = sm.tile_prefix + sm.tile_total;
        if (REPL) {
            if (DESER) sm.tot_pool = total; else sm.tot_payload = total;
        } else {
            volatile WsHead* vh = p.ws.head;
            if (DESER) vh->pool_bytes = total; else vh->payload_bytes = total;
        }
    }
}

// ---- one thread, once every item is complete: final checks, sentinel, head, result -------------------------------------------
// write_head: this CTA owns the workspace head and the result (always, but for CTAs other than 0 of a replicated pass)
template <bool DESER, bool REPL>
__device__ __forceinline__ void finalize(const ScanParams& p, const Shape& s, int status, Shared& sm, bool write_head)
{
    volatile WsHead* vh = p.ws.head;
    const bool ok = s.code == 0;
    uint64_t P = DESER ? s.P_hdr : (REPL ? sm.tot_payload : vh->payload_bytes);
    uint64_t pool = DESER ? (REPL ? sm.tot_pool : vh->pool_bytes) : 0;
    if (!ok) { P = 0; pool = 0; }
    const uint64_t hb = s.hb, B = s.B;
    const uint64_t total = hb + P;
    const uint64_t ng = (P + kGranule - 1) / kGranule;
    if (status == 0) {
        // no block carries the link check `offset + stored == next`, so an empty table must own an empty payload
        if (DESER && ok && B == 0 && s.P_hdr != 0) status = BS_ERR_CORRUPT;
        else if (!DESER && total > p.capacity) status = BS_ERR_CAPACITY;
        else if (!DESER && p.expect_total != 0 && total != p.expect_total) status = BS_ERR_ARG;
        else if (ng + 1 > p.ws.n_granules_cap) status = BS_ERR_CAPACITY;
        else if (DESER && (p.flags & 1u) == BS_LAYOUT_POOL && pool > p.pool_bytes) status = BS_ERR_CAPACITY;
    }
    if (ok) {
        Blk e; e.off = P; e.addr = 0;
        p.ws.blk[B] = e;
        if (ng < p.ws.n_granules_cap) p.ws.tile_first[ng] = (uint32_t)B;
    }
    HeadView hv;
    hv.status = status; hv.T = (uint32_t)(ok ? s.T : s.rep_T); hv.B = (uint32_t)(ok ? B : s.rep_B);
    hv.dtype = s.dtype | (s.align == 8u ? BS_ALIGN8 : 0u) | (s.legs == 4u ? BS_RANK4 : 0u);
    hv.hb = hb; hv.P = P; hv.ng = ng;
    sm.out = hv;
    if (!write_head) return;
    vh->n_tensors = hv.T;
    vh->n_blocks = hv.B;
    vh->header_bytes = hb;
    vh->dtype = hv.dtype;
    vh->payload_bytes = P;
    vh->pool_bytes = pool;
    vh->n_granules = ng;
    vh->status = status;
    if (p.result != nullptr) {
        bs_result r;
        r.total_bytes = total; r.header_bytes = hb; r.payload_bytes = P; r.pool_bytes = pool;
        r.status = status; r.n_tensors = hv.T; r.n_blocks = hv.B;
        for (int z = 0; z < 5; ++z) r.reserved[z] = 0;
        r.reserved[2] = hv.dtype;
        *p.result = r;
    }
}

// One thread per CTA, when the CTA is done with the launch's counters.  Every CTA has its last (out of range) ticket by the
// time the last one is here: that one puts the counters back for the next launch.  A fused kernel calls this when the CTA
// has SEEN the completion count (wait_done): the last CTA to say so resets ep_done, and by then nobody polls it any more.
__device__ __forceinline__ void leave(const ScanParams& p, uint64_t tag)
{
    (void)tag;
    WsHead* head = p.ws.head;
    if (tagged_inc(&head->ep_exit, kIdleTag) == gridDim.x - 1) {
        volatile uint64_t* c = &head->ep_ticket;
        *c = kIdleTag;
        c = &head->ep_done;
        *c = kIdleTag;
        c = &head->ep_exit;
        *c = kIdleTag;
        __threadfence();
    }
}

// The pass, run by threads 0 .. kScanThreads-1 of every CTA of the grid.  Returns with those threads synchronised.
// replicated (fused kernels only; s.n_items == 1): sm.out holds the outcome on return, nothing to wait for.
template <bool DESER>
__device__ __forceinline__ void run(const ScanParams& p, const Shape& s, uint64_t tag, Shared& sm, bool replicated, bool defer_exit = false)
{
    const uint32_t tid = threadIdx.x;
    WsHead* head = p.ws.head;
    if (tid == 0) sm.err = 0;
    bar();
    if (replicated) {
        if (s.code == 0) {
            tensor_slice<DESER>(p, s, 0, sm);
            block_tile<DESER, true>(p, s, 0, tag, sm);
        }
        bar();
        if (tid == 0) finalize<DESER, true>(p, s, s.code ? s.code : sm.err, sm, blockIdx.x == 0);
        __threadfence_block();  // the table this CTA wrote is read back by its own data-movement warps
        bar();
        return;
    }
    for (;;) {
        bar();
        if (tid == 0) sm.item = tagged_inc(&head->ep_ticket, kIdleTag);
        bar();
        const uint32_t item = sm.item;
        if (item >= s.n_items) break;
        if (s.code == 0) {  // the block tile first: later tiles look back at its aggregate
            if (item < s.n_tiles) block_tile<DESER, false>(p, s, item, tag, sm);
            if ((uint64_t)item * kScanTile < s.T || item == 0) tensor_slice<DESER>(p, s, item, sm);
        }
        bar();
        if (tid == 0) {
            const int code = s.code ? s.code : sm.err;
            if (code) post_err(head, tag, code);
            __threadfence();  // this item's table entries and its error are visible before it counts as done
            if (tagged_inc(&head->ep_done, kIdleTag) == s.n_items - 1) {  // every item is complete: finalise
                __threadfence();
                finalize<DESER, false>(p, s, read_err(head, tag), sm, true);
                __threadfence();
            }
        }
    }
    if (!defer_exit && tid == 0) leave(p, tag);
}

// fused kernels, after run(): wait until every item of the pass is complete (one thread per CTA polls the completion
// count, which a fused kernel leaves standing until its end), then work the outcome out HERE, from the shape every CTA
// derived for itself, the totals the last tile's owner left and the epoch's error word — the CTA that completed the last
// item writes the workspace head and the caller's result meanwhile, and nobody waits for it (round 2: ~2.5 us per call).
template <bool DESER>
__device__ __forceinline__ HeadView wait_done(const ScanParams& p, const Shape& s, uint64_t tag, Shared& sm, HeadView* s_out)
{
    if (threadIdx.x == 0) {
        const WsHead* head = p.ws.head;
        uint32_t ns = 32;
        for (;;) {
            const uint64_t w = ld_acquire_u64(&head->ep_done);
            if ((w & ~kCountMask) == kIdleTag && (w & kCountMask) >= s.n_items) break;
            __nanosleep(ns);
            if (ns < 256) ns *= 2;
        }
        finalize<DESER, false>(p, s, read_err(head, tag), sm, false);  // also writes the two sentinels (everybody: same values)
        *s_out = sm.out;
        __threadfence();
    }
    __syncthreads();
    return *s_out;
}

}  // namespace scan
}  // namespace bs
