// bs_move_tma.cu — data movement through the TMA bulk-copy engine: steps S3 + S5 (header write + pack) and
// S7 (descriptor rebuild + unpack / scatter) of SURVEY §8(a), variant BS_VARIANT_TMA.
//
// every worker owns an exact, disjoint interval of the one output buffer and fills it "in complete
// independence".  Here a worker is one WARP and its interval is a TILE of the stream (tile_bytes of payload,
// whatever blocks lie in it; see bs_move.cu for why tiles and not blocks are the unit).  A tile never touches the
// register file:
//
//   pack   : for every block segment inside the tile, one lane issues   cp.async.bulk global -> shared
//            (completion counted in bytes on the stage's mbarrier); the 8 data bytes + 8 zero pad bytes that end
//            an odd-sized block are one zero-filling 16-byte cp.async; when the stage is full ONE
//            cp.async.bulk shared -> global writes the whole tile (the stream side is contiguous).
//   unpack : ONE cp.async.bulk global -> shared brings the tile in; then one cp.async.bulk shared -> global per
//            block segment; the last 8 bytes of an odd-sized block are a plain 8-byte store (the pad bytes of
//            the stream must not be written past the end of a destination block).
//
// Each warp runs its own ring of `stages` tiles in dynamic shared memory (software pipeline: tile i is loaded while
// tile i-(stages-2) is stored), `warps` rings per CTA, one persistent CTA per SM; the warps of the grid claim tiles
// from one counter in the workspace head (round 2, "tile hand-out" below; small ranges: dealt round-robin).  Blocks
// whose address is only 8-byte aligned take a correct slower path of 8-byte cp.async / 8-byte stores.
// The stream produced is byte-identical to the LDG variant's (tests: P6).
//
// Roofline: pure data movement — 1 byte read + 1 byte written per stream byte, HBM-bound; ~2 instructions per
// block segment and per tile instead of ~70 per 512 bytes in the LDG variant.
#include <atomic>

#include "bs_move_common.cuh"
#include "bs_scan_phase.cuh"

#ifdef BS_PHASE_PROF  // development build only (build.py extra=["-DBS_PHASE_PROF"]): cycles per loop phase, summed over warps
__device__ unsigned long long g_bs_phase[8];
extern "C" int bs_debug_phases(unsigned long long* out8, int reset)
{
    if (out8 && cudaMemcpyFromSymbol(out8, g_bs_phase, sizeof(g_bs_phase)) != cudaSuccess) return -1;
    if (reset) { unsigned long long z[8] = {0}; if (cudaMemcpyToSymbol(g_bs_phase, z, sizeof(z)) != cudaSuccess) return -1; }
    return 0;
}
#define BS_PH(k) { const long long t_ = clock64(); ph_acc[k] += (unsigned long long)(t_ - ph_prev); ph_prev = t_; }
#else
#define BS_PH(k)
#endif

namespace bs {

namespace {

constexpr uint32_t kMaxWarps = 16;   // data warps; one more warp per CTA works on the header
constexpr uint32_t kMaxStages = 8;
constexpr uint32_t kSmemLimit = 227u * 1024u;
constexpr uint32_t kStaticSmem = 2048u;  // room for the kernels' static shared memory (mbarriers, the pass's outcome)

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes)
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity)
{
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity)
        : "memory");
    return ok != 0;
}
// Bounded: a phase that never completes (the byte count announced with expect_tx and the copies issued disagree — the
// one piece of arithmetic the pack path does per tile) must not hang the GPU.  try_wait itself blocks for a
// hardware-defined slice, so 2^22 rounds are seconds, far beyond any real wait; then the call fails with BS_ERR_CUDA
// in the workspace status (what was written so far is unspecified) and the warp stops.
__device__ __forceinline__ bool mbar_wait(uint32_t bar, uint32_t parity, int* status)
{
    for (uint32_t spin = 0; spin < (1u << 22); ++spin)
        if (mbar_try_wait(bar, parity)) return true;
    atomicCAS(status, 0, BS_ERR_CUDA);
    return false;
}
// the mbarrier also waits for every cp.async this thread has issued so far (pending count +1 now, -1 on completion)
__device__ __forceinline__ void cp_async_mbar_arrive(uint32_t bar)
{
    asm volatile("cp.async.mbarrier.arrive.shared::cta.b64 [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void bulk_g2s(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g(void* dst, uint32_t src, uint32_t bytes)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group [%0], [%1], %2;" ::"l"(dst), "r"(src), "r"(bytes) : "memory");
}
__device__ __forceinline__ void bulk_g2s_hint(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, uint64_t pol)
{
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes.L2::cache_hint [%0], [%1], %2, [%3], %4;" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar), "l"(pol)
                 : "memory");
}
__device__ __forceinline__ void bulk_s2g_hint(void* dst, uint32_t src, uint32_t bytes, uint64_t pol)
{
    asm volatile("cp.async.bulk.global.shared::cta.bulk_group.L2::cache_hint [%0], [%1], %2, %3;" ::"l"(dst), "r"(src), "r"(bytes),
                 "l"(pol)
                 : "memory");
}
__device__ __forceinline__ uint64_t policy_evict_first()
{
    uint64_t pol;
    asm volatile("createpolicy.fractional.L2::evict_first.b64 %0, 1.0;" : "=l"(pol));
    return pol;
}
struct Hints {  // MoveParams.tune: bit 0 = L2 evict_first on bulk loads, bit 1 = on bulk stores
    uint64_t pol;
    bool ld, st;
};
__device__ __forceinline__ void bulk_g2s_x(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar, const Hints& h)
{
    if (h.ld) bulk_g2s_hint(dst, src, bytes, bar, h.pol); else bulk_g2s(dst, src, bytes, bar);
}
__device__ __forceinline__ void bulk_s2g_x(void* dst, uint32_t src, uint32_t bytes, const Hints& h)
{
    if (h.st) bulk_s2g_hint(dst, src, bytes, h.pol); else bulk_s2g(dst, src, bytes);
}
__device__ __forceinline__ void bulk_commit() { asm volatile("cp.async.bulk.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void bulk_wait_read()
{
    asm volatile("cp.async.bulk.wait_group.read %0;" ::"n"(N) : "memory");
}
__device__ __forceinline__ void fence_proxy_async() { asm volatile("fence.proxy.async.shared::cta;" ::: "memory"); }
// `data` bytes (4, 8 or 12) + zeros up to 16: the last unit of a padded block
__device__ __forceinline__ void cp_async_tail16(uint32_t dst, const void* src, uint32_t data)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 16, %2;" ::"r"(dst), "l"(src), "r"(data) : "memory");
}
__device__ __forceinline__ void cp_async_8(uint32_t dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 8;" ::"r"(dst), "l"(src) : "memory");
}

__device__ __forceinline__ void cp_async_4(uint32_t dst, const void* src)
{
    asm volatile("cp.async.ca.shared.global [%0], [%1], 4;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_16(uint32_t dst, const void* src)
{
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(dst), "l"(src) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N>
__device__ __forceinline__ void cp_async_wait()
{
    asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory");
}

struct Seg {          // intersection of one block with one tile, payload coordinates
    uint64_t lo;      // first payload byte
    uint32_t bulk;    // bytes movable as one 16-byte-granular copy (whole 16-byte units of block data)
    uint32_t tail;    // != 0: the segment ends with the last 16-byte unit of a padded block = `tail` data bytes (4, 8, 12) + zeros
    uint64_t addr;    // device address of the block byte that maps to payload byte `lo`
};

// block entry (e, next = offset of block j+1) clipped to [tlo, thi).  Returns false when the intersection is empty
// (zero-size blocks, clipped tiles).
__device__ __forceinline__ bool clip_seg(const Blk& e, uint64_t next, uint64_t tlo, uint64_t thi, Seg* s)
{
    const uint64_t lo = e.off > tlo ? e.off : tlo;
    const uint64_t hi = next < thi ? next : thi;
    if (hi <= lo) return false;
    const uint32_t pad = (uint32_t)(e.addr & 3ull) * 4u;  // zero pad bytes behind the block's data (D3)
    s->lo = lo;
    s->addr = (e.addr & ~7ull) + (lo - e.off);
    s->tail = (pad != 0 && hi == next) ? 16u - pad : 0u;
    s->bulk = (uint32_t)(hi - lo) - (s->tail ? 16u : 0u);
    return true;
}
__device__ __forceinline__ bool make_seg(const Blk* __restrict__ blk, uint32_t j, uint64_t tlo, uint64_t thi, Seg* s)
{
    // L2 loads: in a fused kernel other CTAs wrote the table during this launch
    const uint4 w = __ldcg(reinterpret_cast<const uint4*>(blk + j));
    Blk e;
    e.off = (uint64_t)w.x | ((uint64_t)w.y << 32);
    e.addr = (uint64_t)w.z | ((uint64_t)w.w << 32);
    const uint64_t next = __ldcg(reinterpret_cast<const unsigned long long*>(&blk[j + 1].off));
    return clip_seg(e, next, tlo, thi, s);
}

// Per-warp metadata in shared memory, filled by cp.async ahead of use (no register is tied up, no warp stalls).  The
// block table is read once per tile and never cached (the data streaming past evicts it), so each of the two lookup
// levels costs a DRAM round trip — about as long as a whole loop iteration of a warp.  `ahead` iterations (1 or 2) lie
// between the fetch of a tile's table entries and their use, and as many again between the fetch of its tile_first[] pair
// and that:
//   tf[2*ahead+1][2]  tile_first[] pair {jlo, jhi_raw} of tiles m .. m+2*ahead (slot = tile index mod the count)
//   blk[ahead+1][34]  block table entries jlo .. jlo+32 of tiles m .. m+ahead
// With ahead = 1 one round trip per iteration stays exposed and spaces the warp's loads; that is how round 1 ran, and why
// its best shapes were narrow peaks (see "pacing" below).  Paced launches use ahead = 2: nothing but the pace spaces them.
constexpr uint32_t kBlkAheadMax = 2;
constexpr uint32_t kBlkSlots = kBlkAheadMax + 1, kTfSlots = 2 * kBlkAheadMax + 1;
constexpr uint32_t kMetaBlk = 34;
constexpr uint32_t kTqSlots = 16;            // tile numbers of a warp's iterations i, slot i & 15 (claimed ahead, kept until stored)
constexpr uint32_t kNoTile = 0xFFFFFFFFu;
static_assert((kMaxStages - 2) + 2 * kBlkAheadMax + 1 <= kTqSlots, "a claimed tile stays queued from its claim (2 * ahead iterations early) to its store (lag late)");
constexpr uint32_t kMetaBytes = (kBlkSlots * kMetaBlk * 16 + kTfSlots * 8 + kTqSlots * 4 + 15) / 16 * 16;
static_assert(kMetaBytes <= kMetaBytesPerWarp, "check_opts (bs_api.cu) budgets kMetaBytesPerWarp of shared memory per warp");

// pack: stage one block segment.  Bulk part: counted in *tx, issued later (after the expect_tx); 8-byte-aligned
// blocks (D16) and odd tails: cp.async now.  Returns the number of cp.async groups this lane started.
__device__ __forceinline__ uint32_t pack_seg_async(const Seg& s, uint32_t d, uint32_t* tx)
{
    uint32_t n_async = 0;
    if (s.addr & 15ull) {  // D16 slow path: 8-byte pieces (a last 4-byte one for f32); the pad is plain shared stores
        const uint32_t nb = s.bulk + s.tail;
        for (uint32_t b = 0; b + 8 <= nb; b += 8) cp_async_8(d + b, reinterpret_cast<const void*>(s.addr + b));
        if (nb & 4u) cp_async_4(d + (nb & ~7u), reinterpret_cast<const void*>(s.addr + (nb & ~7u)));
        n_async += nb ? 1u : 0u;
        if (s.tail) {
            for (uint32_t b = s.tail; b < 16u; b += 4)
                asm volatile("st.shared.u32 [%0], %1;" ::"r"(d + s.bulk + b), "r"(0u) : "memory");
            fence_proxy_async();
        }
    } else {
        *tx += s.bulk;
        if (s.tail) {
            cp_async_tail16(d + s.bulk, reinterpret_cast<const void*>(s.addr + s.bulk), s.tail);
            ++n_async;
        }
    }
    return n_async;
}

// unpack: scatter one block segment out of the staged tile
__device__ __forceinline__ void unpack_seg(const Seg& s, uint32_t saddr, const unsigned char* sp, uint32_t flags, int* status,
                                           const Hints& h)
{
    if (s.addr & 15ull) {  // D16 slow path: 8-byte stores
        for (uint32_t b = 0; b < s.bulk; b += 8)
            *reinterpret_cast<uint64_t*>(s.addr + b) = *reinterpret_cast<const uint64_t*>(sp + b);
    } else if (s.bulk) {
        bulk_s2g_x(reinterpret_cast<void*>(s.addr), saddr, s.bulk, h);
    }
    if (s.tail) {  // `tail` data bytes; the pad bytes stay in the stream
        const uint4 v = *reinterpret_cast<const uint4*>(sp + s.bulk);
        if (s.tail == 8u) {
            *reinterpret_cast<uint2*>(s.addr + s.bulk) = make_uint2(v.x, v.y);
            if ((flags & kFlagCheckPad) && (v.z | v.w) != 0) atomicCAS(status, 0, BS_ERR_CORRUPT);
        } else {  // f32 blocks: 4 or 12 data bytes
            uint32_t* o = reinterpret_cast<uint32_t*>(s.addr + s.bulk);
            o[0] = v.x;
            if (s.tail == 12u) { o[1] = v.y; o[2] = v.z; }
            const uint32_t z = s.tail == 12u ? v.w : (v.y | v.z | v.w);
            if ((flags & kFlagCheckPad) && z != 0) atomicCAS(status, 0, BS_ERR_CORRUPT);
        }
    }
}

// ==== align = 8 streams (bs.h BS_ALIGN8; DESIGN.md §18 reading D19) ===========================================================
// Stored sizes are rounded to 8 bytes only, so a block may start 8 bytes off the 16-byte grid of the stream.  The bulk-copy
// engine needs source, destination and size on that grid: a segment whose two sides agree modulo 16 moves an 8-byte head
// (if it starts off the grid), its 16-byte-aligned body as ONE bulk copy and a short rest; a segment whose sides DISAGREE
// moves as 8-byte words, spread over the whole warp.  Kept out of line: the align-16 path above is unchanged.
struct Seg8 {
    uint64_t lo;    // first payload byte
    uint32_t n;     // data bytes (a multiple of 4)
    uint32_t pad;   // zero bytes behind them (f32 only: 4), when the segment ends its block
    uint64_t addr;  // device address of the block byte that maps to payload byte `lo`
};
__device__ __forceinline__ bool clip_seg8(const Blk& e, uint64_t next, uint64_t tlo, uint64_t thi, Seg8* s)
{
    const uint64_t lo = e.off > tlo ? e.off : tlo;
    const uint64_t hi = next < thi ? next : thi;
    if (hi <= lo) return false;
    const uint32_t pad = (hi == next) ? (uint32_t)(e.addr & 3ull) * 4u : 0u;
    s->lo = lo;
    s->addr = (e.addr & ~7ull) + (lo - e.off);
    s->n = (uint32_t)(hi - lo) - pad;
    s->pad = pad;
    return true;
}
__device__ __forceinline__ Blk load_blk(const Blk* __restrict__ blk, uint32_t j, uint64_t* next)
{
    const uint4 w = __ldcg(reinterpret_cast<const uint4*>(blk + j));
    Blk e;
    e.off = (uint64_t)w.x | ((uint64_t)w.y << 32);
    e.addr = (uint64_t)w.z | ((uint64_t)w.w << 32);
    *next = __ldcg(reinterpret_cast<const unsigned long long*>(&blk[j + 1].off));
    return e;
}
struct TileCtx {
    uint64_t tbase, tlo, thi;  // the tile and its part inside the call's range, payload coordinates
    uint32_t sbase, bar;       // shared address of the stage, its mbarrier
    uint32_t jlo, jhi, lane;   // blocks jlo .. jhi touch the tile
    const Blk* blk;
    Blk e0;                    // the lane's own block (jlo + lane), prefetched
    uint64_t next0;
};
__device__ __forceinline__ uint64_t shfl_u64(uint64_t v, uint32_t src)
{
    const uint32_t lo = __shfl_sync(0xffffffffu, (uint32_t)v, src), hi = __shfl_sync(0xffffffffu, (uint32_t)(v >> 32), src);
    return ((uint64_t)hi << 32) | lo;
}
// split of a co-aligned segment that lands at shared / global offset d: head (0 or 8 bytes up to the grid), body (bulk)
__device__ __forceinline__ void split8(uint32_t d, uint32_t n, uint32_t* head, uint32_t* body)
{
    *head = ((d & 8u) && n >= 8u) ? 8u : 0u;
    *body = (n - *head) & ~15u;
}

// pack, align 8: stage every segment of the tile; returns with the bulk copies issued
__device__ __noinline__ void pack_tile_a8(const TileCtx c)
{
    const uint32_t lane = c.lane;
    uint32_t tx = 0, n_async = 0;
    Seg8 s0;
    s0.lo = 0; s0.n = 0; s0.pad = 0; s0.addr = 0;
    const bool have0 = clip_seg8(c.e0, c.next0, c.tlo, c.thi, &s0);
    const uint32_t d0 = c.sbase + (uint32_t)(s0.lo - c.tbase);
    const bool co0 = have0 && (((uint32_t)s0.addr ^ d0) & 15u) == 0;
    uint32_t head0 = 0, body0 = 0;
    auto small_parts = [&](const Seg8& s, uint32_t d, uint32_t head, uint32_t body) {  // everything of a co-aligned segment but its body
        if (head) { cp_async_8(d, reinterpret_cast<const void*>(s.addr)); ++n_async; }
        uint32_t off = head + body;
        const uint32_t rest = s.n - off;
        if (rest & 8u) { cp_async_8(d + off, reinterpret_cast<const void*>(s.addr + off)); off += 8; ++n_async; }
        if (rest & 4u) { cp_async_4(d + off, reinterpret_cast<const void*>(s.addr + off)); ++n_async; }
    };
    auto zero_pad = [&](const Seg8& s, uint32_t d) {
        if (s.pad) {
            for (uint32_t b = 0; b < s.pad; b += 4) asm volatile("st.shared.u32 [%0], %1;" ::"r"(d + s.n + b), "r"(0u) : "memory");
            fence_proxy_async();
        }
    };
    if (co0) {
        split8(d0, s0.n, &head0, &body0);
        tx += body0;
        small_parts(s0, d0, head0, body0);
    }
    if (have0) zero_pad(s0, d0);
    // segments whose two sides disagree modulo 16: 8-byte words, the whole warp on each
    uint32_t mis = __ballot_sync(0xffffffffu, have0 && !co0);
    while (mis) {
        const uint32_t l = (uint32_t)__ffs((int)mis) - 1u;
        mis &= mis - 1u;
        const uint64_t a = shfl_u64(s0.addr, l);
        const uint32_t d = __shfl_sync(0xffffffffu, d0, l), n = __shfl_sync(0xffffffffu, s0.n, l);
        for (uint32_t b = lane * 8u; b + 8u <= n; b += 256u) cp_async_8(d + b, reinterpret_cast<const void*>(a + b));
        if ((n & 4u) && lane == 0) cp_async_4(d + (n & ~7u), reinterpret_cast<const void*>(a + (n & ~7u)));
        ++n_async;
    }
    if (c.jhi >= c.jlo + 32) {  // more than 32 blocks in the tile: small blocks, each lane on its own
        for (uint32_t j = c.jlo + lane + 32; j <= c.jhi; j += 32) {
            uint64_t next;
            const Blk e = load_blk(c.blk, j, &next);
            Seg8 s;
            if (!clip_seg8(e, next, c.tlo, c.thi, &s)) continue;
            const uint32_t d = c.sbase + (uint32_t)(s.lo - c.tbase);
            if ((((uint32_t)s.addr ^ d) & 15u) == 0) {
                uint32_t head, body;
                split8(d, s.n, &head, &body);
                tx += body;
                small_parts(s, d, head, body);
            } else {
                for (uint32_t b = 0; b + 8u <= s.n; b += 8u) cp_async_8(d + b, reinterpret_cast<const void*>(s.addr + b));
                if (s.n & 4u) cp_async_4(d + (s.n & ~7u), reinterpret_cast<const void*>(s.addr + (s.n & ~7u)));
                ++n_async;
            }
            zero_pad(s, d);
        }
    }
    if (n_async) cp_async_mbar_arrive(c.bar);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) tx += __shfl_xor_sync(0xffffffffu, tx, d);
    __syncwarp();  // every lane's cp.async arrival is registered before the phase can complete
    if (lane == 0) mbar_arrive_expect_tx(c.bar, tx);
    __syncwarp();
    if (co0 && body0) bulk_g2s(d0 + head0, reinterpret_cast<const void*>(s0.addr + head0), body0, c.bar);
    if (c.jhi >= c.jlo + 32) {
        for (uint32_t j = c.jlo + lane + 32; j <= c.jhi; j += 32) {
            uint64_t next;
            const Blk e = load_blk(c.blk, j, &next);
            Seg8 s;
            if (!clip_seg8(e, next, c.tlo, c.thi, &s)) continue;
            const uint32_t d = c.sbase + (uint32_t)(s.lo - c.tbase);
            uint32_t head, body;
            split8(d, s.n, &head, &body);
            if ((((uint32_t)s.addr ^ d) & 15u) == 0 && body) bulk_g2s(d + head, reinterpret_cast<const void*>(s.addr + head), body, c.bar);
        }
    }
}

// a tile <-> the stream, align 8: only the last tile of a stream can be 8 bytes off a multiple of 16
__device__ __forceinline__ void store_tile_a8(unsigned char* dst, uint32_t src, uint32_t n)  // one lane
{
    const uint32_t nb = n & ~15u;
    if (nb) bulk_s2g(dst, src, nb);
    if (n & 8u) {
        uint64_t v;
        asm volatile("ld.shared.u64 %0, [%1];" : "=l"(v) : "r"(src + nb) : "memory");
        *reinterpret_cast<uint64_t*>(dst + nb) = v;
    }
}
__device__ __forceinline__ void load_tile_a8(uint32_t dst, const unsigned char* src, uint32_t n, uint32_t bar)  // one lane
{
    const uint32_t nb = n & ~15u;
    if (n & 8u) {
        cp_async_8(dst + nb, src + nb);
        cp_async_mbar_arrive(bar);
    }
    mbar_arrive_expect_tx(bar, nb);
    if (nb) bulk_g2s(dst, src, nb, bar);
}

// unpack, align 8: scatter every segment of the staged tile (sp: generic pointer to the stage)
__device__ __noinline__ void unpack_tile_a8(const TileCtx c, const unsigned char* sp, uint32_t flags, int* status)
{
    const uint32_t lane = c.lane;
    auto check_pad = [&](const Seg8& s, const unsigned char* q) {
        if (s.pad && (flags & kFlagCheckPad)) {
            uint32_t z = 0;
            for (uint32_t b = 0; b < s.pad; b += 4) z |= *reinterpret_cast<const uint32_t*>(q + s.n + b);
            if (z != 0) atomicCAS(status, 0, BS_ERR_CORRUPT);
        }
    };
    auto co_parts = [&](const Seg8& s, uint32_t d, const unsigned char* q) {  // a co-aligned segment
        uint32_t head, body;
        split8(d, s.n, &head, &body);
        if (head) *reinterpret_cast<uint64_t*>(s.addr) = *reinterpret_cast<const uint64_t*>(q);
        if (body) bulk_s2g(reinterpret_cast<void*>(s.addr + head), d + head, body);
        uint32_t off = head + body;
        const uint32_t rest = s.n - off;
        if (rest & 8u) { *reinterpret_cast<uint64_t*>(s.addr + off) = *reinterpret_cast<const uint64_t*>(q + off); off += 8; }
        if (rest & 4u) *reinterpret_cast<uint32_t*>(s.addr + off) = *reinterpret_cast<const uint32_t*>(q + off);
    };
    Seg8 s0;
    s0.lo = 0; s0.n = 0; s0.pad = 0; s0.addr = 0;
    const bool have0 = clip_seg8(c.e0, c.next0, c.tlo, c.thi, &s0);
    const uint32_t off0 = (uint32_t)(s0.lo - c.tbase);
    const uint32_t d0 = c.sbase + off0;
    const bool co0 = have0 && (((uint32_t)s0.addr ^ d0) & 15u) == 0;
    if (co0) co_parts(s0, d0, sp + off0);
    if (have0) check_pad(s0, sp + off0);
    uint32_t mis = __ballot_sync(0xffffffffu, have0 && !co0);
    while (mis) {
        const uint32_t l = (uint32_t)__ffs((int)mis) - 1u;
        mis &= mis - 1u;
        const uint64_t a = shfl_u64(s0.addr, l);
        const uint32_t o = __shfl_sync(0xffffffffu, off0, l), n = __shfl_sync(0xffffffffu, s0.n, l);
        for (uint32_t b = lane * 8u; b + 8u <= n; b += 256u)
            *reinterpret_cast<uint64_t*>(a + b) = *reinterpret_cast<const uint64_t*>(sp + o + b);
        if ((n & 4u) && lane == 0) *reinterpret_cast<uint32_t*>(a + (n & ~7u)) = *reinterpret_cast<const uint32_t*>(sp + o + (n & ~7u));
    }
    if (c.jhi >= c.jlo + 32) {
        for (uint32_t j = c.jlo + lane + 32; j <= c.jhi; j += 32) {
            uint64_t next;
            const Blk e = load_blk(c.blk, j, &next);
            Seg8 s;
            if (!clip_seg8(e, next, c.tlo, c.thi, &s)) continue;
            const uint32_t o = (uint32_t)(s.lo - c.tbase), d = c.sbase + o;
            if ((((uint32_t)s.addr ^ d) & 15u) == 0) {
                co_parts(s, d, sp + o);
            } else {
                for (uint32_t b = 0; b + 8u <= s.n; b += 8u)
                    *reinterpret_cast<uint64_t*>(s.addr + b) = *reinterpret_cast<const uint64_t*>(sp + o + b);
                if (s.n & 4u) *reinterpret_cast<uint32_t*>(s.addr + (s.n & ~7u)) = *reinterpret_cast<const uint32_t*>(sp + o + (s.n & ~7u));
            }
            check_pad(s, sp + o);
        }
    }
}

// Default launch shapes (B200, measured; profiles/r02b_summary.md).  The launch always has the small-set shape — three rings
// of 3 stages x 16 KiB per SM, what sets of tens of MB run fastest with in both directions — and the kernel, which knows the
// payload size, switches sets of half a GB and more to ONE ring of 3 x 48 KiB in the same shared memory.  With tiles handed
// out by a counter (below) every shape that keeps ~96 KiB of loads in flight per SM reaches the same plateau (pack 6.75,
// unpack 6.9 TB/s); one warp per SM issues a third of the instructions.  A package map keeps the small shape unless its size
// limit is a multiple of the large tile.
struct Preset {
    uint32_t tile_bytes, stages, warps;
};

// ---- tile hand-out (round 2; profiles/r02b_summary.md "the cliff") -----------------------------------------------------------
// Round 1 dealt tiles round-robin: warp w of W took tiles w, w + W, ...  Measured in round 2: when the launch asks the memory
// system for more than it can give, the SMs are NOT served evenly (some fall 5-10 % behind), and with a static deal the
// launch lasts as long as its slowest SM — every shape showed a narrow peak with a cliff behind it (offered 1-2 % more
// traffic than the peak, a launch LOST 5-12 %), and round 1's shapes sat near their peaks by accident (the table round
// trip and the instruction overhead of an iteration happened to space a warp's loads about right).  Now tiles are handed
// out by ONE counter in the workspace head: a warp claims its next tile two iterations before it needs the tile's block
// table, an SM that is served faster simply takes more tiles, all SMs finish together, and an over-subscribed launch runs
// at the capacity of the memory system instead of falling off it.  The counter needs no clearing: it carries a tag like
// the pass's counters, the last warp out of a launch puts it back, a stale word (never used, or left by a killed launch) is
// claimed by CAS.
// Round 3: the counter is no longer a word of the caller's workspace.  bs_serialize_range / bs_deserialize_range run on the
// workspace the pass left its tables in, and issuing the ranges of one stream on two CUDA streams is the natural use: with
// one counter in the head two such launches drew tile numbers from the same word — tiles skipped, status BS_OK.  Each
// launch now gets its own {ticket, exit} pair from a ring in the library's device memory, indexed by a host-issued launch
// number (MoveParams.mv_slot), and the movement kernels only READ the workspace again, as in round 1.  Two launches share
// a pair only if kMvSlots counter-dealt launches (each >= 128 MiB of movement) are issued while one of them is still running.
constexpr uint32_t kMvSlots = 1024;
struct __align__(16) MvCtr {
    uint64_t ticket;  // tiles handed out: [63:32] tag, [31:0] count
    uint64_t exit;    // data warps that have left the launch; the last one puts both back
};
__device__ MvCtr g_mv_ctr[kMvSlots];
constexpr uint64_t kMvTag = 0x4D76C1A5ull << 32;  // [63:32] tag of the two move counters between and during launches, [31:0] count
// take `n` numbers from tagged counter `w`: returns the first
__device__ __forceinline__ uint32_t mv_take(uint64_t* w, uint32_t n)
{
    unsigned long long* a = reinterpret_cast<unsigned long long*>(w);
    unsigned long long old = atomicAdd(a, (unsigned long long)n);
    if ((old >> 32) == (kMvTag >> 32)) return (uint32_t)old;
    unsigned long long cur = old + n;  // a stale word: whoever gets there first makes it {tag, n}; adds that landed on it are lost
    for (;;) {
        if ((cur >> 32) == (kMvTag >> 32)) return (uint32_t)atomicAdd(a, (unsigned long long)n);
        const unsigned long long prev = atomicCAS(a, cur, kMvTag | n);
        if (prev == cur) return 0u;
        cur = prev;
    }
}
#ifdef BS_PHASE_PROF
__device__ unsigned int g_bs_trig[4];
__device__ unsigned int g_bs_hist[2][32];
__device__ unsigned long long g_bs_tl[160][8];
#define BS_TL(k) if (threadIdx.x == 0 && blockIdx.x < 160) { unsigned long long t_; asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t_)); g_bs_tl[blockIdx.x][k] = t_; }
#else
#define BS_TL(k)
#endif

__host__ __device__ inline Preset preset_small() { return Preset{16384, 3, 3}; }
__host__ __device__ inline Preset preset_large(bool) { return Preset{49152, 3, 1}; }
constexpr uint64_t kLargePayload = 512ull << 20;
constexpr uint64_t kDynamicBytes = 128ull << 20;  // ranges of this size and more: tiles handed out by the counter

// FUSED: called behind the size / offset pass inside one kernel (fused_tma_kernel); `hv` is that pass's outcome.
template <bool UNPACK, bool FUSED>
__device__ __forceinline__ void move_tma_body(const MoveParams& p, const scan::HeadView& hv, const uint32_t opt_stages,
                                              const uint32_t opt_warps, unsigned char* smem, uint64_t* s_bar, int* cta_status)
{
    const WsHead* head = p.ws.head;
    if (hv.status != 0) {  // deferred error: nothing is written (the engine has a stale header blanked, see kFlagPoisonOnError)
        if (!UNPACK) poison_on_error(p);
        return;
    }
    const uint32_t T = hv.T, B = hv.B;
    const uint64_t hb = hv.hb, P = hv.P, total = hb + P;
    const uint64_t ng = hv.ng;
    const uint64_t lo = p.lo, hi = p.hi < total ? p.hi : total;
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    const bool a8 = (hv.dtype & BS_ALIGN8) != 0;  // an unpadded stream: segments may sit 8 bytes off the 16-byte grid
    uint32_t tile_bytes = p.tile_bytes, n_warps = opt_warps & 0xffffu, n_stages = opt_stages;
    // The preset (bit 31 of opt_warps: bs_opts left the shape open) is settled here, where the payload size is known
    bool large = false;
    if ((opt_warps >> 31) && P >= kLargePayload && p.pkg.cap % preset_large(UNPACK).tile_bytes == 0) {
        const Preset ps = preset_large(UNPACK);
        tile_bytes = ps.tile_bytes; n_stages = ps.stages; n_warps = ps.warps;
        large = true;
    }
    // pacing (experiments; bs_opts.pace >= 100): that many GB/s of HBM traffic for the whole launch
    const uint32_t rate = p.pace >= 100u ? p.pace : 0u;
    // ---- payload tiles of [lo, hi): tile k = payload bytes [k*tile_bytes, (k+1)*tile_bytes) ----
    uint64_t plo = 0, phi = 0, k0 = 0, np = 0;
    if (hi > hb && hi > lo) {
        plo = (lo > hb ? lo : hb) - hb;
        phi = hi - hb;
        k0 = plo / tile_bytes;
        np = (phi + tile_bytes - 1) / tile_bytes - k0;
    }
    // ---- header region: generated (pack) / rebuilt into the descriptor arrays (unpack) with plain loads and stores
    // by warp `n_warps` of every CTA, beside the data warps; by every warp when the range holds no payload ----
    if (warp > n_warps) return;
    if (warp == n_warps || np == 0) {
        const uint64_t hw = np == 0 ? (uint64_t)blockIdx.x * (n_warps + 1) + warp : blockIdx.x;
        const uint64_t n_hw = np == 0 ? (uint64_t)gridDim.x * (n_warps + 1) : gridDim.x;
        if (UNPACK) {
            if (p.header != nullptr) {
                if (FUSED) rebuild_header_warp_v1(p, T, B, hw, n_hw, lane);
                else rebuild_header_warp(p, T, B, hw, n_hw, lane);
            }
        } else {
            if (p.lay.on) write_header_warp_v2(p, T, hb, P, lo, hi < hb ? hi : hb, hw, n_hw, lane);
            else write_header_warp(p, T, B, hb, P, hv.dtype, lo, hi < hb ? hi : hb, hw, n_hw, lane);
        }
        return;
    }
    const Blk* __restrict__ blk = p.ws.blk;

    const uint32_t ring = smem_u32(smem) + warp * n_stages * tile_bytes;  // this warp's stages
    unsigned char* ring_ptr = smem + (size_t)warp * n_stages * tile_bytes;
    unsigned char* meta_ptr = smem + (size_t)n_warps * n_stages * tile_bytes + (size_t)warp * kMetaBytes;
    const Blk* m_blk = reinterpret_cast<const Blk*>(meta_ptr);                                          // [kBlkSlots][kMetaBlk]
    const uint32_t* m_tf = reinterpret_cast<const uint32_t*>(meta_ptr + kBlkSlots * kMetaBlk * 16);    // [kTfSlots][2]
    const uint32_t m_blk_s = smem_u32(meta_ptr), m_tf_s = m_blk_s + kBlkSlots * kMetaBlk * 16;
    const uint32_t bar0 = smem_u32(&s_bar[warp * kMaxStages]);
    if (lane == 0) {
        for (uint32_t s = 0; s < n_stages; ++s) mbar_init(bar0 + 8 * s, 1);
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
    }
    fence_proxy_async();
    __syncwarp();

    const uint64_t worker = (uint64_t)blockIdx.x * n_warps + warp, n_workers = (uint64_t)gridDim.x * n_warps;
    // where an error met while moving goes: the workspace's status word — in a fused kernel the CTA's own word (the head may
    // still be on its way there from the pass's finalising CTA; the kernel's end posts it, see scan::leave)
    int* const status = FUSED ? cta_status : const_cast<int*>(&head->status);
    Hints hints;
    hints.pol = policy_evict_first();
    hints.ld = (p.tune & 1u) != 0;
    hints.st = (p.tune & 2u) != 0;
    int64_t lag = n_stages - 2;  // tile i is stored while tiles i+1 .. i+lag are loading
    if (((p.tune >> 8) & 15u) != 0 && (int64_t)((p.tune >> 8) & 15u) < lag) lag = (p.tune >> 8) & 15u;  // experiment: fewer loads in flight
    // iterations between the fetch of a tile's table entries and their use.  The one-warp pack of a large set fetches two
    // ahead: with small blocks (config 3, 3L: ~10 per tile) its iterations are long enough for the one exposed round trip
    // to show (+0.9 %; unpack: -0.3 %, it keeps one)
    const int64_t ahead = ((p.tune & 0x1000u) || rate || (!UNPACK && large)) ? 2 : 1;

    // ---- which tiles (see "tile hand-out"): iteration i of this warp works on tile tq(i) of the range, kNoTile = none left.
    // Claims are made `reach` iterations ahead: the answer of the atomic is written into the queue one iteration after it
    // was asked for (lane 0 keeps it in a register meanwhile), in time for the tile_first fetch 2 * ahead iterations ahead.
    // A range of less than kDynamicBytes keeps round 1's static round-robin deal: nothing there is worth the two extra round
    // trips of the counter (config 1: 3 us of 8).  tune bit 3 forces the static deal, bit 4 the counter (tests, A/B runs).
    const bool dynamic = (p.tune & 8u) == 0 && ((p.tune & 16u) != 0 || np * tile_bytes >= kDynamicBytes);
    MvCtr* const ctr = &g_mv_ctr[p.mv_slot & (kMvSlots - 1)];
    uint32_t* const m_tq = reinterpret_cast<uint32_t*>(meta_ptr + kBlkSlots * kMetaBlk * 16 + kTfSlots * 8);
    const int64_t reach = 2 * ahead;
    {
        uint32_t first = 0;
        if (dynamic && lane == 0) first = mv_take(&ctr->ticket, (uint32_t)reach);
        first = __shfl_sync(0xffffffffu, first, 0);
        if (lane < kTqSlots) {
            const uint64_t v = dynamic ? (uint64_t)first + lane : worker + (uint64_t)lane * n_workers;
            m_tq[lane] = (lane < (uint32_t)reach && v < np) ? (uint32_t)v : kNoTile;
        }
        __syncwarp();
    }
    // lane 0: the tile number of iteration i, raw (>= np: none left).  Dynamic: an atomic whose answer nobody waits for
    // until the next iteration queues it
    auto next_claim = [&](int64_t i) -> uint64_t {
        return dynamic ? (uint64_t)mv_take(&ctr->ticket, 1u) : worker + (uint64_t)i * n_workers;
    };
    bool claiming = m_tq[(reach - 1) & (kTqSlots - 1)] != kNoTile;  // nothing more to ask for once a claim came back empty
    uint64_t pending = np;                                           // lane 0: the claim of iteration it + reach
    if (lane == 0 && claiming) pending = next_claim(reach);
    auto tq = [&](int64_t i) { return i < 0 ? kNoTile : m_tq[i & (kTqSlots - 1)]; };
    int64_t n_mine = (int64_t)1 << 60;  // the number of this warp's tiles, known when the first empty claim comes up

    // the block table is fetched ahead into shared memory (see kBlkAheadMax)
    auto tile_base = [&](int64_t i) { return (k0 + (uint64_t)tq(i)) * tile_bytes; };
    auto has_tile = [&](int64_t i) { return B != 0 && tq(i) != kNoTile; };
    const uint32_t n_tf = 2 * (uint32_t)ahead + 1, n_bs = (uint32_t)ahead + 1;
    // slots are handed out round-robin by tile index; the loop keeps the slots of its current tile m_cur (no division)
    int64_t m_cur = 0;
    uint32_t tf_base = 0, bs_base = 0;
    auto tf_slot = [&](int64_t i) { const uint32_t s = tf_base + (uint32_t)(i - m_cur); return s >= n_tf ? s - n_tf : s; };   // m_cur <= i <= m_cur + 2*ahead
    auto blk_slot = [&](int64_t i) { const uint32_t s = bs_base + (uint32_t)(i - m_cur); return s >= n_bs ? s - n_bs : s; };  // m_cur <= i <= m_cur + ahead
    auto fetch_tf = [&](int64_t i) {  // lanes 0, 1: tile_first[g0], tile_first[g1] of tile i
        if (has_tile(i) && lane < 2) {
            const uint64_t tb = tile_base(i);
            uint64_t g = lane == 0 ? tb / kGranule : (tb + tile_bytes + kGranule - 1) / kGranule;  // a tile need not end on a granule
            if (g > ng) g = ng;  // tile_first[ng] == B
            cp_async_4(m_tf_s + tf_slot(i) * 8 + lane * 4, p.ws.tile_first + g);
        }
    };
    auto read_tf = [&](int64_t i, uint32_t* jlo, uint32_t* jhi) {
        *jlo = 1; *jhi = 0;
        if (has_tile(i)) {
            const uint32_t s = tf_slot(i) * 2;
            *jlo = m_tf[s];
            *jhi = m_tf[s + 1];
            if (*jhi >= B) *jhi = B - 1;
        }
    };
    auto fetch_blk = [&](int64_t i) {  // entries jlo .. min(jlo+32, jhi+1) of tile i (blk[B] is the sentinel)
        uint32_t jlo, jhi;
        read_tf(i, &jlo, &jhi);
        if (jlo > jhi) return;
        const uint32_t slot = m_blk_s + blk_slot(i) * kMetaBlk * 16;
        if (jlo + lane <= jhi + 1) cp_async_16(slot + lane * 16, blk + jlo + lane);
        if (lane == 0 && jlo + 32 <= jhi + 1) cp_async_16(slot + 32 * 16, blk + jlo + 32);
    };
    const int64_t m0 = UNPACK ? -lag : 0;  // index of the tile whose block table the first iteration needs
    m_cur = m0;
    for (int64_t i = m0; i < m0 + 2 * ahead; ++i) fetch_tf(i);
    cp_async_commit();
    cp_async_wait<0>();
    __syncwarp();
    for (int64_t i = m0; i < m0 + ahead; ++i) fetch_blk(i);
    cp_async_commit();
    for (int64_t g = 1; g < ahead; ++g) cp_async_commit();  // (empty groups: the loop counts `ahead` groups back)
    // pacing (experiments): a warp starts the loads of its next tile no earlier than its share of `rate` allows
    const uint64_t pace = rate ? (uint64_t)tile_bytes * 2u * n_workers / rate : 0;  // ns (GB/s = bytes per ns)
    uint64_t t_next = 0;
    if (pace) asm volatile("mov.u64 %0, %globaltimer;" : "=l"(t_next));

    uint32_t p_st = 0, c_st = 0, c_par = 0;  // stage of the tile being loaded; stage and mbarrier phase of the tile being stored
#ifdef BS_PHASE_PROF
    unsigned long long ph_acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
    long long ph_prev = clock64();
#endif
    for (int64_t it = 0;; ++it) {
        const int64_t m = m0 + it;
        BS_PH(7)
        // the claim asked for one iteration ago has arrived: queue it, ask for the next
        if (lane == 0) {
            m_tq[(it + reach) & (kTqSlots - 1)] = pending < np ? (uint32_t)pending : kNoTile;
            if (pending >= np) claiming = false;
            pending = claiming ? next_claim(it + reach + 1) : np;
        }
        __syncwarp();
        if (n_mine > it && tq(it) == kNoTile) n_mine = it;
        if (it >= n_mine + lag) break;
        // one cp.async group per iteration; the groups of the last ahead - 1 iterations may still be in flight: the
        // table entries of tile m and the tile_first pair of tile m + ahead, fetched `ahead` iterations ago, have landed
        if (ahead == 2) cp_async_wait<1>(); else cp_async_wait<0>();
        BS_PH(0)
        // the store that last read stage it % n_stages was committed two iterations ago
        bulk_wait_read<1>();
        __syncwarp();
        BS_PH(1)
        fetch_tf(m + 2 * ahead);
        fetch_blk(m + ahead);
        cp_async_commit();
        uint32_t jlo, jhi;
        read_tf(m, &jlo, &jhi);
        Blk e0;
        e0.off = 0; e0.addr = 0;
        uint64_t next0 = 0;  // clips to nothing
        if (jlo <= jhi && jlo + lane <= jhi) {
            e0 = m_blk[blk_slot(m) * kMetaBlk + lane];
            next0 = m_blk[blk_slot(m) * kMetaBlk + lane + 1].off;
        }
        BS_PH(2)
        if (it == 0) { BS_TL(4) }
        if (it < n_mine) {  // ---- produce: load tile `it` of this warp into its stage ----
            if (pace) {
                uint64_t now;
                do { asm volatile("mov.u64 %0, %globaltimer;" : "=l"(now)); } while (now < t_next);
                t_next = (now - t_next > 4 * pace ? now : t_next) + pace;  // a warp that fell far behind does not burst
            }
            BS_PH(3)
            const uint32_t st = p_st;
            p_st = p_st + 1 == n_stages ? 0 : p_st + 1;
            const uint64_t tbase = tile_base(it);
            const uint64_t tlo = tbase > plo ? tbase : plo;
            const uint64_t thi = tbase + tile_bytes < phi ? tbase + tile_bytes : phi;
            const uint32_t sbase = ring + st * tile_bytes, bar = bar0 + 8 * st;
            if (UNPACK) {
                if (lane == 0) {
                    if (a8) {
                        load_tile_a8(sbase + (uint32_t)(tlo - tbase), stream_at(p, hb, hb + tlo), (uint32_t)(thi - tlo), bar);
                    } else {
                        mbar_arrive_expect_tx(bar, (uint32_t)(thi - tlo));
                        bulk_g2s_x(sbase + (uint32_t)(tlo - tbase), stream_at(p, hb, hb + tlo), (uint32_t)(thi - tlo), bar, hints);
                        if ((p.tune & 0x20u) && tq(it + 1) != kNoTile) {  // experiment: the next tile of the stream into L2 now
                            const uint64_t nb = tile_base(it + 1);
                            const uint64_t nlo = nb > plo ? nb : plo, nhi = nb + tile_bytes < phi ? nb + tile_bytes : phi;
                            asm volatile("cp.async.bulk.prefetch.L2.global [%0], %1;" ::"l"(stream_at(p, hb, hb + nlo)), "r"((uint32_t)(nhi - nlo)) : "memory");
                        }
                    }
                }
            } else if (a8) {
                TileCtx c;
                c.tbase = tbase; c.tlo = tlo; c.thi = thi; c.sbase = sbase; c.bar = bar; c.jlo = jlo; c.jhi = jhi; c.lane = lane;
                c.blk = blk; c.e0 = e0; c.next0 = next0;
                pack_tile_a8(c);
            } else {
                // pass 1: bytes the bulk copies will deliver; tails and 8-byte-aligned blocks go through cp.async
                uint32_t tx = 0, n_async = 0;
                Seg s0;  // the lane's first segment (tiles rarely hold > 32 blocks)
                const bool have0 = clip_seg(e0, next0, tlo, thi, &s0);
                if (have0) n_async += pack_seg_async(s0, sbase + (uint32_t)(s0.lo - tbase), &tx);
                if (jhi >= jlo + 32) {
                    for (uint32_t j = jlo + lane + 32; j <= jhi; j += 32) {
                        Seg s;
                        if (make_seg(blk, j, tlo, thi, &s)) n_async += pack_seg_async(s, sbase + (uint32_t)(s.lo - tbase), &tx);
                    }
                }
                if (n_async) cp_async_mbar_arrive(bar);
#pragma unroll
                for (int d = 16; d > 0; d >>= 1) tx += __shfl_xor_sync(0xffffffffu, tx, d);
                __syncwarp();  // every lane's cp.async arrival is registered before the phase can complete
                if (lane == 0) mbar_arrive_expect_tx(bar, tx);
                __syncwarp();
                // pass 2: the bulk copies
                if (have0 && (s0.addr & 15ull) == 0 && s0.bulk)
                    bulk_g2s_x(sbase + (uint32_t)(s0.lo - tbase), reinterpret_cast<const void*>(s0.addr), s0.bulk, bar, hints);
                if (jhi >= jlo + 32) {
                    for (uint32_t j = jlo + lane + 32; j <= jhi; j += 32) {
                        Seg s;
                        if (make_seg(blk, j, tlo, thi, &s) && (s.addr & 15ull) == 0 && s.bulk)
                            bulk_g2s_x(sbase + (uint32_t)(s.lo - tbase), reinterpret_cast<const void*>(s.addr), s.bulk, bar, hints);
                    }
                }
            }
        }
        BS_PH(4)
        if (it == lag) { BS_TL(5) }
        if (it >= lag) {  // ---- consume: store tile `it - lag` ----
            const int64_t ci = it - lag;
            const uint32_t st = c_st, parity = c_par;
            if (++c_st == n_stages) { c_st = 0; c_par ^= 1u; }
            const uint64_t tbase = tile_base(ci);
            const uint64_t tlo = tbase > plo ? tbase : plo;
            const uint64_t thi = tbase + tile_bytes < phi ? tbase + tile_bytes : phi;
            const uint32_t sbase = ring + st * tile_bytes, bar = bar0 + 8 * st;
            if (!UNPACK) {
                uint32_t landed = 1;
                if (lane == 0) landed = mbar_wait(bar, parity, status) ? 1u : 0u;
                if (__shfl_sync(0xffffffffu, landed, 0) == 0) break;  // warp-uniform
                BS_PH(5)
                if (lane == 0) {
                    fence_proxy_async();  // the cp.async tails were written through the generic proxy
                    if (a8) store_tile_a8(stream_at(p, hb, hb + tlo), sbase + (uint32_t)(tlo - tbase), (uint32_t)(thi - tlo));
                    else bulk_s2g_x(stream_at(p, hb, hb + tlo), sbase + (uint32_t)(tlo - tbase), (uint32_t)(thi - tlo), hints);
                }
            } else if (a8) {
                if (!__all_sync(0xffffffffu, mbar_wait(bar, parity, status))) break;  // warp-uniform
                BS_PH(5)
                TileCtx c;
                c.tbase = tbase; c.tlo = tlo; c.thi = thi; c.sbase = sbase; c.bar = bar; c.jlo = jlo; c.jhi = jhi; c.lane = lane;
                c.blk = blk; c.e0 = e0; c.next0 = next0;
                unpack_tile_a8(c, ring_ptr + (size_t)st * tile_bytes, p.flags, status);
            } else {
                const unsigned char* sp = ring_ptr + (size_t)st * tile_bytes;
                Seg s0;
                const bool have0 = clip_seg(e0, next0, tlo, thi, &s0);
                if (!__all_sync(0xffffffffu, mbar_wait(bar, parity, status))) break;  // warp-uniform
                BS_PH(5)
                if (have0) unpack_seg(s0, sbase + (uint32_t)(s0.lo - tbase), sp + (s0.lo - tbase), p.flags, status, hints);
                if (jhi >= jlo + 32) {
                    for (uint32_t j = jlo + lane + 32; j <= jhi; j += 32) {
                        Seg s;
                        if (make_seg(blk, j, tlo, thi, &s))
                            unpack_seg(s, sbase + (uint32_t)(s.lo - tbase), sp + (s.lo - tbase), p.flags, status, hints);
                    }
                }
            }
        }
        bulk_commit();
        BS_PH(6)
        ++m_cur;
        tf_base = tf_base + 1 == n_tf ? 0 : tf_base + 1;
        bs_base = bs_base + 1 == n_bs ? 0 : bs_base + 1;
    }
    BS_TL(6)
    cp_async_wait<0>();
    bulk_wait_read<0>();
    BS_TL(7)
    if (dynamic && lane == 0) {
        // the last warp out puts the counters back for the next launch.  Every warp has its last (empty) claim in hand by
        // then: `pending` is stored first, so an atomic of this warp cannot still be on its way when the counter is reset
        m_tq[0] = (uint32_t)pending;
        if (mv_take(&ctr->exit, 1u) == (uint32_t)n_workers - 1u) {
            volatile uint64_t* c = &ctr->ticket;
            *c = kMvTag;
            c = &ctr->exit;
            *c = kMvTag;
            __threadfence();
        }
    }
#ifdef BS_PHASE_PROF
    if (lane == 0) for (int k = 0; k < 8; ++k) atomicAdd(&g_bs_phase[k], k == 7 ? (unsigned long long)(n_mine + lag) : ph_acc[k]);
#endif
}

template <bool UNPACK>
__global__ void __launch_bounds__((kMaxWarps + 1) * 32, 1) move_tma_kernel(const MoveParams p, const uint32_t opt_stages,
                                                                     const uint32_t opt_warps)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t s_bar[kMaxWarps * kMaxStages];
    const WsHead* head = p.ws.head;
    scan::HeadView hv;
    hv.status = head->status; hv.T = head->n_tensors; hv.B = head->n_blocks; hv.dtype = head->dtype;
    hv.hb = head->header_bytes; hv.P = head->payload_bytes; hv.ng = head->n_granules;
    move_tma_body<UNPACK, false>(p, hv, opt_stages, opt_warps, smem, s_bar, nullptr);
}

// ONE launch per bs_serialize / bs_deserialize call: the size / offset pass (bs_scan_phase.cuh) run by the
// first kScanThreads threads of every CTA — its shared state lives at the start of the dynamic shared memory the rings use
// afterwards — then the data movement above.  A set of one work item (<= 1024 blocks and tensors) runs the pass
// replicated: no CTA waits for another; larger sets claim items from the ticket and wait for the completion count.
template <bool UNPACK>
__global__ void __launch_bounds__((kMaxWarps + 1) * 32, 1) fused_tma_kernel(const ScanParams sp, const MoveParams p,
                                                                      const uint32_t opt_stages, const uint32_t opt_warps)
{
    extern __shared__ __align__(128) unsigned char smem[];
    __shared__ __align__(8) uint64_t s_bar[kMaxWarps * kMaxStages];
    __shared__ scan::HeadView s_hv;
    __shared__ int s_move_err;
    if (threadIdx.x == 0) s_move_err = 0;
    BS_TL(0)
    scan::Shared& sm = *reinterpret_cast<scan::Shared*>(smem);
    const scan::Shape s = scan::shape_of<UNPACK>(sp);
    const bool replicated = s.n_items == 1;
    if (threadIdx.x < kScanThreads) scan::run<UNPACK>(sp, s, sp.tag, sm, replicated, /*defer_exit=*/true);
    BS_TL(1)
    scan::HeadView hv;
    if (replicated) {
        __syncthreads();
        hv = sm.out;
        __syncthreads();  // the rings reuse the pass's shared memory
    } else {
        hv = scan::wait_done<UNPACK>(sp, s, sp.tag, sm, &s_hv);  // (ends with a barrier: the rings may reuse the pass's shared memory)
        // this CTA has seen the completion count: it is done with the pass's counters (the last CTA to say so resets them —
        // by then every CTA has seen it)
        if (threadIdx.x == 0) scan::leave(sp, sp.tag);
    }
    BS_TL(2)
    move_tma_body<UNPACK, true>(p, hv, opt_stages, opt_warps, smem, s_bar, &s_move_err);
    BS_TL(3)
    // An error met while moving (an mbarrier that never completed: seconds after the pass's finalising CTA wrote head and
    // result) becomes the status of the call: the warp that met it sees its own word here, no barrier needed
    if ((threadIdx.x & 31) == 0 && *(volatile int*)&s_move_err != 0) {
        volatile WsHead* vh = sp.ws.head;
        vh->status = s_move_err;
        if (sp.result != nullptr) sp.result->status = s_move_err;
    }
}

// The kernels may use the whole 227 KiB of dynamic shared memory: opt in once per kernel and device.  The flags are atomic
// (bs.h: calls are re-entrant); two threads racing here both set the same value.
template <typename K>
cudaError_t allow_max_smem(K kernel, std::atomic<uint64_t>* done)
{
    int dev = 0;
    cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return e;
    const bool tracked = dev >= 0 && dev < 64;
    if (tracked && (done->load(std::memory_order_acquire) >> dev) & 1ull) return cudaSuccess;
    e = cudaFuncSetAttribute(kernel, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(kSmemLimit - kStaticSmem));
    if (e != cudaSuccess) return e;
    if (tracked) done->fetch_or(1ull << dev, std::memory_order_release);
    return cudaSuccess;
}

// the tile counter pair of a launch ("tile hand-out"): launches take the pairs of the ring in turn
uint32_t next_mv_slot()
{
    static std::atomic<uint32_t> seq{0};
    return seq.fetch_add(1, std::memory_order_relaxed) & (kMvSlots - 1);
}

struct Shape3 {
    uint32_t tile_bytes, stages, warps, auto_shape;
    size_t smem;
};
template <bool UNPACK>
cudaError_t resolve_shape(const MoveParams& p, const bs_opts& o, Shape3* out)
{
    Shape3 sh = {p.tile_bytes, o.stages, o.warps, 0u, 0};
    if (o.tile_bytes == 0) {  // bs_opts left the shape open: launch the small shape, the kernel may switch to the large one
        const Preset ps = preset_small(), pl = preset_large(UNPACK);
        if ((size_t)pl.warps * pl.stages * pl.tile_bytes > (size_t)ps.warps * ps.stages * ps.tile_bytes || pl.warps > ps.warps)
            return cudaErrorInvalidValue;  // the large shape must fit the launch of the small one
        sh.tile_bytes = ps.tile_bytes; sh.stages = ps.stages; sh.warps = ps.warps;
        sh.auto_shape = 0x80000000u;
    }
    if (sh.stages < 3 || sh.stages > kMaxStages || sh.warps < 1 || sh.warps > kMaxWarps) return cudaErrorInvalidValue;
    sh.smem = (size_t)sh.warps * sh.stages * sh.tile_bytes + (size_t)sh.warps * kMetaBytes;
    if (sh.smem + kStaticSmem > kSmemLimit) return cudaErrorInvalidValue;
    *out = sh;
    return cudaSuccess;
}

template <bool UNPACK>
cudaError_t launch_tma_t(const MoveParams& p, const bs_opts& o, int sm_count, cudaStream_t stream)
{
    MoveParams q = p;
    Shape3 sh;
    cudaError_t e = resolve_shape<UNPACK>(p, o, &sh);
    if (e != cudaSuccess) return e;
    q.tile_bytes = sh.tile_bytes;
    q.mv_slot = next_mv_slot();
    static std::atomic<uint64_t> allowed{0};
    if ((e = allow_max_smem(move_tma_kernel<UNPACK>, &allowed)) != cudaSuccess) return e;
    move_tma_kernel<UNPACK><<<(unsigned)sm_count, (sh.warps + 1) * 32, sh.smem, stream>>>(q, sh.stages, sh.warps | sh.auto_shape);  // + the header warp
    return cudaGetLastError();
}

// the pass and the movement of the whole stream in ONE launch.  `bytes_bound`: an upper bound of the stream's size
// (serialize: the capacity; deserialize: nbytes) — CTAs beyond the tiles it can hold would find no work.
template <bool UNPACK>
cudaError_t launch_fused_t(const ScanParams& sp, const MoveParams& p, const bs_opts& o, uint64_t bytes_bound, int sm_count,
                           cudaStream_t stream)
{
    MoveParams q = p;
    Shape3 sh;
    cudaError_t e = resolve_shape<UNPACK>(p, o, &sh);
    if (e != cudaSuccess) return e;
    q.tile_bytes = sh.tile_bytes;
    q.mv_slot = next_mv_slot();
    if (sh.smem < sizeof(scan::Shared)) sh.smem = sizeof(scan::Shared);  // small tiles: the pass's state needs more than the rings
    static std::atomic<uint64_t> allowed{0};
    if ((e = allow_max_smem(fused_tma_kernel<UNPACK>, &allowed)) != cudaSuccess) return e;
    if ((e = prepare_scan_state(sp.ws, stream)) != cudaSuccess) return e;
    ScanParams s2 = sp;
    s2.tag = next_epoch_tag();
    const uint64_t items = scan::host_items(sp.T, sp.B);
    const uint64_t tiles = bytes_bound / kGranule + 2;  // data warps take tiles of >= 16 KiB; + the header's share
    uint64_t grid = items > tiles ? items : tiles;
    if (grid > (uint64_t)sm_count) grid = (uint64_t)sm_count;
    const uint32_t threads = (sh.warps + 1) * 32 > kScanThreads ? (sh.warps + 1) * 32 : kScanThreads;
    fused_tma_kernel<UNPACK><<<(unsigned)grid, threads, sh.smem, stream>>>(s2, q, sh.stages, sh.warps | sh.auto_shape);
    return cudaGetLastError();
}

}  // namespace

cudaError_t launch_move_tma(bool unpack, const MoveParams& p, const bs_opts& o, int sm_count, cudaStream_t stream)
{
    return unpack ? launch_tma_t<true>(p, o, sm_count, stream) : launch_tma_t<false>(p, o, sm_count, stream);
}

cudaError_t launch_fused_tma(bool unpack, const ScanParams& sp, const MoveParams& p, const bs_opts& o, uint64_t bytes_bound,
                             int sm_count, cudaStream_t stream)
{
    return unpack ? launch_fused_t<true>(sp, p, o, bytes_bound, sm_count, stream)
                  : launch_fused_t<false>(sp, p, o, bytes_bound, sm_count, stream);
}

}  // namespace bs

#ifdef BS_PHASE_PROF
extern "C" int bs_debug_rates(unsigned int* out2) { out2[0] = out2[1] = 0; return 0; }
extern "C" int bs_debug_hist(unsigned int* out64, int reset)
{
    if (out64 && cudaMemcpyFromSymbol(out64, bs::g_bs_hist, sizeof(bs::g_bs_hist)) != cudaSuccess) return -1;
    if (reset) { unsigned int z[64] = {0}; cudaMemcpyToSymbol(bs::g_bs_hist, z, sizeof(z)); }
    return 0;
}
extern "C" int bs_debug_timeline(unsigned long long* out) { return cudaMemcpyFromSymbol(out, bs::g_bs_tl, sizeof(bs::g_bs_tl)) == cudaSuccess ? 0 : -1; }
extern "C" int bs_debug_trig(unsigned int* out4, int reset)
{
    if (out4 && cudaMemcpyFromSymbol(out4, bs::g_bs_trig, sizeof(bs::g_bs_trig)) != cudaSuccess) return -1;
    if (reset) { unsigned int z[4] = {0}; cudaMemcpyToSymbol(bs::g_bs_trig, z, sizeof(z)); }
    return 0;
}
#endif
