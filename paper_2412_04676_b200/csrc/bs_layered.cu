// bs_layered.cu — wire format v2, structure-shared layers (include/bs.h).
//
// PAPER Fig 4(a) (L75): "Layers indicate position dependent operators which have the same block-sparse structure,
// but the dense sector matrices take different values for the different layers."  The meta data of a structure
// (L63: sector indices, quantum numbers, sector dimensions) is stored once; every layer adds 16 bytes.  The
// "pointer structure ... grid structure of the serialized data" (L90-92) is built by ONE launch before any data moves
// (lplan_kernel; work items of three phases are claimed in order from one ticket, see there):
//   phase 1 : chained scan over the STRUCTURE block table (Bs entries): stored sizes -> gs[] (serialize); header
//             validation, stored sizes + pool slot sizes -> gs[], gp[] (deserialize)
//   phase 2 : chained scan over the LAYERS (T entries): bytes and block count of every layer's structure
//             -> lpos[] = {payload (or pool) offset, index of the layer's first block}; totals, checks, result
//   phase 3 : the flat work table the data-movement kernels already use (blk[] = {payload offset, block address},
//             tile_first[]) — B entries, 16 bytes each, one thread per block (its layer found by binary search in lpos[])
// after which the payload moves through the SAME pack / unpack kernels as wire format v1 (bs_move_tma.cu, bs_move.cu);
// only their header generator / parser differs (bs_move_common.cuh, *_v2).
// Roofline: HBM-bound; the plan touches 8 B (address) + 16 B (table entry) per block plus the structure tables,
// < 0.5 % of the payload traffic; the header itself shrinks from 48 B per block to 48 B per structure block.
#include <string.h>

#include "bs_internal.cuh"

namespace bs {

namespace {

constexpr uint32_t kV2Struct = 32, kV2Layer = 16;
constexpr uint64_t kFlagAgg = 1ull << 62;
constexpr uint64_t kFlagPrefix = 2ull << 62;
constexpr uint64_t kValMask = (1ull << 62) - 1;
constexpr uint32_t kLThreads = 256, kLItems = 4, kLTile = kLThreads * kLItems;

struct LwLayout {
    WsLayout ws;        // head, blk, tile_first: what the move kernels see
    uint64_t* st1[2];   // chained-scan state of the block pass
    uint64_t* st2[2];   // chained-scan state of the layer pass
    uint64_t* gs;       // [Bs+1] exclusive prefix of stored sizes over the structure block table | pad code (bits 0-1)
    uint64_t* gp;       // [Bs+1] exclusive prefix of pool slot sizes (deserialize)
    LayerPos* lpos;     // [T+1]
    uint64_t blk_cap;   // B the blk[] table can hold (plus the sentinel)
};

uint64_t lw_fixed_bytes(uint32_t Bs, uint32_t T, uint64_t B)
{
    const uint64_t t1 = ((uint64_t)Bs + kLTile) / kLTile + 1, t2 = ((uint64_t)T + kLTile) / kLTile + 1;
    return sizeof(WsHead) + 2 * align_up(t1 * 8, 256) + 2 * align_up(t2 * 8, 256) + 2 * align_up(((uint64_t)Bs + 1) * 8, 256) +
           align_up(((uint64_t)T + 1) * sizeof(LayerPos), 256) + align_up((B + 1) * sizeof(Blk), 256);
}

bool lw_layout(void* d_ws, uint64_t ws_bytes, uint32_t Bs, uint32_t T, uint64_t B, LwLayout* L)
{
    const uint64_t fixed = lw_fixed_bytes(Bs, T, B);
    if (d_ws == nullptr || ((uintptr_t)d_ws & 255) != 0 || ws_bytes < fixed + 16) return false;
    const uint64_t t1 = ((uint64_t)Bs + kLTile) / kLTile + 1, t2 = ((uint64_t)T + kLTile) / kLTile + 1;
    unsigned char* p = (unsigned char*)d_ws;
    L->ws.head = (WsHead*)p;
    p += sizeof(WsHead);
    L->ws.scan_state = (ScanState*)p;  // unused by the layered plan (st1 / st2 below are its chains)
    for (int c = 0; c < 2; ++c) { L->st1[c] = (uint64_t*)p; p += align_up(t1 * 8, 256); }
    for (int c = 0; c < 2; ++c) { L->st2[c] = (uint64_t*)p; p += align_up(t2 * 8, 256); }
    L->ws.zero_bytes = (uint64_t)(p - (unsigned char*)d_ws);
    L->gs = (uint64_t*)p; p += align_up(((uint64_t)Bs + 1) * 8, 256);
    L->gp = (uint64_t*)p; p += align_up(((uint64_t)Bs + 1) * 8, 256);
    L->lpos = (LayerPos*)p; p += align_up(((uint64_t)T + 1) * sizeof(LayerPos), 256);
    L->ws.blk = (Blk*)p; p += align_up((B + 1) * sizeof(Blk), 256);
    L->ws.tile_first = (uint32_t*)p;
    L->ws.n_granules_cap = (ws_bytes - fixed) / 4;
    L->blk_cap = B;
    return true;
}

struct LPlanParams {
    LwLayout lw;
    bs_result* result;        // device, may be null
    uint64_t capacity;        // serialize: stream capacity
    uint64_t expect_total;    // serialize: if nonzero the total must equal it (engine re-check of the size prediction)
    // serialize inputs (descriptor arrays, device)
    const bs_struct_rec* structs;
    const bs_layer_rec* layers;
    const uint32_t* dim;
    const uint64_t* addr;
    uint32_t C, Bs, T;        // serialize: counts; deserialize: capacities of the out arrays
    uint32_t dtype;           // serialize: element type of the set (deserialize reads it from the header)
    uint64_t n_addr;          // entries of addr[] (deserialize: capacity of out addr)
    // deserialize inputs
    const unsigned char* header;   // stream byte 0 .. header_bytes
    const unsigned char* payload;  // stream byte 0 when the payload is resident behind the header, else null
    uint64_t nbytes;
    uint64_t pool_base, pool_bytes;
    const uint32_t* out_dim;       // BS_SCATTER_TO_ADDR: caller's extents [Bs][3]
    uint64_t* out_addr;            // pool layout: written; scatter: read
    uint32_t flags;
};

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
__device__ __forceinline__ void set_err(WsHead* h, bs_result* r, int code)
{
    if (code == 0) return;
    atomicCAS(&h->status, 0, code);
    if (r != nullptr) atomicCAS(&r->status, 0, code);  // the plan result may already have been written
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

// ---- single-pass chained (decoupled look-back) exclusive scan of NV u64 components over tiles claimed in order ----
template <int NV>
struct ChainSmem {
    uint64_t warp_sum[NV][kLThreads / 32];
    uint64_t prefix[NV];
    uint64_t total[NV];
};

// tsum: this thread's sum per component; on return excl = exclusive prefix of the thread over the whole sequence.
// Must be called by all kLThreads threads of the CTA; ends with the CTA synchronised.
template <int NV>
__device__ __forceinline__ void chained_scan(const uint64_t (&tsum)[NV], uint64_t (&excl)[NV], uint64_t tile, uint64_t* st0,
                                             uint64_t* st1, ChainSmem<NV>& sm)
{
    const uint32_t lane = threadIdx.x & 31, warp = threadIdx.x >> 5;
    uint64_t incl[NV];
#pragma unroll
    for (int c = 0; c < NV; ++c) {
        incl[c] = warp_incl_scan(tsum[c], lane);
        if (lane == 31) sm.warp_sum[c][warp] = incl[c];
    }
    __syncthreads();
    if (warp < (uint32_t)NV) {  // warp c looks back for component c
        const int c = (int)warp;
        uint64_t* state = c == 0 ? st0 : st1;
        const uint64_t ws = (lane < kLThreads / 32) ? sm.warp_sum[c][lane] : 0;
        const uint64_t agg = warp_sum(ws);
        uint64_t pre = 0;
        if (tile == 0) {
            if (lane == 0) st_release_u64(state, kFlagPrefix | (agg & kValMask));
        } else {
            if (lane == 0) st_release_u64(state + tile, kFlagAgg | (agg & kValMask));
            int64_t look = (int64_t)tile - 1;
            for (;;) {
                const int64_t idx = look - (int64_t)lane;
                uint64_t w = (idx >= 0) ? ld_acquire_u64(state + idx) : kFlagPrefix;
                while (__any_sync(0xffffffffu, (w >> 62) == 0)) {
                    if ((w >> 62) == 0) w = ld_acquire_u64(state + idx);
                }
                const uint32_t is_prefix = __ballot_sync(0xffffffffu, (w >> 62) == 2);
                const uint32_t first = is_prefix ? (uint32_t)__ffs((int)is_prefix) - 1u : 32u;
                pre += warp_sum(lane <= first ? (w & kValMask) : 0ull);
                if (is_prefix) break;
                look -= 32;
            }
            if (lane == 0) st_release_u64(state + tile, kFlagPrefix | ((pre + agg) & kValMask));
        }
        if (lane == 0) { sm.prefix[c] = pre; sm.total[c] = agg; }
    }
    __syncthreads();
#pragma unroll
    for (int c = 0; c < NV; ++c) {
        uint64_t run = sm.prefix[c] + (incl[c] - tsum[c]);
        for (uint32_t w = 0; w < warp; ++w) run += sm.warp_sum[c][w];
        excl[c] = run;
    }
}

struct StructHead {
    uint32_t rank, first, n;
    uint64_t layer_bytes;
};
__device__ __forceinline__ StructHead load_struct(const void* recs, uint64_t s)
{
    const uint4* r = reinterpret_cast<const uint4*>(recs) + 2 * s;
    const uint4 a = __ldg(r), b = __ldg(r + 1);
    StructHead h;
    h.rank = a.x; h.first = a.y; h.n = a.z;
    h.layer_bytes = (uint64_t)b.z | ((uint64_t)b.w << 32);
    return h;
}

// ---- the plan kernel: ONE launch, three phases of work items claimed in order from one ticket ------------------------------
//   phase 1 (n1 items): a tile of the structure block table (+ the same slice of the structure records)
//   phase 2 (n2 items): a tile of the layers; the CTA that finishes the last one writes totals, checks, sentinel, result
//   phase 3          : a chunk of kLTile blocks of the flat work table blk[] / tile_first[]
// An item of phase 2 waits until every item of phase 1 is done, an item of phase 3 until the plan is ready.  Items are
// claimed in order and a claimed item is being executed by a resident CTA, so whatever an item waits for is already
// running and never waits for a later item: forward progress needs no co-residency of the whole grid (the argument of the
// chained scan's look-back).
__device__ __forceinline__ uint32_t ld_acquire_u32(const uint32_t* p)
{
    uint32_t v;
    asm volatile("ld.acquire.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory");
    return v;
}
__device__ __forceinline__ void cta_wait_until(const uint32_t* counter, uint32_t target)
{
    if (threadIdx.x == 0) {
        while (ld_acquire_u32(counter) < target) __nanosleep(64);
    }
    __syncthreads();
}

struct PlanShape {  // uniform over the grid: derived from the call's arguments / the fixed header alone
    uint64_t C, Bs, T, hb, P_hdr;
    uint32_t dtype;     // element type (bs.h): the element size is all it decides (reading E-2)
    bool ok;
    uint32_t n1, n2;
};

template <bool DESER>
__device__ __forceinline__ PlanShape plan_shape(const LPlanParams& p, WsHead* head)
{
    PlanShape s;
    s.C = p.C; s.Bs = p.Bs; s.T = p.T; s.hb = 0; s.P_hdr = 0; s.ok = true; s.dtype = p.dtype;
    if (DESER) {  // the fixed header, field by field in stream order
        int code = 0;
        s.C = s.Bs = s.T = 0;
        if (p.nbytes < kFixedHeader) {
            code = BS_ERR_CORRUPT;
        } else {
            const uint4* f = reinterpret_cast<const uint4*>(p.header);
            const uint4 w0 = __ldg(f), w1 = __ldg(f + 1), w2 = __ldg(f + 2), w3 = __ldg(f + 3);
            const uint64_t hC = w2.x, hBs = w2.y, hT = (uint64_t)w2.z | ((uint64_t)w2.w << 32);
            const uint64_t hH = (uint64_t)w3.x | ((uint64_t)w3.y << 32), hP = (uint64_t)w3.z | ((uint64_t)w3.w << 32);
            if (w0.x != 0x41505342u || w0.y != 0x31455352u)      code = BS_ERR_CORRUPT;  // "BSPARSE1"
            else if (w0.z != 2u)                                  code = BS_ERR_CORRUPT;  // version
            else if (w0.w != 0x01020304u)                         code = BS_ERR_CORRUPT;  // endian_tag
            else if (w1.x > (uint32_t)BS_C128)                    code = BS_ERR_CORRUPT;  // dtype
            else if (w1.y != 2u)                                  code = BS_ERR_CORRUPT;  // n_qn
            else if (w1.z != 3u)                                  code = BS_ERR_CORRUPT;  // max_rank
            else if (w1.w != 16u)                                 code = BS_ERR_CORRUPT;  // align
            else if (hT >= (1ull << 32))                          code = BS_ERR_CORRUPT;
            else if (hH != align_up(kFixedHeader + kV2Struct * hC + kV2Layer * hT + kBlockRec * hBs, kHeaderAlign)) code = BS_ERR_CORRUPT;
            else if (hH > p.nbytes || hP != p.nbytes - hH)        code = BS_ERR_CORRUPT;
            else if (hC > p.C || hBs > p.Bs || hT > p.T)          code = BS_ERR_CAPACITY;  // out arrays too small
            else { s.C = hC; s.Bs = hBs; s.T = hT; s.hb = hH; s.P_hdr = hP; s.dtype = w1.x; }
            if (code == BS_ERR_CAPACITY && blockIdx.x == 0 && threadIdx.x == 0) {  // report the counts
                head->n_structs = (uint32_t)hC; head->n_struct_blocks = (uint32_t)hBs; head->n_tensors = (uint32_t)hT;
            }
        }
        if (code != 0) {
            s.ok = false;
            if (blockIdx.x == 0 && threadIdx.x == 0) set_err(head, nullptr, code);
        }
    } else {
        s.hb = align_up(kFixedHeader + kV2Struct * s.C + kV2Layer * s.T + kBlockRec * s.Bs, kHeaderAlign);
    }
    const uint64_t m = s.Bs > s.C ? s.Bs : s.C;
    const uint64_t t1 = (m + kLTile - 1) / kLTile, t2 = (s.T + kLTile - 1) / kLTile;
    s.n1 = s.ok ? (uint32_t)(t1 ? t1 : 1) : 0u;
    s.n2 = s.ok ? (uint32_t)(t2 ? t2 : 1) : 1u;  // the last item of phase 2 always writes the result
    return s;
}

// ---- phase 1: tile `tile` of the structure block table and of the structure records -----------------------------------------
template <bool DESER>
__device__ __forceinline__ void plan_blocks_tile(const LPlanParams& p, const PlanShape& s, uint64_t tile, ChainSmem<2>& sm)
{
    WsHead* head = p.lw.ws.head;
    const uint32_t tid = threadIdx.x;
    constexpr int kErrBad = DESER ? BS_ERR_CORRUPT : BS_ERR_ARG;
    constexpr int kErrRank = DESER ? BS_ERR_CORRUPT : BS_ERR_UNSUPPORTED;
    const uint64_t C = s.C, Bs = s.Bs, T = s.T;
    const void* srecs = DESER ? (const void*)(p.header + kFixedHeader) : (const void*)p.structs;
    const unsigned char* brec = DESER ? p.header + kFixedHeader + kV2Struct * C + kV2Layer * T : nullptr;
    int err = 0;

    // structure records partition the structure block table in order
#pragma unroll
    for (uint32_t k = 0; k < kLItems; ++k) {
        const uint64_t q = tile * kLTile + (uint64_t)k * kLThreads + tid;
        if (q < C) {
            const StructHead h = load_struct(srecs, q);
            uint64_t prev_end = 0;
            if (q > 0) {
                const StructHead g = load_struct(srecs, q - 1);
                prev_end = (uint64_t)g.first + g.n;
            }
            if (h.rank != 2 && h.rank != 3) err = kErrRank;
            else if (h.first != prev_end) err = kErrBad;
            else if ((uint64_t)h.first + h.n > Bs) err = kErrBad;
            else if (q == C - 1 && (uint64_t)h.first + h.n != Bs) err = kErrBad;
        }
    }
    if (tile == 0) {
        if (C == 0 && Bs != 0 && tid == 0) err = kErrBad;
        if (DESER) {  // header slack must be zero
            const uint64_t used = kFixedHeader + kV2Struct * C + kV2Layer * T + kBlockRec * Bs;
            const uint64_t z = used + 16ull * tid;
            if (z < s.hb) {
                const uint4 w = __ldg(reinterpret_cast<const uint4*>(p.header + z));
                if ((w.x | w.y | w.z | w.w) != 0) err = BS_ERR_CORRUPT;
            }
        }
        if (Bs == 0 && tid == 0) { p.lw.gs[0] = 0; p.lw.gp[0] = 0; }
    }

    uint64_t stored[kLItems], slot[kLItems];
    uint32_t oddf[kLItems];
    uint64_t tsum[2] = {0, 0};
#pragma unroll
    for (uint32_t k = 0; k < kLItems; ++k) {
        const uint64_t j = tile * kLTile + (uint64_t)tid * kLItems + k;
        const bool valid = j < Bs;
        uint32_t d0 = 1, d1 = 1, d2 = 0, owner = 0;
        int32_t q4 = 0, q5 = 0;
        uint64_t offset = 0;
        if (valid) {
            if (DESER) {
                const uint4* r = reinterpret_cast<const uint4*>(brec + kBlockRec * j);
                const uint4 r1 = __ldg(r + 1), r2 = __ldg(r + 2);
                q4 = (int32_t)r1.x; q5 = (int32_t)r1.y;
                d0 = r1.z; d1 = r1.w; d2 = r2.x; owner = r2.y;
                offset = (uint64_t)r2.z | ((uint64_t)r2.w << 32);
            } else {
                d0 = __ldg(p.dim + 3 * j); d1 = __ldg(p.dim + 3 * j + 1); d2 = __ldg(p.dim + 3 * j + 2);
            }
        }
        const uint64_t n01 = (uint64_t)d0 * d1;
        uint64_t n = n01 * d2;
        if (valid && (__umul64hi(n01, (uint64_t)d2) != 0 || n >= (1ull << 57))) { err = kErrBad; n = 0; }
        const uint64_t nbytes = n * elem_bytes(s.dtype);
        const uint64_t st = (nbytes + 15) & ~15ull;
        stored[k] = valid ? st : 0;
        slot[k] = (DESER && valid) ? align_up(nbytes, kPoolAlign) : 0;
        oddf[k] = (uint32_t)(st - nbytes) >> 2;  // pad code: 0..3 words of zero pad (Blk)
        if (DESER && valid) {
            if (owner >= C) err = BS_ERR_CORRUPT;
            else {
                const StructHead h = load_struct(srecs, owner);
                const uint64_t end = (uint64_t)h.first + h.n;
                if (j < h.first || j >= end) err = BS_ERR_CORRUPT;
                else {
                    if (h.rank == 2 && (d2 != 1 || q4 != 0 || q5 != 0)) err = BS_ERR_CORRUPT;
                    // relative offsets = exclusive prefix sum inside the structure, checked link by link
                    uint64_t next = h.layer_bytes;
                    if (j + 1 < end) next = __ldg(reinterpret_cast<const unsigned long long*>(brec + kBlockRec * (j + 1) + 40));
                    if (j == h.first && offset != 0) err = BS_ERR_CORRUPT;
                    if (offset >= (1ull << 62) || offset + st != next) err = BS_ERR_CORRUPT;
                }
            }
            if (p.flags == BS_SCATTER_TO_ADDR &&
                (__ldg(p.out_dim + 3 * j) != d0 || __ldg(p.out_dim + 3 * j + 1) != d1 || __ldg(p.out_dim + 3 * j + 2) != d2)) {
                if (!err) err = BS_ERR_ARG;
            }
        }
        tsum[0] += stored[k];
        tsum[1] += slot[k];
    }
    if (err) set_err(head, nullptr, err);
    if (tile != 0 && tile * kLTile >= Bs) return;  // a tile of structure records only (C > Bs): not part of the chain
    uint64_t excl[2];
    chained_scan<2>(tsum, excl, tile, p.lw.st1[0], p.lw.st1[1], sm);
    uint64_t r0 = excl[0], r1 = excl[1];
#pragma unroll
    for (uint32_t k = 0; k < kLItems; ++k) {
        const uint64_t j = tile * kLTile + (uint64_t)tid * kLItems + k;
        if (j < Bs) {
            p.lw.gs[j] = r0 | oddf[k];
            p.lw.gp[j] = r1;
        }
        r0 += stored[k];
        r1 += slot[k];
    }
    if (Bs != 0 && tile == (Bs - 1) / kLTile && tid == 0) {  // the owner of the last block tile knows the totals
        p.lw.gs[Bs] = sm.prefix[0] + sm.total[0];
        p.lw.gp[Bs] = sm.prefix[1] + sm.total[1];
    }
}

// ---- phase 2: tile `tile` of the layers ----------------------------------------------------------------------------------
// `bad`: the status after phase 1 was not BS_OK.  The tile still takes part in the chain (a later tile looks back at it)
// but scans zeros and dereferences no structure range.
template <bool DESER>
__device__ __forceinline__ void plan_layers_tile(const LPlanParams& p, const PlanShape& s, uint64_t tile, bool bad,
                                                 ChainSmem<2>& sm)
{
    WsHead* head = p.lw.ws.head;
    const uint32_t tid = threadIdx.x;
    const uint64_t C = s.C, T = s.T;
    const void* srecs = DESER ? (const void*)(p.header + kFixedHeader) : (const void*)p.structs;
    const bs_layer_rec* ly = DESER ? reinterpret_cast<const bs_layer_rec*>(p.header + kFixedHeader + kV2Struct * C) : p.layers;
    constexpr int kErrBad = DESER ? BS_ERR_CORRUPT : BS_ERR_ARG;
    uint64_t vb[kLItems], vn[kLItems], woff[kLItems];
    uint32_t sfirst[kLItems];
    uint64_t tsum[2] = {0, 0};
    int err = 0;
#pragma unroll
    for (uint32_t k = 0; k < kLItems; ++k) {
        const uint64_t t = tile * kLTile + (uint64_t)tid * kLItems + k;
        vb[k] = 0; vn[k] = 0; woff[k] = 0; sfirst[k] = 0;
        if (t < T && !bad) {
            const uint4 w = __ldg(reinterpret_cast<const uint4*>(ly + t));  // structure, tag, offset
            const uint32_t st = w.x;
            if (st >= C) err = kErrBad;
            else {
                const StructHead h = load_struct(srecs, st);
                const uint64_t* g = DESER ? p.lw.gp : p.lw.gs;
                vb[k] = (g[(uint64_t)h.first + h.n] & ~15ull) - (g[h.first] & ~15ull);
                vn[k] = h.n;
                sfirst[k] = h.first;
                if (DESER) woff[k] = (uint64_t)w.z | ((uint64_t)w.w << 32);
                if (DESER) {  // layer offsets = exclusive prefix sum of layer_bytes, checked link by link, inside [0, P]
                    const uint64_t off = (uint64_t)w.z | ((uint64_t)w.w << 32);
                    uint64_t next = s.P_hdr;
                    if (t + 1 < T) next = __ldg(reinterpret_cast<const unsigned long long*>(&ly[t + 1].offset));
                    if (t == 0 && off != 0) err = BS_ERR_CORRUPT;
                    if (off > s.P_hdr || h.layer_bytes > s.P_hdr - off || off + h.layer_bytes != next) err = BS_ERR_CORRUPT;
                }
            }
        }
        tsum[0] += vb[k];
        tsum[1] += vn[k];
    }
    if (err) set_err(head, nullptr, err);
    uint64_t excl[2];
    chained_scan<2>(tsum, excl, tile, p.lw.st2[0], p.lw.st2[1], sm);
    uint64_t r0 = excl[0], r1 = excl[1];
#pragma unroll
    for (uint32_t k = 0; k < kLItems; ++k) {
        const uint64_t t = tile * kLTile + (uint64_t)tid * kLItems + k;
        if (t < T) {
            LayerPos lp; lp.off = r0; lp.first_addr = r1;
            lp.stream_off = DESER ? woff[k] : r0; lp.sfirst = sfirst[k]; lp.sn = (uint32_t)vn[k];
            p.lw.lpos[t] = lp;
        }
        r0 += vb[k];
        r1 += vn[k];
    }
    if (tile == s.n2 - 1 && tid == 0) {  // the owner of the last tile knows the totals (T == 0: zeros)
        LayerPos lp; lp.off = sm.prefix[0] + sm.total[0]; lp.first_addr = sm.prefix[1] + sm.total[1];
        lp.stream_off = 0; lp.sfirst = 0; lp.sn = 0;
        p.lw.lpos[T] = lp;
    }
}

// ---- end of phase 2 (one thread): totals, capacity checks, sentinel, result ---------------------------------------------------
template <bool DESER>
__device__ __forceinline__ void plan_finalize(const LPlanParams& p, const PlanShape& s)
{
    volatile WsHead* vh = p.lw.ws.head;
    int status = vh->status;
    const bool bad = !s.ok;
    uint64_t tot_bytes = 0, tot_blocks = 0;
    if (s.ok) {
        const volatile LayerPos* end = p.lw.lpos + s.T;
        tot_bytes = end->off; tot_blocks = end->first_addr;
    }
    uint64_t P = DESER ? s.P_hdr : tot_bytes;
    uint64_t pool = DESER ? tot_bytes : 0;
    if (status != 0) { pool = 0; if (!DESER) P = 0; tot_blocks = 0; }
    if (bad) P = 0;
    const uint64_t hb = s.hb;
    const uint64_t total = hb + P;
    const uint64_t ng = (P + kGranule - 1) / kGranule;
    if (status == 0) {
        if (DESER && s.T == 0 && s.P_hdr != 0) status = BS_ERR_CORRUPT;
        else if (tot_blocks >= (1ull << 32)) status = BS_ERR_UNSUPPORTED;
        else if (!DESER && total > p.capacity) status = BS_ERR_CAPACITY;
        else if (!DESER && p.expect_total != 0 && total != p.expect_total) status = BS_ERR_ARG;
        else if (ng + 1 > p.lw.ws.n_granules_cap) status = BS_ERR_CAPACITY;
        else if (tot_blocks > p.lw.blk_cap || tot_blocks > p.n_addr) status = BS_ERR_CAPACITY;
        else if (DESER && p.flags == BS_LAYOUT_POOL && pool > p.pool_bytes) status = BS_ERR_CAPACITY;
    }
    if (s.ok && tot_blocks <= p.lw.blk_cap) {
        Blk e; e.off = P; e.addr = 0;
        p.lw.ws.blk[tot_blocks] = e;
        if (ng < p.lw.ws.n_granules_cap) p.lw.ws.tile_first[ng] = (uint32_t)tot_blocks;
    }
    if (s.ok) {
        vh->n_structs = (uint32_t)s.C;
        vh->n_struct_blocks = (uint32_t)s.Bs;
        vh->n_tensors = (uint32_t)s.T;
    }
    vh->n_blocks = (uint32_t)tot_blocks;
    vh->dtype = s.dtype;
    vh->header_bytes = hb;
    vh->payload_bytes = P;
    vh->pool_bytes = pool;
    vh->n_granules = ng;
    vh->status = status;
    if (p.result != nullptr) {
        bs_result r;
        r.total_bytes = total; r.header_bytes = hb; r.payload_bytes = P; r.pool_bytes = pool;
        r.status = status; r.n_tensors = vh->n_tensors; r.n_blocks = (uint32_t)tot_blocks;
        r.reserved[0] = vh->n_structs; r.reserved[1] = vh->n_struct_blocks;
        for (int z = 2; z < 5; ++z) r.reserved[z] = 0;
        r.reserved[2] = s.dtype;
        *p.result = r;
    }
}

// ---- phase 3: blocks [chunk*kLTile, +kLTile) of the flat work table ------------------------------------------------------------
// Block i belongs to the last layer t with first_addr[t] <= i (binary search over lpos[], L2-resident; four searches per
// thread in flight).  Writes blk[i] = {payload offset, address | odd} and the granule boundaries inside the block.
template <bool DESER>
__device__ __forceinline__ void plan_expand_chunk(const LPlanParams& p, uint64_t chunk, uint64_t B, uint64_t T, uint64_t hb,
                                                  const uint32_t* s_index, uint32_t n_index, uint32_t stride,
                                                  uint32_t* big_idx, uint32_t* big_cnt, uint64_t* big_g0)
{
    WsHead* head = p.lw.ws.head;
    const uint32_t tid = threadIdx.x, lane = tid & 31;
    const LayerPos* lpos = p.lw.lpos;

    uint64_t idx[kLItems];
    uint32_t lo[kLItems], hi[kLItems];
#pragma unroll
    for (uint32_t k = 0; k < kLItems; ++k) {  // level 1: the sampled index in shared memory
        idx[k] = chunk * kLTile + (uint64_t)k * kLThreads + tid;
        uint32_t a = 0, b = n_index;  // answer in [a, b): s_index[0] == 0 <= i
        while (b - a > 1) {
            const uint32_t mid = (a + b) >> 1;
            if ((uint64_t)s_index[mid] <= idx[k]) a = mid; else b = mid;
        }
        lo[k] = a * stride;
        hi[k] = (uint64_t)(a + 1) * stride < T ? (a + 1) * stride : (uint32_t)T;
    }
    for (uint32_t span = stride; span > 1; span = (span + 1) >> 1) {  // level 2: ceil(log2 stride) rounds in lpos[]
#pragma unroll
        for (uint32_t k = 0; k < kLItems; ++k) {
            if (hi[k] - lo[k] > 1) {
                const uint32_t mid = (lo[k] + hi[k]) >> 1;
                if (lpos[mid].first_addr <= idx[k]) lo[k] = mid; else hi[k] = mid;
            }
        }
    }
#pragma unroll
    for (uint32_t k = 0; k < kLItems; ++k) {
        const uint64_t i = idx[k];
        bool big = false;
        uint64_t g0 = 0, cnt = 0;
        if (i < B) {
            const LayerPos lp = lpos[lo[k]];
            const uint64_t j = (uint64_t)lp.sfirst + (i - lp.first_addr);
            const uint64_t g = p.lw.gs[j], gn = p.lw.gs[j + 1], gf = p.lw.gs[lp.sfirst];
            const uint64_t off = lp.stream_off + ((g & ~15ull) - (gf & ~15ull));
            const uint64_t stored = (gn & ~15ull) - (g & ~15ull);
            const uint64_t padc = g & 3ull;  // words of zero pad behind the block's data
            uint64_t address;
            if (!DESER) {
                address = __ldg(reinterpret_cast<const unsigned long long*>(p.addr + i));
                if (address & 7) set_err(head, p.result, BS_ERR_ARG);  // D16
            } else if (p.flags == BS_SCATTER_TO_ADDR) {
                address = __ldg(reinterpret_cast<const unsigned long long*>(p.out_addr + i));
                if (address & 7) set_err(head, p.result, BS_ERR_ARG);
            } else {
                address = p.pool_base + lp.off + (p.lw.gp[j] - p.lw.gp[lp.sfirst]);
                p.out_addr[i] = address;
            }
            if (DESER && padc && p.payload != nullptr) {  // pad bytes are zero: the last 16-byte unit of the block
                const uint4 u = __ldg(reinterpret_cast<const uint4*>(p.payload + hb + off + stored - 16));
                const uint32_t w[4] = {u.x, u.y, u.z, u.w};
                uint32_t pad = 0;
#pragma unroll
                for (uint32_t q = 0; q < 4; ++q) pad |= (q >= 4u - (uint32_t)padc) ? w[q] : 0u;
                if (pad != 0) set_err(head, p.result, BS_ERR_CORRUPT);
            }
            Blk e;
            e.off = off;
            e.addr = (address & ~7ull) | padc;  // pad code (Blk): e.g. 2 words = the 8 zero bytes of an odd f64 block
            p.lw.ws.blk[i] = e;
            // granule boundaries g*kGranule inside [off, off + stored)
            g0 = (off + kGranule - 1) / kGranule;
            const uint64_t g1 = (off + stored + kGranule - 1) / kGranule;
            cnt = g1 > g0 ? g1 - g0 : 0;
            if (cnt <= 4) {
                for (uint64_t q = 0; q < cnt; ++q)
                    if (g0 + q < p.lw.ws.n_granules_cap) p.lw.ws.tile_first[g0 + q] = (uint32_t)i;
            } else {
                big = true;
            }
        }
        // large blocks: the whole warp fills their boundaries
        const uint32_t bigs = __ballot_sync(0xffffffffu, big);
        if (bigs) {
            if (big) {
                const uint32_t slot = __popc(bigs & ((1u << lane) - 1u));
                big_idx[slot] = (uint32_t)i;
                big_g0[slot] = g0;
                big_cnt[slot] = cnt > 0xffffffffull ? 0xffffffffu : (uint32_t)cnt;
            }
            __syncwarp();
            const uint32_t nb = __popc(bigs);
            for (uint32_t sl = 0; sl < nb; ++sl) {
                const uint64_t b0 = big_g0[sl];
                const uint32_t c = big_cnt[sl], ix = big_idx[sl];
                for (uint64_t q = lane; q < c; q += 32)
                    if (b0 + q < p.lw.ws.n_granules_cap) p.lw.ws.tile_first[b0 + q] = ix;
            }
            __syncwarp();
        }
    }
}

template <bool DESER>
__global__ void __launch_bounds__(kLThreads) lplan_kernel(const LPlanParams p)
{
    __shared__ uint32_t s_item;
    __shared__ uint32_t s_flag;
    __shared__ ChainSmem<2> sm;
    __shared__ uint32_t s_big_idx[kLThreads];
    __shared__ uint32_t s_big_cnt[kLThreads];
    __shared__ uint64_t s_big_g0[kLThreads];
    __shared__ uint32_t s_index[kLTile];  // first_addr of every stride-th layer: level 1 of the layer search of phase 3
    WsHead* head = p.lw.ws.head;
    const uint32_t tid = threadIdx.x, warp = tid >> 5;
    const PlanShape s = plan_shape<DESER>(p, head);
    const uint32_t n12 = s.n1 + s.n2;
    uint32_t n_index = 0, stride = 1;

    for (;;) {
        __syncthreads();
        if (tid == 0) s_item = atomicAdd(&head->scan_ticket, 1u);
        __syncthreads();
        const uint32_t item = s_item;
        if (item < s.n1) {
            plan_blocks_tile<DESER>(p, s, item, sm);
            __syncthreads();
            if (tid == 0) {
                __threadfence();
                if (atomicAdd(&head->ctas_done, 1u) == s.n1 - 1) {  // phase 1 is complete: hand its status to phase 2
                    __threadfence();
                    const uint32_t st = (*(volatile int*)&head->status != 0) ? 1u : 0u;
                    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(&head->status_pass1), "r"(st | 2u) : "memory");
                }
            }
        } else if (item < n12) {
            if (tid == 0) {
                uint32_t v = 3u;  // no phase 1 (the fixed header was rejected): nothing to scan
                if (s.n1 != 0)
                    while (((v = ld_acquire_u32(&head->status_pass1)) & 2u) == 0) __nanosleep(64);
                s_flag = v & 1u;
            }
            __syncthreads();
            plan_layers_tile<DESER>(p, s, item - s.n1, s_flag != 0, sm);
            __syncthreads();
            if (tid == 0) {
                __threadfence();
                if (atomicAdd(&head->ctas_done2, 1u) == s.n2 - 1) {  // every layer tile is done
                    __threadfence();
                    plan_finalize<DESER>(p, s);
                    __threadfence();
                    asm volatile("st.release.gpu.global.u32 [%0], %1;" ::"l"(&head->scan_ticket2), "r"(1u) : "memory");
                }
            }
        } else {
            cta_wait_until(&head->scan_ticket2, 1u);  // the plan is ready
            const volatile WsHead* vh = head;
            if (vh->status != 0) return;  // deferred error: no table, and the move kernels will write nothing
            const uint64_t B = vh->n_blocks;
            const uint64_t chunk = item - n12;
            if (chunk * kLTile >= B) return;  // every later item is out of range too
            const uint64_t T = vh->n_tensors;
            if (n_index == 0) {  // first chunk of this CTA
                stride = (uint32_t)((T + kLTile - 1) / kLTile);
                n_index = (uint32_t)((T + stride - 1) / stride);
                for (uint32_t q = tid; q < n_index; q += kLThreads) s_index[q] = (uint32_t)p.lw.lpos[(uint64_t)q * stride].first_addr;
                __syncthreads();
            }
            plan_expand_chunk<DESER>(p, chunk, B, T, vh->header_bytes, s_index, n_index, stride, s_big_idx + warp * 32,
                                     s_big_cnt + warp * 32, s_big_g0 + warp * 32);
        }
    }
}

int check_layered(const bs_layered_desc* s)
{
    if (s == nullptr) return BS_ERR_ARG;
    if (s->n_qn != 2 || s->dtype > (uint32_t)BS_C128) return BS_ERR_UNSUPPORTED;
    auto al = [](const void* q, uintptr_t a) { return ((uintptr_t)q & (a - 1)) == 0; };
    if (s->n_structs && (s->structs == nullptr || !al(s->structs, 16))) return BS_ERR_ARG;
    if (s->n_layers && (s->layers == nullptr || !al(s->layers, 16))) return BS_ERR_ARG;
    if (s->n_struct_blocks && (s->qn == nullptr || !al(s->qn, 8))) return BS_ERR_ARG;
    if (s->n_struct_blocks && (s->dim == nullptr || !al(s->dim, 4))) return BS_ERR_ARG;
    if (s->n_addr && (s->addr == nullptr || !al(s->addr, 8))) return BS_ERR_ARG;
    if (s->n_addr >= (1ull << 32)) return BS_ERR_UNSUPPORTED;
    return BS_OK;
}

// one CTA per work item, at most a few waves' worth resident (items are claimed dynamically)
unsigned plan_grid(const LPlanParams& p, int sms)
{
    const uint64_t m = p.Bs > p.C ? p.Bs : p.C;
    uint64_t want = (m + kLTile - 1) / kLTile + (p.T + kLTile - 1) / kLTile + (p.n_addr + kLTile - 1) / kLTile + 3;
    const uint64_t cap = (uint64_t)sms * 8;
    if (want > cap) want = cap;
    return (unsigned)want;
}

}  // namespace

// ---- entry points used by bs_engine.cu -----------------------------------------------------------------------------------
int check_layered_desc(const bs_layered_desc* s) { return check_layered(s); }

bool layered_ws(void* d_ws, uint64_t ws_bytes, uint32_t Bs, uint32_t T, uint64_t B, WsLayout* out)
{
    LwLayout L;
    if (!lw_layout(d_ws, ws_bytes, Bs, T, B, &L)) return false;
    *out = L.ws;
    return true;
}

LayeredView layered_view(const bs_layered_desc* d, void* d_ws, uint64_t ws_bytes)
{
    LayeredView v;
    memset(&v, 0, sizeof(v));
    LwLayout L;
    if (!lw_layout(d_ws, ws_bytes, d->n_struct_blocks, d->n_layers, d->n_addr, &L)) return v;
    v.on = 1;
    v.C = d->n_structs;
    v.Bs = d->n_struct_blocks;
    v.structs = d->structs;
    v.layers = d->layers;
    v.gs = L.gs;
    v.lpos = L.lpos;
    return v;
}

// the three plan launches of a layered serialize (S1, S2, S4 for wire format v2)
int run_layered_serialize_plan(const bs_layered_desc* set, void* d_ws, uint64_t ws_bytes, uint64_t capacity,
                               uint64_t expect_total, bs_result* d_result, int sms, cudaStream_t stream)
{
    LPlanParams p;
    memset(&p, 0, sizeof(p));
    if (!lw_layout(d_ws, ws_bytes, set->n_struct_blocks, set->n_layers, set->n_addr, &p.lw)) return BS_ERR_CAPACITY;
    cudaError_t e = cudaMemsetAsync(p.lw.ws.head, 0, p.lw.ws.zero_bytes, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    p.result = d_result;
    p.capacity = capacity;
    p.expect_total = expect_total;
    p.structs = set->structs;
    p.layers = set->layers;
    p.dim = set->dim;
    p.addr = set->addr;
    p.C = set->n_structs;
    p.Bs = set->n_struct_blocks;
    p.T = set->n_layers;
    p.dtype = set->dtype;
    p.n_addr = set->n_addr;
    lplan_kernel<false><<<plan_grid(p, sms), kLThreads, 0, stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

int run_layered_deserialize_plan(const void* d_header, const void* d_payload, uint64_t nbytes, const bs_layered_desc* out,
                                 void* d_pool, uint64_t pool_bytes, uint32_t flags, void* d_ws, uint64_t ws_bytes,
                                 bs_result* d_result, int sms, cudaStream_t stream)
{
    LPlanParams p;
    memset(&p, 0, sizeof(p));
    if (!lw_layout(d_ws, ws_bytes, out->n_struct_blocks, out->n_layers, out->n_addr, &p.lw)) return BS_ERR_CAPACITY;
    cudaError_t e = cudaMemsetAsync(p.lw.ws.head, 0, p.lw.ws.zero_bytes, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    p.result = d_result;
    p.C = out->n_structs;
    p.Bs = out->n_struct_blocks;
    p.T = out->n_layers;
    p.n_addr = out->n_addr;
    p.header = (const unsigned char*)d_header;
    p.payload = (const unsigned char*)d_payload;
    p.nbytes = nbytes;
    p.pool_base = (uint64_t)(uintptr_t)d_pool;
    p.pool_bytes = pool_bytes;
    p.out_dim = out->dim;
    p.out_addr = out->addr;
    p.flags = flags;
    lplan_kernel<true><<<plan_grid(p, sms), kLThreads, 0, stream>>>(p);
    e = cudaGetLastError();
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

// pm != null: the stream side is a set of package slots (bs_pkg.cu); d_dst is then unused
int run_layered_pack_range(const bs_layered_desc* set, void* d_ws, uint64_t ws_bytes, void* d_dst, uint64_t lo, uint64_t hi,
                           const bs_opts& o, int sms, cudaStream_t stream, const PkgMap* pm, uint32_t flags)
{
    MoveParams mp;
    memset(&mp, 0, sizeof(mp));
    if (!layered_ws(d_ws, ws_bytes, set->n_struct_blocks, set->n_layers, set->n_addr, &mp.ws)) return BS_ERR_CAPACITY;
    mp.lay = layered_view(set, d_ws, ws_bytes);
    mp.qn = set->qn;
    mp.dim = set->dim;
    mp.addr = set->addr;
    mp.stream = (unsigned char*)d_dst;
    mp.lo = lo;
    mp.hi = hi;
    mp.tile_bytes = o.tile_bytes;
    mp.tune = o.tune;
    mp.pace = o.pace;
    mp.flags = flags;
    if (pm) mp.pkg = *pm;
    cudaError_t e = launch_move(false, mp, o, sms, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

int run_layered_unpack_range(const bs_layered_desc* out, void* d_ws, uint64_t ws_bytes, const void* d_src,
                             const void* d_header, uint64_t lo, uint64_t hi, uint32_t flags, const bs_opts& o, int sms,
                             cudaStream_t stream, const PkgMap* pm)
{
    MoveParams mp;
    memset(&mp, 0, sizeof(mp));
    if (!layered_ws(d_ws, ws_bytes, out->n_struct_blocks, out->n_layers, out->n_addr, &mp.ws)) return BS_ERR_CAPACITY;
    mp.lay = layered_view(out, d_ws, ws_bytes);
    mp.qn = out->qn;
    mp.dim = out->dim;
    mp.addr = out->addr;
    mp.stream = (unsigned char*)const_cast<void*>(d_src);
    mp.header = (const unsigned char*)d_header;
    mp.lo = lo;
    mp.hi = hi;
    mp.tile_bytes = o.tile_bytes;
    mp.tune = o.tune;
    mp.pace = o.pace;
    mp.flags = flags;
    if (pm) mp.pkg = *pm;
    cudaError_t e = launch_move(true, mp, o, sms, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    return BS_OK;
}

}  // namespace bs

using namespace bs;

extern "C" {

uint64_t bs_layered_header_bytes(uint64_t n_structs, uint64_t n_layers, uint64_t n_struct_blocks)
{
    return align_up(kFixedHeader + kV2Struct * n_structs + kV2Layer * n_layers + kBlockRec * n_struct_blocks, kHeaderAlign);
}

uint64_t bs_layered_workspace_bytes(uint32_t n_structs, uint32_t n_struct_blocks, uint32_t n_layers, uint64_t n_addr,
                                    uint64_t stream_capacity)
{
    (void)n_structs;
    return lw_fixed_bytes(n_struct_blocks, n_layers, n_addr) + align_up(4 * (stream_capacity / kGranule + 4), 256);
}

int bs_layered_stream_info(const void* h, bs_layered_stream_info_t* out)
{
    if (h == nullptr || out == nullptr) return BS_ERR_ARG;
    const unsigned char* s = (const unsigned char*)h;
    uint32_t w[10];
    uint64_t q[3];
    memcpy(w, s, 40);
    memcpy(q, s + 40, 24);
    if (memcmp(s, "BSPARSE1", 8) != 0) return BS_ERR_CORRUPT;
    if (w[2] != 2u || w[3] != 0x01020304u || w[4] > (uint32_t)BS_C128 || w[5] != 2u || w[6] != 3u || w[7] != 16u) return BS_ERR_CORRUPT;
    if (q[0] >= (1ull << 32)) return BS_ERR_CORRUPT;
    if (q[1] != bs_layered_header_bytes(w[8], q[0], w[9])) return BS_ERR_CORRUPT;
    out->dtype = w[4];
    out->n_structs = w[8];
    out->n_struct_blocks = w[9];
    out->n_layers = q[0];
    out->header_bytes = q[1];
    out->payload_bytes = q[2];
    out->total_bytes = q[1] + q[2];
    return BS_OK;
}

int bs_layered_serialized_size(const bs_layered_desc* set, void* d_ws, uint64_t ws_bytes, uint64_t* header_bytes,
                               uint64_t* total_bytes, cudaStream_t stream)
{
    int rc = check_layered(set);
    if (rc) return rc;
    if (header_bytes == nullptr || total_bytes == nullptr) return BS_ERR_ARG;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    if ((rc = run_layered_serialize_plan(set, d_ws, ws_bytes, UINT64_MAX, 0, nullptr, sms, stream))) return rc;
    WsHead h;
    cudaError_t e = cudaMemcpyAsync(&h, d_ws, sizeof(h), cudaMemcpyDeviceToHost, stream);
    if (e != cudaSuccess) return cuda_fail(e);
    e = cudaStreamSynchronize(stream);
    if (e != cudaSuccess) return cuda_fail(e);
    *header_bytes = h.header_bytes;
    *total_bytes = h.header_bytes + h.payload_bytes;
    if (h.status == BS_ERR_CAPACITY) return BS_OK;  // a workspace too small for the tile index is fine for a size query
    return h.status;
}

int bs_layered_serialize_range(const bs_layered_desc* set, void* d_dst, uint64_t lo, uint64_t hi, int run_scan, void* d_ws,
                               uint64_t ws_bytes, bs_result* d_result, const bs_opts* opts, cudaStream_t stream)
{
    int rc = check_layered(set);
    if (rc) return rc;
    if (d_dst == nullptr || ((uintptr_t)d_dst & 15) || (lo & 15) || (hi & 15) || lo > hi) return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    if ((rc = check_opts(o))) return rc;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    if (run_scan && (rc = run_layered_serialize_plan(set, d_ws, ws_bytes, UINT64_MAX, 0, d_result, sms, stream))) return rc;
    return run_layered_pack_range(set, d_ws, ws_bytes, d_dst, lo, hi, o, sms, stream, nullptr, 0);
}

int bs_layered_serialize(const bs_layered_desc* set, void* d_stream, uint64_t capacity, void* d_ws, uint64_t ws_bytes,
                         bs_result* d_result, const bs_opts* opts, cudaStream_t stream)
{
    int rc = check_layered(set);
    if (rc) return rc;
    if (d_stream == nullptr || ((uintptr_t)d_stream & 15)) return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    if ((rc = check_opts(o))) return rc;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    if ((rc = run_layered_serialize_plan(set, d_ws, ws_bytes, capacity, 0, d_result, sms, stream))) return rc;
    return run_layered_pack_range(set, d_ws, ws_bytes, d_stream, 0, capacity & ~15ull, o, sms, stream, nullptr, 0);
}

int bs_layered_deserialize(const void* d_stream, uint64_t nbytes, bs_layered_desc* out, void* d_pool, uint64_t pool_bytes,
                           uint32_t flags, void* d_ws, uint64_t ws_bytes, bs_result* d_result, const bs_opts* opts,
                           cudaStream_t stream)
{
    int rc = check_layered(out);
    if (rc) return rc;
    if (d_stream == nullptr || ((uintptr_t)d_stream & 15)) return BS_ERR_ARG;
    if (flags != BS_LAYOUT_POOL && flags != BS_SCATTER_TO_ADDR) return BS_ERR_ARG;
    if (flags == BS_LAYOUT_POOL && pool_bytes && (d_pool == nullptr || ((uintptr_t)d_pool & 255))) return BS_ERR_ARG;
    bs_opts o;
    resolve_opts(opts, &o);
    if ((rc = check_opts(o))) return rc;
    int sms;
    if ((rc = device_sm_count(&sms))) return rc;
    const unsigned char* s = (const unsigned char*)d_stream;
    if ((rc = run_layered_deserialize_plan(s, s, nbytes, out, d_pool, pool_bytes, flags, d_ws, ws_bytes, d_result, sms, stream)))
        return rc;
    return run_layered_unpack_range(out, d_ws, ws_bytes, s, s, 0, nbytes & ~15ull, flags, o, sms, stream, nullptr);
}

}  // extern "C"
