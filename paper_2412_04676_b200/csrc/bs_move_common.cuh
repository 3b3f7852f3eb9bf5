// bs_move_common.cuh — device helpers shared by the data-movement kernels (bs_move.cu: LDG variant,
// bs_move_tma.cu: TMA bulk variant): wire-format v1 header generation (S3) and descriptor rebuild (S7).
#pragma once
#include "bs_internal.cuh"

namespace bs {


// pack with a deferred error, engine path: the staging buffer goes to the host whatever happened, and it may still hold
// the stream of an earlier call — blank the 64 bytes where this call's fixed header would be
__device__ __forceinline__ void poison_on_error(const MoveParams& p)
{
    if ((p.flags & kFlagPoisonOnError) && p.lo == 0 && p.pkg.cap == 0 && blockIdx.x == 0 && threadIdx.x < 4)
        reinterpret_cast<uint4*>(p.stream)[threadIdx.x] = make_uint4(0, 0, 0, 0);
}

// owner of block r: the last tensor t with first_block[t] <= r (tensors partition the blocks in order)
__device__ __forceinline__ uint32_t tensor_of_block(const bs_tensor_rec* tensors, uint32_t T, uint32_t r)
{
    uint32_t lo = 0, hi = T;  // invariant: first_block[lo] <= r (tensor 0 starts at 0), answer in [lo, hi)
    while (hi - lo > 1) {
        uint32_t mid = (lo + hi) >> 1;
        if (__ldg(&tensors[mid].first_block) <= r) lo = mid; else hi = mid;
    }
    return lo;
}

// ---- S3: one 16-byte unit of the header region (wire format v1) -------------------------------------------
__device__ __forceinline__ uint4 header_unit(const MoveParams& p, uint64_t u, uint32_t T, uint32_t B, uint64_t hb,
                                             uint64_t P, uint32_t dtype)
{
    uint4 v = make_uint4(0, 0, 0, 0);
    const bool r4 = (dtype & BS_RANK4) != 0;  // wire format v3: four legs, 64-byte block records
    if (u < 4) {
        if (u == 0) v = make_uint4(0x41505342u, 0x31455352u, r4 ? 3u : 1u, 0x01020304u);  // "BSPARSE1", version, endian_tag
        else if (u == 1) v = make_uint4(dtype & BS_DTYPE_MASK, 2u, r4 ? 4u : 3u, (dtype & BS_ALIGN8) ? 8u : 16u);  // dtype, n_qn, max_rank, align
        else if (u == 2) v = make_uint4(T, 0u, B, 0u);                           // u64 n_tensors, u64 n_blocks
        else v = make_uint4((uint32_t)hb, (uint32_t)(hb >> 32), (uint32_t)P, (uint32_t)(P >> 32));
        return v;
    }
    u -= 4;
    if (u < 2ull * T) {  // tensor records travel byte for byte
        return __ldg(reinterpret_cast<const uint4*>(p.tensors) + u);
    }
    u -= 2ull * T;
    if (r4) {  // i32 qn[4][2] (two units); u32 dim[4]; u32 tensor, u32 reserved, u64 offset
        if (u < 4ull * B) {
            const uint32_t r = (uint32_t)(u >> 2), part = (uint32_t)(u & 3);
            if (part < 2) {
                v = __ldg(reinterpret_cast<const uint4*>(p.qn + 8ull * r) + part);
            } else if (part == 2) {
                v = __ldg(reinterpret_cast<const uint4*>(p.dim + 4ull * r));
            } else {
                const uint64_t off = __ldcg(reinterpret_cast<const unsigned long long*>(&p.ws.blk[r].off));
                v = make_uint4(tensor_of_block(p.tensors, T, r), 0u, (uint32_t)off, (uint32_t)(off >> 32));
            }
        }
        return v;
    }
    if (u < 3ull * B) {
        const uint32_t r = (uint32_t)(u / 3), part = (uint32_t)(u % 3);
        const int32_t* q = p.qn + 6ull * r;
        const uint32_t* d = p.dim + 3ull * r;
        if (part == 0) {
            int2 a = __ldg(reinterpret_cast<const int2*>(q)), b = __ldg(reinterpret_cast<const int2*>(q + 2));
            v = make_uint4((uint32_t)a.x, (uint32_t)a.y, (uint32_t)b.x, (uint32_t)b.y);
        } else if (part == 1) {
            int2 a = __ldg(reinterpret_cast<const int2*>(q + 4));
            v = make_uint4((uint32_t)a.x, (uint32_t)a.y, __ldg(d), __ldg(d + 1));
        } else {
            const uint64_t off = __ldcg(reinterpret_cast<const unsigned long long*>(&p.ws.blk[r].off));
            v = make_uint4(__ldg(d + 2), tensor_of_block(p.tensors, T, r), (uint32_t)off, (uint32_t)(off >> 32));
        }
    }
    return v;  // slack up to header_bytes: zeros
}

// ---- S7 (descriptor part): one record of the header -> the out descriptor arrays ------------------------------
__device__ __forceinline__ void rebuild_record(const MoveParams& p, uint64_t rec, uint32_t T, uint32_t B)
{
    if (rec < T) {
        const uint4* s = reinterpret_cast<const uint4*>(p.header + kFixedHeader + kTensorRec * rec);
        uint4* d = reinterpret_cast<uint4*>(p.tensors + rec);
        d[0] = __ldg(s);
        d[1] = __ldg(s + 1);
        return;
    }
    const uint64_t r = rec - T;
    if (r >= B) return;
    if (p.rank4) {  // wire format v3: 64-byte records, out arrays with four legs
        const uint4* s = reinterpret_cast<const uint4*>(p.header + kFixedHeader + kTensorRec * (uint64_t)T + kBlockRec4 * r);
        uint4* q = reinterpret_cast<uint4*>(p.qn + 8 * r);
        q[0] = __ldg(s);
        q[1] = __ldg(s + 1);
        if ((p.flags & 1u) == BS_LAYOUT_POOL) {
            *reinterpret_cast<uint4*>(p.dim + 4 * r) = __ldg(s + 2);
            p.addr[r] = __ldcg(reinterpret_cast<const unsigned long long*>(&p.ws.blk[r].addr)) & ~7ull;
        }
        return;
    }
    const uint4* s = reinterpret_cast<const uint4*>(p.header + kFixedHeader + kTensorRec * (uint64_t)T + kBlockRec * r);
    const uint4 r0 = __ldg(s), r1 = __ldg(s + 1), r2 = __ldg(s + 2);
    int2* q = reinterpret_cast<int2*>(p.qn + 6 * r);
    q[0] = make_int2((int)r0.x, (int)r0.y);
    q[1] = make_int2((int)r0.z, (int)r0.w);
    q[2] = make_int2((int)r1.x, (int)r1.y);
    if ((p.flags & 1u) == BS_LAYOUT_POOL) {  // scatter mode: dim / addr are caller inputs, already checked equal
        p.dim[3 * r + 0] = r1.z;
        p.dim[3 * r + 1] = r1.w;
        p.dim[3 * r + 2] = r2.x;
        p.addr[r] = __ldcg(reinterpret_cast<const unsigned long long*>(&p.ws.blk[r].addr)) & ~7ull;
    }
}


// ==== wire format v2 (structure-shared layers; include/bs.h) ==========================================================
// owner of structure block j: the last structure s with first_block[s] <= j and a non-empty range holding j
__device__ __forceinline__ uint32_t struct_of_block(const bs_struct_rec* st, uint32_t C, uint32_t j)
{
    uint32_t lo = 0, hi = C;
    while (hi - lo > 1) {
        uint32_t mid = (lo + hi) >> 1;
        if (__ldg(&st[mid].first_block) <= j) lo = mid; else hi = mid;
    }
    return lo;
}

// S3, v2: one 16-byte unit of the header region.  The plan kernel of bs_layered.cu left gs[] (prefix of stored sizes
// over the structure block table, pad code in bits 0-1), lpos[] (payload offset of every layer) and the set's dtype.
__device__ __forceinline__ uint4 header_unit_v2(const MoveParams& p, uint64_t u, uint32_t T, uint64_t hb, uint64_t P)
{
    const uint32_t C = p.lay.C, Bs = p.lay.Bs;
    uint4 v = make_uint4(0, 0, 0, 0);
    if (u < 4) {
        if (u == 0) v = make_uint4(0x41505342u, 0x31455352u, 2u, 0x01020304u);  // "BSPARSE1", version 2, endian_tag
        else if (u == 1) v = make_uint4(p.ws.head->dtype, 2u, 3u, 16u);          // dtype, n_qn, max_rank, align
        else if (u == 2) v = make_uint4(C, Bs, T, 0u);                           // u32 C, u32 Bs, u64 n_layers
        else v = make_uint4((uint32_t)hb, (uint32_t)(hb >> 32), (uint32_t)P, (uint32_t)(P >> 32));
        return v;
    }
    u -= 4;
    if (u < 2ull * C) {
        const uint32_t s = (uint32_t)(u >> 1);
        const uint4 w = __ldg(reinterpret_cast<const uint4*>(p.lay.structs) + u);
        if ((u & 1) == 0) return w;  // rank, first_block, n_blocks, dq[0]
        const uint32_t f = __ldg(&p.lay.structs[s].first_block), n = __ldg(&p.lay.structs[s].n_blocks);
        const uint64_t lb = (p.lay.gs[f + n] & ~15ull) - (p.lay.gs[f] & ~15ull);
        return make_uint4(w.x, w.y, (uint32_t)lb, (uint32_t)(lb >> 32));  // dq[1], sign, layer_bytes
    }
    u -= 2ull * C;
    if (u < T) {
        const uint2 w = __ldg(reinterpret_cast<const uint2*>(p.lay.layers + u));  // structure, tag
        const uint64_t off = p.lay.lpos[u].off;
        return make_uint4(w.x, w.y, (uint32_t)off, (uint32_t)(off >> 32));
    }
    u -= T;
    if (u < 3ull * Bs) {
        const uint32_t r = (uint32_t)(u / 3), part = (uint32_t)(u % 3);
        const int32_t* q = p.qn + 6ull * r;
        const uint32_t* d = p.dim + 3ull * r;
        if (part == 0) {
            int2 a = __ldg(reinterpret_cast<const int2*>(q)), b = __ldg(reinterpret_cast<const int2*>(q + 2));
            v = make_uint4((uint32_t)a.x, (uint32_t)a.y, (uint32_t)b.x, (uint32_t)b.y);
        } else if (part == 1) {
            int2 a = __ldg(reinterpret_cast<const int2*>(q + 4));
            v = make_uint4((uint32_t)a.x, (uint32_t)a.y, __ldg(d), __ldg(d + 1));
        } else {
            const uint32_t s = struct_of_block(p.lay.structs, C, r);
            const uint64_t rel = (p.lay.gs[r] & ~15ull) - (p.lay.gs[__ldg(&p.lay.structs[s].first_block)] & ~15ull);
            v = make_uint4(__ldg(d + 2), s, (uint32_t)rel, (uint32_t)(rel >> 32));
        }
    }
    return v;
}

// S7, v2 (descriptor part): record `rec` of the header -> structs / layers / qn / dim.  addr[] was written by the
// expansion kernel of bs_layered.cu.
__device__ __forceinline__ void rebuild_record_v2(const MoveParams& p, uint64_t rec, uint32_t C, uint32_t T, uint32_t Bs)
{
    const unsigned char* h = p.header + kFixedHeader;
    if (rec < C) {
        const uint4* s = reinterpret_cast<const uint4*>(h + 32 * rec);
        uint4* d = reinterpret_cast<uint4*>(p.lay.structs + rec);
        d[0] = __ldg(s);
        d[1] = __ldg(s + 1);
        return;
    }
    rec -= C;
    if (rec < T) {
        *reinterpret_cast<uint4*>(p.lay.layers + rec) = __ldg(reinterpret_cast<const uint4*>(h + 32ull * C + 16 * rec));
        return;
    }
    rec -= T;
    if (rec >= Bs) return;
    const uint4* s = reinterpret_cast<const uint4*>(h + 32ull * C + 16ull * T + kBlockRec * rec);
    const uint4 r0 = __ldg(s), r1 = __ldg(s + 1), r2 = __ldg(s + 2);
    int2* q = reinterpret_cast<int2*>(p.qn + 6 * rec);
    q[0] = make_int2((int)r0.x, (int)r0.y);
    q[1] = make_int2((int)r0.z, (int)r0.w);
    q[2] = make_int2((int)r1.x, (int)r1.y);
    if ((p.flags & 1u) == BS_LAYOUT_POOL) {  // scatter mode: dim is a caller input, already checked equal
        p.dim[3 * rec + 0] = r1.z;
        p.dim[3 * rec + 1] = r1.w;
        p.dim[3 * rec + 2] = r2.x;
    }
}

// ---- format dispatch used by both move kernels ---------------------------------------------------------------------------
__device__ __forceinline__ uint4 header_unit_any(const MoveParams& p, uint64_t u, uint32_t T, uint32_t B, uint64_t hb,
                                                 uint64_t P)
{
    return p.lay.on ? header_unit_v2(p, u, T, hb, P) : header_unit(p, u, T, B, hb, P, p.ws.head->dtype);
}
__device__ __forceinline__ uint64_t n_rebuild_records(const MoveParams& p, const WsHead* head)
{
    return p.lay.on ? (uint64_t)head->n_structs + head->n_tensors + head->n_struct_blocks
                    : (uint64_t)head->n_tensors + head->n_blocks;
}
__device__ __forceinline__ void rebuild_record_any(const MoveParams& p, const WsHead* head, uint64_t rec)
{
    if (p.lay.on) rebuild_record_v2(p, rec, head->n_structs, head->n_tensors, head->n_struct_blocks);
    else rebuild_record(p, rec, head->n_tensors, head->n_blocks);
}

// ---- warp-level header workers (TMA variant: a dedicated warp per CTA runs these beside the data warps) -------
// Header worker `hw` of `n_hw` (one warp each).  Nothing here depends on another worker.

// S3 for stream bytes [lo, hend), hend <= header_bytes: fixed header, tensor records and zero slack unit by unit
// (few); block records one LANE per record, four records per lane in flight, each worker a contiguous run of
// records so the owning tensor is found by one binary search and then only ever steps forward.
__device__ __forceinline__ void write_header_warp(const MoveParams& p, uint32_t T, uint32_t B, uint64_t hb, uint64_t P,
                                                  uint32_t dtype, uint64_t lo, uint64_t hend, uint64_t hw, uint64_t n_hw,
                                                  uint32_t lane)
{
    if (lo >= hend) return;
    if (dtype & BS_RANK4) {  // wire format v3: unit by unit (sets of order-4 tensors are small beside the operator sets)
        const uint64_t u0 = lo / 16, n = (hend - lo) / 16;
        for (uint64_t i = hw * 32 + lane; i < n; i += n_hw * 32)
            __stcs(reinterpret_cast<uint4*>(stream_at(p, hb, lo + i * 16)), header_unit(p, u0 + i, T, B, hb, P, dtype));
        return;
    }
    const uint64_t rec0 = kFixedHeader + kTensorRec * (uint64_t)T;  // stream offset of block record 0
    const uint64_t rec_end = rec0 + kBlockRec * (uint64_t)B;
    {   // everything that is not a block record
        const uint64_t n_head = rec0 / 16, n_slack = (hb - rec_end) / 16;
        for (uint64_t i = hw * 32 + lane; i < n_head + n_slack; i += n_hw * 32) {
            const uint64_t u = i < n_head ? i : rec_end / 16 + (i - n_head);
            const uint64_t s = u * 16;
            if (s >= lo && s < hend) __stcs(reinterpret_cast<uint4*>(stream_at(p, hb, s)), header_unit(p, u, T, B, hb, P, dtype));
        }
    }
    if (B == 0 || hend <= rec0 || lo >= rec_end) return;
    const uint64_t r_lo = lo > rec0 ? (lo - rec0) / kBlockRec : 0;                        // first record touching [lo, hend)
    const uint64_t r_hi = hend < rec_end ? (hend - rec0 + kBlockRec - 1) / kBlockRec : B;  // one past the last
    const uint64_t per = (r_hi - r_lo + n_hw - 1) / n_hw;
    const uint64_t my0 = r_lo + hw * per, my1 = my0 + per < r_hi ? my0 + per : r_hi;
    if (my0 >= my1) return;
    uint32_t t = tensor_of_block(p.tensors, T, (uint32_t)my0);  // warp-uniform; each lane then walks forward
    constexpr int K = 4;
    for (uint64_t base = my0; base < my1; base += 32 * K) {
        int2 q0[K], q1[K], q2[K];
        uint32_t d0[K], d1[K], d2[K];
        uint64_t off[K];
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint64_t r = base + (uint64_t)k * 32 + lane;
            if (r < my1) {
                const int2* q = reinterpret_cast<const int2*>(p.qn + 6 * r);
                q0[k] = __ldg(q); q1[k] = __ldg(q + 1); q2[k] = __ldg(q + 2);
                d0[k] = __ldg(p.dim + 3 * r); d1[k] = __ldg(p.dim + 3 * r + 1); d2[k] = __ldg(p.dim + 3 * r + 2);
                off[k] = __ldcg(reinterpret_cast<const unsigned long long*>(&p.ws.blk[r].off));  // L2: fused kernels
            }
        }
#pragma unroll
        for (int k = 0; k < K; ++k) {
            const uint64_t r = base + (uint64_t)k * 32 + lane;
            if (r < my1) {
                while (t + 1 < T && __ldg(&p.tensors[t + 1].first_block) <= r) ++t;  // tensors partition the blocks in order
                const uint64_t s = rec0 + kBlockRec * r;
                const uint4 v0 = make_uint4((uint32_t)q0[k].x, (uint32_t)q0[k].y, (uint32_t)q1[k].x, (uint32_t)q1[k].y);
                const uint4 v1 = make_uint4((uint32_t)q2[k].x, (uint32_t)q2[k].y, d0[k], d1[k]);
                const uint4 v2 = make_uint4(d2[k], t, (uint32_t)off[k], (uint32_t)(off[k] >> 32));
                if (s >= lo && s < hend) __stcs(reinterpret_cast<uint4*>(stream_at(p, hb, s)), v0);
                if (s + 16 >= lo && s + 16 < hend) __stcs(reinterpret_cast<uint4*>(stream_at(p, hb, s + 16)), v1);
                if (s + 32 >= lo && s + 32 < hend) __stcs(reinterpret_cast<uint4*>(stream_at(p, hb, s + 32)), v2);
            }
        }
    }
}

// S3, v2: the header is small when layers share structures (48 bytes per STRUCTURE block); unit by unit
__device__ __forceinline__ void write_header_warp_v2(const MoveParams& p, uint32_t T, uint64_t hb, uint64_t P, uint64_t lo,
                                                     uint64_t hend, uint64_t hw, uint64_t n_hw, uint32_t lane)
{
    if (lo >= hend) return;
    const uint64_t u0 = lo / 16, n = (hend - lo) / 16;
    for (uint64_t i = hw * 32 + lane; i < n; i += n_hw * 32)
        __stcs(reinterpret_cast<uint4*>(stream_at(p, hb, lo + i * 16)), header_unit_v2(p, u0 + i, T, hb, P));
}

// S7 (descriptor part): records [0, T+B) of p.header -> the out descriptor arrays, 128 records per step
__device__ __forceinline__ void rebuild_header_warp(const MoveParams& p, uint32_t T, uint32_t B, uint64_t hw, uint64_t n_hw,
                                                    uint32_t lane)
{
    (void)T; (void)B;
    const WsHead* head = p.ws.head;
    const uint64_t n_rec = n_rebuild_records(p, head);
    for (uint64_t base = hw * 128; base < n_rec; base += n_hw * 128) {
#pragma unroll
        for (int k = 0; k < 4; ++k) rebuild_record_any(p, head, base + (uint64_t)k * 32 + lane);
    }
}


// the same for wire format v1 with the counts in registers (fused kernels: the workspace head may not be written yet)
__device__ __forceinline__ void rebuild_header_warp_v1(const MoveParams& p, uint32_t T, uint32_t B, uint64_t hw, uint64_t n_hw,
                                                       uint32_t lane)
{
    const uint64_t n_rec = (uint64_t)T + B;
    for (uint64_t base = hw * 128; base < n_rec; base += n_hw * 128) {
#pragma unroll
        for (int k = 0; k < 4; ++k) rebuild_record(p, base + (uint64_t)k * 32 + lane, T, B);
    }
}

}  // namespace bs
