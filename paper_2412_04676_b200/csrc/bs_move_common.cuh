// bs_move_common.cuh — device helpers shared by the data-movement kernels (bs_move.cu: LDG variant,
// bs_move_tma.cu: TMA bulk variant): wire-format v1 header generation (S3) and descriptor rebuild (S7).
#pragma once
#include "bs_internal.cuh"

namespace bs {

constexpr uint32_t kFlagCheckPad = 0x100u;  // unpack: pad bytes must be zero (engine path; see bs_engine.cu)

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
                                             uint64_t P)
{
    uint4 v = make_uint4(0, 0, 0, 0);
    if (u < 4) {
        if (u == 0) v = make_uint4(0x41505342u, 0x31455352u, 1u, 0x01020304u);  // "BSPARSE1", version, endian_tag
        else if (u == 1) v = make_uint4(0u, 2u, 3u, 16u);                        // dtype, n_qn, max_rank, align
        else if (u == 2) v = make_uint4(T, 0u, B, 0u);                           // u64 n_tensors, u64 n_blocks
        else v = make_uint4((uint32_t)hb, (uint32_t)(hb >> 32), (uint32_t)P, (uint32_t)(P >> 32));
        return v;
    }
    u -= 4;
    if (u < 2ull * T) {  // tensor records travel byte for byte
        return __ldg(reinterpret_cast<const uint4*>(p.tensors) + u);
    }
    u -= 2ull * T;
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
            const uint64_t off = p.ws.blk[r].off;
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
        p.addr[r] = p.ws.blk[r].addr & ~7ull;
    }
}

}  // namespace bs
