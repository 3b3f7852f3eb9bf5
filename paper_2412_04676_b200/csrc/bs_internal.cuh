// bs_internal.cuh — shared declarations of libbsstream's translation units (not part of the C ABI).
//
// Data layout in HBM:
//   workspace := bs_wshead (256 B) | scan_state[n_scan_tiles+1] {word, tag} (16 B each) | blk[B_cap+1] (16 B each)
//                | tile_first[n_granules_cap] u32
//   Nothing in the workspace needs clearing between calls of the v1 scan (bs_scan_phase.cuh): every word the scan
//   synchronises on carries the call's EPOCH tag, so whatever an earlier call (or nobody) left there reads as "not yet
//   written".  (The layered plan of bs_layered.cu still clears its own head + state.)
//   blk[i]        = { payload offset of block i , device address of block i | odd-flag in bit 0 }
//                   — the paper's "pointer structure ... grid structure of the serialized data"
//                   (PAPER L90-92), built before any data moves;  blk[B] = { P, 0 } sentinel.
//   tile_first[g] = index of the block that holds payload byte g*BS_GRANULE  (work partition, S4)
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>

#include "bs.h"

namespace bs {

constexpr uint32_t kFixedHeader = 64;
constexpr uint32_t kTensorRec = 32;
constexpr uint32_t kBlockRec = 48;
constexpr uint32_t kBlockRec4 = 64;  // wire format v3 (BS_RANK4): four legs per block record
constexpr uint32_t kHeaderAlign = 128;
constexpr uint32_t kPoolAlign = 256;
constexpr uint32_t kGranule = 16384;  // bytes of payload per tile_first entry
constexpr uint32_t kMetaBytesPerWarp = 2048;  // TMA variant: shared memory per data warp beside its ring (prefetched block table)

constexpr uint32_t kScanThreads = 256;
constexpr uint32_t kScanItems = 4;
constexpr uint32_t kScanTile = kScanThreads * kScanItems;

struct __align__(16) Blk {
    uint64_t off;   // payload offset (exclusive prefix sum of stored sizes)
    uint64_t addr;  // device address of the dense block (8-byte aligned); bits 0-1 = c: nbytes = stored - 4*c (zero pad)
};

// element size of a dtype (bs.h): f64 8, f32 4, c64 8, c128 16
__host__ __device__ inline uint32_t elem_bytes(uint32_t dtype) { return dtype == BS_F32 ? 4u : (dtype == BS_C128 ? 16u : 8u); }
// legs per block and bytes per block record of a set / stream, from the flags of its dtype word (bs.h BS_RANK4)
__host__ __device__ inline uint32_t legs_of(uint32_t dtype_word) { return (dtype_word & BS_RANK4) ? 4u : 3u; }
__host__ __device__ inline uint32_t block_rec_bytes(uint32_t dtype_word) { return (dtype_word & BS_RANK4) ? kBlockRec4 : kBlockRec; }
__host__ __device__ inline uint64_t header_bytes_of(uint64_t T, uint64_t B, uint32_t dtype_word)
{
    return (kFixedHeader + kTensorRec * T + (uint64_t)block_rec_bytes(dtype_word) * B + (kHeaderAlign - 1)) / kHeaderAlign * kHeaderAlign;
}

struct __align__(16) ScanState {  // one tile of the chained scan: {flag | value, epoch tag}, read and written as ONE 16-byte access
    uint64_t word;
    uint64_t tag;
};

struct __align__(256) WsHead {
    // ---- line 0: what the pass leaves for the data-movement kernels (plain fields, final once the pass is complete) ----
    uint32_t scan_ticket;    // layered plan (bs_layered.cu): dynamic item id
    uint32_t ctas_done;      // layered plan: items of phase 1 done
    int32_t status;          // BS_OK or the first error (the unpack kernels may still flip it: pad check)
    uint32_t n_tensors;
    uint32_t n_blocks;
    uint32_t status_pass1;   // layered sets: status after the first plan pass (read by the second)
    uint64_t header_bytes;
    uint64_t payload_bytes;
    uint64_t pool_bytes;
    uint64_t n_granules;     // ceil(P / kGranule)
    // layered sets (wire format v2, bs_layered.cu): counts and the tickets of the second plan kernel
    uint32_t n_structs;
    uint32_t n_struct_blocks;
    uint32_t scan_ticket2;
    uint32_t ctas_done2;
    uint32_t dtype;          // element type of the set the tables describe (bs.h BS_F64 ..)
    uint32_t pad0[13];
    // ---- the v1 pass's own synchronisation words (bs_scan_phase.cuh), one 128-byte line each: the CTAs of a fused kernel
    // that poll `ready` must not slow the atomics of those still working down ----
    ScanState ready;         // line 1: unused since round 2 (fused kernels poll ep_done and finalise for themselves)
    uint64_t pad1[14];
    uint64_t ep_ticket;      // line 2: work items handed out.  [63:24] a fixed "idle" tag, [23:0] count: the last CTA out of
    uint64_t pad2[15];       //         a launch puts the three counters back to {tag, 0}, so the next launch pays ONE atomic
    uint64_t ep_done;        // line 3: work items completed; the CTA that completes the last one finalises
    uint64_t ep_exit;        //         CTAs that have left the item loop; the last one resets the counters
    uint64_t ep_err;         //         first error of the call: [63:24] epoch tag, [7:0] = -code
    uint64_t unused_r2[2];   //         (round 2 kept the movement's tile counter here; it now lives in the library's own
                             //         device memory, one pair per launch: bs_move_tma.cu "tile hand-out")
    uint64_t pad3[11];
};
static_assert(sizeof(WsHead) == 512, "WsHead is four 128-byte lines");

struct WsLayout {
    WsHead* head;
    ScanState* scan_state;
    Blk* blk;
    uint32_t* tile_first;
    uint64_t n_granules_cap;
    uint64_t zero_bytes;  // head + scan_state: cleared in front of a scan only while a CUDA graph is being captured
};

__host__ __device__ inline uint64_t align_up(uint64_t x, uint64_t a) { return (x + (a - 1)) / a * a; }

inline uint64_t ws_fixed_bytes(uint32_t n_blocks)
{
    uint64_t n_scan_tiles = ((uint64_t)n_blocks + kScanTile) / kScanTile + 1;
    return sizeof(WsHead) + align_up(n_scan_tiles * sizeof(ScanState), 256) + align_up(((uint64_t)n_blocks + 1) * sizeof(Blk), 256);
}

inline bool ws_layout(void* d_ws, uint64_t ws_bytes, uint32_t n_blocks, WsLayout* L)
{
    uint64_t n_scan_tiles = ((uint64_t)n_blocks + kScanTile) / kScanTile + 1;
    uint64_t fixed = ws_fixed_bytes(n_blocks);
    if (d_ws == nullptr || ((uintptr_t)d_ws & 255) != 0 || ws_bytes < fixed + 16) return false;
    unsigned char* p = (unsigned char*)d_ws;
    L->head = (WsHead*)p;
    L->scan_state = (ScanState*)(p + sizeof(WsHead));
    L->zero_bytes = sizeof(WsHead) + align_up(n_scan_tiles * sizeof(ScanState), 256);
    L->blk = (Blk*)(p + L->zero_bytes);
    L->tile_first = (uint32_t*)(p + fixed);
    L->n_granules_cap = (ws_bytes - fixed) / 4;
    return true;
}

// ---- scan pass (S1, S2, S4 / S6): sizes -> offsets -> blk table + tile_first; validation -------------
struct ScanParams {
    WsLayout ws;
    bs_result* result;       // device, may be null
    uint64_t capacity;       // SER: stream capacity; DESER: unused
    uint64_t expect_total;   // SER: if nonzero, total must equal it (engine re-check of the size prediction)
    // SER inputs (descriptor, device arrays)
    const bs_tensor_rec* tensors;
    const uint32_t* dim;
    const uint64_t* addr;
    uint32_t T, B;           // SER: counts; DESER: capacities of the out arrays
    uint32_t dtype;          // SER: element type of the set | BS_ALIGN8 | BS_RANK4; DESER: BS_RANK4 = the shape of the out arrays
    // DESER inputs
    const unsigned char* header;  // stream byte 0 .. header_bytes (device)
    const unsigned char* payload; // stream byte 0 when the payload is resident behind the header (pad-zero check), else null
    uint64_t nbytes;              // total stream length
    uint64_t pool_base;           // BS_LAYOUT_POOL: device address of the pool
    uint64_t pool_bytes;
    const uint32_t* out_dim;      // BS_SCATTER_TO_ADDR inputs
    const uint64_t* out_addr;
    uint32_t flags;
    uint64_t tag;                 // the call's epoch tag (bs_scan_phase.cuh); filled in by the launchers
};

uint64_t next_epoch_tag();
cudaError_t prepare_scan_state(const WsLayout& L, cudaStream_t stream);
cudaError_t launch_scan(bool deser, const ScanParams& p, int sm_count, cudaStream_t stream);

// ---- layered sets (wire format v2): what the header generator / parser of the move kernels needs ---------
struct __align__(32) LayerPos {
    uint64_t off;         // serialize: payload offset of the layer; deserialize: pool offset of the layer
    uint64_t first_addr;  // index of the layer's first block in addr[] / blk[]
    uint64_t stream_off;  // payload offset of the layer (deserialize: from the wire)
    uint32_t sfirst, sn;  // block range of the layer's structure in the structure block table
};
struct LayeredView {
    uint32_t on;                   // 0: wire format v1
    uint32_t C, Bs;                // serialize: counts (deserialize reads them from WsHead)
    bs_struct_rec* structs;        // descriptor arrays: serialize inputs, deserialize outputs
    bs_layer_rec* layers;
    const uint64_t* gs;            // [Bs+1] exclusive prefix of stored sizes over the structure block table | odd bit
    const LayerPos* lpos;          // [T+1]
};

// ---- self-contained packages (bs.h "packages"): the stream is not one buffer but lies cut into slots -------
// cap != 0: stream byte s lives at base + slot(k)*slot_bytes + 64 + (s - lo_k), k = its package under the cut of `cap`,
// slot(k) = slot_of[k] (device table) or k.  The kernels then ignore MoveParams.stream / lo (lo must be 0).  Every
// work tile lies inside one package because cap is a multiple of the tile size and the payload is cut from its start.
struct PkgMap {
    uint64_t cap;
    uint64_t slot_bytes;
    unsigned char* base;
    const uint32_t* slot_of;
    uint64_t k_base;  // without a slot table: package k lies in slot k - k_base (a batch of packages in a staging buffer)
};

// ---- data movement (S3, S5 / S7): stream bytes [lo,hi) <-> blocks ------------------------------------------
struct MoveParams {
    WsLayout ws;
    // descriptor arrays: SER inputs, DESER outputs
    bs_tensor_rec* tensors;
    int32_t* qn;
    uint32_t* dim;
    uint64_t* addr;
    unsigned char* stream;        // p with p[s - lo] = stream byte s   (pack: destination; unpack: source)
    const unsigned char* header;  // DESER: stream byte 0.. (whole header region), null = no descriptor rebuild
    uint64_t lo, hi;
    uint32_t tile_bytes;
    uint32_t flags;
    uint32_t tune;                // bs_opts.tune: launch-shape switches of the TMA variant (bs.h BS_TUNE_*)
    uint32_t pace;                // bs_opts.pace: >= 100: pace the launch at that many GB/s of HBM traffic (experiments)
    uint32_t rank4;               // != 0: qn / dim have four legs per block (BS_RANK4; wire format v3)
    uint32_t mv_slot;             // which tile-counter pair of the library's ring this launch uses (filled in by the launchers)
    LayeredView lay;              // lay.on != 0: qn / dim are the structure block table, header is wire format v2
    PkgMap pkg;                   // pkg.cap != 0: the stream side is a set of package slots
};

// where stream byte s lives (valid for a run of bytes that does not leave s's package; hb = header_bytes)
__device__ __forceinline__ unsigned char* stream_at(const MoveParams& p, uint64_t hb, uint64_t s)
{
    if (p.pkg.cap == 0) return p.stream + (s - p.lo);
    uint64_t k, within;
    if (s < hb) {
        k = s / p.pkg.cap;
        within = s - k * p.pkg.cap;
    } else {
        const uint64_t x = s - hb, j = x / p.pkg.cap;
        k = (hb + p.pkg.cap - 1) / p.pkg.cap + j;
        within = x - j * p.pkg.cap;
    }
    const uint64_t slot = p.pkg.slot_of ? (uint64_t)__ldg(p.pkg.slot_of + k) : k - p.pkg.k_base;
    return p.pkg.base + slot * p.pkg.slot_bytes + 64 + within;
}

cudaError_t launch_move(bool unpack, const MoveParams& p, const bs_opts& opts, int sm_count, cudaStream_t stream);
cudaError_t launch_move_tma(bool unpack, const MoveParams& p, const bs_opts& opts, int sm_count, cudaStream_t stream);
// the size / offset pass and the movement of the whole stream in one launch (TMA variant; bs_move_tma.cu)
cudaError_t launch_fused_tma(bool unpack, const ScanParams& sp, const MoveParams& p, const bs_opts& opts, uint64_t bytes_bound,
                             int sm_count, cudaStream_t stream);

void resolve_opts(const bs_opts* in, bs_opts* out);

// ---- host-side runners shared by the translation units (bs_api.cu, bs_layered.cu) -------------------------------------------
constexpr uint32_t kFlagCheckPad = 0x100u;       // unpack: pad bytes must be zero (engine path; the payload is not resident at parse time)
constexpr uint32_t kFlagNoAlign8 = 0x400u;       // parse pass: the movement that follows cannot take an align-8 stream (LDG variant)
constexpr uint32_t kFlagPoisonOnError = 0x200u;  // pack (engine): a deferred error zeroes the first 64 bytes of the range that holds
                                                 // stream byte 0, so a host buffer never keeps a stale but valid header
int cuda_fail(cudaError_t e);
int device_sm_count(int* out);
int check_set(const bs_set_desc* s);
int check_layered_desc(const bs_layered_desc* s);
int check_opts(const bs_opts& o);
int run_serialize_scan(const bs_set_desc* set, const WsLayout& L, uint64_t capacity, uint64_t expect_total,
                       bs_result* d_result, int sms, cudaStream_t stream);
int run_pack_range(const bs_set_desc* set, const WsLayout& L, void* d_dst, uint64_t lo, uint64_t hi, const bs_opts& o,
                   int sms, cudaStream_t stream, uint32_t flags = 0);
int run_deserialize_scan(const void* d_header, const void* d_payload, uint64_t nbytes, const bs_set_desc* out,
                         void* d_pool, uint64_t pool_bytes, uint32_t flags, const WsLayout& L, bs_result* d_result,
                         int sms, cudaStream_t stream);
int run_unpack_range(const bs_set_desc* out, const WsLayout& L, const void* d_src, const void* d_header, uint64_t lo,
                     uint64_t hi, uint32_t flags, const bs_opts& o, int sms, cudaStream_t stream);
int run_pack_packages(const bs_set_desc* set, const WsLayout& L, const PkgMap& pm, const bs_opts& o, int sms, cudaStream_t stream);
int run_pack_packages_range(const bs_set_desc* set, const WsLayout& L, const PkgMap& pm, uint64_t lo, uint64_t hi, const bs_opts& o,
                            int sms, cudaStream_t stream);
int run_unpack_packages(const bs_set_desc* out, const WsLayout& L, const PkgMap& pm, uint64_t header_bytes, uint32_t flags,
                        const bs_opts& o, int sms, cudaStream_t stream);
int run_unpack_packages_range(const bs_set_desc* out, const WsLayout& L, const PkgMap& pm, uint64_t lo, uint64_t hi, uint32_t flags,
                              const bs_opts& o, int sms, cudaStream_t stream);
// wire format v2 (bs_layered.cu)
bool layered_ws(void* d_ws, uint64_t ws_bytes, uint32_t Bs, uint32_t T, uint64_t B, WsLayout* out);
int run_layered_serialize_plan(const bs_layered_desc* set, void* d_ws, uint64_t ws_bytes, uint64_t capacity,
                               uint64_t expect_total, bs_result* d_result, int sms, cudaStream_t stream);
int run_layered_deserialize_plan(const void* d_header, const void* d_payload, uint64_t nbytes, const bs_layered_desc* out,
                                 void* d_pool, uint64_t pool_bytes, uint32_t flags, void* d_ws, uint64_t ws_bytes,
                                 bs_result* d_result, int sms, cudaStream_t stream);
int run_layered_pack_range(const bs_layered_desc* set, void* d_ws, uint64_t ws_bytes, void* d_dst, uint64_t lo, uint64_t hi,
                           const bs_opts& o, int sms, cudaStream_t stream, const PkgMap* pm = nullptr, uint32_t flags = 0);
int run_layered_unpack_range(const bs_layered_desc* out, void* d_ws, uint64_t ws_bytes, const void* d_src,
                             const void* d_header, uint64_t lo, uint64_t hi, uint32_t flags, const bs_opts& o, int sms,
                             cudaStream_t stream, const PkgMap* pm = nullptr);

}  // namespace bs
