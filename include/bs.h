/*
 * bs.h — C ABI of libbsstream: serialize / deserialize / offload / prefetch of symmetry-blocked
 * (U(1) quantum-number-labelled) block-sparse matrices and rank-3 tensors (fp64; also f32 / c64 / c128) on one NVIDIA B200.
 *
 * The operations are those of arXiv 2412.04676 (Menczer & Legeza), /root/reference/PAPER.md:
 *   - §III (L85): saving scratch data = (1) serialization, "generating long continuous stripes in
 *     memory", (2) transfer to a storage medium; loading = transfer + deserialization.
 *   - §III.B.2 (L104-108): exact size prediction before serialization; every worker gets an exact,
 *     disjoint interval of one output buffer; independent parallel fill; the single stream
 *     "deserializes into an object identical to the one used as the original input".
 *   - §II.B (L63): blocks travel with their meta data (sector indices, quantum numbers, sector dims).
 *   - §III.A (L89-92), §III.B.4 (L132-138): segment-wise synchronous IO, asynchronous save / load
 *     overlapped with computation, with a completion point ("checkpoint") before the data is used.
 * The paper defines no byte format; "wire format v1" below is this project's.
 *
 * Conventions
 *   - Every function returns int: BS_OK (0), BS_PENDING (1) or a negative BS_ERR_*.
 *   - Pointers named d_* are DEVICE pointers, h_* are HOST pointers (h_pinned: page-locked).  Structs
 *     passed by pointer (bs_set_desc, bs_opts, bs_engine_cfg, bs_stream_info_t) live on the HOST.
 *   - Ownership: the caller owns every buffer it passes (descriptor arrays, blocks, stream, pool,
 *     workspace, pinned host memory) and keeps it alive and unmodified until the stream work / ticket
 *     of the call has completed.  The library owns only what bs_engine_create allocates.
 *   - Calls enqueue work on the given cudaStream_t and return without synchronising unless stated.
 *     Errors detected on the device (capacity, corrupt header, bad descriptor) are DEFERRED: they land
 *     in bs_result.status (device memory) and, for engine calls, in the ticket.  When status != BS_OK
 *     no stream / block / descriptor output has been written by the data-movement kernels.
 *   - The path does no floating-point arithmetic: values move as opaque words of their element size; results
 *     are bit-exact (tolerance 0).
 *   - Thread-safety: functions are re-entrant; one bs_engine must be driven by one host thread.
 *   - There is no CPU fallback: without a CUDA device every device-touching call fails with BS_ERR_CUDA.
 *
 * Wire format v1 (little-endian, no implicit padding):
 *   stream  := fixed_header(64) | tensor_rec[T](32 each) | block_rec[B](48 each) | zeros to a multiple
 *              of 128 | payload(P)
 *   fixed_header: char magic[8]="BSPARSE1"; u32 version=1; u32 endian_tag=0x01020304; u32 dtype (0 f64,
 *                 1 f32, 2 c64, 3 c128: element size e = 8, 4, 8, 16); u32 n_qn=2; u32 max_rank=3; u32 align=16 (8: BS_ALIGN8
 *                 below, then read align8 for align16 in the payload rule); u64 n_tensors; u64 n_blocks;
 *                 u64 header_bytes; u64 payload_bytes
 *   tensor_rec  : bs_tensor_rec, byte for byte
 *   block_rec   : i32 qn[3][2]; u32 dim[3]; u32 tensor; u64 offset
 *   payload     : block i's e*prod(dim_i) raw bytes at payload+offset_i, then zeros up to the next
 *                 multiple of 16; offset_i = sum_{j<i} align16(e*prod(dim_j))   (descriptor order)
 */
#ifndef BS_H_
#define BS_H_

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

#if defined(__CUDACC__) || defined(CUDART_VERSION) || defined(__DRIVER_TYPES_H__)
/* cudaStream_t comes from the CUDA headers */
#else
typedef struct CUstream_st *cudaStream_t;
#endif

#define BS_VERSION 0x00010200u /* library 1.2 (1.1 = round 2: bs_stream_info_t grew by align / max_rank, bs_layered_stream_info_t by
                                  dtype, bs_workspace_bytes grew: rebuild callers against this header); wire formats v1, v2, v3 */

enum {
    BS_OK = 0,
    BS_PENDING = 1,          /* bs_ticket_query: work still in flight */
    BS_ERR_ARG = -1,         /* NULL / misaligned pointer, bad descriptor partition, size overflow */
    BS_ERR_CAPACITY = -2,    /* stream / pool / workspace / descriptor arrays too small */
    BS_ERR_CORRUPT = -3,     /* header validation failed; nothing was written */
    BS_ERR_UNSUPPORTED = -4, /* rank not in {2,3} ({2,3,4} in a BS_RANK4 set), unknown dtype, n_qn != 2 */
    BS_ERR_CUDA = -5,        /* a CUDA runtime call failed; see bs_last_cuda_error() */
    BS_ERR_IO = -6           /* the storage tier of a bs_queue: open / read / write of a file failed (errno is the C library's) */
};

/* Element type of every block of a set (bs_set_desc.dtype; the header's dtype word).  The path does no arithmetic on the
 * values: the type only fixes the element size e, nbytes = e * prod(dim).  Both wire formats carry
 * every type (a stream holds blocks of ONE type). */
enum { BS_F64 = 0 /* e = 8 */, BS_F32 = 1 /* e = 4 */, BS_C64 = 2 /* e = 8 */, BS_C128 = 3 /* e = 16 */ };

/* Stream alignment (DESIGN.md §18 reading D19).  OR-ed into bs_set_desc.dtype of a set that
 * is SERIALIZED: the stream is written with the header's align word = 8 instead of 16, i.e. stored_i = align8(nbytes_i) — no
 * pad byte at all for f64 / c64 / c128 blocks (f32: 0 or 4) — so block offsets are the literal exclusive prefix sum of the
 * block byte sizes and the stream's total is a multiple of 8, not of 16.  Deserialize / prefetch take the alignment from the
 * stream; bs_result.reserved[2] and bs_stream_info_t report it.  Wire format v1 and the TMA variant only (BS_ERR_UNSUPPORTED
 * for layered sets and for BS_VARIANT_LDG).  Blocks whose stream offset and address differ by 8 modulo 16 cannot go through
 * the bulk-copy engine and move as 8-byte words: expect roughly half the bandwidth of the padded format on sets with many
 * odd-sized blocks (DESIGN.md §18 has the numbers). */
#define BS_ALIGN8 0x100u
/* Tensors of rank up to 4 ("tree-like tensor network state methods": the nodes of a tree
 * tensor network state are order-4; DESIGN.md §19 reading D20).  OR-ed into bs_set_desc.dtype it says that the per-block
 * arrays have FOUR legs — qn [B][4][2], dim [B][4] — and that tensors may have rank 2, 3 or 4 (unused legs: dim 1, labels 0).
 * The stream is then WIRE FORMAT v3 = v1 with a fourth leg:
 *   fixed_header: as v1 with version = 3 and max_rank = 4;  tensor_rec: as v1;
 *   block_rec   : i32 qn[4][2]; u32 dim[4]; u32 tensor; u32 reserved = 0; u64 offset      (64 bytes)
 *   header_bytes = align128(64 + 32*T + 64*B) = bs_header_bytes_rank4(T, B);  payload and pool layout as v1.
 * For deserialize / prefetch outputs the flag says how the caller shaped `out`'s arrays: a v3 stream needs it, a v1 stream must
 * not have it (BS_ERR_ARG otherwise).  qn and dim of such a set must be 16-byte aligned (BS_ERR_ARG at once otherwise: their
 * rows move as 16-byte words).  Not combined with BS_ALIGN8 or layered sets (BS_ERR_UNSUPPORTED). */
#define BS_RANK4 0x200u
#define BS_DTYPE_MASK 0xffu

/* bs_deserialize / bs_prefetch_async destination layout */
enum {
    BS_LAYOUT_POOL = 0,     /* out->addr[i] = d_pool + sum_{j<i} align256(nbytes_j); written by the call */
    BS_SCATTER_TO_ADDR = 1  /* out->addr[i] and out->dim are INPUTS: caller-chosen destinations; extents
                               must equal the stream's, else BS_ERR_ARG */
};

/* One tensor of the set; 32 bytes; identical bytes on the wire (PAPER L63 meta data). */
typedef struct bs_tensor_rec {
    uint32_t rank;        /* 2 (operator matrix) or 3 (MPS site tensor, PAPER Eq. 2); 4 in a BS_RANK4 set (tree node) */
    uint32_t first_block; /* index of its first block in the per-block arrays */
    uint32_t n_blocks;    /* tensors partition the block table in order: first_block[t+1] = first_block[t] + n_blocks[t] */
    int32_t dq[2];        /* conserved charge (dN, d2Sz): sum_k sign[k]*qn[k] == dq for every block */
    int8_t sign[4];       /* leg arrows +-1; unused legs 0 */
    uint32_t tag;         /* opaque user id */
    uint32_t reserved;    /* 0 */
} bs_tensor_rec;

/* A set of block-sparse tensors.  HOST struct; every pointer is a DEVICE pointer. */
typedef struct bs_set_desc {
    uint32_t n_tensors;     /* T.  For bs_deserialize / bs_prefetch_async outputs: CAPACITY of tensors[] */
    uint32_t n_blocks;      /* B.  For outputs: CAPACITY of qn / dim / addr */
    uint32_t n_qn;          /* 2: (N, 2Sz) */
    uint32_t dtype;         /* BS_F64, BS_F32, BS_C64 or BS_C128, optionally | BS_ALIGN8 or | BS_RANK4; for outputs: 0 or
                               BS_RANK4 (the shape of qn / dim), the stream's type comes back in bs_result */
    bs_tensor_rec *tensors; /* [T]        */
    int32_t *qn;            /* [B][3][2]  labels per leg; unused legs 0; 8-byte aligned   (BS_RANK4: [B][4][2], 16-byte aligned) */
    uint32_t *dim;          /* [B][3]     extents; unused legs 1; 4-byte aligned          (BS_RANK4: [B][4], 16-byte aligned)    */
    uint64_t *addr;         /* [B]        device address of each dense, contiguous, row-major (last index
                                          fastest) block; must be 8-byte aligned, 16-byte aligned for the
                                          vector fast path */
} bs_set_desc;

/* Deferred outcome of one call; 64 bytes in DEVICE memory, written by the call's kernels. */
typedef struct bs_result {
    uint64_t total_bytes;   /* header_bytes + payload_bytes (required capacity, also on BS_ERR_CAPACITY) */
    uint64_t header_bytes;
    uint64_t payload_bytes;
    uint64_t pool_bytes;    /* deserialize: bytes BS_LAYOUT_POOL needs = sum align256(nbytes_i) */
    int32_t status;         /* BS_OK or BS_ERR_* */
    uint32_t n_tensors;
    uint32_t n_blocks;
    uint32_t reserved[5];   /* [0], [1]: see bs_layered_*; [2] = dtype of the stream (| BS_ALIGN8 / BS_RANK4 as the stream is);
                               [3]: see bs_package_emit */
} bs_result;

typedef struct bs_stream_info_t {
    uint64_t n_tensors, n_blocks, header_bytes, payload_bytes, total_bytes;
    uint64_t dtype; /* BS_F64 .. BS_C128 */
    uint64_t align; /* 16 or 8 (BS_ALIGN8) */
    uint64_t max_rank; /* 3 (wire format v1) or 4 (wire format v3, BS_RANK4) */
} bs_stream_info_t;

/* Launch tuning.  NULL everywhere means defaults.  The stream produced never depends on these
 * (decomposition independence; tests/test_gpu_parity.py P6). */
typedef struct bs_opts {
    uint32_t variant;     /* 0 = default; 1 = BS_VARIANT_LDG (16-byte vector loads/stores);
                             2 = BS_VARIANT_TMA (cp.async.bulk global<->shared staging, one ring of tiles per warp) */
    uint32_t tile_bytes;  /* stream bytes per work tile; 0 = default; <= 65536 and a multiple of 16384 (LDG) or of 1024, >= 4096 (TMA) */
    uint32_t ctas_per_sm; /* LDG: persistent CTAs per SM; 0 = default (occupancy limit) */
    uint32_t stages;      /* TMA: ring depth (tiles) per warp, 3..8; 0 = default */
    uint32_t warps;       /* TMA: warps (rings) per CTA, 1..16; warps*stages*tile_bytes <= 225 KiB; 0 = default */
    uint32_t tune;        /* TMA: how tiles are handed out and how far ahead a tile's block table is fetched — OR of BS_TUNE_* below;
                             0 = by size.  The static deal and the forced counter are what the decomposition tests (P6) and
                             bench.py --ab compare; the remaining bits are measurement switches of DESIGN.md §20 (each measured and
                             left off by default).  Bits outside BS_TUNE_KNOWN_BITS: BS_ERR_ARG. */
    uint32_t fuse;        /* bs_serialize / bs_deserialize as ONE launch (size / offset pass + movement in one kernel): 0 = by size
                             (sets of up to ~150 k blocks), 1 = never, 2 = always; > 2: BS_ERR_ARG */
    uint32_t pace;        /* TMA, measurements only: a warp starts the loads of its next tile no earlier than its share of a target
                             traffic rate allows; 0 (and anything < 100) = none, >= 100 = that many GB/s of HBM traffic for the launch */
} bs_opts;
enum { BS_VARIANT_DEFAULT = 0, BS_VARIANT_LDG = 1, BS_VARIANT_TMA = 2 };
/* bs_opts.tune (until round 2 these rode in a field called `reserved`; same offsets, so the struct layout is unchanged) */
#define BS_TUNE_EVICT_FIRST_LD 0x1u    /* L2 evict_first hint on bulk loads (measured: no gain) */
#define BS_TUNE_EVICT_FIRST_ST 0x2u    /* ... on bulk stores */
#define BS_TUNE_DEAL_STATIC    0x8u    /* tiles dealt round-robin (round 1) whatever the size */
#define BS_TUNE_DEAL_COUNTER   0x10u   /* tiles from the launch's counter whatever the size (default: ranges of >= 128 MiB) */
#define BS_TUNE_L2_PREFETCH    0x20u   /* unpack asks the next stream tile into L2 (measured: inside the spread) */
#define BS_TUNE_MAX_LOADS_MASK 0xf00u  /* at most ((tune >> 8) & 15) tiles loading beside the one being stored; 0 = ring depth - 2 */
#define BS_TUNE_TABLE_AHEAD_2  0x1000u /* block table fetched two iterations ahead (default: pack of sets >= 512 MiB) */
#define BS_TUNE_KNOWN_BITS     0x1f3bu

/* ---- host-only helpers ------------------------------------------------------------------------ */
uint32_t bs_version(void);
const char *bs_strerror(int code);
int bs_last_cuda_error(void); /* cudaError_t of the last BS_ERR_CUDA on this thread */

/* align128(64 + 32*T + 48*B): the header size is known from the counts alone. */
uint64_t bs_header_bytes(uint64_t n_tensors, uint64_t n_blocks);
/* align128(64 + 32*T + 64*B): the same for a BS_RANK4 set (wire format v3). */
uint64_t bs_header_bytes_rank4(uint64_t n_tensors, uint64_t n_blocks);

/* Bytes of device workspace a call needs for a set of up to n_blocks blocks whose stream is at most
 * stream_capacity bytes: the offset table ("pointer structure"), scan state and the calls' work counters.
 * 256-byte aligned; it may be uninitialised memory (every word the kernels synchronise on carries a tag) and is reusable
 * from call to call, but it serves ONE pass at a time: calls that run the size / offset or parse pass (bs_serialized_size,
 * bs_serialize, bs_deserialize, a range call with run_scan) and may run concurrently (two streams) need a workspace each.
 * Range calls behind a completed pass only read it and may overlap one another (see bs_deserialize_range). */
uint64_t bs_workspace_bytes(uint32_t n_tensors, uint32_t n_blocks, uint64_t stream_capacity);

/* Parse the 64-byte fixed header (HOST memory).  BS_ERR_CORRUPT if it is not a v1 or v3 header. */
int bs_stream_info(const void *h_first_64_bytes, bs_stream_info_t *out);

/* ---- serialize ------------------------------------------------------------ */

/* Exact size of the stream before any data moves.  Runs the size/offset pass on `stream`
 * and SYNCHRONISES it.  header_bytes / total_bytes are HOST outputs. */
int bs_serialized_size(const bs_set_desc *set, void *d_workspace, uint64_t workspace_bytes,
                       uint64_t *header_bytes, uint64_t *total_bytes, cudaStream_t stream);

/* Write the stream of `set` to d_stream[0 .. total).  d_stream 16-byte aligned, `capacity` bytes.
 * Asynchronous.  d_result (DEVICE, 64 bytes) receives total/header/payload bytes and the status:
 * BS_ERR_CAPACITY if total > capacity (total_bytes = required size), BS_ERR_ARG for a descriptor that
 * does not partition its blocks, a block address not 8-byte aligned or a size overflow,
 * BS_ERR_UNSUPPORTED for rank not in {2,3} (BS_RANK4 sets: {2,3,4}).  Every byte of [0,total) is written, including padding. */
int bs_serialize(const bs_set_desc *set, void *d_stream, uint64_t capacity, void *d_workspace,
                 uint64_t workspace_bytes, bs_result *d_result, const bs_opts *opts, cudaStream_t stream);

/* Segment form (Fig 4(b)): write stream bytes [lo, hi) to d_dst[0 .. hi-lo).  lo, hi
 * multiples of 16 (hi is clipped to the total).  The size/offset pass must have run on the same
 * workspace (bs_serialized_size, bs_serialize or a previous range call with lo == 0 runs it).
 * run_scan != 0 runs it first.  concat over a partition of [0,total) == the bs_serialize stream. */
int bs_serialize_range(const bs_set_desc *set, void *d_dst, uint64_t lo, uint64_t hi, int run_scan,
                       void *d_workspace, uint64_t workspace_bytes, bs_result *d_result,
                       const bs_opts *opts, cudaStream_t stream);

/* bs_serialize without a workspace argument and without any allocation: for callers that cannot get device memory at the
 * moment they must save a set.  That is the normal state of the solver this library serves — it hands whatever HBM is
 * left to its own block pool, and the memory peaks of PAPER L132-136 are the very reason data is pushed out, so a
 * cudaMalloc then fails or is forbidden (a plug-in may not allocate behind the host program's pool) — and of any caller
 * that cannot afford the device-wide synchronisation a cudaMalloc / cudaFree brings while side streams are busy.
 *   - The workspace is a fixed array of bs_noalloc_scratch_bytes() = 1.5 MiB of device memory inside the library, held
 *     on every GPU the library is used on from the moment its code is loaded there until the process exits.  The call
 *     itself calls no cudaMalloc, cudaFree or other allocating routine; set, d_stream and d_result are still the
 *     caller's, exactly as for bs_serialize, and the stream written is byte for byte bs_serialize's.
 *   - Limits: set->n_blocks <= BS_NOALLOC_MAX_BLOCKS and capacity <= BS_NOALLOC_MAX_STREAM_BYTES (pass the smaller of
 *     your buffer size and the limit).  Beyond either the call returns BS_ERR_CAPACITY at once and enqueues nothing;
 *     a stream that turns out larger than `capacity` is the usual deferred BS_ERR_CAPACITY in d_result.
 *   - The FIRST call on each device looks the array's device address up (cudaGetSymbolAddress with that device current;
 *     BS_ERR_CUDA if the runtime refuses, BS_ERR_UNSUPPORTED for a device ordinal >= 64).  Make that first call during
 *     set-up, before any stream capture is begun; later calls only read the cached address.
 *   - Every call on a device uses the SAME array and finds in it whatever the previous call left.  Nothing in it has to
 *     start at zero (each word the kernels synchronise on carries a per-call tag), so calls one after the other on one
 *     stream, or ordered by events, need no clearing in between.  Calls that can overlap on the GPU (two streams, no
 *     event between them) race on it and produce garbage with status BS_OK: give such callers a workspace each
 *     (bs_serialize).  The array is also what bs_serialize_range would need to follow up on this call: it is not
 *     exposed, so there is no range form. */
#define BS_NOALLOC_MAX_BLOCKS 65536u
#define BS_NOALLOC_MAX_STREAM_BYTES (1ull << 30)
uint64_t bs_noalloc_scratch_bytes(void); /* host-only: the size of the built-in array */
int bs_serialize_noalloc(const bs_set_desc *set, void *d_stream, uint64_t capacity, bs_result *d_result,
                         const bs_opts *opts, cudaStream_t stream);

/* ---- deserialize ---------------------------------------------------------------- */

/* Validate the header of d_stream[0..nbytes) (every check of DESIGN.md "deserialize"), rebuild the
 * descriptor into out's device arrays (capacities out->n_tensors / out->n_blocks) and copy every
 * block out: to d_pool (BS_LAYOUT_POOL) or to out->addr (BS_SCATTER_TO_ADDR).  Asynchronous.
 * d_result: status BS_ERR_CORRUPT (nothing written), BS_ERR_CAPACITY (arrays / pool / workspace too
 * small; pool_bytes = required), BS_ERR_ARG (scatter extents differ); n_tensors / n_blocks = counts. */
int bs_deserialize(const void *d_stream, uint64_t nbytes, bs_set_desc *out, void *d_pool,
                   uint64_t pool_bytes, uint32_t flags, void *d_workspace, uint64_t workspace_bytes,
                   bs_result *d_result, const bs_opts *opts, cudaStream_t stream);

/* Segment form (Fig 4(b); the mirror image of bs_serialize_range): scatter the payload bytes of stream range
 * [lo, hi), found at d_src[0 .. hi-lo), to their blocks.  lo, hi multiples of 16 (hi is clipped to the total).  The
 * parse / validate pass must have run on the same workspace with the same `out` and destination (a bs_deserialize call;
 * the tables it leaves are what this call uses) and its status is honoured: nothing is written unless it was BS_OK.
 * d_header: stream byte 0 .. header_bytes to rebuild the descriptor arrays from as well, or NULL (payload only).
 * The union over a partition of [header_bytes, total) rebuilds every block.  BS_VARIANT_LDG on the tables of an unpadded
 * (BS_ALIGN8) stream writes nothing and leaves BS_ERR_UNSUPPORTED as the workspace's status, which later range calls honour.
 * Both range forms only READ the workspace: once the pass has completed, the ranges of one stream may be issued on several
 * CUDA streams at once on the same workspace (order them behind the pass with an event). */
int bs_deserialize_range(const void *d_src, uint64_t lo, uint64_t hi, const void *d_header, bs_set_desc *out, uint32_t flags,
                         void *d_workspace, uint64_t workspace_bytes, const bs_opts *opts, cudaStream_t stream);


/* ==== wire format v2: structure-shared layers (PAPER Fig 4(a), L75) =============================
 *
 * "Layers indicate position dependent operators which have the same block-sparse structure, but the dense sector
 * matrices take different values for the different layers" (L75).  A layered set is C STRUCTURES (one table of
 * labelled sectors each: the meta data of L63, stored once) and T LAYERS, each naming its structure and owning one
 * dense block per sector of it.  The payload is byte-identical to the v1 payload of the same tensors; only the header
 * differs (48 bytes per structure block + 16 per layer instead of 48 per block of every tensor).
 *
 *   stream      := fixed_header(64) | struct_rec[C](32) | layer_rec[T](16) | block_rec[Bs](48) | zeros to a multiple
 *                  of 128 | payload(P)
 *   fixed_header: char magic[8]="BSPARSE1"; u32 version=2; u32 endian_tag=0x01020304; u32 dtype (as v1: element size e);
 *                 u32 n_qn=2; u32 max_rank=3; u32 align=16; u32 n_structs=C; u32 n_struct_blocks=Bs; u64 n_layers=T;
 *                 u64 header_bytes; u64 payload_bytes
 *   struct_rec  : bs_struct_rec, byte for byte (layer_bytes = sum over its blocks of align16(e*prod(dim)))
 *   layer_rec   : bs_layer_rec, byte for byte  (offset = sum over earlier layers of their structure's layer_bytes)
 *   block_rec   : i32 qn[3][2]; u32 dim[3]; u32 structure; u64 offset   (offset relative to the start of a layer =
 *                 sum over earlier blocks of the same structure of align16(e*prod(dim)))
 *   payload     : layer t at payload + offset_t, block j of its structure at + offset_j, zero padded to 16
 *   header_bytes = align128(64 + 32*C + 16*T + 48*Bs)
 */
typedef struct bs_struct_rec {
    uint32_t rank;        /* 2 or 3 */
    uint32_t first_block; /* structures partition the structure block table (qn / dim) in order */
    uint32_t n_blocks;
    int32_t dq[2];        /* conserved charge: sum_k sign[k]*qn[k] == dq for every block */
    int8_t sign[4];
    uint64_t layer_bytes; /* OUTPUT of deserialize (from the wire); ignored by serialize */
} bs_struct_rec;

typedef struct bs_layer_rec {
    uint32_t structure;   /* index into structs[] */
    uint32_t tag;         /* opaque user id (operator index / site) */
    uint64_t offset;      /* OUTPUT of deserialize (payload offset of the layer, from the wire); ignored by serialize */
} bs_layer_rec;

/* HOST struct; every pointer is a DEVICE pointer.  addr[] lists the blocks layer by layer (descriptor order), inside
 * a layer in the order of its structure's block table: B = sum_t structs[layers[t].structure].n_blocks entries. */
typedef struct bs_layered_desc {
    uint32_t n_structs;       /* C.   For deserialize / prefetch outputs: CAPACITY of structs[] */
    uint32_t n_struct_blocks; /* Bs.  For outputs: CAPACITY of qn / dim */
    uint32_t n_layers;        /* T.   For outputs: CAPACITY of layers[] */
    uint32_t n_qn;            /* 2 */
    uint32_t dtype;           /* BS_F64, BS_F32, BS_C64 or BS_C128 (for outputs: 0; the stream's type comes back in bs_result) */
    uint32_t reserved;        /* 0 */
    uint64_t n_addr;          /* entries of addr[]: must be >= B (serialize: B is checked on the device) */
    bs_struct_rec *structs;   /* [C]         */
    bs_layer_rec *layers;     /* [T]         */
    int32_t *qn;              /* [Bs][3][2]  */
    uint32_t *dim;            /* [Bs][3]     */
    uint64_t *addr;           /* [B]         8-byte aligned block addresses (16 for the fast path) */
} bs_layered_desc;

typedef struct bs_layered_stream_info_t {
    uint64_t n_structs, n_struct_blocks, n_layers, header_bytes, payload_bytes, total_bytes;
    uint64_t dtype; /* BS_F64 .. BS_C128 */
} bs_layered_stream_info_t;

/* align128(64 + 32*C + 16*T + 48*Bs) */
uint64_t bs_layered_header_bytes(uint64_t n_structs, uint64_t n_layers, uint64_t n_struct_blocks);
/* workspace for a layered set of up to these counts (n_addr = B) whose stream is at most stream_capacity bytes */
uint64_t bs_layered_workspace_bytes(uint32_t n_structs, uint32_t n_struct_blocks, uint32_t n_layers, uint64_t n_addr,
                                    uint64_t stream_capacity);
int bs_layered_stream_info(const void *h_first_64_bytes, bs_layered_stream_info_t *out); /* HOST memory */

/* As bs_serialized_size / bs_serialize / bs_serialize_range / bs_deserialize, for wire format v2.  bs_result:
 * n_tensors = T, n_blocks = B, reserved[0] = C, reserved[1] = Bs, reserved[2] = dtype.  Deferred statuses as for v1; additionally
 * BS_ERR_ARG for a layer naming a structure >= C and BS_ERR_CAPACITY for n_addr < B.  bs_layered_deserialize writes
 * structs / layers (wire records), qn / dim (BS_LAYOUT_POOL; with BS_SCATTER_TO_ADDR dim [Bs][3] and addr [B] are
 * INPUTS) and addr. */
int bs_layered_serialized_size(const bs_layered_desc *set, void *d_workspace, uint64_t workspace_bytes,
                               uint64_t *header_bytes, uint64_t *total_bytes, cudaStream_t stream);
int bs_layered_serialize(const bs_layered_desc *set, void *d_stream, uint64_t capacity, void *d_workspace,
                         uint64_t workspace_bytes, bs_result *d_result, const bs_opts *opts, cudaStream_t stream);
int bs_layered_serialize_range(const bs_layered_desc *set, void *d_dst, uint64_t lo, uint64_t hi, int run_scan,
                               void *d_workspace, uint64_t workspace_bytes, bs_result *d_result, const bs_opts *opts,
                               cudaStream_t stream);
int bs_layered_deserialize(const void *d_stream, uint64_t nbytes, bs_layered_desc *out, void *d_pool,
                           uint64_t pool_bytes, uint32_t flags, void *d_workspace, uint64_t workspace_bytes,
                           bs_result *d_result, const bs_opts *opts, cudaStream_t stream);

/* ---- asynchronous offload / prefetch engine ------------------- */

typedef struct bs_engine bs_engine;
typedef struct bs_ticket bs_ticket;

typedef struct bs_engine_cfg {
    uint64_t chunk_bytes;      /* staging chunk ("segment", PAPER Fig 4(b)); 0 = 256 MiB; multiple of 65536 */
    uint32_t n_staging;        /* staging buffers; 0 = 2 (double buffering) */
    uint32_t max_tensors;      /* largest T the engine will see */
    uint32_t max_blocks;       /* largest B the engine will see */
    uint64_t max_stream_bytes; /* largest stream the engine will see */
    bs_opts opts;
} bs_engine_cfg;

typedef struct bs_ticket_stats {
    uint64_t bytes;    /* stream bytes moved over PCIe */
    uint32_t n_chunks;
    int32_t status;
    float dma_ms;      /* first DMA start -> last DMA end, device-timed */
    float total_ms;    /* first engine kernel -> completion, device-timed */
} bs_ticket_stats;

/* Allocates the side streams (highest priority), events, n_staging staging chunks, the workspace and
 * a header buffer sized for max_blocks.  Device memory use = n_staging*chunk_bytes + O(max_blocks). */
int bs_engine_create(bs_engine **out, const bs_engine_cfg *cfg);
int bs_engine_destroy(bs_engine *e); /* waits for in-flight work */

/* Save: after everything already enqueued on `producer`, pack the stream of `set` chunk by chunk into
 * the staging buffers and DMA each chunk to h_pinned[0..total).  Returns at once; `producer` is not
 * blocked.  total_bytes = the value bs_serialized_size returned for this set (the paper's size
 * prediction, L106; it fixes the chunk count on the host and is re-checked on the device);
 * total_bytes == 0 makes the call compute it, which SYNCHRONISES `producer`.
 * BS_ERR_CAPACITY at once if total_bytes > h_capacity or exceeds the engine's limits. */
int bs_offload_async(bs_engine *e, const bs_set_desc *set, uint64_t total_bytes, void *h_pinned,
                     uint64_t h_capacity, cudaStream_t producer, bs_ticket **ticket);

/* Load: DMA the stream h_pinned[0..nbytes) chunk by chunk to the staging buffers, validate the header,
 * rebuild `out` and scatter every block (flags as bs_deserialize).  `consumer` is made to wait for
 * completion (cudaStreamWaitEvent — the "checkpoint" of PAPER L138); the host is not blocked. */
int bs_prefetch_async(bs_engine *e, const void *h_pinned, uint64_t nbytes, bs_set_desc *out, void *d_pool,
                      uint64_t pool_bytes, uint32_t flags, cudaStream_t consumer, bs_ticket **ticket);


/* The same two calls for layered sets (wire format v2).  The engine must have been created with max_tensors >= C and
 * >= T, max_blocks >= Bs and >= B. */
int bs_offload_layered_async(bs_engine *e, const bs_layered_desc *set, uint64_t total_bytes, void *h_pinned,
                             uint64_t h_capacity, cudaStream_t producer, bs_ticket **ticket);
int bs_prefetch_layered_async(bs_engine *e, const void *h_pinned, uint64_t nbytes, bs_layered_desc *out, void *d_pool,
                              uint64_t pool_bytes, uint32_t flags, cudaStream_t consumer, bs_ticket **ticket);

/* ==== self-contained packages (PAPER §III.B.3) =========================================
 *
 * "Each serialized component is self contained in the sense that the string contains not only the deserializable data,
 * but also metadata which pinpoints the location of the component within the original, whole object.  As a result,
 * these packages can be sent, mixed with other packages and received back without the need to keep track of their
 * order" (L124); they "can be cut down into even smaller packages ... to keep MPI package sizes below an implementation
 * or self imposed upper limit" (L126).  A package is a 64-byte header followed by a range of a wire-format-v1 stream:
 *
 *   package        := package_header(64) | stream bytes [lo, lo + nbytes)
 *   package_header : char magic[8]="BSPKG001"; u32 version=1; u32 index; u32 count; u32 first_block; u64 stream_id;
 *                    u64 total_bytes; u64 lo; u64 nbytes; u64 first_block_offset
 *     first_block        = the block holding the package's first payload byte (the largest i with offset_i <= lo -
 *                          header_bytes); BS_PKG_NO_BLOCK for a package of the header region
 *     first_block_offset = lo - header_bytes - offset_{first_block}   (0 for a package of the header region)
 *   the cut (a function of header_bytes, total_bytes and the size limit `cap`, a multiple of 16): the header region
 *   [0, header_bytes) is cut into ceil(header_bytes/cap) packages of cap bytes (the last one shorter), then the payload
 *   likewise; index counts them in stream order.  No package straddles the header / payload boundary, so the packages
 *   of the header region rebuild the block table and every payload package is then unpacked on its own, in any order.
 *
 * Packages live in SLOTS: n_slots buffers of slot_bytes each (slot_bytes a multiple of 16, >= 64 + cap), slot s at
 * base + s*slot_bytes.  A slot whose magic is not "BSPKG001" or whose stream_id differs is foreign and is skipped
 * ("mixed with other packages").  Who checks what on the receiving side: the HOST reads the 64-byte package headers to
 * plan the copies and checks what that plan relies on (version, agreement on count and total_bytes, every index exactly
 * once, ranges tiling [0,total) in index order, each fitting its slot, none straddling the header boundary) and fails at
 * once with BS_ERR_CORRUPT; the DEVICE checks each package against the parsed stream (total_bytes, first_block and
 * first_block_offset against the offset table) and every v1 header check of bs_deserialize, deferred as usual, before
 * any block is written. */
enum { BS_PKG_HEADER = 64 };
#define BS_PKG_NO_BLOCK 0xFFFFFFFFu

/* number of packages of a stream; 0 for an invalid cut (cap == 0, cap % 16 != 0, header_bytes > total_bytes) */
uint64_t bs_package_count(uint64_t header_bytes, uint64_t total_bytes, uint64_t cap);
/* stream range [*lo, *hi) of package `index`; BS_ERR_ARG for an invalid cut or index */
int bs_package_range(uint64_t header_bytes, uint64_t total_bytes, uint64_t cap, uint64_t index, uint64_t *lo, uint64_t *hi);
/* workspace for bs_package_emit / bs_package_unpack: bs_workspace_bytes + room for the assembled header region and for
 * the slot table of the one-launch path.  (bs_package_emit also accepts a plain bs_workspace_bytes workspace, and
 * bs_package_unpack one with room for the header region only; the slot table is then a stream-ordered allocation.)
 * Limits that are a multiple of the work tile (bs_opts.tile_bytes, 16 KiB by default) cost a fixed number of launches
 * whatever the number of packages; any other multiple of 16 is served package by package. */
uint64_t bs_package_workspace_bytes(uint32_t n_tensors, uint32_t n_blocks, uint64_t stream_capacity);

/* Serialize `set` straight into packages in DEVICE slots: package k -> d_slots + slot(k)*slot_bytes with
 * slot(k) = h_slot_of[k] (HOST array of `count` entries, each < n_slots, all different) or k when h_slot_of is NULL.
 * total_bytes = the size prediction (bs_serialized_size; re-checked on the device); 0 computes it, which SYNCHRONISES
 * `stream`.  Bytes of a slot behind its package are not written.  bs_result: as bs_serialize, reserved[3] = count.
 * At once: BS_ERR_ARG (cap, slot_bytes, slot map), BS_ERR_CAPACITY (count > n_slots, workspace). */
int bs_package_emit(const bs_set_desc *set, uint64_t total_bytes, uint64_t cap, uint64_t stream_id, void *d_slots,
                    uint64_t slot_bytes, uint64_t n_slots, const uint32_t *h_slot_of, void *d_workspace,
                    uint64_t workspace_bytes, bs_result *d_result, const bs_opts *opts, cudaStream_t stream);

/* Deserialize from packages lying in DEVICE slots in any order, foreign slots skipped.  Copies the n_slots package
 * headers to the host and SYNCHRONISES `stream` once to plan; then as bs_deserialize (same outputs, flags, deferred
 * statuses; BS_ERR_CORRUPT also for a package that disagrees with the parsed stream). */
int bs_package_unpack(const void *d_slots, uint64_t slot_bytes, uint64_t n_slots, uint64_t stream_id, bs_set_desc *out,
                      void *d_pool, uint64_t pool_bytes, uint32_t flags, void *d_workspace, uint64_t workspace_bytes,
                      bs_result *d_result, const bs_opts *opts, cudaStream_t stream);

/* The same for layered sets: packages of a wire-format-v2 stream (first_block counts the blocks in the order of the
 * layered descriptor's addr[]: layer by layer, inside a layer in the order of its structure's block table).
 * bs_layered_package_workspace_bytes = bs_layered_workspace_bytes + room for the assembled header region. */
uint64_t bs_layered_package_workspace_bytes(uint32_t n_structs, uint32_t n_struct_blocks, uint32_t n_layers, uint64_t n_addr,
                                            uint64_t stream_capacity);
int bs_layered_package_emit(const bs_layered_desc *set, uint64_t total_bytes, uint64_t cap, uint64_t stream_id, void *d_slots,
                            uint64_t slot_bytes, uint64_t n_slots, const uint32_t *h_slot_of, void *d_workspace,
                            uint64_t workspace_bytes, bs_result *d_result, const bs_opts *opts, cudaStream_t stream);
int bs_layered_package_unpack(const void *d_slots, uint64_t slot_bytes, uint64_t n_slots, uint64_t stream_id,
                              bs_layered_desc *out, void *d_pool, uint64_t pool_bytes, uint32_t flags, void *d_workspace,
                              uint64_t workspace_bytes, bs_result *d_result, const bs_opts *opts, cudaStream_t stream);

/* The same through the engine, slots in pinned HOST memory (the receive buffers of L126): package k is packed into a
 * staging buffer behind its header and DMA'd to h_slots + slot(k)*slot_bytes; cap + 64 <= chunk_bytes.  Prefetch takes
 * the slots in the order they lie (arrival order): header-region packages first, then every payload package is unpacked
 * on its own.  A staging buffer takes a batch of packages: with slot_bytes == 64 + cap, packages whose host slots are
 * consecutive cross the link in one DMA (a short package ends its batch, so nothing behind it is written), and limits that
 * are a multiple of the work tile cost two launches per batch.  ticket n_chunks = number of packages, bytes = stream bytes
 * + 64 per package.  Ticket / checkpoint semantics as bs_offload_async / bs_prefetch_async. */
int bs_offload_packages_async(bs_engine *e, const bs_set_desc *set, uint64_t total_bytes, uint64_t cap, uint64_t stream_id,
                              void *h_slots, uint64_t slot_bytes, uint64_t n_slots, const uint32_t *h_slot_of,
                              cudaStream_t producer, bs_ticket **ticket);
int bs_prefetch_packages_async(bs_engine *e, const void *h_slots, uint64_t slot_bytes, uint64_t n_slots, uint64_t stream_id,
                               bs_set_desc *out, void *d_pool, uint64_t pool_bytes, uint32_t flags, cudaStream_t consumer,
                               bs_ticket **ticket);
/* and for layered sets (packages of a wire-format-v2 stream) */
int bs_offload_layered_packages_async(bs_engine *e, const bs_layered_desc *set, uint64_t total_bytes, uint64_t cap,
                                      uint64_t stream_id, void *h_slots, uint64_t slot_bytes, uint64_t n_slots,
                                      const uint32_t *h_slot_of, cudaStream_t producer, bs_ticket **ticket);
int bs_prefetch_layered_packages_async(bs_engine *e, const void *h_slots, uint64_t slot_bytes, uint64_t n_slots,
                                       uint64_t stream_id, bs_layered_desc *out, void *d_pool, uint64_t pool_bytes,
                                       uint32_t flags, cudaStream_t consumer, bs_ticket **ticket);

/* ==== save / load queue with checkpoints (PAPER §III.B.4) ============================
 *
 * "organizing asynchronous load and save into a kind of queuing system together with checkpoints to make sure that
 * required data of a given computational task are already available in the memory, could maximize performance rate
 * regarding IO operations" (L136-138).  A bs_queue is two engines — a SAVE lane and a LOAD lane, each with its own side
 * streams, staging buffers and workspace — so a save (device -> host) and a load (host -> device) run at the same time,
 * one in each direction of the PCIe link, and a table of KEYS that orders what must be ordered:
 *   - what a caller observes is per-key PROGRAM ORDER: a load of `key` returns the object of the last save of `key`
 *     submitted before it (the load lane waits, on the device, for that save's completion event); a save over a key
 *     whose load is still running waits for the load (the host buffer is being read); operations on different keys
 *     are independent and overlap.  Host buffers of different keys must not overlap.
 *   - checkpoints are events, never host waits: bs_queue_load makes `consumer` wait for the loaded blocks,
 *     bs_queue_checkpoint makes any stream wait until every operation submitted so far on `key` has completed (after
 *     it, the saved blocks may be overwritten).
 * Device memory held = 2 x (n_staging x chunk_bytes + O(max_blocks)), fixed at creation, whatever is in flight — not
 * the extra serialized + deserialized buffers of the paper's Fig 3(c) (L136).  One queue is driven by one host thread. */
typedef struct bs_queue bs_queue;

typedef struct bs_queue_stats {
    uint64_t saves, loads;             /* accepted calls */
    uint64_t bytes_saved, bytes_loaded; /* stream bytes they move */
    uint64_t host_bytes_live;          /* sum of the streams the live keys hold in host memory */
    uint64_t host_bytes_peak;
    uint64_t keys_live;
    uint64_t device_bytes;             /* staging + workspace + header buffers of both lanes */
    uint32_t in_flight;                /* operations submitted and not yet complete (at the time of the call) */
    uint32_t max_in_flight;
    uint64_t bytes_spilled, bytes_filled; /* storage tier: stream bytes written to / read from files (completed jobs) */
} bs_queue_stats;

int bs_queue_create(bs_queue **out, const bs_engine_cfg *lane_cfg); /* both lanes get lane_cfg */
int bs_queue_destroy(bs_queue *q);                                  /* drains first */

/* Save `set` under `key` into h_pinned (as bs_offload_async: total_bytes = the size prediction, 0 computes it and
 * synchronises `producer`).  A previous stream of `key` is replaced. */
int bs_queue_save(bs_queue *q, uint64_t key, const bs_set_desc *set, uint64_t total_bytes, void *h_pinned,
                  uint64_t h_capacity, cudaStream_t producer);
/* The same for layered sets (wire format v2); a key holds a stream of ONE format: loading it with the other call is
 * BS_ERR_ARG.  Element types other than fp64 (v1) travel through bs_queue_save / bs_queue_load unchanged. */
int bs_queue_save_layered(bs_queue *q, uint64_t key, const bs_layered_desc *set, uint64_t total_bytes, void *h_pinned,
                          uint64_t h_capacity, cudaStream_t producer);
int bs_queue_load_layered(bs_queue *q, uint64_t key, bs_layered_desc *out, void *d_pool, uint64_t pool_bytes, uint32_t flags,
                          cudaStream_t consumer);
/* Register a complete stream (either wire format) that is already in pinned host memory (it came from elsewhere) under `key`. */
int bs_queue_adopt(bs_queue *q, uint64_t key, const void *h_pinned, uint64_t nbytes);
/* Load the stream of `key` (as bs_prefetch_async).  BS_ERR_ARG for an unknown key. */
int bs_queue_load(bs_queue *q, uint64_t key, bs_set_desc *out, void *d_pool, uint64_t pool_bytes, uint32_t flags,
                  cudaStream_t consumer);
int bs_queue_checkpoint(bs_queue *q, uint64_t key, cudaStream_t stream); /* device-side wait; BS_ERR_ARG: unknown key */
/* Host-blocking: waits for the last save and the last load of `key`; returns the first deferred status that is not
 * BS_OK.  Either stats pointer may be NULL; stats of an operation that never happened have n_chunks = 0, bytes = 0. */
int bs_queue_wait(bs_queue *q, uint64_t key, bs_ticket_stats *save_stats, bs_ticket_stats *load_stats);
int bs_queue_query(bs_queue *q, uint64_t key);   /* BS_OK | BS_PENDING | BS_ERR_* (BS_ERR_ARG: unknown key) */
int bs_queue_forget(bs_queue *q, uint64_t key);  /* waits for the key's operations, then drops it: the host buffer is the caller's again */
int bs_queue_drain(bs_queue *q);                 /* host-blocking: everything submitted so far has completed */
int bs_queue_get_stats(bs_queue *q, bs_queue_stats *out);

/* ---- the storage tier below pinned host RAM (PAPER §III: saving = serialization, then "writing the serialized data
 * to a storage media"; L90: "a single CPU thread takes care of saving the serialized data while the remaining CPU
 * threads ... proceed with subsequent computational tasks"; L144/L202: data spilled to a local disk in the background;
 * SURVEY §8(f) NEXT-4).  The queue owns ONE host IO thread (started by the first call); jobs run in submission order.
 *   bs_queue_spill   : once the save of `key` has completed, write its stream to the file `path` (created / truncated).
 *                      Returns at once.  The key stays loadable from host RAM; after bs_queue_io_wait + bs_queue_forget the
 *                      host buffer is the caller's again and the file is the only copy.
 *   bs_queue_fill    : read the file `path` (a stream written by bs_queue_spill, either wire format) into h_pinned and
 *                      register it under `key` (as bs_queue_adopt).  Returns at once; BS_ERR_CAPACITY if the file is larger
 *                      than h_capacity, BS_ERR_IO if it cannot be opened.  A bs_queue_load of the key submitted before the
 *                      read has finished BLOCKS THE HOST until it has (the "fetching" stall of L132) — a DMA cannot wait
 *                      for a host thread.
 *   bs_queue_io_wait : host-blocking; the outcome of the key's last storage job (BS_OK | BS_ERR_IO), the bytes it moved and
 *                      the seconds its reads / writes took.
 * A save over a key, bs_queue_forget and bs_queue_destroy wait for the key's pending storage job (its buffer is in use). */
int bs_queue_spill(bs_queue *q, uint64_t key, const char *path);
int bs_queue_fill(bs_queue *q, uint64_t key, const char *path, void *h_pinned, uint64_t h_capacity);
int bs_queue_io_wait(bs_queue *q, uint64_t key, uint64_t *bytes, double *seconds);

int bs_ticket_wait(bs_ticket *t, bs_ticket_stats *stats /* may be NULL */); /* blocks the host; returns the deferred status */
int bs_ticket_query(const bs_ticket *t);                                   /* BS_OK | BS_PENDING | BS_ERR_* */
int bs_ticket_stream_wait(const bs_ticket *t, cudaStream_t stream);        /* make `stream` wait for completion (no host block):
                                                                               after an offload the blocks may be overwritten */
int bs_ticket_destroy(bs_ticket *t);                                       /* after completion */

#ifdef __cplusplus
}
#endif
#endif /* BS_H_ */
