/*
 * bs_oracle_v2.c — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded CPU serializer /
 * deserializer for wire format v2: STRUCTURE-SHARED LAYERS.
 *
 * What it follows.  PAPER.md Fig 4(a) caption (L75): "Layers indicate position dependent operators which
 * have the same block-sparse structure, but the dense sector matrices take different values for the
 * different layers."  A set is therefore C *structures* (one table of labelled sectors each: the meta data
 * of L63) and T *layers*, each layer naming its structure and owning one dense block per sector of it.
 * Format v1 repeats the 48-byte block record for every layer; v2 stores each structure's records once.
 * The paper prints no byte format: v2 below is this project's own, DESIGN.md "Wire format v2",
 * and this file is its definition.  The other properties are the paper's and are kept: exact size prediction
 * (L106), a pointer/grid structure built before any data moves (L90-92), one contiguous stream that
 * deserializes into an identical object (L108), meta data that locates every component (L124).
 *
 * Wire format v2 (little-endian, no implicit padding):
 *   stream     := fixed_header(64) | struct_rec[C](32) | layer_rec[T](16) | block_rec[Bs](48)
 *                 | zeros to a multiple of 128 | payload(P)
 *   fixed_header: char magic[8]="BSPARSE1"; u32 version=2; u32 endian_tag=0x01020304; u32 dtype (0 f64,
 *                 1 f32, 2 c64, 3 c128: element size e = 8, 4, 8, 16 — reading E-2 below);
 *                 u32 n_qn=2; u32 max_rank=3; u32 align=16; u32 n_structs=C; u32 n_struct_blocks=Bs;
 *                 u64 n_layers=T; u64 header_bytes; u64 payload_bytes
 *   struct_rec  : u32 rank; u32 first_block; u32 n_blocks; i32 dq[2]; i8 sign[4]; u64 layer_bytes
 *   layer_rec   : u32 structure; u32 tag; u64 offset
 *   block_rec   : i32 qn[3][2]; u32 dim[3]; u32 structure; u64 offset     (offset relative to the layer)
 *   payload     : layer t at payload + offset_t; inside it block j of its structure at + offset_j: the
 *                 e*prod(dim_j) raw bytes of that layer's block, then zeros to the next multiple of 16
 *     offset_j      = sum over earlier blocks j' of the SAME structure of align16(e*prod(dim_j'))
 *     layer_bytes_s = sum over the blocks of structure s of align16(e*prod(dim))
 *     offset_t      = sum_{t' < t} layer_bytes[structure[t']]                 (descriptor order)
 *     header_bytes  = align128(64 + 32*C + 16*T + 48*Bs)
 * Block addresses: addr[] lists the blocks layer by layer (descriptor order), inside a layer in the
 * order of its structure's block table; it has B = sum_t n_blocks[structure[t]] entries.
 *
 * Reading E-2 (round 2; SURVEY §8(f) NEXT-4 "complex128 / fp32 dtypes", applied to layered sets; the paper's Fig 4(a)
 * layers (L75) are value layers of one structure whatever the element type): exactly as reading E-1 did for wire
 * format v1, the header's dtype word selects the element size e and nothing else changes —
 * nbytes = e*prod(dim), stored = align16(nbytes) (an f32 block carries 0, 4, 8 or 12 zero pad bytes), pool slots stay
 * align256(nbytes).  Every function below that computed 8*prod(dim) computes e*prod(dim); dtype = 0 gives the bytes
 * round 1 gave.  Pins of the element types (tests/test_oracle_v2.py): G6 hand-typed f32 golden stream; payload ==
 * the payload of the independently written numpy oracle bs_oracle_dtype.py (v1) on the expanded set for every type;
 * the c64 stream == the f64 stream but for the dtype word; offsets against numpy.cumsum of e-sized blocks.
 *
 * Relation to v1 (a pin, tests/test_oracle_v2.py): expanding every layer into a v1 tensor with its
 * structure's records gives a v1 set whose PAYLOAD is byte-identical to the v2 payload.
 *
 * Pins (-m "not gpu"): G2 hand-typed 320-byte golden stream + independent struct reader; payload ==
 * v1 payload of the expanded set (v1 oracle is pinned on its own); offsets vs numpy.cumsum; size
 * prediction; round trip / fixpoint; conservation from the stream alone; dense brute force per layer;
 * fault injection on every validated field.  Unpinned: nothing in this file.
 *
 * Shares no code with bs_oracle.c or with paper_2412_04676_b200/ (helpers are re-typed).
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>

#define ORC_OK               0
#define ORC_ERR_ARG        (-1)
#define ORC_ERR_CAPACITY   (-2)
#define ORC_ERR_CORRUPT    (-3)
#define ORC_ERR_UNSUPPORTED (-4)

#define V2_FIXED_HEADER 64u
#define V2_STRUCT_REC   32u
#define V2_LAYER_REC    16u
#define V2_BLOCK_REC    48u
#define V2_HEADER_ALIGN 128u
#define V2_BLOCK_ALIGN  16u
#define V2_POOL_ALIGN   256u

typedef struct {
    uint32_t rank;          /* 2 or 3 */
    uint32_t first_block;   /* into the structure block table */
    uint32_t n_blocks;
    int32_t  dq[2];
    int8_t   sign[4];
    uint64_t layer_bytes;   /* wire / output: stored bytes of one layer; ignored on input */
} orc2_struct;

typedef struct {
    uint32_t structure;
    uint32_t tag;
    uint64_t offset;        /* wire / output: payload offset of the layer; ignored on input */
} orc2_layer;

typedef char orc2_struct_is_32_bytes[(sizeof(orc2_struct) == 32) ? 1 : -1];
typedef char orc2_layer_is_16_bytes[(sizeof(orc2_layer) == 16) ? 1 : -1];

static uint64_t up(uint64_t x, uint64_t a) { return (x + (a - 1)) / a * a; }
static void w32(unsigned char *p, uint32_t v) { memcpy(p, &v, 4); }
static void w64(unsigned char *p, uint64_t v) { memcpy(p, &v, 8); }
static uint32_t r32(const unsigned char *p) { uint32_t v; memcpy(&v, p, 4); return v; }
static uint64_t r64(const unsigned char *p) { uint64_t v; memcpy(&v, p, 8); return v; }
static int32_t  ri32(const unsigned char *p) { int32_t v; memcpy(&v, p, 4); return v; }

uint64_t orc2_header_bytes(uint64_t C, uint64_t T, uint64_t Bs)
{
    return up(V2_FIXED_HEADER + V2_STRUCT_REC * C + V2_LAYER_REC * T + V2_BLOCK_REC * Bs, V2_HEADER_ALIGN);
}

/* structures partition the structure block table in order; every layer names a structure */
static int check_desc(uint64_t C, uint64_t Bs, uint64_t T, const orc2_struct *st, const orc2_layer *ly)
{
    if (C >= (1ull << 32) || Bs >= (1ull << 32) || T >= (1ull << 32)) return ORC_ERR_UNSUPPORTED;
    uint64_t next = 0;
    for (uint64_t s = 0; s < C; ++s) {
        if (st[s].rank != 2 && st[s].rank != 3) return ORC_ERR_UNSUPPORTED;
        if (st[s].first_block != next) return ORC_ERR_ARG;
        next += st[s].n_blocks;
    }
    if (next != Bs) return ORC_ERR_ARG;
    for (uint64_t t = 0; t < T; ++t)
        if (ly[t].structure >= C) return ORC_ERR_ARG;
    return ORC_OK;
}

/* element size of a dtype word (reading E-2): f64 8, f32 4, c64 8, c128 16 */
static uint64_t elem_size(uint32_t dtype) { return dtype == 1u ? 4u : (dtype == 3u ? 16u : 8u); }

static int block_bytes(const uint32_t *dim3, uint32_t dtype, uint64_t *nbytes)
{
    uint64_t d0 = dim3[0], d1 = dim3[1], d2 = dim3[2];
    uint64_t n01 = d0 * d1;
    if (d2 != 0 && n01 > (UINT64_MAX / 16u) / d2) return ORC_ERR_ARG;
    *nbytes = elem_size(dtype) * n01 * d2;
    return ORC_OK;
}

/* ---- the "pointer structure" (L90-92) of a layered set ----------------------------------------------
 * rel_offset[j] (j over the structure block table), layer_bytes[s], layer_offset[t], n_addr = B, P.
 * Any output pointer may be NULL. */
int orc2_plan(uint64_t C, uint64_t Bs, uint64_t T, const orc2_struct *st, const orc2_layer *ly,
              const uint32_t *dim /*[Bs][3]*/, uint32_t dtype, uint64_t *rel_offset, uint64_t *layer_bytes,
              uint64_t *layer_offset, uint64_t *n_addr, uint64_t *payload_bytes)
{
    int rc = check_desc(C, Bs, T, st, ly);
    if (rc) return rc;
    if (dtype > 3u) return ORC_ERR_UNSUPPORTED;
    for (uint64_t s = 0; s < C; ++s) {
        uint64_t run = 0;
        for (uint64_t j = st[s].first_block; j < (uint64_t)st[s].first_block + st[s].n_blocks; ++j) {
            uint64_t nb = 0;
            rc = block_bytes(dim + 3 * j, dtype, &nb);
            if (rc) return rc;
            if (rel_offset) rel_offset[j] = run;
            run += up(nb, V2_BLOCK_ALIGN);
        }
        if (layer_bytes) layer_bytes[s] = run;
    }
    uint64_t run = 0, na = 0;
    for (uint64_t t = 0; t < T; ++t) {
        const orc2_struct *s = &st[ly[t].structure];
        uint64_t lb = 0;
        for (uint64_t j = s->first_block; j < (uint64_t)s->first_block + s->n_blocks; ++j) {
            uint64_t nb = 0;
            block_bytes(dim + 3 * j, dtype, &nb);
            lb += up(nb, V2_BLOCK_ALIGN);
        }
        if (layer_offset) layer_offset[t] = run;
        run += lb;
        na += s->n_blocks;
    }
    if (n_addr) *n_addr = na;
    if (payload_bytes) *payload_bytes = run;
    return ORC_OK;
}

int orc2_serialized_size(uint64_t C, uint64_t Bs, uint64_t T, const orc2_struct *st, const orc2_layer *ly,
                         const uint32_t *dim, uint32_t dtype, uint64_t *header_bytes, uint64_t *total_bytes)
{
    uint64_t P;
    int rc = orc2_plan(C, Bs, T, st, ly, dim, dtype, NULL, NULL, NULL, NULL, &P);
    if (rc) return rc;
    *header_bytes = orc2_header_bytes(C, T, Bs);
    *total_bytes = *header_bytes + P;
    return ORC_OK;
}

/* ---- serialize: header, then layer by layer, block by block ---------------------------------------- */
int orc2_serialize(uint64_t C, uint64_t Bs, uint64_t T, const orc2_struct *st, const orc2_layer *ly,
                   const int32_t *qn /*[Bs][3][2]*/, const uint32_t *dim /*[Bs][3]*/,
                   const uint64_t *addr /*[B] host addresses, layer-major*/, uint32_t dtype, unsigned char *out,
                   uint64_t capacity, uint64_t *written)
{
    uint64_t hb, total;
    int rc = orc2_serialized_size(C, Bs, T, st, ly, dim, dtype, &hb, &total);
    if (rc) return rc;
    *written = total;
    if (capacity < total) return ORC_ERR_CAPACITY;

    unsigned char *p = out;
    memcpy(p, "BSPARSE1", 8);
    w32(p + 8, 2u);               /* version */
    w32(p + 12, 0x01020304u);     /* endian_tag */
    w32(p + 16, dtype);           /* dtype (reading E-2) */
    w32(p + 20, 2u);              /* n_qn */
    w32(p + 24, 3u);              /* max_rank */
    w32(p + 28, 16u);             /* align */
    w32(p + 32, (uint32_t)C);
    w32(p + 36, (uint32_t)Bs);
    w64(p + 40, T);
    w64(p + 48, hb);
    w64(p + 56, total - hb);
    p += V2_FIXED_HEADER;

    for (uint64_t s = 0; s < C; ++s) {                       /* struct records, with layer_bytes */
        uint64_t lb = 0;
        for (uint64_t j = st[s].first_block; j < (uint64_t)st[s].first_block + st[s].n_blocks; ++j) {
            uint64_t nb = 0;
            block_bytes(dim + 3 * j, dtype, &nb);
            lb += up(nb, V2_BLOCK_ALIGN);
        }
        w32(p + 0, st[s].rank);
        w32(p + 4, st[s].first_block);
        w32(p + 8, st[s].n_blocks);
        memcpy(p + 12, &st[s].dq[0], 4);
        memcpy(p + 16, &st[s].dq[1], 4);
        memcpy(p + 20, st[s].sign, 4);
        w64(p + 24, lb);
        p += V2_STRUCT_REC;
    }
    {                                                         /* layer records, with payload offsets */
        uint64_t run = 0;
        for (uint64_t t = 0; t < T; ++t) {
            w32(p + 0, ly[t].structure);
            w32(p + 4, ly[t].tag);
            w64(p + 8, run);
            p += V2_LAYER_REC;
            const orc2_struct *s = &st[ly[t].structure];
            for (uint64_t j = s->first_block; j < (uint64_t)s->first_block + s->n_blocks; ++j) {
                uint64_t nb = 0;
                block_bytes(dim + 3 * j, dtype, &nb);
                run += up(nb, V2_BLOCK_ALIGN);
            }
        }
    }
    for (uint64_t s = 0; s < C; ++s) {                       /* block records, offsets relative to the layer */
        uint64_t run = 0;
        for (uint64_t j = st[s].first_block; j < (uint64_t)st[s].first_block + st[s].n_blocks; ++j) {
            uint64_t nb = 0;                                  /* (initialised for gcc, as below) */
            block_bytes(dim + 3 * j, dtype, &nb);
            memcpy(p, qn + 6 * j, 24);
            w32(p + 24, dim[3 * j + 0]);
            w32(p + 28, dim[3 * j + 1]);
            w32(p + 32, dim[3 * j + 2]);
            w32(p + 36, (uint32_t)s);
            w64(p + 40, run);
            run += up(nb, V2_BLOCK_ALIGN);
            p += V2_BLOCK_REC;
        }
    }
    memset(p, 0, (size_t)(out + hb - p));                    /* slack */

    unsigned char *q = out + hb;                              /* payload */
    uint64_t a = 0;
    for (uint64_t t = 0; t < T; ++t) {
        const orc2_struct *s = &st[ly[t].structure];
        for (uint64_t j = s->first_block; j < (uint64_t)s->first_block + s->n_blocks; ++j, ++a) {
            uint64_t nb = 0;                                  /* (initialised for gcc; block_bytes always sets it here: the plan passed) */
            block_bytes(dim + 3 * j, dtype, &nb);
            uint64_t sb = up(nb, V2_BLOCK_ALIGN);
            memcpy(q, (const void *)(uintptr_t)addr[a], (size_t)nb);
            memset(q + nb, 0, (size_t)(sb - nb));
            q += sb;
        }
    }
    if ((uint64_t)(q - out) != total) return ORC_ERR_ARG;    /* prediction == written (L106) */
    return ORC_OK;
}

/* ---- the fixed header alone ------------------------------------------------------------------------ */
int orc2_stream_info(const unsigned char *s, uint64_t n, uint64_t *C, uint64_t *Bs, uint64_t *T,
                     uint64_t *header_bytes, uint64_t *payload_bytes)
{
    if (n < V2_FIXED_HEADER) return ORC_ERR_CORRUPT;
    if (memcmp(s, "BSPARSE1", 8) != 0) return ORC_ERR_CORRUPT;
    if (r32(s + 8) != 2u) return ORC_ERR_CORRUPT;
    if (r32(s + 12) != 0x01020304u) return ORC_ERR_CORRUPT;
    if (r32(s + 16) > 3u) return ORC_ERR_CORRUPT;               /* dtype: one of the four element types */
    if (r32(s + 20) != 2u) return ORC_ERR_CORRUPT;
    if (r32(s + 24) != 3u) return ORC_ERR_CORRUPT;
    if (r32(s + 28) != 16u) return ORC_ERR_CORRUPT;
    *C = r32(s + 32);
    *Bs = r32(s + 36);
    *T = r64(s + 40);
    *header_bytes = r64(s + 48);
    *payload_bytes = r64(s + 56);
    if (*T >= (1ull << 32)) return ORC_ERR_CORRUPT;
    if (*header_bytes != orc2_header_bytes(*C, *T, *Bs)) return ORC_ERR_CORRUPT;
    return ORC_OK;
}

/* the element type of a stream whose fixed header orc2_stream_info accepts */
int orc2_stream_dtype(const unsigned char *s, uint64_t n, uint32_t *dtype)
{
    uint64_t C, Bs, T, hb, P;
    int rc = orc2_stream_info(s, n, &C, &Bs, &T, &hb, &P);
    if (rc) return rc;
    *dtype = r32(s + 16);
    return ORC_OK;
}

/* ---- validate: every field, in stream order ----------------------------------------------------------
 * fixed header; header_bytes + payload_bytes == n; struct records partition the block table, rank in {2,3};
 * block records: owner, unused legs (dim 1, labels 0), offset == running sum inside the structure, the
 * structure's total == its layer_bytes; layer records: structure < C, offset == running sum of layer_bytes,
 * final sum == payload_bytes; header slack zero; pad bytes of every block of every layer zero. */
int orc2_validate_stream(const unsigned char *s, uint64_t n)
{
    uint64_t C, Bs, T, hb, P;
    int rc = orc2_stream_info(s, n, &C, &Bs, &T, &hb, &P);
    if (rc) return rc;
    if (hb > n || hb + P != n) return ORC_ERR_CORRUPT;
    const uint32_t dtype = r32(s + 16);
    const unsigned char *srec = s + V2_FIXED_HEADER;
    const unsigned char *lrec = srec + V2_STRUCT_REC * C;
    const unsigned char *brec = lrec + V2_LAYER_REC * T;
    uint64_t next = 0;
    for (uint64_t k = 0; k < C; ++k) {
        const unsigned char *r = srec + V2_STRUCT_REC * k;
        uint32_t rank = r32(r), first = r32(r + 4), nb = r32(r + 8);
        if (rank != 2 && rank != 3) return ORC_ERR_CORRUPT;
        if (first != next) return ORC_ERR_CORRUPT;
        if ((uint64_t)first + nb > Bs) return ORC_ERR_CORRUPT;
        uint64_t run = 0;
        for (uint64_t j = first; j < (uint64_t)first + nb; ++j) {
            const unsigned char *b = brec + V2_BLOCK_REC * j;
            if (r32(b + 36) != (uint32_t)k) return ORC_ERR_CORRUPT;
            for (uint32_t leg = rank; leg < 3; ++leg) {
                if (r32(b + 24 + 4 * leg) != 1) return ORC_ERR_CORRUPT;
                if (ri32(b + 8 * leg) != 0 || ri32(b + 8 * leg + 4) != 0) return ORC_ERR_CORRUPT;
            }
            uint32_t d3[3] = { r32(b + 24), r32(b + 28), r32(b + 32) };
            uint64_t nbytes;
            if (block_bytes(d3, dtype, &nbytes)) return ORC_ERR_CORRUPT;
            if (r64(b + 40) != run) return ORC_ERR_CORRUPT;
            uint64_t sb = up(nbytes, V2_BLOCK_ALIGN);
            if (sb < nbytes || run + sb < run) return ORC_ERR_CORRUPT;   /* a structure no layer uses may exceed P */
            run += sb;
        }
        if (r64(r + 24) != run) return ORC_ERR_CORRUPT;            /* layer_bytes */
        next += nb;
    }
    if (next != Bs) return ORC_ERR_CORRUPT;
    uint64_t run = 0;
    for (uint64_t t = 0; t < T; ++t) {
        const unsigned char *r = lrec + V2_LAYER_REC * t;
        uint32_t k = r32(r);
        if (k >= C) return ORC_ERR_CORRUPT;
        if (r64(r + 8) != run) return ORC_ERR_CORRUPT;
        uint64_t lb = r64(srec + V2_STRUCT_REC * k + 24);
        if (run + lb < run || run + lb > P) return ORC_ERR_CORRUPT;
        run += lb;
    }
    if (run != P) return ORC_ERR_CORRUPT;
    for (uint64_t z = V2_FIXED_HEADER + V2_STRUCT_REC * C + V2_LAYER_REC * T + V2_BLOCK_REC * Bs; z < hb; ++z)
        if (s[z] != 0) return ORC_ERR_CORRUPT;
    for (uint64_t t = 0; t < T; ++t) {                              /* pad bytes */
        const unsigned char *r = lrec + V2_LAYER_REC * t;
        const unsigned char *sr = srec + V2_STRUCT_REC * r32(r);
        uint64_t base = hb + r64(r + 8);
        for (uint64_t j = r32(sr + 4); j < (uint64_t)r32(sr + 4) + r32(sr + 8); ++j) {
            const unsigned char *b = brec + V2_BLOCK_REC * j;
            uint64_t nbytes = elem_size(dtype) * r32(b + 24) * r32(b + 28) * r32(b + 32);
            for (uint64_t z = nbytes; z < up(nbytes, V2_BLOCK_ALIGN); ++z)
                if (s[base + r64(b + 40) + z] != 0) return ORC_ERR_CORRUPT;
        }
    }
    return ORC_OK;
}

/* counts a receiver needs to size its arrays: B = number of blocks over all layers, and the pool bytes
 * BS_LAYOUT_POOL needs = sum over all layers and blocks of align256(nbytes) */
int orc2_counts(const unsigned char *s, uint64_t n, uint64_t *n_addr, uint64_t *pool_bytes)
{
    uint64_t C, Bs, T, hb, P;
    int rc = orc2_stream_info(s, n, &C, &Bs, &T, &hb, &P);
    if (rc) return rc;
    if (hb > n) return ORC_ERR_CORRUPT;
    const unsigned char *srec = s + V2_FIXED_HEADER;
    const unsigned char *lrec = srec + V2_STRUCT_REC * C;
    const unsigned char *brec = lrec + V2_LAYER_REC * T;
    uint64_t na = 0, pool = 0;
    for (uint64_t t = 0; t < T; ++t) {
        uint32_t k = r32(lrec + V2_LAYER_REC * t);
        if (k >= C) return ORC_ERR_CORRUPT;
        const unsigned char *sr = srec + V2_STRUCT_REC * k;
        uint64_t first = r32(sr + 4), nb = r32(sr + 8);
        if (first + nb > Bs) return ORC_ERR_CORRUPT;
        for (uint64_t j = first; j < first + nb; ++j) {
            const unsigned char *b = brec + V2_BLOCK_REC * j;
            pool += up(elem_size(r32(s + 16)) * r32(b + 24) * r32(b + 28) * r32(b + 32), V2_POOL_ALIGN);
        }
        na += nb;
    }
    *n_addr = na;
    *pool_bytes = pool;
    return ORC_OK;
}

/* ---- deserialize -----------------------------------------------------------------------------------------
 * flags 0 (pool layout): addr_out[a] = pool + sum over earlier (layer, block) pairs of align256(nbytes).
 * flags 1 (scatter): addr_out[a] is an input; dim_out [Bs][3] is an input and must equal the stream's.
 * structs_out / layers_out receive the wire records (layer_bytes and offsets included). */
int orc2_deserialize(const unsigned char *s, uint64_t n, orc2_struct *structs_out, orc2_layer *layers_out,
                     int32_t *qn_out, uint32_t *dim_out, uint64_t *addr_out, unsigned char *pool,
                     uint64_t pool_bytes, uint32_t flags)
{
    int rc = orc2_validate_stream(s, n);
    if (rc) return rc;
    uint64_t C, Bs, T, hb, P, na, need;
    orc2_stream_info(s, n, &C, &Bs, &T, &hb, &P);
    orc2_counts(s, n, &na, &need);
    const unsigned char *srec = s + V2_FIXED_HEADER;
    const unsigned char *lrec = srec + V2_STRUCT_REC * C;
    const unsigned char *brec = lrec + V2_LAYER_REC * T;
    if (flags == 0) {
        if (need > pool_bytes) return ORC_ERR_CAPACITY;
    } else if (flags == 1) {
        for (uint64_t j = 0; j < Bs; ++j)
            for (int leg = 0; leg < 3; ++leg)
                if (dim_out[3 * j + leg] != r32(brec + V2_BLOCK_REC * j + 24 + 4 * leg)) return ORC_ERR_ARG;
    } else {
        return ORC_ERR_ARG;
    }
    for (uint64_t k = 0; k < C; ++k) memcpy(&structs_out[k], srec + V2_STRUCT_REC * k, V2_STRUCT_REC);
    for (uint64_t t = 0; t < T; ++t) memcpy(&layers_out[t], lrec + V2_LAYER_REC * t, V2_LAYER_REC);
    for (uint64_t j = 0; j < Bs; ++j) {
        const unsigned char *b = brec + V2_BLOCK_REC * j;
        memcpy(qn_out + 6 * j, b, 24);
        dim_out[3 * j + 0] = r32(b + 24);
        dim_out[3 * j + 1] = r32(b + 28);
        dim_out[3 * j + 2] = r32(b + 32);
    }
    uint64_t a = 0, cursor = 0;
    for (uint64_t t = 0; t < T; ++t) {
        const unsigned char *sr = srec + V2_STRUCT_REC * layers_out[t].structure;
        uint64_t base = hb + layers_out[t].offset;
        for (uint64_t j = r32(sr + 4); j < (uint64_t)r32(sr + 4) + r32(sr + 8); ++j, ++a) {
            const unsigned char *b = brec + V2_BLOCK_REC * j;
            uint64_t nbytes = elem_size(r32(s + 16)) * r32(b + 24) * r32(b + 28) * r32(b + 32);
            unsigned char *dst;
            if (flags == 0) {
                dst = pool + cursor;
                addr_out[a] = (uint64_t)(uintptr_t)dst;
                cursor += up(nbytes, V2_POOL_ALIGN);
            } else {
                dst = (unsigned char *)(uintptr_t)addr_out[a];
            }
            memcpy(dst, s + base + r64(b + 40), (size_t)nbytes);
        }
    }
    return ORC_OK;
}
