/*
 * bs_oracle.c — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded CPU serializer /
 * deserializer for symmetry-blocked (U(1)-labelled) block-sparse fp64 tensors.
 *
 * This file DEFINES what the CUDA path must produce, byte for byte (tolerance 0).  It shares no
 * code, header, table or helper with paper_2412_04676_b200/: every struct layout is re-typed here.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 * build, load or call it.
 *
 * What it follows.  PAPER.md (arxiv 2412.04676) states *properties* of its serializer and no
 * byte format:
 *   L85   serialization = "generating long continuous stripes in memory"
 *   L63   non-zero sectors go "together with series of meta data ... sector indices, related
 *         quantum numbers, and sector dimensions"
 *   L90-92 a "pointer structure ... grid structure of the serialized data" is determined first,
 *         buffers are "filled with actual data only afterward"
 *   L106  "low cost and exact prediction of post-serialization data size before the actual
 *         serialization"; each worker gets an exact interval of the single output buffer
 *   L108  workers fill independently, yet "produce a single, continuos stream of bytes, which
 *         deserializes into an object identical to the one used as the original input"
 *   L124  each component carries "metadata which pinpoints the location of the component within
 *         the original, whole object"
 *   L134  deserialization restores "the block sparse matrix and tensor structures"
 * The byte format ("wire format v1") that realises these is this project's own reading, listed in
 * DESIGN.md "Readings" D1-D18.  The steps below are written in the order of
 * SURVEY §8(c) serialize(X) 1-5 and deserialize(S, n), with no blocking, threading or reordering.
 *
 * Pins (tests/test_oracle_*.py, -m "not gpu"): P7 hand-checked 288-byte golden stream + an
 * independent Python struct reader; P3 offsets vs numpy.cumsum; P1 round trip / fixpoint; P2 size
 * prediction; P4 conservation read from the stream alone; P5 dense brute-force reconstruction;
 * P8 memcpy special cases; P9 placement invariance; P10 fault injection; P11 special bit patterns.
 * Unpinned: nothing in this file.  (The paper's GB/s figures are "parity unpinned": no number in
 * the paper is tied to a byte format.)
 *
 * Reading D19 (round 2; SURVEY §8(c) D3 kept `align` as a header field "so a future align=8 (no pad, literal unpadded
 * reading) is representable"; SURVEY §8(f) NEXT-4 "align = 8 unpadded streams"; BASELINE.json north_star: "offsets equal to
 * the exclusive prefix sum of the block byte sizes"): the header's align word is 16 or 8 and is the ONLY thing that
 * changes — stored_i = align_up(nbytes_i, align), offset_i = the exclusive prefix sum of stored_i, payload_bytes = their sum.
 * With align = 8 an fp64 block is stored without any pad byte, offsets are the literal prefix sum of the block byte sizes,
 * and the stream's total is a multiple of 8 (not of 16).  Every function that took no alignment keeps its round-1 meaning
 * (16) and has an `_al` twin that takes it; the readers take it from the header.  Pins (tests/test_oracle_align8.py): G7
 * hand-typed 280-byte golden stream (the P7 example unpadded: offsets 0, 8); offsets vs numpy.cumsum of the unpadded sizes;
 * byte equality with the independently written numpy oracle (bs_oracle_dtype.py) at align 8; payload == the plain
 * concatenation of the blocks; round trip, fixpoint, fault injection.
 *
 * All integers little-endian; the host is assumed little-endian (checked in orc_selftest_endian).
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>

#define ORC_OK               0
#define ORC_ERR_ARG        (-1)
#define ORC_ERR_CAPACITY   (-2)
#define ORC_ERR_CORRUPT    (-3)
#define ORC_ERR_UNSUPPORTED (-4)

#define ORC_FIXED_HEADER 64u
#define ORC_TENSOR_REC   32u
#define ORC_BLOCK_REC    48u
#define ORC_HEADER_ALIGN 128u
#define ORC_BLOCK_ALIGN  16u
#define ORC_POOL_ALIGN   256u

/* descriptor record of one tensor; identical bytes on the wire (format v1 "tensor_rec") */
typedef struct {
    uint32_t rank;          /* 2 or 3 */
    uint32_t first_block;
    uint32_t n_blocks;
    int32_t  dq[2];         /* conserved charge (dN, d2Sz) */
    int8_t   sign[4];       /* leg arrows, unused legs 0 */
    uint32_t tag;
    uint32_t reserved;      /* 0 */
} orc_tensor;

typedef char orc_tensor_is_32_bytes[(sizeof(orc_tensor) == 32) ? 1 : -1];

static uint64_t align_up(uint64_t x, uint64_t a) { return (x + (a - 1)) / a * a; }

static void put_u32(unsigned char *p, uint32_t v) { memcpy(p, &v, 4); }
static void put_u64(unsigned char *p, uint64_t v) { memcpy(p, &v, 8); }
static uint32_t get_u32(const unsigned char *p) { uint32_t v; memcpy(&v, p, 4); return v; }
static uint64_t get_u64(const unsigned char *p) { uint64_t v; memcpy(&v, p, 8); return v; }
static int32_t  get_i32(const unsigned char *p) { int32_t v; memcpy(&v, p, 4); return v; }

int orc_selftest_endian(void) { uint32_t x = 0x01020304u; unsigned char b[4]; memcpy(b, &x, 4); return b[0] == 4; }

/* ---- serialize, step 1: header size is known from the counts alone (L106) ------------------- */
uint64_t orc_header_bytes(uint64_t T, uint64_t B)
{
    return align_up(ORC_FIXED_HEADER + ORC_TENSOR_REC * T + ORC_BLOCK_REC * B, ORC_HEADER_ALIGN);
}

/* ---- serialize, step 2: the "pointer structure" (L90-92): sizes, stored sizes, offsets ------ */
/* nbytes[i] = 8*prod(dim[i]);  stored[i] = align_up(nbytes[i], align);  offset[i] = sum_{j<i} stored[j];
 * align = 16 (wire format v1 as round 1 defined it) or 8 (reading D19: unpadded for fp64) */
int orc_plan_al(uint64_t B, const uint32_t *dim /*[B][3]*/, uint32_t align, uint64_t *nbytes, uint64_t *stored,
                uint64_t *offset, uint64_t *payload_bytes)
{
    uint64_t run = 0;
    if (align != 16u && align != 8u) return ORC_ERR_UNSUPPORTED;
    for (uint64_t i = 0; i < B; ++i) {
        uint64_t d0 = dim[3 * i + 0], d1 = dim[3 * i + 1], d2 = dim[3 * i + 2];
        uint64_t n01 = d0 * d1;                         /* < 2^64 always (u32*u32) */
        if (d2 != 0 && n01 > (UINT64_MAX / 8u) / d2) return ORC_ERR_ARG;
        uint64_t nb = 8u * n01 * d2;
        uint64_t st = align_up(nb, align);
        if (nbytes) nbytes[i] = nb;
        if (stored) stored[i] = st;
        if (offset) offset[i] = run;
        run += st;
    }
    *payload_bytes = run;
    return ORC_OK;
}

int orc_plan(uint64_t B, const uint32_t *dim /*[B][3]*/, uint64_t *nbytes, uint64_t *stored,
             uint64_t *offset, uint64_t *payload_bytes)
{
    return orc_plan_al(B, dim, ORC_BLOCK_ALIGN, nbytes, stored, offset, payload_bytes);
}

int orc_serialized_size_al(uint64_t T, uint64_t B, const uint32_t *dim, uint32_t align, uint64_t *header_bytes,
                           uint64_t *total_bytes)
{
    uint64_t P;
    int rc = orc_plan_al(B, dim, align, NULL, NULL, NULL, &P);
    if (rc) return rc;
    *header_bytes = orc_header_bytes(T, B);
    *total_bytes = *header_bytes + P;
    return ORC_OK;
}

int orc_serialized_size(uint64_t T, uint64_t B, const uint32_t *dim, uint64_t *header_bytes,
                        uint64_t *total_bytes)
{
    return orc_serialized_size_al(T, B, dim, ORC_BLOCK_ALIGN, header_bytes, total_bytes);
}

/* the descriptor must partition the block table into tensors in order (D5, D8) */
static int check_descriptor(uint64_t T, uint64_t B, const orc_tensor *t)
{
    uint64_t next = 0;
    if (T >= (1ull << 32) || B >= (1ull << 32)) return ORC_ERR_UNSUPPORTED;   /* D13 */
    for (uint64_t k = 0; k < T; ++k) {
        if (t[k].rank != 2 && t[k].rank != 3) return ORC_ERR_UNSUPPORTED;
        if (t[k].first_block != next) return ORC_ERR_ARG;
        next += t[k].n_blocks;
    }
    if (next != B) return ORC_ERR_ARG;
    return ORC_OK;
}

/* ---- serialize, step 3: fixed header, tensor records, block records, zero slack ------------- */
int orc_emit_header_al(uint64_t T, uint64_t B, const orc_tensor *tensors, const int32_t *qn /*[B][3][2]*/,
                       const uint32_t *dim /*[B][3]*/, uint32_t align, unsigned char *out, uint64_t capacity)
{
    int rc = check_descriptor(T, B, tensors);
    if (rc) return rc;
    uint64_t hb = orc_header_bytes(T, B), P;
    if (capacity < hb) return ORC_ERR_CAPACITY;
    rc = orc_plan_al(B, dim, align, NULL, NULL, NULL, &P);
    if (rc) return rc;

    unsigned char *p = out;
    memcpy(p, "BSPARSE1", 8);
    put_u32(p + 8, 1u);              /* version */
    put_u32(p + 12, 0x01020304u);    /* endian_tag */
    put_u32(p + 16, 0u);             /* dtype f64 */
    put_u32(p + 20, 2u);             /* n_qn */
    put_u32(p + 24, 3u);             /* max_rank */
    put_u32(p + 28, align);          /* align: 16, or 8 (reading D19) */
    put_u64(p + 32, T);
    put_u64(p + 40, B);
    put_u64(p + 48, hb);
    put_u64(p + 56, P);
    p += ORC_FIXED_HEADER;

    for (uint64_t k = 0; k < T; ++k) {
        put_u32(p + 0, tensors[k].rank);
        put_u32(p + 4, tensors[k].first_block);
        put_u32(p + 8, tensors[k].n_blocks);
        memcpy(p + 12, &tensors[k].dq[0], 4);
        memcpy(p + 16, &tensors[k].dq[1], 4);
        memcpy(p + 20, tensors[k].sign, 4);
        put_u32(p + 24, tensors[k].tag);
        put_u32(p + 28, tensors[k].reserved);
        p += ORC_TENSOR_REC;
    }

    uint64_t run = 0;
    for (uint64_t k = 0; k < T; ++k) {
        for (uint64_t i = tensors[k].first_block; i < (uint64_t)tensors[k].first_block + tensors[k].n_blocks; ++i) {
            memcpy(p, qn + 6 * i, 24);                  /* i32 qn[3][2] */
            put_u32(p + 24, dim[3 * i + 0]);
            put_u32(p + 28, dim[3 * i + 1]);
            put_u32(p + 32, dim[3 * i + 2]);
            put_u32(p + 36, (uint32_t)k);               /* owning tensor (L124) */
            put_u64(p + 40, run);                       /* offset inside the payload */
            run += align_up(8ull * dim[3 * i + 0] * dim[3 * i + 1] * dim[3 * i + 2], align);
            p += ORC_BLOCK_REC;
        }
    }
    memset(p, 0, (size_t)(out + hb - p));               /* slack up to the 128-byte boundary */
    return ORC_OK;
}

int orc_emit_header(uint64_t T, uint64_t B, const orc_tensor *tensors, const int32_t *qn /*[B][3][2]*/,
                    const uint32_t *dim /*[B][3]*/, unsigned char *out, uint64_t capacity)
{
    return orc_emit_header_al(T, B, tensors, qn, dim, ORC_BLOCK_ALIGN, out, capacity);
}

/* ---- serialize, step 4 for blocks of tensors [t0,t1): copy, then pad with zeros ------------- */
/* Writes payload bytes [offset(first block of t0), offset(end of t1-1)) to out[0..).  addr[i] is
 * the host address of block i for i in that range (other entries are not read). */
int orc_emit_payload_range_al(uint64_t T, uint64_t B, const orc_tensor *tensors, const uint32_t *dim,
                              const uint64_t *addr, uint32_t align, uint64_t t0, uint64_t t1, unsigned char *out,
                              uint64_t capacity, uint64_t *first_offset, uint64_t *range_bytes)
{
    int rc = check_descriptor(T, B, tensors);
    if (rc) return rc;
    if (align != 16u && align != 8u) return ORC_ERR_UNSUPPORTED;
    if (t0 > t1 || t1 > T) return ORC_ERR_ARG;
    uint64_t b0 = (t0 < T) ? tensors[t0].first_block : B;
    uint64_t b1 = (t1 < T) ? tensors[t1].first_block : B;
    uint64_t run = 0, start = 0;
    for (uint64_t i = 0; i < b1; ++i) {
        uint64_t nb = 8ull * dim[3 * i + 0] * dim[3 * i + 1] * dim[3 * i + 2];
        uint64_t st = align_up(nb, align);
        if (i == b0) start = run;
        if (i >= b0) {
            if (run - start + st > capacity) return ORC_ERR_CAPACITY;
            memcpy(out + (run - start), (const void *)(uintptr_t)addr[i], (size_t)nb);
            memset(out + (run - start) + nb, 0, (size_t)(st - nb));
        }
        run += st;
    }
    if (b0 >= b1) start = run;
    *first_offset = start;
    *range_bytes = run - start;
    return ORC_OK;
}

int orc_emit_payload_range(uint64_t T, uint64_t B, const orc_tensor *tensors, const uint32_t *dim,
                           const uint64_t *addr, uint64_t t0, uint64_t t1, unsigned char *out,
                           uint64_t capacity, uint64_t *first_offset, uint64_t *range_bytes)
{
    return orc_emit_payload_range_al(T, B, tensors, dim, addr, ORC_BLOCK_ALIGN, t0, t1, out, capacity, first_offset, range_bytes);
}

/* ---- serialize, steps 1-5 --------------------------------------------------------------------- */
int orc_serialize_al(uint64_t T, uint64_t B, const orc_tensor *tensors, const int32_t *qn,
                     const uint32_t *dim, const uint64_t *addr, uint32_t align, unsigned char *out, uint64_t capacity,
                     uint64_t *written)
{
    uint64_t hb, total, first, pb;
    int rc = check_descriptor(T, B, tensors);
    if (rc) return rc;
    rc = orc_serialized_size_al(T, B, dim, align, &hb, &total);          /* steps 1-2 */
    if (rc) return rc;
    *written = total;                                                     /* required size, also on failure */
    if (capacity < total) return ORC_ERR_CAPACITY;
    rc = orc_emit_header_al(T, B, tensors, qn, dim, align, out, capacity); /* step 3 */
    if (rc) return rc;
    rc = orc_emit_payload_range_al(T, B, tensors, dim, addr, align, 0, T, out + hb, capacity - hb, &first, &pb);  /* step 4 */
    if (rc) return rc;
    if (first != 0 || hb + pb != total) return ORC_ERR_ARG;               /* step 5: prediction == written */
    return ORC_OK;
}

int orc_serialize(uint64_t T, uint64_t B, const orc_tensor *tensors, const int32_t *qn,
                  const uint32_t *dim, const uint64_t *addr, unsigned char *out, uint64_t capacity,
                  uint64_t *written)
{
    return orc_serialize_al(T, B, tensors, qn, dim, addr, ORC_BLOCK_ALIGN, out, capacity, written);
}

/* ---- stream_info: the fixed header alone ----------------------------------------------------- */
int orc_stream_info(const unsigned char *s, uint64_t n, uint64_t *T, uint64_t *B, uint64_t *header_bytes,
                    uint64_t *payload_bytes)
{
    if (n < ORC_FIXED_HEADER) return ORC_ERR_CORRUPT;
    if (memcmp(s, "BSPARSE1", 8) != 0) return ORC_ERR_CORRUPT;
    if (get_u32(s + 8) != 1u) return ORC_ERR_CORRUPT;
    if (get_u32(s + 12) != 0x01020304u) return ORC_ERR_CORRUPT;
    if (get_u32(s + 16) != 0u) return ORC_ERR_CORRUPT;
    if (get_u32(s + 20) != 2u) return ORC_ERR_CORRUPT;
    if (get_u32(s + 24) != 3u) return ORC_ERR_CORRUPT;
    if (get_u32(s + 28) != 16u && get_u32(s + 28) != 8u) return ORC_ERR_CORRUPT;   /* align (reading D19) */
    *T = get_u64(s + 32);
    *B = get_u64(s + 40);
    *header_bytes = get_u64(s + 48);
    *payload_bytes = get_u64(s + 56);
    if (*T >= (1ull << 32) || *B >= (1ull << 32)) return ORC_ERR_CORRUPT;
    if (*header_bytes != orc_header_bytes(*T, *B)) return ORC_ERR_CORRUPT;
    return ORC_OK;
}

/* the align word of a stream whose fixed header orc_stream_info accepts */
int orc_stream_align(const unsigned char *s, uint64_t n, uint32_t *align)
{
    uint64_t T, B, hb, P;
    int rc = orc_stream_info(s, n, &T, &B, &hb, &P);
    if (rc) return rc;
    *align = get_u32(s + 28);
    return ORC_OK;
}

/* ---- validate: every check of SURVEY §8(c) deserialize(S, n), in that order ------------------ */
int orc_validate_stream(const unsigned char *s, uint64_t n)
{
    uint64_t T, B, hb, P;
    int rc = orc_stream_info(s, n, &T, &B, &hb, &P);
    if (rc) return rc;
    if (hb > n || hb + P != n) return ORC_ERR_CORRUPT;
    const uint32_t align = get_u32(s + 28);
    const unsigned char *trec = s + ORC_FIXED_HEADER;
    const unsigned char *brec = trec + ORC_TENSOR_REC * T;
    uint64_t next = 0, run = 0;
    for (uint64_t k = 0; k < T; ++k) {
        const unsigned char *t = trec + ORC_TENSOR_REC * k;
        uint32_t rank = get_u32(t), first = get_u32(t + 4), nb = get_u32(t + 8);
        if (rank != 2 && rank != 3) return ORC_ERR_CORRUPT;
        if (get_u32(t + 28) != 0) return ORC_ERR_CORRUPT;           /* reserved */
        if (first != next) return ORC_ERR_CORRUPT;
        if ((uint64_t)first + nb > B) return ORC_ERR_CORRUPT;
        for (uint64_t i = first; i < (uint64_t)first + nb; ++i) {
            const unsigned char *b = brec + ORC_BLOCK_REC * i;
            if (get_u32(b + 36) != (uint32_t)k) return ORC_ERR_CORRUPT;   /* owner */
            for (uint32_t leg = rank; leg < 3; ++leg) {                   /* unused legs */
                if (get_u32(b + 24 + 4 * leg) != 1) return ORC_ERR_CORRUPT;
                if (get_i32(b + 8 * leg) != 0 || get_i32(b + 8 * leg + 4) != 0) return ORC_ERR_CORRUPT;
            }
            uint64_t d0 = get_u32(b + 24), d1 = get_u32(b + 28), d2 = get_u32(b + 32);
            uint64_t n01 = d0 * d1;
            if (d2 != 0 && n01 > (UINT64_MAX / 8u) / d2) return ORC_ERR_CORRUPT;
            uint64_t nbytes = 8u * n01 * d2;
            if (get_u64(b + 40) != run) return ORC_ERR_CORRUPT;           /* offsets = exclusive sum */
            uint64_t st = align_up(nbytes, align);
            if (st < nbytes || run + st < run || run + st > P) return ORC_ERR_CORRUPT;
            for (uint64_t z = nbytes; z < st; ++z)                         /* pad bytes are zero */
                if (s[hb + run + z] != 0) return ORC_ERR_CORRUPT;
            run += st;
        }
        next += nb;
    }
    if (next != B) return ORC_ERR_CORRUPT;
    if (run != P) return ORC_ERR_CORRUPT;
    for (uint64_t z = ORC_FIXED_HEADER + ORC_TENSOR_REC * T + ORC_BLOCK_REC * B; z < hb; ++z)  /* slack */
        if (s[z] != 0) return ORC_ERR_CORRUPT;
    return ORC_OK;
}

/* pool bytes BS_LAYOUT_POOL needs: sum align256(nbytes_i)  (D14) */
int orc_pool_bytes(const unsigned char *s, uint64_t n, uint64_t *pool_bytes)
{
    uint64_t T, B, hb, P, sum = 0;
    int rc = orc_stream_info(s, n, &T, &B, &hb, &P);
    if (rc) return rc;
    if (hb > n) return ORC_ERR_CORRUPT;
    const unsigned char *brec = s + ORC_FIXED_HEADER + ORC_TENSOR_REC * T;
    for (uint64_t i = 0; i < B; ++i) {
        const unsigned char *b = brec + ORC_BLOCK_REC * i;
        sum += align_up(8ull * get_u32(b + 24) * get_u32(b + 28) * get_u32(b + 32), ORC_POOL_ALIGN);
    }
    *pool_bytes = sum;
    return ORC_OK;
}

/* ---- deserialize ------------------------------------------------------------------------------
 * flags 0 (pool layout): addr_out[i] = pool + sum_{j<i} align256(nbytes_j); block data copied there.
 * flags 1 (scatter):     addr_out[i] is an input (caller-chosen host address); dim_out is an input and
 *                        must equal the stream's extents.
 * On any validation failure nothing is written. */
int orc_deserialize(const unsigned char *s, uint64_t n, orc_tensor *tensors_out, int32_t *qn_out,
                    uint32_t *dim_out, uint64_t *addr_out, unsigned char *pool, uint64_t pool_bytes,
                    uint32_t flags)
{
    int rc = orc_validate_stream(s, n);
    if (rc) return rc;
    uint64_t T, B, hb, P;
    orc_stream_info(s, n, &T, &B, &hb, &P);
    const unsigned char *trec = s + ORC_FIXED_HEADER;
    const unsigned char *brec = trec + ORC_TENSOR_REC * T;
    if (flags == 0) {
        uint64_t need;
        orc_pool_bytes(s, n, &need);
        if (need > pool_bytes) return ORC_ERR_CAPACITY;
    } else if (flags == 1) {
        for (uint64_t i = 0; i < B; ++i)
            for (int leg = 0; leg < 3; ++leg)
                if (dim_out[3 * i + leg] != get_u32(brec + ORC_BLOCK_REC * i + 24 + 4 * leg)) return ORC_ERR_ARG;
    } else {
        return ORC_ERR_ARG;
    }
    for (uint64_t k = 0; k < T; ++k) memcpy(&tensors_out[k], trec + ORC_TENSOR_REC * k, ORC_TENSOR_REC);
    uint64_t cursor = 0;
    for (uint64_t i = 0; i < B; ++i) {
        const unsigned char *b = brec + ORC_BLOCK_REC * i;
        memcpy(qn_out + 6 * i, b, 24);
        uint32_t d0 = get_u32(b + 24), d1 = get_u32(b + 28), d2 = get_u32(b + 32);
        dim_out[3 * i + 0] = d0; dim_out[3 * i + 1] = d1; dim_out[3 * i + 2] = d2;
        uint64_t nbytes = 8ull * d0 * d1 * d2;
        unsigned char *dst;
        if (flags == 0) {
            dst = pool + cursor;
            addr_out[i] = (uint64_t)(uintptr_t)dst;
            cursor += align_up(nbytes, ORC_POOL_ALIGN);
        } else {
            dst = (unsigned char *)(uintptr_t)addr_out[i];
        }
        memcpy(dst, s + hb + get_u64(b + 40), (size_t)nbytes);
    }
    return ORC_OK;
}

/* ---- helpers outside the hot path -------------------------------------------------------------
 * D10/P4: every block satisfies sum_k sign[k]*qn[k] == dq.  D12: duplicate label tuples inside a
 * tensor are flagged here, never by the serializer.  Returns 0 if clean, 1 conservation violated,
 * 2 duplicate labels, <0 on a malformed descriptor. */
int orc_validate_set(uint64_t T, uint64_t B, const orc_tensor *tensors, const int32_t *qn)
{
    int rc = check_descriptor(T, B, tensors);
    if (rc) return rc;
    for (uint64_t k = 0; k < T; ++k) {
        uint64_t lo = tensors[k].first_block, hi = lo + tensors[k].n_blocks;
        for (uint64_t i = lo; i < hi; ++i) {
            for (int c = 0; c < 2; ++c) {
                int64_t acc = 0;
                for (int leg = 0; leg < 3; ++leg) acc += (int64_t)tensors[k].sign[leg] * qn[6 * i + 2 * leg + c];
                if (acc != tensors[k].dq[c]) return 1;
            }
            for (uint64_t j = lo; j < i; ++j)
                if (memcmp(qn + 6 * i, qn + 6 * j, 24) == 0) return 2;
        }
    }
    return 0;
}
