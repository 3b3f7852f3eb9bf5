/*
 * bs_oracle_v3.c — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded CPU serializer / deserializer for wire
 * format v3: block-sparse tensors of rank 2, 3 or 4 (SURVEY.md §8(f) NEXT-4 "rank-4 tensors").
 *
 * What it follows.  PAPER.md L41: the block-sparse machinery serves "tree-like tensor network state methods" as well —
 * the nodes of a tree tensor network state are order-4 tensors (three virtual legs and a physical one, or four virtual
 * legs), symmetry-blocked exactly like the order-3 MPS tensors of Eq. 2 (L47): a block exists where the quantum numbers
 * of its legs are conserved, and travels with "sector indices, related quantum numbers, and sector dimensions" (L63).
 * The paper prints no byte format; wire format v1 (bs_oracle.c) has room for three legs per block record.
 * Reading D20: v3 is v1 with a fourth leg and nothing else changed —
 *
 *   stream  := fixed_header(64) | tensor_rec[T](32) | block_rec[B](64) | zeros to a multiple of 128 | payload(P)
 *   fixed_header: char magic[8]="BSPARSE1"; u32 version=3; u32 endian_tag=0x01020304; u32 dtype (0 f64, 1 f32, 2 c64,
 *                 3 c128: element size e = 8, 4, 8, 16); u32 n_qn=2; u32 max_rank=4; u32 align=16; u64 n_tensors;
 *                 u64 n_blocks; u64 header_bytes; u64 payload_bytes
 *   tensor_rec  : u32 rank (2, 3 or 4); u32 first_block; u32 n_blocks; i32 dq[2]; i8 sign[4]; u32 tag; u32 reserved=0
 *                 (byte for byte the v1 record: it always had four leg arrows)
 *   block_rec   : i32 qn[4][2]; u32 dim[4]; u32 tensor; u32 reserved=0; u64 offset            (32+16+4+4+8 = 64 bytes)
 *   payload     : block i's e*prod(dim_i[0..3]) raw bytes (row-major, last index fastest) at payload+offset_i, then zeros
 *                 up to the next multiple of 16; offset_i = sum_{j<i} align16(e*prod(dim_j)), descriptor order
 *   header_bytes = align128(64 + 32*T + 64*B);  unused legs of a block (leg >= rank of its tensor): dim 1, labels 0
 *   pool layout on deserialize: addr_i = pool + sum_{j<i} align256(nbytes_j)                  (as v1, D14)
 *
 * The steps are those of SURVEY §8(c) serialize(X) 1-5 and deserialize(S, n) (L90-92 pointer structure first, L106 exact
 * size prediction, L108 identical object back), written in that order with no blocking, threading or reordering.
 *
 * Pins (tests/test_oracle_v3.py, -m "not gpu"): G8 hand-typed golden stream + an independent struct reader
 * (tests/streamreader.py read_stream_v3); offsets vs numpy.cumsum; the PAYLOAD of a set of rank <= 3 tensors == the payload
 * of the separately pinned v1 oracle (the fourth leg has extent 1); dense brute-force reconstruction of order-4 arrays
 * (blocks cut out of a dense 4-index array by a conservation rule, round trip, scattered back, compared bitwise);
 * conservation read from the stream alone; round trip / fixpoint; fault injection on every validated field.
 * Unpinned: nothing in this file.  Shares no code with bs_oracle.c, bs_oracle_v2.c or paper_2412_04676_b200/.
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>

#define ORC_OK               0
#define ORC_ERR_ARG        (-1)
#define ORC_ERR_CAPACITY   (-2)
#define ORC_ERR_CORRUPT    (-3)
#define ORC_ERR_UNSUPPORTED (-4)

#define V3_FIXED   64u
#define V3_TENSOR  32u
#define V3_BLOCK   64u
#define V3_LEGS     4u

typedef struct {
    uint32_t rank;          /* 2, 3 or 4 */
    uint32_t first_block;
    uint32_t n_blocks;
    int32_t  dq[2];
    int8_t   sign[4];
    uint32_t tag;
    uint32_t reserved;      /* 0 */
} orc3_tensor;
typedef char orc3_tensor_is_32_bytes[(sizeof(orc3_tensor) == 32) ? 1 : -1];

static uint64_t up(uint64_t x, uint64_t a) { return (x + (a - 1)) / a * a; }
static void w32(unsigned char *p, uint32_t v) { memcpy(p, &v, 4); }
static void w64(unsigned char *p, uint64_t v) { memcpy(p, &v, 8); }
static uint32_t r32(const unsigned char *p) { uint32_t v; memcpy(&v, p, 4); return v; }
static uint64_t r64(const unsigned char *p) { uint64_t v; memcpy(&v, p, 8); return v; }
static int32_t ri32(const unsigned char *p) { int32_t v; memcpy(&v, p, 4); return v; }
static uint64_t esize(uint32_t dtype) { return dtype == 1u ? 4u : (dtype == 3u ? 16u : 8u); }

uint64_t orc3_header_bytes(uint64_t T, uint64_t B) { return up(V3_FIXED + V3_TENSOR * T + V3_BLOCK * B, 128u); }

/* e * d0*d1*d2*d3 with overflow refused (D13: sizes are u64) */
static int block_bytes(const uint32_t *d, uint32_t dtype, uint64_t *nbytes)
{
    uint64_t n = 1;
    for (uint32_t k = 0; k < V3_LEGS; ++k) {
        if (d[k] != 0 && n > (UINT64_MAX / 16u) / d[k]) return ORC_ERR_ARG;
        n *= d[k];
    }
    *nbytes = esize(dtype) * n;
    return ORC_OK;
}

static int check_desc(uint64_t T, uint64_t B, const orc3_tensor *t, uint32_t dtype)
{
    if (T >= (1ull << 32) || B >= (1ull << 32) || dtype > 3u) return ORC_ERR_UNSUPPORTED;
    uint64_t next = 0;
    for (uint64_t k = 0; k < T; ++k) {
        if (t[k].rank < 2 || t[k].rank > 4) return ORC_ERR_UNSUPPORTED;
        if (t[k].first_block != next) return ORC_ERR_ARG;
        next += t[k].n_blocks;
    }
    return next == B ? ORC_OK : ORC_ERR_ARG;
}

/* step 2, the "pointer structure" (L90-92): nbytes, stored = align16(nbytes), offset = exclusive prefix sum */
int orc3_plan(uint64_t B, const uint32_t *dim /*[B][4]*/, uint32_t dtype, uint64_t *nbytes, uint64_t *stored, uint64_t *offset,
              uint64_t *payload_bytes)
{
    if (dtype > 3u) return ORC_ERR_UNSUPPORTED;
    uint64_t run = 0;
    for (uint64_t i = 0; i < B; ++i) {
        uint64_t nb;
        int rc = block_bytes(dim + 4 * i, dtype, &nb);
        if (rc) return rc;
        if (nbytes) nbytes[i] = nb;
        if (stored) stored[i] = up(nb, 16u);
        if (offset) offset[i] = run;
        run += up(nb, 16u);
    }
    *payload_bytes = run;
    return ORC_OK;
}

int orc3_serialized_size(uint64_t T, uint64_t B, const uint32_t *dim, uint32_t dtype, uint64_t *header_bytes, uint64_t *total_bytes)
{
    uint64_t P;
    int rc = orc3_plan(B, dim, dtype, NULL, NULL, NULL, &P);
    if (rc) return rc;
    *header_bytes = orc3_header_bytes(T, B);
    *total_bytes = *header_bytes + P;
    return ORC_OK;
}

/* steps 1-5 */
int orc3_serialize(uint64_t T, uint64_t B, const orc3_tensor *tensors, const int32_t *qn /*[B][4][2]*/, const uint32_t *dim /*[B][4]*/,
                   const uint64_t *addr /*[B] host addresses*/, uint32_t dtype, unsigned char *out, uint64_t capacity, uint64_t *written)
{
    uint64_t hb, total;
    int rc = check_desc(T, B, tensors, dtype);
    if (rc) return rc;
    rc = orc3_serialized_size(T, B, dim, dtype, &hb, &total);
    if (rc) return rc;
    *written = total;
    if (capacity < total) return ORC_ERR_CAPACITY;

    unsigned char *p = out;
    memcpy(p, "BSPARSE1", 8);
    w32(p + 8, 3u);               /* version */
    w32(p + 12, 0x01020304u);     /* endian_tag */
    w32(p + 16, dtype);
    w32(p + 20, 2u);              /* n_qn */
    w32(p + 24, 4u);              /* max_rank */
    w32(p + 28, 16u);             /* align */
    w64(p + 32, T);
    w64(p + 40, B);
    w64(p + 48, hb);
    w64(p + 56, total - hb);
    p += V3_FIXED;
    for (uint64_t k = 0; k < T; ++k) {                  /* tensor records travel field by field */
        w32(p + 0, tensors[k].rank);
        w32(p + 4, tensors[k].first_block);
        w32(p + 8, tensors[k].n_blocks);
        memcpy(p + 12, &tensors[k].dq[0], 4);
        memcpy(p + 16, &tensors[k].dq[1], 4);
        memcpy(p + 20, tensors[k].sign, 4);
        w32(p + 24, tensors[k].tag);
        w32(p + 28, tensors[k].reserved);
        p += V3_TENSOR;
    }
    uint64_t run = 0;
    for (uint64_t k = 0; k < T; ++k) {
        for (uint64_t i = tensors[k].first_block; i < (uint64_t)tensors[k].first_block + tensors[k].n_blocks; ++i) {
            uint64_t nb = 0;
            block_bytes(dim + 4 * i, dtype, &nb);
            memcpy(p, qn + 8 * i, 32);                  /* i32 qn[4][2] */
            for (uint32_t leg = 0; leg < V3_LEGS; ++leg) w32(p + 32 + 4 * leg, dim[4 * i + leg]);
            w32(p + 48, (uint32_t)k);                   /* owning tensor (L124) */
            w32(p + 52, 0u);                            /* reserved */
            w64(p + 56, run);                           /* offset inside the payload */
            run += up(nb, 16u);
            p += V3_BLOCK;
        }
    }
    memset(p, 0, (size_t)(out + hb - p));               /* slack up to the 128-byte boundary */
    unsigned char *q = out + hb;                         /* step 4: copy, then pad with zeros */
    for (uint64_t i = 0; i < B; ++i) {
        uint64_t nb = 0;
        block_bytes(dim + 4 * i, dtype, &nb);
        memcpy(q, (const void *)(uintptr_t)addr[i], (size_t)nb);
        memset(q + nb, 0, (size_t)(up(nb, 16u) - nb));
        q += up(nb, 16u);
    }
    if ((uint64_t)(q - out) != total) return ORC_ERR_ARG;   /* step 5: prediction == written (L106) */
    return ORC_OK;
}

int orc3_stream_info(const unsigned char *s, uint64_t n, uint64_t *T, uint64_t *B, uint64_t *header_bytes, uint64_t *payload_bytes,
                     uint32_t *dtype)
{
    if (n < V3_FIXED) return ORC_ERR_CORRUPT;
    if (memcmp(s, "BSPARSE1", 8) != 0) return ORC_ERR_CORRUPT;
    if (r32(s + 8) != 3u) return ORC_ERR_CORRUPT;
    if (r32(s + 12) != 0x01020304u) return ORC_ERR_CORRUPT;
    if (r32(s + 16) > 3u) return ORC_ERR_CORRUPT;
    if (r32(s + 20) != 2u) return ORC_ERR_CORRUPT;
    if (r32(s + 24) != 4u) return ORC_ERR_CORRUPT;
    if (r32(s + 28) != 16u) return ORC_ERR_CORRUPT;
    *dtype = r32(s + 16);
    *T = r64(s + 32);
    *B = r64(s + 40);
    *header_bytes = r64(s + 48);
    *payload_bytes = r64(s + 56);
    if (*T >= (1ull << 32) || *B >= (1ull << 32)) return ORC_ERR_CORRUPT;
    if (*header_bytes != orc3_header_bytes(*T, *B)) return ORC_ERR_CORRUPT;
    return ORC_OK;
}

/* every check of SURVEY §8(c) deserialize(S, n), in that order, with a fourth leg */
int orc3_validate_stream(const unsigned char *s, uint64_t n)
{
    uint64_t T, B, hb, P;
    uint32_t dtype;
    int rc = orc3_stream_info(s, n, &T, &B, &hb, &P, &dtype);
    if (rc) return rc;
    if (hb > n || hb + P != n) return ORC_ERR_CORRUPT;
    const unsigned char *trec = s + V3_FIXED, *brec = trec + V3_TENSOR * T;
    uint64_t next = 0, run = 0;
    for (uint64_t k = 0; k < T; ++k) {
        const unsigned char *t = trec + V3_TENSOR * k;
        uint32_t rank = r32(t), first = r32(t + 4), nb = r32(t + 8);
        if (rank < 2 || rank > 4) return ORC_ERR_CORRUPT;
        if (r32(t + 28) != 0) return ORC_ERR_CORRUPT;
        if (first != next) return ORC_ERR_CORRUPT;
        if ((uint64_t)first + nb > B) return ORC_ERR_CORRUPT;
        for (uint64_t i = first; i < (uint64_t)first + nb; ++i) {
            const unsigned char *b = brec + V3_BLOCK * i;
            if (r32(b + 48) != (uint32_t)k) return ORC_ERR_CORRUPT;          /* owner */
            if (r32(b + 52) != 0) return ORC_ERR_CORRUPT;                    /* reserved */
            for (uint32_t leg = rank; leg < V3_LEGS; ++leg) {                 /* unused legs */
                if (r32(b + 32 + 4 * leg) != 1) return ORC_ERR_CORRUPT;
                if (ri32(b + 8 * leg) != 0 || ri32(b + 8 * leg + 4) != 0) return ORC_ERR_CORRUPT;
            }
            uint32_t d[4] = { r32(b + 32), r32(b + 36), r32(b + 40), r32(b + 44) };
            uint64_t nbytes;
            if (block_bytes(d, dtype, &nbytes)) return ORC_ERR_CORRUPT;
            if (r64(b + 56) != run) return ORC_ERR_CORRUPT;                   /* offsets = exclusive prefix sum */
            uint64_t st = up(nbytes, 16u);
            if (st < nbytes || run + st < run || run + st > P) return ORC_ERR_CORRUPT;
            for (uint64_t z = nbytes; z < st; ++z)
                if (s[hb + run + z] != 0) return ORC_ERR_CORRUPT;             /* pad bytes are zero */
            run += st;
        }
        next += nb;
    }
    if (next != B || run != P) return ORC_ERR_CORRUPT;
    for (uint64_t z = V3_FIXED + V3_TENSOR * T + V3_BLOCK * B; z < hb; ++z)
        if (s[z] != 0) return ORC_ERR_CORRUPT;
    return ORC_OK;
}

int orc3_pool_bytes(const unsigned char *s, uint64_t n, uint64_t *pool_bytes)
{
    uint64_t T, B, hb, P, sum = 0;
    uint32_t dtype;
    int rc = orc3_stream_info(s, n, &T, &B, &hb, &P, &dtype);
    if (rc) return rc;
    if (hb > n) return ORC_ERR_CORRUPT;
    const unsigned char *brec = s + V3_FIXED + V3_TENSOR * T;
    for (uint64_t i = 0; i < B; ++i) {
        const unsigned char *b = brec + V3_BLOCK * i;
        sum += up(esize(dtype) * r32(b + 32) * r32(b + 36) * r32(b + 40) * r32(b + 44), 256u);
    }
    *pool_bytes = sum;
    return ORC_OK;
}

/* flags 0: pool layout (addr_out written); flags 1: scatter (addr_out, dim_out are inputs; extents must match) */
int orc3_deserialize(const unsigned char *s, uint64_t n, orc3_tensor *tensors_out, int32_t *qn_out /*[B][4][2]*/,
                     uint32_t *dim_out /*[B][4]*/, uint64_t *addr_out, unsigned char *pool, uint64_t pool_bytes, uint32_t flags)
{
    int rc = orc3_validate_stream(s, n);
    if (rc) return rc;
    uint64_t T, B, hb, P;
    uint32_t dtype;
    orc3_stream_info(s, n, &T, &B, &hb, &P, &dtype);
    const unsigned char *trec = s + V3_FIXED, *brec = trec + V3_TENSOR * T;
    if (flags == 0) {
        uint64_t need;
        orc3_pool_bytes(s, n, &need);
        if (need > pool_bytes) return ORC_ERR_CAPACITY;
    } else if (flags == 1) {
        for (uint64_t i = 0; i < B; ++i)
            for (uint32_t leg = 0; leg < V3_LEGS; ++leg)
                if (dim_out[4 * i + leg] != r32(brec + V3_BLOCK * i + 32 + 4 * leg)) return ORC_ERR_ARG;
    } else {
        return ORC_ERR_ARG;
    }
    for (uint64_t k = 0; k < T; ++k) memcpy(&tensors_out[k], trec + V3_TENSOR * k, V3_TENSOR);
    uint64_t cursor = 0;
    for (uint64_t i = 0; i < B; ++i) {
        const unsigned char *b = brec + V3_BLOCK * i;
        memcpy(qn_out + 8 * i, b, 32);
        uint64_t nbytes = esize(dtype);
        for (uint32_t leg = 0; leg < V3_LEGS; ++leg) {
            dim_out[4 * i + leg] = r32(b + 32 + 4 * leg);
            nbytes *= dim_out[4 * i + leg];
        }
        unsigned char *dst;
        if (flags == 0) {
            dst = pool + cursor;
            addr_out[i] = (uint64_t)(uintptr_t)dst;
            cursor += up(nbytes, 256u);
        } else {
            dst = (unsigned char *)(uintptr_t)addr_out[i];
        }
        memcpy(dst, s + hb + r64(b + 56), (size_t)nbytes);
    }
    return ORC_OK;
}

/* D10 / P4 with four legs: every block satisfies sum_k sign[k]*qn[k] == dq.  0 clean, 1 violated, <0 malformed */
int orc3_validate_set(uint64_t T, uint64_t B, const orc3_tensor *tensors, const int32_t *qn)
{
    int rc = check_desc(T, B, tensors, 0);
    if (rc) return rc;
    for (uint64_t k = 0; k < T; ++k)
        for (uint64_t i = tensors[k].first_block; i < (uint64_t)tensors[k].first_block + tensors[k].n_blocks; ++i)
            for (int c = 0; c < 2; ++c) {
                int64_t acc = 0;
                for (uint32_t leg = 0; leg < V3_LEGS; ++leg) acc += (int64_t)tensors[k].sign[leg] * qn[8 * i + 2 * leg + c];
                if (acc != tensors[k].dq[c]) return 1;
            }
    return 0;
}
