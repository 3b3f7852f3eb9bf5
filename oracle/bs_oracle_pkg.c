/*
 * bs_oracle_pkg.c — TEST INFRASTRUCTURE ONLY.  Plain, slow, single-threaded CPU definition of SELF-CONTAINED
 * PACKAGES.
 *
 * What it follows.  PAPER.md §III.B.3:
 *   L124  "Each serialized component is self contained in the sense that the string contains not only the
 *         deserializable data, but also metadata which pinpoints the location of the component within the
 *         original, whole object.  As a result, these packages can be sent, mixed with other packages and
 *         received back without the need to keep track of their order"
 *   L126  "these packages can be cut down into even smaller packages ... to keep MPI package sizes below an
 *         implementation or self imposed upper limit.  The packages produced by the same serialization call
 *         are kept together ... in the end all packages are stored in a way that the whole, deserializable
 *         byte strings are stored continuously in memory."
 * The paper prints no byte layout; the one below is this project's.  A package carries
 * a range of a wire-format-v1 or -v2 stream; for v2 the blocks are counted in the order of the layered descriptor's addr[]:
 *
 *   package     := package_header(64) | stream bytes [lo, lo + nbytes)
 *   package_header: char magic[8]="BSPKG001"; u32 version=1; u32 index; u32 count; u32 first_block;
 *                   u64 stream_id; u64 total_bytes; u64 lo; u64 nbytes; u64 first_block_offset
 *     stream_id          label of the serialization call the package belongs to ("kept together", L126)
 *     total_bytes        length of the whole stream;  [lo, lo+nbytes) = the package's place in it (L124)
 *     first_block        index of the block that holds the package's first payload byte, i.e. the LARGEST i with
 *                        offset_i <= lo - header_bytes; 0xFFFFFFFF for a package of the header region
 *     first_block_offset lo - header_bytes - offset_{first_block}  (0 for a package of the header region)
 *   cutting (a function of header_bytes, total_bytes and the size limit `cap`, a multiple of 16): the header
 *   region [0, header_bytes) is cut into ceil(header_bytes/cap) packages of cap bytes (the last one shorter),
 *   then the payload [header_bytes, total) likewise; index counts them in stream order; count = their number.
 *   A package never straddles the header / payload boundary, so the packages of the header region alone rebuild
 *   the block table and every payload package can then be unpacked on its own, in any order.
 *
 * Pins (tests/test_oracle_pkg.py): hand-typed golden package headers of the 288-byte v1 golden stream; the cut
 * against a numpy restatement; first_block against numpy.searchsorted over the offsets an independent struct
 * reader extracts; reassembly from shuffled slots == the stream (the paper's property); fault injection.
 * Unpinned: nothing in this file.  Shares no code with the CUDA path or with the other oracle files.
 */
#include <stdint.h>
#include <stddef.h>
#include <string.h>

#define ORC_OK               0
#define ORC_ERR_ARG        (-1)
#define ORC_ERR_CAPACITY   (-2)
#define ORC_ERR_CORRUPT    (-3)

#define PKG_HEADER 64u
#define PKG_NO_BLOCK 0xFFFFFFFFu

static uint32_t g32(const unsigned char *p) { uint32_t v; memcpy(&v, p, 4); return v; }
static uint64_t g64(const unsigned char *p) { uint64_t v; memcpy(&v, p, 8); return v; }
static void p32(unsigned char *p, uint32_t v) { memcpy(p, &v, 4); }
static void p64(unsigned char *p, uint64_t v) { memcpy(p, &v, 8); }

/* ---- the cut ---------------------------------------------------------------------------------------- */
uint64_t orcp_count(uint64_t header_bytes, uint64_t total_bytes, uint64_t cap)
{
    if (cap == 0 || (cap & 15) || header_bytes > total_bytes) return 0;
    uint64_t P = total_bytes - header_bytes;
    return (header_bytes + cap - 1) / cap + (P + cap - 1) / cap;
}

int orcp_range(uint64_t header_bytes, uint64_t total_bytes, uint64_t cap, uint64_t index, uint64_t *lo,
               uint64_t *hi)
{
    if (cap == 0 || (cap & 15) || header_bytes > total_bytes) return ORC_ERR_ARG;
    uint64_t nh = (header_bytes + cap - 1) / cap;
    if (index >= orcp_count(header_bytes, total_bytes, cap)) return ORC_ERR_ARG;
    if (index < nh) {
        *lo = index * cap;
        *hi = (*lo + cap < header_bytes) ? *lo + cap : header_bytes;
    } else {
        *lo = header_bytes + (index - nh) * cap;
        *hi = (*lo + cap < total_bytes) ? *lo + cap : total_bytes;
    }
    return ORC_OK;
}

/* ---- first_block of a wire-format-v2 (structure-shared layers) stream -------------------------------- */
/* The blocks of a layered set are counted layer by layer, inside a layer in the order of its structure's block table
 * (the order of the descriptor's addr[]); block a of layer t, structure block j, starts at payload offset
 * layer_rec[t].offset + block_rec[j].offset.  first_block = the largest a whose start is <= plo, as for v1. */
static void first_block_v2(const unsigned char *s, uint64_t plo, uint32_t *first_block, uint64_t *intra)
{
    uint64_t C = g32(s + 32), T = g64(s + 40);
    const unsigned char *srec = s + 64, *lrec = srec + 32 * C, *brec = lrec + 16 * T;
    uint64_t a = 0;
    for (uint64_t t = 0; t < T; ++t) {
        uint64_t st = g32(lrec + 16 * t), loff = g64(lrec + 16 * t + 8);
        uint64_t fb = g32(srec + 32 * st + 4), nb = g32(srec + 32 * st + 8);
        for (uint64_t j = fb; j < fb + nb; ++j, ++a) {
            uint64_t off = loff + g64(brec + 48 * j + 40);
            if (off <= plo) { *first_block = (uint32_t)a; *intra = plo - off; }
        }
    }
}

/* ---- emit package `index` of a wire-format-v1 or v2 stream into out[0 .. 64 + nbytes) ---------------- */
/* Reads header_bytes, the counts and the block records' offsets from the stream itself. */
int orcp_emit(const unsigned char *s, uint64_t n, uint64_t cap, uint64_t stream_id, uint64_t index,
              unsigned char *out, uint64_t capacity, uint64_t *written)
{
    if (n < 64 || memcmp(s, "BSPARSE1", 8) != 0 || (g32(s + 8) != 1u && g32(s + 8) != 2u)) return ORC_ERR_ARG;
    const int v2 = g32(s + 8) == 2u;
    uint64_t T = v2 ? 0 : g64(s + 32), B = v2 ? 0 : g64(s + 40), hb = g64(s + 48);
    if (hb > n) return ORC_ERR_ARG;
    uint64_t lo, hi;
    int rc = orcp_range(hb, n, cap, index, &lo, &hi);
    if (rc) return rc;
    uint64_t nbytes = hi - lo;
    *written = PKG_HEADER + nbytes;
    if (capacity < PKG_HEADER + nbytes) return ORC_ERR_CAPACITY;
    uint32_t first_block = PKG_NO_BLOCK;
    uint64_t intra = 0;
    if (lo >= hb && v2) {
        first_block_v2(s, lo - hb, &first_block, &intra);
    } else if (lo >= hb) {                            /* largest i with offset_i <= lo - hb */
        const unsigned char *brec = s + 64 + 32 * T;
        uint64_t plo = lo - hb;
        for (uint64_t i = 0; i < B; ++i) {
            uint64_t off = g64(brec + 48 * i + 40);
            if (off <= plo) { first_block = (uint32_t)i; intra = plo - off; }
        }
    }
    memcpy(out, "BSPKG001", 8);
    p32(out + 8, 1u);
    p32(out + 12, (uint32_t)index);
    p32(out + 16, (uint32_t)orcp_count(hb, n, cap));
    p32(out + 20, first_block);
    p64(out + 24, stream_id);
    p64(out + 32, n);
    p64(out + 40, lo);
    p64(out + 48, nbytes);
    p64(out + 56, intra);
    memcpy(out + PKG_HEADER, s + lo, (size_t)nbytes);
    return ORC_OK;
}

/* ---- reassemble: slots in any order -> the whole stream, stored continuously (L126) ------------------ */
/* slots: n_slots slots of slot_bytes each; a slot whose magic is not "BSPKG001" or whose stream_id differs is
 * skipped ("mixed with other packages", L124).  The packages found must carry the same total_bytes and count,
 * every index 0..count-1 exactly once, ranges inside [0,total) that tile it in index order, and fit their slot. */
int orcp_assemble(const unsigned char *slots, uint64_t slot_bytes, uint64_t n_slots, uint64_t stream_id,
                  unsigned char *out, uint64_t capacity, uint64_t *total_bytes)
{
    uint64_t total = 0, count = 0, found = 0;
    if (slot_bytes < PKG_HEADER) return ORC_ERR_ARG;
    for (uint64_t k = 0; k < n_slots; ++k) {          /* pass 1: agree on total and count */
        const unsigned char *h = slots + k * slot_bytes;
        if (memcmp(h, "BSPKG001", 8) != 0 || g64(h + 24) != stream_id) continue;
        if (g32(h + 8) != 1u) return ORC_ERR_CORRUPT;
        if (found == 0) { total = g64(h + 32); count = g32(h + 16); }
        else if (g64(h + 32) != total || g32(h + 16) != count) return ORC_ERR_CORRUPT;
        ++found;
    }
    if (found == 0 || found != count) return ORC_ERR_CORRUPT;
    *total_bytes = total;
    if (capacity < total) return ORC_ERR_CAPACITY;
    uint64_t next = 0;
    for (uint64_t want = 0; want < count; ++want) {   /* pass 2: index order; each index exactly once */
        uint64_t hits = 0;
        for (uint64_t k = 0; k < n_slots; ++k) {
            const unsigned char *h = slots + k * slot_bytes;
            if (memcmp(h, "BSPKG001", 8) != 0 || g64(h + 24) != stream_id) continue;
            if (g32(h + 12) != want) continue;
            uint64_t lo = g64(h + 40), nb = g64(h + 48);
            if (++hits > 1) return ORC_ERR_CORRUPT;
            if (lo != next || nb == 0 || nb > total - lo || nb > slot_bytes - PKG_HEADER) return ORC_ERR_CORRUPT;
            memcpy(out + lo, h + PKG_HEADER, (size_t)nb);
            next = lo + nb;
        }
        if (hits != 1) return ORC_ERR_CORRUPT;
    }
    if (next != total) return ORC_ERR_CORRUPT;
    return ORC_OK;
}
