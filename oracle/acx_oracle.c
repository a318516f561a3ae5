/* ORACLE — test infrastructure, not product code.
 *
 * A plain, slow, single-threaded CPU decoder of the ACX-B200 archive format, version 3 (FORMAT.md), written from FORMAT.md
 * and the paper's description of the method (§2: absolute-offset LZ77, fixed-size blocks, four streams
 * per block: literals, match lengths, absolute offsets, command sequence; §5: 64-bit sizes/offsets;
 * PAPER.md:125 §6.2: literal classes stored separately).
 * It shares no code, header, table generator or helper with the CUDA path (paper_2606_18900_b200/csrc) or with the
 * encoder.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * The method reaches exactly the original bytes, so the final pin is decode(encode(x)) == x against the ORIGINAL
 * bytes (tests/test_oracle_*.py); the byte-serial copy loop below is the definition of LZ77 copy semantics
 * (FORMAT.md §2) and the rANS step is FORMAT.md §1.7 written out symbol by symbol.  Segments are decoded in index
 * order, which is always valid because every source precedes its destination.
 *
 * Parity status: every function here is pinned (hand-built archives with hand-written expected bytes, an
 * independent pure-Python rANS encoder and byte-serial reference in the tests, closed-form compressed size,
 * final-state invariant, round trips against the original bytes; each rule of FORMAT.md §3 has a hand-built archive
 * that violates only that rule).  Nothing is "parity unpinned".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { OK = 0, E_MAGIC = -1, E_VERSION = -2, E_TRUNCATED = -3, E_CORRUPT = -4, E_RANGE = -5, E_LEVEL = -6, E_NOMEM = -7 };

static uint64_t rd64(const uint8_t* p) { uint64_t v = 0; for (int i = 7; i >= 0; i--) v = (v << 8) | p[i]; return v; }
static uint32_t rd32(const uint8_t* p) { return (uint32_t)p[0] | ((uint32_t)p[1] << 8) | ((uint32_t)p[2] << 16) | ((uint32_t)p[3] << 24); }
static uint32_t rd16(const uint8_t* p) { return (uint32_t)p[0] | ((uint32_t)p[1] << 8); }

typedef struct {
    uint64_t N, n_blocks, n_segs, tables_off, qtab_off, blocktab_off, dir_off, fnv_off, payload_off, archive_bytes;
    uint64_t total_lit, total_match_bytes, total_matches, total_cmds, total_litq, src_window;
    uint32_t log2_bs, min_match, W, prob_bits, n_tables, max_level, max_cmds, flags, log2_seg, q_min, q_mode, n_qpairs;
} hdr_t;

#define TAIL_PAD 128u
#define HEADER_BYTES 192u
#define MAX_TABLES 12          /* 4 + W, W <= 8 */

/* FORMAT.md §1.1 */
static int parse_header(const uint8_t* a, uint64_t n, hdr_t* h) {
    static const uint8_t magic[8] = {0x41, 0x43, 0x58, 0x42, 0x32, 0x30, 0x30, 0x00};
    if (n < HEADER_BYTES) return E_TRUNCATED;
    if (memcmp(a, magic, 8)) return E_MAGIC;
    if (rd32(a + 8) != 3) return E_VERSION;
    if (rd32(a + 12) != HEADER_BYTES) return E_CORRUPT;
    h->N = rd64(a + 16); h->n_blocks = rd64(a + 24); h->n_segs = rd64(a + 32);
    h->log2_bs = rd32(a + 40); h->min_match = rd32(a + 44); h->W = rd32(a + 48); h->prob_bits = rd32(a + 52);
    h->n_tables = rd32(a + 56); h->max_level = rd32(a + 60); h->max_cmds = rd32(a + 64); h->flags = rd32(a + 68);
    h->log2_seg = rd32(a + 72); h->q_min = rd32(a + 76); h->q_mode = rd32(a + 80); h->n_qpairs = rd32(a + 84);
    h->tables_off = rd64(a + 88); h->qtab_off = rd64(a + 96); h->blocktab_off = rd64(a + 104); h->dir_off = rd64(a + 112);
    h->fnv_off = rd64(a + 120); h->payload_off = rd64(a + 128); h->archive_bytes = rd64(a + 136);
    h->total_lit = rd64(a + 144); h->total_match_bytes = rd64(a + 152); h->total_matches = rd64(a + 160);
    h->total_cmds = rd64(a + 168); h->total_litq = rd64(a + 176); h->src_window = rd64(a + 184);
    if (h->log2_bs < 3 || h->log2_bs > 20 || h->min_match < 1 || h->W < 4 || h->W > 8) return E_CORRUPT;
    if (h->prob_bits != 11 || h->n_tables != 4 + h->W) return E_CORRUPT;
    if (h->W < 8 && h->N > (1ull << (8 * h->W))) return E_CORRUPT;
    if (h->log2_seg < 3 || h->log2_seg > 14 || h->log2_seg > h->log2_bs) return E_CORRUPT;
    if (h->q_min == 1 || h->q_mode > 1 || (h->q_min == 0 && h->q_mode != 0)) return E_CORRUPT;
    if (h->q_mode == 1 ? (h->n_qpairs < 1 || h->n_qpairs > 4096) : h->n_qpairs != 0) return E_CORRUPT;
    if (h->max_cmds > 510) return E_CORRUPT;
    uint64_t BS = 1ull << h->log2_bs;
    if (h->n_blocks != (h->N + BS - 1) / BS) return E_CORRUPT;
    if (h->n_segs < h->n_blocks || h->n_segs >= (1ull << 32)) return E_CORRUPT;
    if (h->archive_bytes > n) return E_TRUNCATED;
    if (h->archive_bytes % 16 || h->archive_bytes < HEADER_BYTES + TAIL_PAD) return E_CORRUPT;
    /* sections in order, 16-byte aligned, non-overlapping */
    uint64_t at = HEADER_BYTES;
    if (h->tables_off < at || h->tables_off % 16) return E_CORRUPT;
    at = h->tables_off + 528ull * h->n_tables;
    if (h->qtab_off < at || h->qtab_off % 16) return E_CORRUPT;
    at = h->qtab_off + 4ull * h->n_qpairs;
    if (h->blocktab_off < at || h->blocktab_off % 16) return E_CORRUPT;
    at = h->blocktab_off + 8 * (h->n_blocks + 1);
    if (h->dir_off < at || h->dir_off % 16) return E_CORRUPT;
    at = h->dir_off + 32 * h->n_segs;
    if (h->flags & 1) { if (h->fnv_off < at || h->fnv_off % 8) return E_CORRUPT; at = h->fnv_off + 8 * h->n_blocks; }
    if (h->payload_off < at || h->payload_off % 16 || h->payload_off > h->archive_bytes - TAIL_PAD) return E_CORRUPT;
    if (h->total_lit + h->total_match_bytes != h->N || h->total_litq > h->total_lit) return E_CORRUPT;
    return OK;
}

/* A decode table: byte tables have 256 symbols and 2^11 slots; the Q pair table up to 4096 symbols and 2^12 slots.
 * value[s] = what symbol s stands for (the byte, or the pair v0 | v1 << 8). */
typedef struct {
    uint32_t mode, pb, n_sym;
    uint32_t freq[4096], cum[4097];
    uint16_t value[4096];
    uint16_t sym_of_slot[4096];
} table_t;

/* slot -> the symbol s with cum[s] <= slot < cum[s] + freq[s] (FORMAT.md §1.2, §1.3), written out as a table */
static void fill_slots(table_t* t) {
    for (uint32_t s = 0; s < t->n_sym; s++)
        for (uint32_t k = t->cum[s]; k < t->cum[s] + t->freq[s] && k < (1u << t->pb); k++) t->sym_of_slot[k] = (uint16_t)s;
}

/* FORMAT.md §1.2 and §1.3.  T has n_tables + 1 entries: T[n_tables] is the pair table (mode 2 = unused when q_mode = 0). */
static int parse_tables(const uint8_t* a, const hdr_t* h, table_t* T) {
    for (uint32_t t = 0; t < h->n_tables; t++) {
        const uint8_t* p = a + h->tables_off + 528ull * t;
        T[t].mode = rd32(p); T[t].pb = h->prob_bits; T[t].n_sym = 256;
        if (T[t].mode > 2) return E_CORRUPT;
        if (T[t].mode == 1 && !(t >= 2 && t < 2 + h->W)) return E_CORRUPT; /* raw is for OFF planes only */
        int litq_unused = (t == 3 + h->W) && (h->q_min == 0 || h->q_mode == 1);
        if ((T[t].mode == 2) != litq_unused) return E_CORRUPT;           /* unused: exactly the byte table of LITQ when it has no use */
        uint32_t sum = 0;
        T[t].cum[0] = 0;
        for (int s = 0; s < 256; s++) { T[t].freq[s] = rd16(p + 16 + 2 * s); T[t].value[s] = (uint16_t)s; sum += T[t].freq[s]; T[t].cum[s + 1] = sum; }
        if (T[t].mode == 0 && sum != (1u << h->prob_bits)) return E_CORRUPT;
        if (T[t].mode != 0 && sum != 0) return E_CORRUPT;
        if (T[t].mode == 0) fill_slots(&T[t]);
    }
    table_t* Q = &T[h->n_tables];
    Q->mode = 2; Q->pb = 12; Q->n_sym = h->n_qpairs;
    if (h->q_mode == 1) {
        Q->mode = 0;
        uint32_t sum = 0; Q->cum[0] = 0;
        for (uint32_t i = 0; i < h->n_qpairs; i++) {
            const uint8_t* p = a + h->qtab_off + 4ull * i;
            Q->value[i] = (uint16_t)rd16(p); Q->freq[i] = rd16(p + 2);
            if (Q->freq[i] < 1 || (i > 0 && Q->value[i] <= Q->value[i - 1])) return E_CORRUPT;
            sum += Q->freq[i]; Q->cum[i + 1] = sum;
        }
        if (sum != 4096) return E_CORRUPT;
        fill_slots(Q);
    }
    return OK;
}

typedef struct { uint64_t payload_off, out_start, out_end; uint32_t n_cmd, n_match, n_lit_a, n_lit_q, n_sym_q, n_words, n_ext, level; } seg_t;

/* FORMAT.md §1.4 */
static int read_block(const uint8_t* a, const hdr_t* h, uint64_t b, uint64_t* first_seg, uint64_t* end_seg, uint32_t* level) {
    const uint8_t* p = a + h->blocktab_off + 8 * b;
    *first_seg = rd32(p); *level = rd16(p + 4); *end_seg = rd32(p + 8);
    if (rd16(p + 6) != 0) return E_CORRUPT;
    if (b == 0 && *first_seg != 0) return E_CORRUPT;
    if (*end_seg <= *first_seg || *end_seg > h->n_segs) return E_CORRUPT;                 /* at least one segment per block */
    if (b + 1 == h->n_blocks && (*end_seg != h->n_segs || rd32(p + 12) != 0)) return E_CORRUPT;
    if (*level > h->max_level) return E_CORRUPT;
    return OK;
}

/* FORMAT.md §1.5: segment s of block b (segments [first_seg, end_seg)) */
static int read_seg(const uint8_t* a, const hdr_t* h, uint64_t s, uint64_t b, uint64_t first_seg, uint64_t end_seg, uint32_t level,
                    seg_t* d, uint64_t* payload_end) {
    const uint8_t* p = a + h->dir_off + 32 * s;
    uint64_t BS = 1ull << h->log2_bs, bstart = b * BS, bend = bstart + BS < h->N ? bstart + BS : h->N;
    d->payload_off = rd64(p); d->out_start = rd64(p + 8);
    d->n_cmd = rd16(p + 16); d->n_match = rd16(p + 18); d->n_lit_a = rd16(p + 20); d->n_lit_q = rd16(p + 22);
    d->n_sym_q = rd16(p + 24); d->n_words = rd16(p + 26); d->n_ext = rd16(p + 28); d->level = rd16(p + 30);
    *payload_end = (s + 1 < h->n_segs) ? rd64(p + 32) : h->archive_bytes - TAIL_PAD;
    if (d->payload_off % 16 || d->payload_off < h->payload_off || *payload_end <= d->payload_off || *payload_end > h->archive_bytes - TAIL_PAD) return E_CORRUPT;
    if (d->n_cmd < 1 || d->n_cmd > 510 || d->n_cmd > h->max_cmds || !(d->n_match == d->n_cmd || d->n_match + 1 == d->n_cmd)) return E_CORRUPT;
    if (d->level != level) return E_CORRUPT;
    if (d->n_lit_a + d->n_lit_q > 16384) return E_CORRUPT;
    if (h->q_min == 0 && (d->n_lit_q || d->n_sym_q)) return E_CORRUPT;
    if (h->q_mode == 0 && d->n_sym_q != d->n_lit_q) return E_CORRUPT;
    if (s == first_seg ? d->out_start != bstart : !(d->out_start > bstart && d->out_start < bend)) return E_CORRUPT;
    d->out_end = bend;
    if (s + 1 < end_seg) {
        d->out_end = rd64(p + 32 + 8);
        if (!(d->out_end > d->out_start && d->out_end < bend)) return E_CORRUPT;
    }
    return OK;
}

/* FORMAT.md §1.7: decode n_sym symbols; tid[i] = table of symbol i.  Scalar loop over symbols, 32 states; state k
 * renormalises from its own stream words[word_off[k] .. word_off[k+1]) (word_off has 33 entries).  used[k] = number of
 * words state k consumed.  sym[i] = the table's symbol index.  Returns OK, or E_TRUNCATED when a state would read past
 * the end of its stream. */
static int rans_decode(const table_t* T, const uint8_t* tid, uint64_t n_sym, uint32_t X[32],
                       const uint8_t* words, const uint64_t word_off[33], uint16_t* sym, uint64_t used[32]) {
    for (int k = 0; k < 32; k++) used[k] = 0;
    for (uint64_t i = 0; i < n_sym; i++) {
        int k = (int)(i & 31);
        const table_t* t = &T[tid[i]];
        uint32_t pb = t->pb;
        uint32_t x = X[k];
        uint32_t slot = x & ((1u << pb) - 1);
        uint32_t s = t->sym_of_slot[slot];
        x = t->freq[s] * (x >> pb) + slot - t->cum[s];
        if (x < (1u << 16)) {
            if (word_off[k] + used[k] >= word_off[k + 1]) return E_TRUNCATED;
            x = (x << 16) | rd16(words + 2 * (word_off[k] + used[k]));
            used[k]++;
        }
        X[k] = x;
        sym[i] = (uint16_t)s;
    }
    return OK;
}

typedef struct {
    uint8_t *cmd, *mlen, *lit_a;     /* tokens / LITA bytes                               */
    uint16_t* lit_q;                 /* LITQ symbols: bytes (byte mode) or pairs v0 | v1 << 8 */
    uint64_t* src;                   /* assembled absolute offsets                        */
    uint32_t *lit_len, *match_len;   /* decoded lengths per command (match_len 0 = none)  */
    uint16_t* sym; uint8_t* tid;
    uint64_t cap_cmd, cap_lit, cap_sym;
} scratch_t;

static int ensure(scratch_t* s, uint64_t n_cmd, uint64_t n_lit, uint64_t n_sym) {
    if (n_cmd > s->cap_cmd) {
        s->cap_cmd = n_cmd * 2 + 16;
        s->cmd = realloc(s->cmd, s->cap_cmd); s->mlen = realloc(s->mlen, s->cap_cmd);
        s->src = realloc(s->src, 8 * s->cap_cmd);
        s->lit_len = realloc(s->lit_len, 4 * s->cap_cmd); s->match_len = realloc(s->match_len, 4 * s->cap_cmd);
        if (!s->cmd || !s->mlen || !s->src || !s->lit_len || !s->match_len) return E_NOMEM;
    }
    if (n_lit > s->cap_lit) {
        s->cap_lit = n_lit * 2 + 16;
        s->lit_a = realloc(s->lit_a, s->cap_lit); s->lit_q = realloc(s->lit_q, 2 * s->cap_lit);
        if (!s->lit_a || !s->lit_q) return E_NOMEM;
    }
    if (n_sym > s->cap_sym) {
        s->cap_sym = n_sym * 2 + 16;
        s->sym = realloc(s->sym, 2 * s->cap_sym); s->tid = realloc(s->tid, s->cap_sym);
        if (!s->sym || !s->tid) return E_NOMEM;
    }
    return OK;
}
static void release(scratch_t* s) {
    free(s->cmd); free(s->mlen); free(s->lit_a); free(s->lit_q); free(s->src); free(s->lit_len); free(s->match_len); free(s->sym); free(s->tid);
    memset(s, 0, sizeof *s);
}

/* FORMAT.md §1.6-1.7: the logical streams of a segment, then the per-command lengths and sources. */
static int decode_streams(const uint8_t* a, const hdr_t* h, const table_t* T, const seg_t* d, uint64_t payload_end, scratch_t* s) {
    uint32_t W = h->W, n_coded = 0, n_raw = 0;
    for (uint32_t p = 0; p < W; p++) { if (T[2 + p].mode == 0) n_coded++; else n_raw++; }
    uint64_t n_sym = (uint64_t)d->n_cmd + (uint64_t)d->n_match * (1 + n_coded) + d->n_lit_a + d->n_sym_q;
    int rc = ensure(s, d->n_cmd, (uint64_t)d->n_lit_a + d->n_sym_q, n_sym);
    if (rc) return rc;
    /* payload geometry */
    uint64_t rans_bytes = 256 + 2ull * d->n_words;   /* head: 32 x (state, word_off) */
    uint64_t ext_off = d->payload_off + ((rans_bytes + 3) & ~3ull);
    uint64_t raw_off = ext_off + 4ull * d->n_ext;
    uint64_t need = raw_off + (uint64_t)n_raw * d->n_match;
    if (need > payload_end) return E_TRUNCATED;
    /* symbol order: CMD, MLEN, coded OFF planes from high to low, LITA, LITQ */
    uint32_t q_table = h->q_mode == 1 ? h->n_tables : 3 + W;
    uint64_t k = 0;
    for (uint32_t i = 0; i < d->n_cmd; i++) s->tid[k++] = 0;
    for (uint32_t i = 0; i < d->n_match; i++) s->tid[k++] = 1;
    for (int p = (int)W - 1; p >= 0; p--) if (T[2 + p].mode == 0) for (uint32_t i = 0; i < d->n_match; i++) s->tid[k++] = (uint8_t)(2 + p);
    for (uint32_t i = 0; i < d->n_lit_a; i++) s->tid[k++] = (uint8_t)(2 + W);
    for (uint32_t i = 0; i < d->n_sym_q; i++) s->tid[k++] = (uint8_t)q_table;
    uint32_t X[32]; uint64_t woff[33], used[32];
    for (int j = 0; j < 32; j++) { X[j] = rd32(a + d->payload_off + 8 * j); woff[j] = rd32(a + d->payload_off + 8 * j + 4); }
    woff[32] = d->n_words;
    if (woff[0] != 0) return E_CORRUPT;
    for (int j = 0; j < 32; j++) if (woff[j] > woff[j + 1]) return E_CORRUPT;
    for (int j = 0; j < 32; j++) if (X[j] < (1u << 16)) return E_CORRUPT;
    rc = rans_decode(T, s->tid, n_sym, X, a + d->payload_off + 256, woff, s->sym, used);
    if (rc) return rc;
    for (int j = 0; j < 32; j++) if (used[j] != woff[j + 1] - woff[j]) return E_CORRUPT; /* every stream fully consumed */
    for (int j = 0; j < 32; j++) if (X[j] != (1u << 16)) return E_CORRUPT; /* encoder started every state at 2^16 */
    /* split */
    k = 0;
    for (uint32_t i = 0; i < d->n_cmd; i++) s->cmd[i] = (uint8_t)s->sym[k + i];
    k += d->n_cmd;
    for (uint32_t i = 0; i < d->n_match; i++) s->mlen[i] = (uint8_t)s->sym[k + i];
    k += d->n_match;
    for (uint32_t i = 0; i < d->n_match; i++) s->src[i] = 0;
    for (int p = (int)W - 1; p >= 0; p--) if (T[2 + p].mode == 0) {
        for (uint32_t i = 0; i < d->n_match; i++) s->src[i] |= (uint64_t)s->sym[k + i] << (8 * p);
        k += d->n_match;
    }
    for (uint32_t i = 0; i < d->n_lit_a; i++) s->lit_a[i] = (uint8_t)s->sym[k + i];
    k += d->n_lit_a;
    for (uint32_t i = 0; i < d->n_sym_q; i++) s->lit_q[i] = T[q_table].value[s->sym[k + i]];   /* the byte, or the pair */
    uint64_t r = raw_off;
    for (uint32_t p = 0; p < W; p++) if (T[2 + p].mode == 1) {
        for (uint32_t i = 0; i < d->n_match; i++) s->src[i] |= (uint64_t)a[r + i] << (8 * p);
        r += d->n_match;
    }
    /* lengths: CMD escapes first in EXT, then MLEN escapes */
    uint64_t e = 0;
    for (uint32_t c = 0; c < d->n_cmd; c++) {
        uint32_t v = s->cmd[c];
        if (v == 255) { if (e >= d->n_ext) return E_CORRUPT; v = 255 + rd32(a + ext_off + 4 * e); e++; }
        s->lit_len[c] = v;
    }
    for (uint32_t c = 0; c < d->n_cmd; c++) {
        if (c >= d->n_match) { s->match_len[c] = 0; continue; }
        uint32_t v = s->mlen[c];
        if (v == 255) { if (e >= d->n_ext) return E_CORRUPT; v = 255 + rd32(a + ext_off + 4 * e); e++; }
        s->match_len[c] = h->min_match + v;
    }
    if (e != d->n_ext) return E_CORRUPT;
    return OK;
}

static int getbit(const uint8_t* m, uint64_t i) { return (m[i >> 3] >> (i & 7)) & 1; }
static void setbit(uint8_t* m, uint64_t i) { m[i >> 3] |= (uint8_t)(1u << (i & 7)); }

/* FORMAT.md §2 (literal classes, byte-serial copy) and §3 (level invariant) for one segment of block b.
 * `matchmap` bit = 1: match byte. */
static int decode_segment(const hdr_t* h, const seg_t* d, const scratch_t* s, uint64_t b, uint8_t* out,
                          uint8_t* matchmap, const uint16_t* levels) {
    uint64_t dst = d->out_start, end = d->out_end, la = 0, lq = 0;   /* lq: next LITQ symbol */
    uint64_t seg_limit = d->out_start + (1ull << h->log2_seg);
    for (uint32_t c = 0; c < d->n_cmd; c++) {
        uint32_t ll = s->lit_len[c], ml = s->match_len[c];
        if (dst >= seg_limit) return E_CORRUPT;                      /* §1.5: a command starts below SEG bytes of its segment */
        if (dst + ll > end) return E_CORRUPT;
        if (h->q_min > 0 && ll >= h->q_min) {                        /* a LITQ run */
            if (h->q_mode == 0) {
                if (lq + ll > d->n_sym_q) return E_CORRUPT;
                for (uint32_t i = 0; i < ll; i++) out[dst + i] = (uint8_t)s->lit_q[lq + i];
                lq += ll;
            } else {                                                 /* pairs k = floor(dst/2) .. floor((dst+ll-1)/2), §1.7 */
                uint64_t k0 = dst >> 1, k1 = (dst + ll - 1) >> 1;
                if (lq + (k1 - k0 + 1) > d->n_sym_q) return E_CORRUPT;
                for (uint64_t k = k0; k <= k1; k++, lq++) {
                    uint16_t pr = s->lit_q[lq];
                    if (2 * k >= dst) out[2 * k] = (uint8_t)(pr & 0xff);                 /* fillers outside the run are dropped */
                    if (2 * k + 1 < dst + ll) out[2 * k + 1] = (uint8_t)(pr >> 8);
                }
            }
        } else {
            if (la + ll > d->n_lit_a) return E_CORRUPT;
            for (uint32_t i = 0; i < ll; i++) out[dst + i] = s->lit_a[la + i];
            la += ll;
        }
        dst += ll;
        if (c < d->n_match) {
            uint64_t src = s->src[c];
            if (!(src < dst) || dst + ml > end) return E_CORRUPT;
            if (src + ml > dst && dst - src > ll) return E_CORRUPT;   /* FORMAT.md §3 (c): the seed of a self-overlapping match is the tail of its own literal run */
            if (matchmap) {
                uint64_t seed_end = src + ml < dst ? src + ml : dst;
                for (uint64_t q = src; q < seed_end; q++) {
                    uint64_t S = q >> h->log2_bs;
                    if (getbit(matchmap, q)) { if (S == b || !(levels[S] < d->level)) return E_LEVEL; }  /* §3 (b) */
                    else if (S != b && !(levels[S] <= d->level)) return E_LEVEL;                          /* §3 (a) */
                }
            }
            for (uint32_t i = 0; i < ml; i++) out[dst + i] = out[src + i]; /* ascending, one byte at a time */
            if (matchmap) for (uint32_t i = 0; i < ml; i++) setbit(matchmap, dst + i);
            dst += ml;
        }
    }
    if (dst != end || la != d->n_lit_a || lq != d->n_sym_q) return E_CORRUPT;
    return OK;
}

/* ------------------------------------------------------------------------------------------------ exports ---- */

#define N_HEADER_FIELDS 28
/* fields: N, n_blocks, n_segs, log2_bs, min_match, W, prob_bits, n_tables, max_level, max_cmds, flags, log2_seg, q_min,
 * q_mode, n_qpairs, tables_off, qtab_off, blocktab_off, dir_off, fnv_off, payload_off, archive_bytes, total_lit,
 * total_match_bytes, total_matches, total_cmds, total_litq, src_window */
int acx_oracle_header(const uint8_t* a, uint64_t n, uint64_t* f) {
    hdr_t h;
    int rc = parse_header(a, n, &h);
    if (rc) return rc;
    uint64_t v[N_HEADER_FIELDS] = {h.N, h.n_blocks, h.n_segs, h.log2_bs, h.min_match, h.W, h.prob_bits, h.n_tables, h.max_level,
                      h.max_cmds, h.flags, h.log2_seg, h.q_min, h.q_mode, h.n_qpairs, h.tables_off, h.qtab_off, h.blocktab_off,
                      h.dir_off, h.fnv_off, h.payload_off, h.archive_bytes, h.total_lit, h.total_match_bytes,
                      h.total_matches, h.total_cmds, h.total_litq, h.src_window};
    memcpy(f, v, sizeof v);
    return OK;
}

/* Decode of blocks [0, n_prefix_blocks) in index order (n_prefix_blocks = 0 or >= n_blocks: the whole archive; a
 * prefix is self-sufficient because every source precedes its destination).  check_levels != 0 also verifies
 * FORMAT.md §3 and the optional FNV section.  out must hold min(N, n_prefix_blocks * BS) bytes. */
int acx_oracle_decode_prefix(const uint8_t* a, uint64_t n, uint8_t* out, uint64_t out_cap, int check_levels, uint64_t n_prefix_blocks) {
    hdr_t h; scratch_t s; seg_t d;
    memset(&s, 0, sizeof s);
    int rc = parse_header(a, n, &h);
    if (rc) return rc;
    uint64_t nb = (n_prefix_blocks == 0 || n_prefix_blocks > h.n_blocks) ? h.n_blocks : n_prefix_blocks;
    uint64_t need_out = (nb << h.log2_bs) < h.N ? (nb << h.log2_bs) : h.N;
    if (out_cap < need_out) return E_RANGE;
    table_t* T = calloc(MAX_TABLES + 1, sizeof(table_t));
    if (!T) return E_NOMEM;
    if ((rc = parse_tables(a, &h, T))) { free(T); return rc; }
    uint8_t* matchmap = NULL; uint16_t* levels = NULL;
    if (check_levels) {
        matchmap = calloc(h.N / 8 + 1, 1); levels = calloc(h.n_blocks + 1, 2);
        if (!matchmap || !levels) { free(matchmap); free(levels); free(T); return E_NOMEM; }
    }
    uint64_t sums[5] = {0, 0, 0, 0, 0}; uint32_t max_level = 0, max_cmds = 0;
    uint64_t prev_end_seg = 0;
    for (uint64_t b = 0; b < nb && !rc; b++) {
        uint64_t s0, s1; uint32_t level;
        if ((rc = read_block(a, &h, b, &s0, &s1, &level))) break;
        if (s0 != prev_end_seg) { rc = E_CORRUPT; break; }
        prev_end_seg = s1;
        if (levels) levels[b] = (uint16_t)level;
        if (level > max_level) max_level = level;
        for (uint64_t sg = s0; sg < s1 && !rc; sg++) {
            uint64_t pend;
            if ((rc = read_seg(a, &h, sg, b, s0, s1, level, &d, &pend))) break;
            if ((rc = decode_streams(a, &h, T, &d, pend, &s))) break;
            if ((rc = decode_segment(&h, &d, &s, b, out, matchmap, levels))) break;
            sums[0] += d.n_lit_a + d.n_lit_q; sums[1] += d.n_match; sums[2] += d.n_cmd; sums[4] += d.n_lit_q;
            for (uint32_t c = 0; c < d.n_cmd; c++) sums[3] += s.match_len[c];
            if (d.n_cmd > max_cmds) max_cmds = d.n_cmd;
        }
        if (!rc && check_levels && (h.flags & 1)) {
            uint64_t BS = 1ull << h.log2_bs, lo = b * BS, hi = lo + BS < h.N ? lo + BS : h.N, f = 0xcbf29ce484222325ull;
            for (uint64_t q = lo; q < hi; q++) { f ^= out[q]; f *= 0x100000001b3ull; }
            if (f != rd64(a + h.fnv_off + 8 * b)) rc = E_CORRUPT;
        }
    }
    if (!rc && nb == h.n_blocks && (sums[0] != h.total_lit || sums[1] != h.total_matches || sums[2] != h.total_cmds || sums[3] != h.total_match_bytes ||
                sums[4] != h.total_litq || max_level != h.max_level || max_cmds != h.max_cmds || prev_end_seg != h.n_segs)) rc = E_CORRUPT;
    if (!rc && nb == h.n_blocks) for (uint64_t q = h.archive_bytes - TAIL_PAD; q < h.archive_bytes; q++) if (a[q]) rc = E_CORRUPT;   /* §1: tail pad */
    free(matchmap); free(levels); release(&s); free(T);
    return rc;
}

int acx_oracle_decode(const uint8_t* a, uint64_t n, uint8_t* out, uint64_t out_cap, int check_levels) {
    return acx_oracle_decode_prefix(a, n, out, out_cap, check_levels, 0);
}

/* Block b: first segment, one-past-last segment, level. */
int acx_oracle_block_segs(const uint8_t* a, uint64_t n, uint64_t b, uint64_t* out3) {
    hdr_t h; uint32_t level;
    int rc = parse_header(a, n, &h);
    if (rc) return rc;
    if (b >= h.n_blocks) return E_RANGE;
    if ((rc = read_block(a, &h, b, &out3[0], &out3[1], &level))) return rc;
    out3[2] = level;
    return OK;
}

/* Stage-level view of segment sg for parity debugging: tokens, literal bytes, sources, and per-command
 * lit_len / match_len / lit_pos (position of the run in ITS literal stream: byte index in LITA, symbol index in LITQ) /
 * out_pos (absolute position of the command's first byte).  lit = the segment's literal bytes in command order (both
 * classes interleaved as they appear in the output).  Arrays must hold n_cmd (n_lit_a + n_lit_q for lit) entries;
 * counts = {n_cmd, n_match, n_lit_a, n_lit_q, n_sym_q, n_words, n_ext, level, block, out_start, out_end}. */
int acx_oracle_segment(const uint8_t* a, uint64_t n, uint64_t sg, uint64_t* counts, uint8_t* cmd, uint8_t* mlen, uint8_t* lit,
                       uint64_t* src, uint32_t* lit_len, uint32_t* match_len, uint32_t* lit_pos, uint64_t* out_pos) {
    hdr_t h; scratch_t s; seg_t d; uint64_t pend;
    memset(&s, 0, sizeof s);
    int rc = parse_header(a, n, &h);
    if (rc) return rc;
    if (sg >= h.n_segs) return E_RANGE;
    uint64_t b = rd64(a + h.dir_off + 32 * sg + 8) >> h.log2_bs, s0, s1; uint32_t level;
    if (b >= h.n_blocks) return E_CORRUPT;
    if ((rc = read_block(a, &h, b, &s0, &s1, &level))) return rc;
    if (sg < s0 || sg >= s1) return E_CORRUPT;
    if ((rc = read_seg(a, &h, sg, b, s0, s1, level, &d, &pend))) return rc;
    uint64_t cv[11] = {d.n_cmd, d.n_match, d.n_lit_a, d.n_lit_q, d.n_sym_q, d.n_words, d.n_ext, d.level, b, d.out_start, d.out_end};
    memcpy(counts, cv, sizeof cv);
    if (!cmd) return OK;
    table_t* T = calloc(MAX_TABLES + 1, sizeof(table_t));
    if (!T) return E_NOMEM;
    if ((rc = parse_tables(a, &h, T)) || (rc = decode_streams(a, &h, T, &d, pend, &s))) { release(&s); free(T); return rc; }
    memcpy(cmd, s.cmd, d.n_cmd); memcpy(mlen, s.mlen, d.n_match);
    uint64_t op = d.out_start, la = 0, lq = 0, lo = 0;
    for (uint32_t c = 0; c < d.n_cmd; c++) {
        uint32_t ll = s.lit_len[c];
        if (c < d.n_match) src[c] = s.src[c];
        lit_len[c] = ll; match_len[c] = s.match_len[c]; out_pos[c] = op;
        if (h.q_min > 0 && ll >= h.q_min) {
            lit_pos[c] = (uint32_t)lq;
            if (h.q_mode == 0) { for (uint32_t i = 0; i < ll; i++) lit[lo + i] = (uint8_t)s.lit_q[lq + i]; lq += ll; }
            else for (uint64_t k = op >> 1; k <= (op + ll - 1) >> 1; k++, lq++) {
                if (2 * k >= op) lit[lo + (2 * k - op)] = (uint8_t)(s.lit_q[lq] & 0xff);
                if (2 * k + 1 < op + ll) lit[lo + (2 * k + 1 - op)] = (uint8_t)(s.lit_q[lq] >> 8);
            }
        } else { lit_pos[c] = (uint32_t)la; memcpy(lit + lo, s.lit_a + la, ll); la += ll; }
        lo += ll; op += (uint64_t)ll + s.match_len[c];
    }
    release(&s); free(T);
    return OK;
}

/* The rANS step alone (FORMAT.md §1.7), for the rANS pins.  freq: n_tables rows of n_sym_per_table u16 (each row sums to
 * 2^prob_bits[t]; at most 4096 symbols).  states: 32 initial states in, final states out.  word_off: 33 entries (u64);
 * words_used: 32 entries out.  sym: u16 symbol indices out. */
int acx_oracle_rans(const uint16_t* freq, uint32_t n_tables, uint32_t n_sym_per_table, const uint32_t* prob_bits, const uint8_t* tid,
                    uint64_t n_sym, uint32_t* states, const uint8_t* words, const uint64_t* word_off, uint16_t* sym, uint64_t* words_used) {
    if (n_tables > MAX_TABLES + 1 || n_sym_per_table > 4096) return E_RANGE;
    table_t* T = calloc(n_tables, sizeof(table_t));
    if (!T) return E_NOMEM;
    for (uint32_t t = 0; t < n_tables; t++) {
        uint32_t sum = 0; T[t].mode = 0; T[t].cum[0] = 0; T[t].pb = prob_bits[t]; T[t].n_sym = n_sym_per_table;
        for (uint32_t s = 0; s < n_sym_per_table; s++) { T[t].freq[s] = freq[(uint64_t)n_sym_per_table * t + s]; sum += T[t].freq[s]; T[t].cum[s + 1] = sum; }
        if (prob_bits[t] > 12 || sum != (1u << prob_bits[t])) { free(T); return E_CORRUPT; }
        fill_slots(&T[t]);
    }
    for (int k = 0; k < 32; k++) if (word_off[k] > word_off[k + 1]) { free(T); return E_CORRUPT; }
    int rc = rans_decode(T, tid, n_sym, states, words, word_off, sym, words_used);
    free(T);
    return rc;
}

/* FNV-1a 64 (FORMAT.md §5; "FNV for device-resident GPU paths"). */
uint64_t acx_oracle_fnv1a64(const uint8_t* p, uint64_t n) {
    uint64_t f = 0xcbf29ce484222325ull;
    for (uint64_t i = 0; i < n; i++) { f ^= p[i]; f *= 0x100000001b3ull; }
    return f;
}
