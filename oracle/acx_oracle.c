/* ORACLE — test infrastructure, not product code.
 *
 * A plain, slow, single-threaded CPU decoder of the ACX-B200 archive format (FORMAT.md), written from FORMAT.md and
 * the paper's description of the method (§2: absolute-offset LZ77, fixed-size blocks, four streams
 * per block: literals, match lengths, absolute offsets, command sequence; §5: 64-bit sizes/offsets).
 * It shares no code, header, table generator or helper with the CUDA path (paper_2606_18900_b200/csrc) or with the
 * encoder.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may use it.
 *
 * The method reaches exactly the original bytes, so the final pin is decode(encode(x)) == x against the ORIGINAL
 * bytes (tests/test_oracle_*.py); the byte-serial copy loop below is the definition of LZ77 copy semantics
 * (FORMAT.md §2) and the rANS step is FORMAT.md §1.5 written out symbol by symbol.  Blocks are decoded in index
 * order, which is always valid because every source precedes its destination.
 *
 * Parity status: every function here is pinned (hand-built archives with hand-written expected bytes, an
 * independent pure-Python rANS encoder and byte-serial reference in the tests, closed-form compressed size,
 * final-state invariant, round trips against the original bytes).  Nothing is "parity unpinned".
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

enum { OK = 0, E_MAGIC = -1, E_VERSION = -2, E_TRUNCATED = -3, E_CORRUPT = -4, E_RANGE = -5, E_LEVEL = -6, E_NOMEM = -7 };

static uint64_t rd64(const uint8_t* p) { uint64_t v = 0; for (int i = 7; i >= 0; i--) v = (v << 8) | p[i]; return v; }
static uint32_t rd32(const uint8_t* p) { return (uint32_t)p[0] | ((uint32_t)p[1] << 8) | ((uint32_t)p[2] << 16) | ((uint32_t)p[3] << 24); }
static uint32_t rd16(const uint8_t* p) { return (uint32_t)p[0] | ((uint32_t)p[1] << 8); }

typedef struct {
    uint64_t N, n_blocks, tables_off, dir_off, fnv_off, payload_off, archive_bytes;
    uint64_t total_lit, total_match_bytes, total_matches, total_cmds, src_window;
    uint32_t log2_bs, min_match, W, prob_bits, n_tables, max_level, max_cmds, flags;
} hdr_t;

/* FORMAT.md §1.1 */
static int parse_header(const uint8_t* a, uint64_t n, hdr_t* h) {
    static const uint8_t magic[8] = {0x41, 0x43, 0x58, 0x42, 0x32, 0x30, 0x30, 0x00};
    if (n < 160) return E_TRUNCATED;
    if (memcmp(a, magic, 8)) return E_MAGIC;
    if (rd32(a + 8) != 2) return E_VERSION;
    if (rd32(a + 12) != 160) return E_CORRUPT;
    h->N = rd64(a + 16); h->n_blocks = rd64(a + 24);
    h->log2_bs = rd32(a + 32); h->min_match = rd32(a + 36); h->W = rd32(a + 40); h->prob_bits = rd32(a + 44);
    h->n_tables = rd32(a + 48); h->max_level = rd32(a + 52); h->max_cmds = rd32(a + 56); h->flags = rd32(a + 60);
    h->tables_off = rd64(a + 64); h->dir_off = rd64(a + 72); h->fnv_off = rd64(a + 80); h->payload_off = rd64(a + 88);
    h->archive_bytes = rd64(a + 96); h->total_lit = rd64(a + 104); h->total_match_bytes = rd64(a + 112);
    h->total_matches = rd64(a + 120); h->total_cmds = rd64(a + 128); h->src_window = rd64(a + 136);
    if (h->log2_bs < 3 || h->log2_bs > 20 || h->min_match < 1 || h->W < 4 || h->W > 8) return E_CORRUPT;
    if (h->prob_bits != 11 || h->n_tables != 3 + h->W) return E_CORRUPT;
    if (h->W < 8 && h->N > (1ull << (8 * h->W))) return E_CORRUPT;
    uint64_t BS = 1ull << h->log2_bs;
    if (h->n_blocks != (h->N + BS - 1) / BS) return E_CORRUPT;
    if (h->archive_bytes > n) return E_TRUNCATED;
    if (h->archive_bytes % 16) return E_CORRUPT;
    if (h->tables_off < 160 || h->tables_off % 16 || h->dir_off < h->tables_off + 528ull * h->n_tables || h->dir_off % 16) return E_CORRUPT;
    uint64_t dir_end = h->dir_off + 32 * h->n_blocks;
    if (h->flags & 1) { if (h->fnv_off < dir_end || h->fnv_off % 8) return E_CORRUPT; dir_end = h->fnv_off + 8 * h->n_blocks; }
    if (h->payload_off < dir_end || h->payload_off % 16 || h->payload_off > h->archive_bytes) return E_CORRUPT;
    if (h->total_lit + h->total_match_bytes != h->N) return E_CORRUPT;
    return OK;
}

typedef struct { uint32_t mode; uint32_t freq[256]; uint32_t cum[257]; uint8_t sym_of_slot[2048]; } table_t;

/* slot -> the symbol s with cum[s] <= slot < cum[s] + freq[s] (FORMAT.md §1.2), written out as a table */
static void fill_slots(table_t* t) {
    for (int s = 0; s < 256; s++) for (uint32_t k = t->cum[s]; k < t->cum[s] + t->freq[s] && k < 2048; k++) t->sym_of_slot[k] = (uint8_t)s;
}

/* FORMAT.md §1.2 */
static int parse_tables(const uint8_t* a, const hdr_t* h, table_t* T) {
    uint32_t M = 1u << h->prob_bits;
    for (uint32_t t = 0; t < h->n_tables; t++) {
        const uint8_t* p = a + h->tables_off + 528ull * t;
        T[t].mode = rd32(p);
        if (T[t].mode > 1) return E_CORRUPT;
        if (T[t].mode == 1 && !(t >= 2 && t < 2 + h->W)) return E_CORRUPT; /* raw is for OFF planes only */
        uint32_t sum = 0;
        T[t].cum[0] = 0;
        for (int s = 0; s < 256; s++) { T[t].freq[s] = rd16(p + 16 + 2 * s); sum += T[t].freq[s]; T[t].cum[s + 1] = sum; }
        if (T[t].mode == 0 && sum != M) return E_CORRUPT;
        if (T[t].mode == 0) fill_slots(&T[t]);
    }
    return OK;
}

typedef struct { uint64_t payload_off; uint32_t n_cmd, n_match, n_lit, n_words, n_ext; uint32_t level; } dir_t;

static int read_dir(const uint8_t* a, const hdr_t* h, uint64_t b, dir_t* d, uint64_t* payload_end) {
    const uint8_t* p = a + h->dir_off + 32 * b;
    d->payload_off = rd64(p); d->n_cmd = rd32(p + 8); d->n_match = rd32(p + 12); d->n_lit = rd32(p + 16);
    d->n_words = rd32(p + 20); d->n_ext = rd32(p + 24); d->level = rd16(p + 28);
    *payload_end = (b + 1 < h->n_blocks) ? rd64(p + 32) : h->archive_bytes;
    if (d->payload_off % 16 || d->payload_off < h->payload_off || *payload_end <= d->payload_off || *payload_end > h->archive_bytes) return E_CORRUPT;
    if (d->n_cmd < 1 || !(d->n_match == d->n_cmd || d->n_match + 1 == d->n_cmd)) return E_CORRUPT;
    if (d->level > h->max_level) return E_CORRUPT;
    return OK;
}

/* FORMAT.md §1.5: decode n_sym symbols; tid[i] = table of symbol i.  Scalar loop over symbols, 32 states; state k
 * renormalises from its own stream words[word_off[k] .. word_off[k+1]) (word_off has 33 entries).  used[k] = number of
 * words state k consumed.  Returns OK, or E_TRUNCATED when a state would read past the end of its stream. */
static int rans_decode(const table_t* T, const uint8_t* tid, uint64_t n_sym, uint32_t prob_bits, uint32_t X[32],
                       const uint8_t* words, const uint64_t word_off[33], uint8_t* sym, uint64_t used[32]) {
    uint32_t M = 1u << prob_bits;
    for (int k = 0; k < 32; k++) used[k] = 0;
    for (uint64_t i = 0; i < n_sym; i++) {
        int k = (int)(i & 31);
        const table_t* t = &T[tid[i]];
        uint32_t x = X[k];
        uint32_t slot = x & (M - 1);
        int s = t->sym_of_slot[slot];
        x = t->freq[s] * (x >> prob_bits) + slot - t->cum[s];
        if (x < (1u << 16)) {
            if (word_off[k] + used[k] >= word_off[k + 1]) return E_TRUNCATED;
            x = (x << 16) | rd16(words + 2 * (word_off[k] + used[k]));
            used[k]++;
        }
        X[k] = x;
        sym[i] = (uint8_t)s;
    }
    return OK;
}

typedef struct {
    uint8_t *cmd, *mlen, *lit;   /* tokens / literal bytes                        */
    uint64_t* src;               /* assembled absolute offsets                    */
    uint32_t *lit_len, *match_len; /* decoded lengths per command (match_len 0 = none) */
    uint8_t *sym, *tid;
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
    if (n_lit > s->cap_lit) { s->cap_lit = n_lit * 2 + 16; s->lit = realloc(s->lit, s->cap_lit); if (!s->lit) return E_NOMEM; }
    if (n_sym > s->cap_sym) {
        s->cap_sym = n_sym * 2 + 16;
        s->sym = realloc(s->sym, s->cap_sym); s->tid = realloc(s->tid, s->cap_sym);
        if (!s->sym || !s->tid) return E_NOMEM;
    }
    return OK;
}
static void release(scratch_t* s) {
    free(s->cmd); free(s->mlen); free(s->lit); free(s->src); free(s->lit_len); free(s->match_len); free(s->sym); free(s->tid);
    memset(s, 0, sizeof *s);
}

/* FORMAT.md §1.4-1.5: the four logical streams of block b, then the per-command lengths and sources. */
static int decode_streams(const uint8_t* a, const hdr_t* h, const table_t* T, const dir_t* d, uint64_t payload_end, scratch_t* s) {
    uint32_t W = h->W, n_coded = 0, n_raw = 0;
    for (uint32_t p = 0; p < W; p++) { if (T[2 + p].mode == 0) n_coded++; else n_raw++; }
    uint64_t n_sym = (uint64_t)d->n_cmd + (uint64_t)d->n_match * (1 + n_coded) + d->n_lit;
    int rc = ensure(s, d->n_cmd, d->n_lit, n_sym);
    if (rc) return rc;
    /* payload geometry */
    uint64_t rans_bytes = 256 + 2ull * d->n_words;   /* head: 32 x (state, word_off) */
    uint64_t ext_off = d->payload_off + ((rans_bytes + 3) & ~3ull);
    uint64_t raw_off = ext_off + 4ull * d->n_ext;
    uint64_t need = raw_off + (uint64_t)n_raw * d->n_match;
    if (need > payload_end) return E_TRUNCATED;
    /* symbol order: CMD, MLEN, coded OFF planes from high to low, LIT */
    uint64_t k = 0;
    for (uint32_t i = 0; i < d->n_cmd; i++) s->tid[k++] = 0;
    for (uint32_t i = 0; i < d->n_match; i++) s->tid[k++] = 1;
    for (int p = (int)W - 1; p >= 0; p--) if (T[2 + p].mode == 0) for (uint32_t i = 0; i < d->n_match; i++) s->tid[k++] = (uint8_t)(2 + p);
    for (uint32_t i = 0; i < d->n_lit; i++) s->tid[k++] = (uint8_t)(2 + W);
    uint32_t X[32]; uint64_t woff[33], used[32];
    for (int j = 0; j < 32; j++) { X[j] = rd32(a + d->payload_off + 8 * j); woff[j] = rd32(a + d->payload_off + 8 * j + 4); }
    woff[32] = d->n_words;
    if (woff[0] != 0) return E_CORRUPT;
    for (int j = 0; j < 32; j++) if (woff[j] > woff[j + 1]) return E_CORRUPT;
    for (int j = 0; j < 32; j++) if (X[j] < (1u << 16)) return E_CORRUPT;
    rc = rans_decode(T, s->tid, n_sym, h->prob_bits, X, a + d->payload_off + 256, woff, s->sym, used);
    if (rc) return rc;
    for (int j = 0; j < 32; j++) if (used[j] != woff[j + 1] - woff[j]) return E_CORRUPT; /* every stream fully consumed */
    for (int j = 0; j < 32; j++) if (X[j] != (1u << 16)) return E_CORRUPT; /* encoder started every state at 2^16 */
    /* split */
    k = 0;
    memcpy(s->cmd, s->sym + k, d->n_cmd); k += d->n_cmd;
    memcpy(s->mlen, s->sym + k, d->n_match); k += d->n_match;
    for (uint32_t i = 0; i < d->n_match; i++) s->src[i] = 0;
    for (int p = (int)W - 1; p >= 0; p--) if (T[2 + p].mode == 0) {
        for (uint32_t i = 0; i < d->n_match; i++) s->src[i] |= (uint64_t)s->sym[k + i] << (8 * p);
        k += d->n_match;
    }
    memcpy(s->lit, s->sym + k, d->n_lit);
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

/* FORMAT.md §2 (byte-serial copy) and §3 (level invariant) for one block.  `matchmap` bit = 1: match byte. */
static int decode_block(const hdr_t* h, const dir_t* d, const scratch_t* s, uint64_t b, uint8_t* out,
                        uint8_t* matchmap, const uint16_t* levels) {
    uint64_t BS = 1ull << h->log2_bs;
    uint64_t dst = b * BS, end = dst + BS < h->N ? dst + BS : h->N, lp = 0;
    for (uint32_t c = 0; c < d->n_cmd; c++) {
        uint32_t ll = s->lit_len[c], ml = s->match_len[c];
        if (lp + ll > d->n_lit || dst + ll > end) return E_CORRUPT;
        for (uint32_t i = 0; i < ll; i++) out[dst + i] = s->lit[lp + i];
        lp += ll; dst += ll;
        if (c < d->n_match) {
            uint64_t src = s->src[c];
            if (!(src < dst) || dst + ml > end) return E_CORRUPT;
            if (src + ml > dst && src < b * BS) return E_CORRUPT;   /* FORMAT.md §3 (c): a self-overlapping match starts in its own block */
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
    if (dst != end || lp != d->n_lit) return E_CORRUPT;
    return OK;
}

/* ------------------------------------------------------------------------------------------------ exports ---- */

/* fields[0..19]: N, n_blocks, log2_bs, min_match, W, prob_bits, n_tables, max_level, max_cmds, flags, tables_off,
 * dir_off, fnv_off, payload_off, archive_bytes, total_lit, total_match_bytes, total_matches, total_cmds, src_window */
int acx_oracle_header(const uint8_t* a, uint64_t n, uint64_t* f) {
    hdr_t h;
    int rc = parse_header(a, n, &h);
    if (rc) return rc;
    uint64_t v[20] = {h.N, h.n_blocks, h.log2_bs, h.min_match, h.W, h.prob_bits, h.n_tables, h.max_level, h.max_cmds,
                      h.flags, h.tables_off, h.dir_off, h.fnv_off, h.payload_off, h.archive_bytes, h.total_lit,
                      h.total_match_bytes, h.total_matches, h.total_cmds, h.src_window};
    memcpy(f, v, sizeof v);
    return OK;
}

/* Decode of blocks [0, n_prefix_blocks) in index order (n_prefix_blocks = 0 or >= n_blocks: the whole archive; a
 * prefix is self-sufficient because every source precedes its destination).  check_levels != 0 also verifies
 * FORMAT.md §3 and the optional FNV section.  out must hold min(N, n_prefix_blocks * BS) bytes. */
int acx_oracle_decode_prefix(const uint8_t* a, uint64_t n, uint8_t* out, uint64_t out_cap, int check_levels, uint64_t n_prefix_blocks);

int acx_oracle_decode(const uint8_t* a, uint64_t n, uint8_t* out, uint64_t out_cap, int check_levels) {
    return acx_oracle_decode_prefix(a, n, out, out_cap, check_levels, 0);
}

int acx_oracle_decode_prefix(const uint8_t* a, uint64_t n, uint8_t* out, uint64_t out_cap, int check_levels, uint64_t n_prefix_blocks) {
    hdr_t h; table_t T[11]; scratch_t s; dir_t d;
    memset(&s, 0, sizeof s);
    int rc = parse_header(a, n, &h);
    if (rc) return rc;
    uint64_t nb = (n_prefix_blocks == 0 || n_prefix_blocks > h.n_blocks) ? h.n_blocks : n_prefix_blocks;
    uint64_t need_out = (nb << h.log2_bs) < h.N ? (nb << h.log2_bs) : h.N;
    if (out_cap < need_out) return E_RANGE;
    if ((rc = parse_tables(a, &h, T))) return rc;
    uint8_t* matchmap = NULL; uint16_t* levels = NULL;
    if (check_levels) {
        matchmap = calloc(h.N / 8 + 1, 1); levels = calloc(h.n_blocks + 1, 2);
        if (!matchmap || !levels) { free(matchmap); free(levels); return E_NOMEM; }
    }
    uint64_t sums[4] = {0, 0, 0, 0}; uint32_t max_level = 0, max_cmds = 0;
    for (uint64_t b = 0; b < nb && !rc; b++) {
        uint64_t pend;
        if ((rc = read_dir(a, &h, b, &d, &pend))) break;
        if ((rc = decode_streams(a, &h, T, &d, pend, &s))) break;
        if (levels) levels[b] = (uint16_t)d.level;
        if ((rc = decode_block(&h, &d, &s, b, out, matchmap, levels))) break;
        sums[0] += d.n_lit; sums[1] += d.n_match; sums[2] += d.n_cmd;
        for (uint32_t c = 0; c < d.n_cmd; c++) sums[3] += s.match_len[c];
        if (d.level > max_level) max_level = d.level;
        if (d.n_cmd > max_cmds) max_cmds = d.n_cmd;
        if (check_levels && (h.flags & 1)) {
            uint64_t BS = 1ull << h.log2_bs, lo = b * BS, hi = lo + BS < h.N ? lo + BS : h.N, f = 0xcbf29ce484222325ull;
            for (uint64_t q = lo; q < hi; q++) { f ^= out[q]; f *= 0x100000001b3ull; }
            if (f != rd64(a + h.fnv_off + 8 * b)) rc = E_CORRUPT;
        }
    }
    if (!rc && nb == h.n_blocks && (sums[0] != h.total_lit || sums[1] != h.total_matches || sums[2] != h.total_cmds || sums[3] != h.total_match_bytes ||
                max_level != h.max_level || max_cmds != h.max_cmds)) rc = E_CORRUPT;
    free(matchmap); free(levels); release(&s);
    return rc;
}

/* Stage-level view of block b for parity debugging: tokens, literal bytes, sources, and per-command
 * lit_len / match_len / lit_pos (exclusive prefix of lit_len) / out_pos (absolute position of the command's first byte).
 * Arrays must hold n_cmd (n_lit for lit) entries; counts = {n_cmd, n_match, n_lit, n_words, n_ext, level}. */
int acx_oracle_block(const uint8_t* a, uint64_t n, uint64_t b, uint32_t* counts, uint8_t* cmd, uint8_t* mlen, uint8_t* lit,
                     uint64_t* src, uint32_t* lit_len, uint32_t* match_len, uint32_t* lit_pos, uint64_t* out_pos) {
    hdr_t h; table_t T[11]; scratch_t s; dir_t d; uint64_t pend;
    memset(&s, 0, sizeof s);
    int rc = parse_header(a, n, &h);
    if (rc) return rc;
    if (b >= h.n_blocks) return E_RANGE;
    if ((rc = parse_tables(a, &h, T))) return rc;
    if ((rc = read_dir(a, &h, b, &d, &pend))) return rc;
    counts[0] = d.n_cmd; counts[1] = d.n_match; counts[2] = d.n_lit; counts[3] = d.n_words; counts[4] = d.n_ext; counts[5] = d.level;
    if (!cmd) return OK;
    if ((rc = decode_streams(a, &h, T, &d, pend, &s))) { release(&s); return rc; }
    memcpy(cmd, s.cmd, d.n_cmd); memcpy(mlen, s.mlen, d.n_match); memcpy(lit, s.lit, d.n_lit);
    uint64_t op = b << h.log2_bs; uint32_t lp = 0;
    for (uint32_t c = 0; c < d.n_cmd; c++) {
        if (c < d.n_match) src[c] = s.src[c];
        lit_len[c] = s.lit_len[c]; match_len[c] = s.match_len[c];
        lit_pos[c] = lp; out_pos[c] = op;
        lp += s.lit_len[c]; op += (uint64_t)s.lit_len[c] + s.match_len[c];
    }
    release(&s);
    return OK;
}

/* The rANS step alone (FORMAT.md §1.5), for the rANS pins: freq is n_tables x 256 u16 (each row sums to 2^prob_bits).
 * states: 32 initial states in, final states out.  word_off: 33 entries (u64); words_used: 32 entries out. */
int acx_oracle_rans(const uint16_t* freq, uint32_t n_tables, uint32_t prob_bits, const uint8_t* tid, uint64_t n_sym,
                    uint32_t* states, const uint8_t* words, const uint64_t* word_off, uint8_t* sym, uint64_t* words_used) {
    if (n_tables > 11) return E_RANGE;
    table_t T[11];
    for (uint32_t t = 0; t < n_tables; t++) {
        uint32_t sum = 0; T[t].mode = 0; T[t].cum[0] = 0;
        for (int s = 0; s < 256; s++) { T[t].freq[s] = freq[256 * t + s]; sum += T[t].freq[s]; T[t].cum[s + 1] = sum; }
        if (sum != (1u << prob_bits) || prob_bits > 11) return E_CORRUPT;
        fill_slots(&T[t]);
    }
    for (int k = 0; k < 32; k++) if (word_off[k] > word_off[k + 1]) return E_CORRUPT;
    return rans_decode(T, tid, n_sym, prob_bits, states, words, word_off, sym, words_used);
}

/* FNV-1a 64 (FORMAT.md §5; "FNV for device-resident GPU paths"). */
uint64_t acx_oracle_fnv1a64(const uint8_t* p, uint64_t n) {
    uint64_t f = 0xcbf29ce484222325ull;
    for (uint64_t i = 0; i < n; i++) { f ^= p[i]; f *= 0x100000001b3ull; }
    return f;
}
