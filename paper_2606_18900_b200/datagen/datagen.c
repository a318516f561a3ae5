/* Seeded synthetic inputs shaped like the paper's workloads (Table 2, §4).
 *
 * This module is the ONLY code shared by the oracle side and the CUDA side of the tests. It holds none of the
 * method's arithmetic (no LZ, no rANS, no format knowledge): it only produces the bytes to be compressed and the
 * read index entries.  Recipes are stated in DESIGN.md §"Input recipe" (BASELINE.json configs[0..4]).
 *
 * Everything is integer arithmetic on a counter-based generator, so bytes are identical across compilers and any
 * window [lo, hi) of a FASTQ file can be produced without producing the rest.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

static inline uint64_t mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}
/* draw k of stream (seed, stream, idx) */
static inline uint64_t draw(uint64_t seed, uint64_t stream, uint64_t idx, uint64_t k) {
    uint64_t key = mix64(seed ^ (stream * 0xD6E8FEB86659FD93ull));
    key = mix64(key ^ (idx * 0xA0761D6478BD642Full));
    return mix64(key + k);
}

enum { ST_REF = 1, ST_POS = 2, ST_SUB = 3, ST_QUAL = 4, ST_PLAN = 5, ST_NOVEL = 6, ST_MUT = 7, ST_REGION = 8 };

/* ---------------------------------------------------------------- FASTQ ---------------------------------- */
/* Record n (n >= 1):  "@SIM.<n> <n>/1\n" + 150 bases + "\n+\n" + 150 quals + "\n";  length 2*digits(n) + 313.   */

#define READ_LEN 150

static int ndigits(uint64_t n) { int d = 1; while (n >= 10) { n /= 10; d++; } return d; }

/* byte offset of record n (1-based) in the untruncated file */
static uint64_t fastq_record_off(uint64_t n) {
    uint64_t off = 0, lo = 1;
    for (int d = 1; d <= 20; d++) {
        uint64_t hi = lo * 10; /* records with d digits: [lo, hi) */
        if (n <= lo) break;
        uint64_t cnt = (n < hi ? n : hi) - lo;
        off += cnt * (uint64_t)(2 * d + 313);
        lo = hi;
    }
    return off;
}
/* largest n with fastq_record_off(n) <= pos */
static uint64_t fastq_record_at(uint64_t pos) {
    uint64_t lo = 1, hi = pos / 315 + 2;
    while (lo < hi) {
        uint64_t mid = lo + (hi - lo + 1) / 2;
        if (fastq_record_off(mid) <= pos) lo = mid; else hi = mid - 1;
    }
    return lo;
}

static inline int ref_base(uint64_t seed, uint64_t i) { /* 0..3, uniform */
    return (int)((draw(seed, ST_REF, i >> 5, 0) >> (2 * (i & 31))) & 3);
}

static int fastq_record(uint64_t seed, uint64_t ref_len, uint64_t n, unsigned char* rec) {
    static const char B[4] = {'A', 'C', 'G', 'T'};
    int d = ndigits(n), p = 0;
    char num[24];
    { uint64_t t = n; for (int i = d - 1; i >= 0; i--) { num[i] = (char)('0' + t % 10); t /= 10; } }
    memcpy(rec + p, "@SIM.", 5); p += 5;
    memcpy(rec + p, num, d); p += d;
    rec[p++] = ' ';
    memcpy(rec + p, num, d); p += d;
    rec[p++] = '/'; rec[p++] = '1'; rec[p++] = '\n';
    uint64_t pos = draw(seed, ST_POS, n, 0) % (ref_len - READ_LEN + 1);
    for (int i = 0; i < READ_LEN; i += 2) { /* one 64-bit draw serves two bases: 2 x (16 + 16) bits */
        uint64_t r = draw(seed, ST_SUB, n, (uint64_t)(i >> 1));
        for (int j = 0; j < 2; j++) {
            unsigned sub = (unsigned)(r & 0xffff), nn = (unsigned)((r >> 16) & 0xffff);
            r >>= 32;
            int b = ref_base(seed, pos + (uint64_t)(i + j));
            if (sub < 655) b = (b + 1 + (int)(sub % 3)) & 3;      /* 1 % substitution, always to another base */
            rec[p++] = (nn < 66) ? 'N' : (unsigned char)B[b];     /* 0.1 % N                                  */
        }
    }
    rec[p++] = '\n'; rec[p++] = '+'; rec[p++] = '\n';
    for (int i = 0; i < READ_LEN; i++) {
        /* Irwin-Hall(12) of bytes: mean 1530, sd 256.0  ->  q = round(36 - 8 i / 149 + 4 z), clipped to [2, 41] */
        uint64_t a = draw(seed, ST_QUAL, n, (uint64_t)(2 * i)), b = draw(seed, ST_QUAL, n, (uint64_t)(2 * i + 1));
        int s = 0;
        for (int k = 0; k < 8; k++) { s += (int)(a & 0xff); a >>= 8; }
        for (int k = 0; k < 4; k++) { s += (int)(b & 0xff); b >>= 8; }
        int64_t num64 = (int64_t)36 * 149 * 64 - (int64_t)8 * i * 64 + (int64_t)(s - 1530) * 149;
        int64_t den = 149 * 64;
        int64_t q = (2 * num64 + den) / (2 * den); /* num64 >= 39038 > 0, so this is round-half-up */
        if (q < 2) q = 2;
        if (q > 41) q = 41;
        rec[p++] = (unsigned char)(33 + q);
    }
    rec[p++] = '\n';
    return p;
}

/* Bytes [lo, hi) of the FASTQ file of total size N (the last record is cut at N). */
int acx_gen_fastq(uint64_t seed, uint64_t ref_len, uint64_t N, uint64_t lo, uint64_t hi, unsigned char* out) {
    if (lo > hi || hi > N || ref_len < READ_LEN) return -1;
    if (lo == hi) return 0;
    unsigned char rec[512];
    uint64_t n = fastq_record_at(lo);
    uint64_t off = fastq_record_off(n);
    while (off < hi) {
        int len = fastq_record(seed, ref_len, n, rec);
        uint64_t a = off < lo ? lo : off, b = off + (uint64_t)len < hi ? off + (uint64_t)len : hi;
        if (b > a) memcpy(out + (a - lo), rec + (a - off), b - a);
        off += (uint64_t)len;
        n++;
    }
    return 0;
}
/* Number of whole records inside [0, N). */
uint64_t acx_fastq_n_reads(uint64_t N) {
    uint64_t n = fastq_record_at(N); /* record n starts at <= N */
    /* records 1..n-1 are complete iff record n starts <= N, which holds */
    return n - 1;
}
/* Read index entries (FORMAT.md §4) for reads [first, first+count) (0-based read id r = record r+1). */
int acx_fastq_index(uint64_t N, uint64_t first, uint64_t count, uint64_t* out) {
    uint64_t total = acx_fastq_n_reads(N);
    if (first + count > total) return -1;
    uint64_t off = fastq_record_off(first + 1);
    for (uint64_t r = 0; r < count; r++) {
        uint64_t len = (uint64_t)(2 * ndigits(first + r + 1) + 313);
        out[r] = off | (len << 40);
        off += len;
    }
    return 0;
}

/* ---------------------------------------------------------------- FASTA genome --------------------------- */
/* 24 sequences ">chr1".."\>chr24", sizes proportional to 249 - 203 i / 23, 60-character lines, scaled so the file
 * has exactly N bytes (the last line/sequence is cut at N).  Base content over the concatenated base space:
 * alternating novel segments (uniform ACGT, length uniform 300..7400) and copy segments (length uniform 300..6000,
 * source uniform over all earlier base positions, per-copy divergence uniform 2..15 %), i.e. ~45 % copied; N-runs of
 * 10,000 every 2.5..7.5 Mbp (uniform gap, mean 5 Mbp).  Needs the whole file in memory (copies read earlier output). */

typedef struct { uint64_t base0, nbases, file0; int hdr; } chr_t;

static void fasta_layout(uint64_t N, chr_t* c, uint64_t* total_bases) {
    /* find the scale (bases per unit) by bisection on the total file size; weights w_i = 249*23 - 203*i */
    uint64_t w[24], wsum = 0;
    for (int i = 0; i < 24; i++) { w[i] = 249 * 23 - 203 * (uint64_t)i; wsum += w[i]; }
    uint64_t lo = 0, hi = N;
    for (;;) { /* largest G (total bases) whose file size <= N */
        uint64_t G = lo + (hi - lo + 1) / 2;
        uint64_t sz = 0;
        for (int i = 0; i < 24; i++) {
            uint64_t nb = G / wsum * w[i] + (G % wsum) * w[i] / wsum;
            int hdr = 4 + (i + 1 >= 10 ? 2 : 1) + 1;
            sz += (uint64_t)hdr + nb + (nb + 59) / 60;
        }
        if (sz <= N) lo = G; else hi = G - 1;
        if (lo >= hi) break;
    }
    uint64_t G = lo, b0 = 0, f0 = 0;
    for (int i = 0; i < 24; i++) {
        uint64_t nb = G / wsum * w[i] + (G % wsum) * w[i] / wsum;
        c[i].hdr = 4 + (i + 1 >= 10 ? 2 : 1) + 1;
        c[i].base0 = b0; c[i].nbases = nb; c[i].file0 = f0;
        b0 += nb; f0 += (uint64_t)c[i].hdr + nb + (nb + 59) / 60;
    }
    /* the remainder of the file (N - f0 bytes, < a few hundred) extends the last sequence */
    if (f0 < N) {
        uint64_t extra = N - f0, nb = c[23].nbases;
        /* add bases one line at a time */
        while (extra > 0) {
            if (nb % 60 == 0) { /* new line: needs base + newline */
                if (extra < 2) break;
                nb++; extra -= 2;
            } else { nb++; extra -= 1; }
        }
        b0 += nb - c[23].nbases; c[23].nbases = nb;
    }
    *total_bases = b0;
}

typedef struct { int ci; uint64_t j, fo; unsigned col; } cur_t;
static void cur_set(cur_t* u, const chr_t* c, uint64_t g) {
    int i = 0;
    while (i < 23 && g >= c[i + 1].base0) i++;
    u->ci = i; u->j = g - c[i].base0; u->col = (unsigned)(u->j % 60);
    u->fo = c[i].file0 + (uint64_t)c[i].hdr + u->j + u->j / 60;
}
static inline void cur_adv(cur_t* u, const chr_t* c) {
    u->j++; u->fo++;
    if (++u->col == 60) { u->col = 0; u->fo++; }
    if (u->j == c[u->ci].nbases && u->ci < 23) { u->ci++; u->j = 0; u->col = 0; u->fo = c[u->ci].file0 + (uint64_t)c[u->ci].hdr; }
}

int acx_gen_fasta(uint64_t seed, uint64_t N, unsigned char* out) {
    static const char B[4] = {'A', 'C', 'G', 'T'};
    chr_t c[24];
    uint64_t G;
    if (N < 4096) return -1;
    fasta_layout(N, c, &G);
    memset(out, '\n', N);
    for (int i = 0; i < 24; i++) {
        char h[16]; int n = 0;
        h[n++] = '>'; h[n++] = 'c'; h[n++] = 'h'; h[n++] = 'r';
        if (i + 1 >= 10) h[n++] = (char)('0' + (i + 1) / 10);
        h[n++] = (char)('0' + (i + 1) % 10); h[n++] = '\n';
        if (c[i].file0 + (uint64_t)n <= N) memcpy(out + c[i].file0, h, (size_t)n);
    }
    /* walk the segment plan */
    uint64_t g = 0, seg = 0;
    uint64_t next_n = 2500000 + draw(seed, ST_PLAN, 0, 99) % 5000001;
    cur_t d; cur_set(&d, c, 0);
    uint64_t nov_i = ~0ull, nov_v = 0, mut_i = ~0ull, mut_v = 0;
    while (g < G) {
        uint64_t r0 = draw(seed, ST_PLAN, seg, 0), r1 = draw(seed, ST_PLAN, seg, 1), r2 = draw(seed, ST_PLAN, seg, 2);
        int kind = (int)(seg & 1); /* 0 novel, 1 copy, 2 N-run */
        uint64_t len;
        if (g >= next_n) { kind = 2; len = 10000; next_n = g + len + 2500000 + r0 % 5000001; }
        else if (kind == 0) len = 300 + r0 % 7101;
        else len = 300 + r0 % 5701;
        if (kind == 1 && g < len) kind = 0;
        if (len > G - g) len = G - g;
        unsigned thr = 0;
        cur_t s; s.ci = 0;
        if (kind == 1) { cur_set(&s, c, r1 % (g - len + 1)); thr = (unsigned)(1311 + r2 % 8520); } /* 2 % .. 15 % of 65536 */
        for (uint64_t k = 0; k < len; k++) {
            uint64_t gi = g + k;
            unsigned char ch;
            if (kind == 2) ch = 'N';
            else if (kind == 0) {
                if ((gi >> 5) != nov_i) { nov_i = gi >> 5; nov_v = draw(seed, ST_NOVEL, nov_i, 0); }
                ch = (unsigned char)B[(nov_v >> (2 * (gi & 31))) & 3];
            } else {
                ch = out[s.fo];
                cur_adv(&s, c);
                if (ch != 'N') {
                    if ((gi >> 2) != mut_i) { mut_i = gi >> 2; mut_v = draw(seed, ST_MUT, mut_i, 0); }
                    uint64_t m = mut_v >> (16 * (gi & 3));
                    if ((unsigned)(m & 0xffff) < thr) {
                        int b = ch == 'A' ? 0 : ch == 'C' ? 1 : ch == 'G' ? 2 : 3;
                        ch = (unsigned char)B[(b + 1 + (int)((m & 0xffff) % 3)) & 3];
                    }
                }
            }
            if (d.fo < N) out[d.fo] = ch;
            cur_adv(&d, c);
        }
        g += len; seg++;
    }
    return 0;
}

/* n region "reads": offsets uniform in [0, N - len], fixed length (configs[2]: 150).  FORMAT.md §4 entries. */
int acx_gen_region_index(uint64_t seed, uint64_t N, uint64_t n, uint64_t len, uint64_t* out) {
    if (len > N || len >= (1ull << 24) || N > (1ull << 40)) return -1;
    for (uint64_t i = 0; i < n; i++) out[i] = (draw(seed, ST_REGION, i, 0) % (N - len + 1)) | (len << 40);
    return 0;
}
