/* CPU BASELINE — test / measurement infrastructure, not product code.
 *
 * A multithreaded CPU decoder of the ACX-B200 format (FORMAT.md version 3), the second reported baseline named by
 * BASELINE.json north_star ("the oracle, and a multithreaded CPU decoder, timed on the B200 box's own host cores").
 * It follows the schedule of FORMAT.md §3 on host threads: pass 1 = every segment in parallel: entropy decode
 * (FORMAT.md §1.7), command lengths, literal placement; pass 2 = dependency levels in order, the segments of a level's
 * blocks in parallel: byte-serial match copies (FORMAT.md §2).  Separate source: it shares no code with the oracle
 * (acx_oracle.c), with the encoder or with the CUDA path.  It assumes a valid archive (the oracle is the validator) and
 * is checked against the original bytes by tests/test_cpu_mt.py.  Only tests/ and bench.py's cpu_baseline leg use it. */
#include <pthread.h>
#include <stdatomic.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct { uint32_t mode, pb; uint16_t freq[4096], cum[4096], value[4096], slot2sym[4096]; } tab_t;
typedef struct { uint32_t lit_len, match_len; uint64_t src; } cmd_t;

typedef struct {
    const uint8_t* a; uint8_t* out;
    uint64_t N, n_blocks, n_segs, dir_off, blocktab_off; uint32_t log2_bs, min_match, W, n_tables, max_level, q_min, q_mode;
    tab_t* T;                                /* n_tables byte tables + the pair table */
    cmd_t* cmds; uint64_t* cmd_off;          /* commands of all segments, segment s at cmds[cmd_off[s] ..] */
    uint32_t* by_level; uint64_t* level_off; /* segment ids sorted by the level of their block */
    atomic_ullong next; uint64_t work_lo, work_hi; int pass; atomic_int err;
} job_t;

static uint64_t g64(const uint8_t* p) { uint64_t v; memcpy(&v, p, 8); return v; }
static uint32_t g32(const uint8_t* p) { uint32_t v; memcpy(&v, p, 4); return v; }
static uint32_t g16(const uint8_t* p) { uint16_t v; memcpy(&v, p, 2); return v; }

/* pass 1 for segment sg: FORMAT.md §1.5-1.7, literal placement of both classes */
static int seg_pass1(job_t* J, uint64_t sg, uint16_t* sym, uint64_t sym_cap) {
    const uint8_t* d = J->a + J->dir_off + 32 * sg;
    uint64_t po = g64(d), out_start = g64(d + 8);
    uint32_t n_cmd = g16(d + 16), n_match = g16(d + 18), n_lit_a = g16(d + 20), n_sym_q = g16(d + 24), n_words = g16(d + 26), n_ext = g16(d + 28);
    uint32_t W = J->W, n_coded = 0;
    for (uint32_t p = 0; p < W; p++) n_coded += J->T[2 + p].mode == 0;
    uint64_t n_sym = (uint64_t)n_cmd + (uint64_t)n_match * (1 + n_coded) + n_lit_a + n_sym_q;
    if (n_sym > sym_cap) return -1;
    const uint8_t* pl = J->a + po;
    uint32_t X[32]; const uint8_t* wp[32];
    for (int k = 0; k < 32; k++) { X[k] = g32(pl + 8 * k); wp[k] = pl + 256 + 2ull * g32(pl + 8 * k + 4); }
    /* table of each region of the symbol sequence: CMD, MLEN, coded planes (high first), LITA, LITQ */
    uint64_t i = 0;
    uint64_t reg_end[14]; const tab_t* reg_tab[14]; int nr = 0;
    reg_end[nr] = n_cmd; reg_tab[nr++] = &J->T[0];
    reg_end[nr] = reg_end[nr - 1] + n_match; reg_tab[nr++] = &J->T[1];
    for (int p = (int)W - 1; p >= 0; p--) if (J->T[2 + p].mode == 0) { reg_end[nr] = reg_end[nr - 1] + n_match; reg_tab[nr++] = &J->T[2 + p]; }
    reg_end[nr] = reg_end[nr - 1] + n_lit_a; reg_tab[nr++] = &J->T[2 + W];
    const tab_t* TQ = &J->T[J->q_mode == 1 ? J->n_tables : 3 + W];
    reg_end[nr] = reg_end[nr - 1] + n_sym_q; reg_tab[nr++] = TQ;
    for (int r = 0; r < nr; r++) {
        const tab_t* t = reg_tab[r];
        const uint32_t pb = t->pb, mask = (1u << pb) - 1;
        for (; i < reg_end[r]; i++) {
            int k = (int)(i & 31);
            uint32_t x = X[k], slot = x & mask, s = t->slot2sym[slot];
            x = t->freq[s] * (x >> pb) + slot - t->cum[s];
            if (x < 65536u) { x = (x << 16) | g16(wp[k]); wp[k] += 2; }
            X[k] = x; sym[i] = t->value[s];
        }
    }
    uint64_t ext_off = (256 + 2ull * n_words + 3) & ~3ull;
    const uint8_t* ext = pl + ext_off;
    const uint16_t *tc = sym, *tm = sym + n_cmd, *planes = sym + n_cmd + n_match, *lit_a = sym + n_sym - n_sym_q - n_lit_a, *lit_q = sym + n_sym - n_sym_q;
    uint32_t n_ext_cmd = 0;
    for (uint32_t c = 0; c < n_cmd; c++) n_ext_cmd += tc[c] == 255;
    const uint8_t* raw = ext + 4ull * n_ext;
    cmd_t* C = J->cmds + J->cmd_off[sg];
    uint32_t ec = 0, em = n_ext_cmd;
    uint64_t dst = out_start, la = 0, lq = 0;
    uint8_t* out = J->out;
    for (uint32_t c = 0; c < n_cmd; c++) {
        uint32_t ll = tc[c]; if (ll == 255) ll = 255 + g32(ext + 4ull * ec++);
        uint32_t ml = 0; uint64_t src = 0;
        if (c < n_match) {
            uint32_t v = tm[c]; if (v == 255) v = 255 + g32(ext + 4ull * em++);
            ml = J->min_match + v;
            uint32_t kc = 0, kr = 0;
            for (int p = (int)W - 1; p >= 0; p--) if (J->T[2 + p].mode == 0) { src |= (uint64_t)planes[(uint64_t)kc * n_match + c] << (8 * p); kc++; }
            for (uint32_t p = 0; p < W; p++) if (J->T[2 + p].mode == 1) { src |= (uint64_t)raw[(uint64_t)kr * n_match + c] << (8 * p); kr++; }
        }
        /* literal placement */
        if (J->q_min && ll >= J->q_min) {
            if (J->q_mode == 0) { for (uint32_t q = 0; q < ll; q++) out[dst + q] = (uint8_t)lit_q[lq + q]; lq += ll; }
            else for (uint64_t k = dst >> 1; k <= (dst + ll - 1) >> 1; k++, lq++) {       /* aligned pairs, fillers dropped */
                if (2 * k >= dst) out[2 * k] = (uint8_t)lit_q[lq];
                if (2 * k + 1 < dst + ll) out[2 * k + 1] = (uint8_t)(lit_q[lq] >> 8);
            }
        } else { for (uint32_t q = 0; q < ll; q++) out[dst + q] = (uint8_t)lit_a[la + q]; la += ll; }
        dst += ll + ml;
        C[c].lit_len = ll; C[c].match_len = ml; C[c].src = src;
    }
    return 0;
}

/* pass 2 for segment sg: FORMAT.md §2 */
static void seg_pass2(job_t* J, uint64_t sg) {
    const uint8_t* d = J->a + J->dir_off + 32 * sg;
    uint32_t n_cmd = g16(d + 16), n_match = g16(d + 18);
    const cmd_t* C = J->cmds + J->cmd_off[sg];
    uint64_t dst = g64(d + 8);
    uint8_t* out = J->out;
    for (uint32_t c = 0; c < n_cmd; c++) {
        dst += C[c].lit_len;
        if (c < n_match) {
            uint64_t src = C[c].src; uint32_t ml = C[c].match_len;
            if (src + ml <= dst) memcpy(out + dst, out + src, ml);
            else for (uint32_t i = 0; i < ml; i++) out[dst + i] = out[src + i];   /* self-overlap: ascending byte by byte */
            dst += ml;
        }
    }
}

static void* worker(void* arg) {
    job_t* J = (job_t*)arg;
    uint64_t cap = 16384 + 16384 + 510ull * 10 + 4096;      /* FORMAT.md §1.5 limits: literals + tokens of a segment */
    uint16_t* sym = J->pass == 1 ? (uint16_t*)malloc(2 * cap) : NULL;
    for (;;) {
        uint64_t i = atomic_fetch_add(&J->next, 64);
        if (i >= J->work_hi) break;
        uint64_t e = i + 64 < J->work_hi ? i + 64 : J->work_hi;
        for (; i < e; i++) {
            if (J->pass == 1) { if (seg_pass1(J, i, sym, cap)) atomic_store(&J->err, -1); }
            else seg_pass2(J, J->by_level[i]);
        }
    }
    free(sym);
    return NULL;
}

static void run(job_t* J, int threads, int pass, uint64_t lo, uint64_t hi) {
    pthread_t th[256];
    if (threads > 256) threads = 256;
    J->pass = pass; J->work_lo = lo; J->work_hi = hi; atomic_store(&J->next, lo);
    for (int t = 0; t < threads; t++) pthread_create(&th[t], NULL, worker, J);
    for (int t = 0; t < threads; t++) pthread_join(th[t], NULL);
}

static void fill_table(tab_t* T) {
    uint32_t cum = 0;
    for (uint32_t s = 0; s < 4096 && cum < (1u << T->pb); s++) {
        T->cum[s] = (uint16_t)cum;
        for (uint32_t k = 0; k < T->freq[s] && cum + k < (1u << T->pb); k++) T->slot2sym[cum + k] = (uint16_t)s;
        cum += T->freq[s];
    }
}

/* Decodes the whole archive into out (>= N bytes) with `threads` host threads.  Returns 0, or a negative error. */
int acx_mt_decode(const uint8_t* a, uint64_t n, uint8_t* out, uint64_t out_cap, int threads) {
    job_t* J = (job_t*)calloc(1, sizeof(job_t));
    if (!J || n < 192 || memcmp(a, "ACXB200", 8) || g32(a + 8) != 3) { free(J); return -1; }
    J->a = a; J->out = out; J->N = g64(a + 16); J->n_blocks = g64(a + 24); J->n_segs = g64(a + 32); J->log2_bs = g32(a + 40);
    J->min_match = g32(a + 44); J->W = g32(a + 48); J->n_tables = g32(a + 56); J->max_level = g32(a + 60);
    J->q_min = g32(a + 76); J->q_mode = g32(a + 80);
    uint32_t n_qpairs = g32(a + 84);
    uint64_t tables_off = g64(a + 88), qtab_off = g64(a + 96), total_cmds = g64(a + 168);
    J->blocktab_off = g64(a + 104); J->dir_off = g64(a + 112);
    if (out_cap < J->N || J->n_tables > 12 || threads < 1 || n_qpairs > 4096) { free(J); return -2; }
    J->T = (tab_t*)calloc(J->n_tables + 1, sizeof(tab_t));
    if (!J->T) { free(J); return -3; }
    for (uint32_t t = 0; t < J->n_tables; t++) {
        const uint8_t* p = a + tables_off + 528ull * t;
        tab_t* T = &J->T[t];
        T->mode = g32(p); T->pb = 11;
        for (int s = 0; s < 256; s++) { T->freq[s] = (uint16_t)g16(p + 16 + 2 * s); T->value[s] = (uint16_t)s; }
        fill_table(T);
    }
    {
        tab_t* T = &J->T[J->n_tables];
        T->pb = 12;
        for (uint32_t i = 0; i < n_qpairs; i++) { T->value[i] = (uint16_t)g16(a + qtab_off + 4ull * i); T->freq[i] = (uint16_t)g16(a + qtab_off + 4ull * i + 2); }
        fill_table(T);
    }
    J->cmds = (cmd_t*)malloc(sizeof(cmd_t) * (total_cmds + 1));
    J->cmd_off = (uint64_t*)malloc(8 * (J->n_segs + 1));
    J->by_level = (uint32_t*)malloc(4 * (J->n_segs + 1));
    J->level_off = (uint64_t*)calloc(J->max_level + 3, 8);
    if (!J->cmds || !J->cmd_off || !J->by_level || !J->level_off) return -3;
    uint64_t acc = 0;
    for (uint64_t s = 0; s < J->n_segs; s++) {
        const uint8_t* d = a + J->dir_off + 32 * s;
        J->cmd_off[s] = acc; acc += g16(d + 16);
        J->level_off[g16(d + 30) + 2]++;
    }
    for (uint32_t l = 2; l < J->max_level + 3; l++) J->level_off[l] += J->level_off[l - 1];
    for (uint64_t s = 0; s < J->n_segs; s++) J->by_level[J->level_off[g16(a + J->dir_off + 32 * s + 30) + 1]++] = (uint32_t)s;
    run(J, threads, 1, 0, J->n_segs);                                          /* pass 1: all segments */
    for (uint32_t l = 0; l <= J->max_level && !atomic_load(&J->err); l++)       /* pass 2: level by level */
        run(J, threads, 2, J->level_off[l], J->level_off[l + 1]);
    int rc = atomic_load(&J->err);
    free(J->cmds); free(J->cmd_off); free(J->by_level); free(J->level_off); free(J->T); free(J);
    return rc;
}
