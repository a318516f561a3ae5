/* CPU BASELINE — test / measurement infrastructure, not product code.
 *
 * A multithreaded CPU decoder of the ACX-B200 format (FORMAT.md version 2), the second reported baseline named by
 * BASELINE.json north_star ("the oracle, and a multithreaded CPU decoder, timed on the B200 box's own host cores").
 * It follows the schedule of FORMAT.md §3 on host threads: pass 1 = every block in parallel: entropy decode
 * (FORMAT.md §1.5), command lengths, literal placement; pass 2 = dependency levels in order, the blocks of a level in
 * parallel: byte-serial match copies (FORMAT.md §2).  Separate source: it shares no code with the oracle
 * (acx_oracle.c), with the encoder or with the CUDA path.  It assumes a valid archive (the oracle is the validator) and
 * is checked against the original bytes by tests/test_cpu_mt.py.  Only tests/ and bench.py's cpu_baseline leg use it. */
#include <pthread.h>
#include <stdatomic.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

typedef struct { uint32_t mode; uint16_t freq[256], cum[256]; uint8_t slot2sym[2048]; } tab_t;
typedef struct { uint32_t lit_len, match_len; uint64_t src; } cmd_t;

typedef struct {
    const uint8_t* a; uint8_t* out;
    uint64_t N, n_blocks, dir_off; uint32_t log2_bs, min_match, W, n_tables, max_level;
    tab_t T[11];
    cmd_t* cmds; uint64_t* cmd_off;          /* commands of all blocks, block b at cmds[cmd_off[b] ..] */
    uint32_t* by_level; uint64_t* level_off; /* block ids sorted by level */
    atomic_ullong next; uint64_t work_lo, work_hi; int pass; atomic_int err;
} job_t;

static uint64_t g64(const uint8_t* p) { uint64_t v; memcpy(&v, p, 8); return v; }
static uint32_t g32(const uint8_t* p) { uint32_t v; memcpy(&v, p, 4); return v; }
static uint32_t g16(const uint8_t* p) { uint16_t v; memcpy(&v, p, 2); return v; }

/* pass 1 for block b: FORMAT.md §1.4-1.5 */
static int block_pass1(job_t* J, uint64_t b, uint8_t* sym, uint64_t sym_cap) {
    const uint8_t* d = J->a + J->dir_off + 32 * b;
    uint64_t po = g64(d); uint32_t n_cmd = g32(d + 8), n_match = g32(d + 12), n_lit = g32(d + 16), n_words = g32(d + 20);
    uint32_t W = J->W, n_coded = 0;
    for (uint32_t p = 0; p < W; p++) n_coded += J->T[2 + p].mode == 0;
    uint64_t n_sym = (uint64_t)n_cmd + (uint64_t)n_match * (1 + n_coded) + n_lit;
    if (n_sym > sym_cap) return -1;
    const uint8_t* pl = J->a + po;
    uint32_t X[32]; const uint8_t* wp[32];
    for (int k = 0; k < 32; k++) { X[k] = g32(pl + 8 * k); wp[k] = pl + 256 + 2ull * g32(pl + 8 * k + 4); }
    /* table of each region of the symbol sequence: CMD, MLEN, coded planes (high first), LIT */
    uint64_t i = 0;
    uint64_t reg_end[12]; const tab_t* reg_tab[12]; int nr = 0;
    reg_end[nr] = n_cmd; reg_tab[nr++] = &J->T[0];
    reg_end[nr] = reg_end[nr - 1] + n_match; reg_tab[nr++] = &J->T[1];
    for (int p = (int)W - 1; p >= 0; p--) if (J->T[2 + p].mode == 0) { reg_end[nr] = reg_end[nr - 1] + n_match; reg_tab[nr++] = &J->T[2 + p]; }
    reg_end[nr] = reg_end[nr - 1] + n_lit; reg_tab[nr++] = &J->T[2 + W];
    for (int r = 0; r < nr; r++) {
        const tab_t* t = reg_tab[r];
        for (; i < reg_end[r]; i++) {
            int k = (int)(i & 31);
            uint32_t x = X[k], slot = x & 2047u, s = t->slot2sym[slot];
            x = t->freq[s] * (x >> 11) + slot - t->cum[s];
            if (x < 65536u) { x = (x << 16) | g16(wp[k]); wp[k] += 2; }
            X[k] = x; sym[i] = (uint8_t)s;
        }
    }
    uint64_t ext_off = (256 + 2ull * n_words + 3) & ~3ull;
    const uint8_t* ext = pl + ext_off;
    const uint8_t *tc = sym, *tm = sym + n_cmd, *planes = sym + n_cmd + n_match, *lit = sym + n_sym - n_lit;
    uint32_t n_ext_cmd = 0;
    for (uint32_t c = 0; c < n_cmd; c++) n_ext_cmd += tc[c] == 255;
    const uint8_t* raw = ext + 4ull * (g32(d + 24));
    cmd_t* C = J->cmds + J->cmd_off[b];
    uint32_t ec = 0, em = n_ext_cmd;
    uint64_t dst = b << J->log2_bs, lp = 0;
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
        memcpy(J->out + dst, lit + lp, ll);       /* literal placement */
        lp += ll; dst += ll + ml;
        C[c].lit_len = ll; C[c].match_len = ml; C[c].src = src;
    }
    return 0;
}

/* pass 2 for block b: FORMAT.md §2 */
static void block_pass2(job_t* J, uint64_t b) {
    const uint8_t* d = J->a + J->dir_off + 32 * b;
    uint32_t n_cmd = g32(d + 8), n_match = g32(d + 12);
    const cmd_t* C = J->cmds + J->cmd_off[b];
    uint64_t dst = b << J->log2_bs;
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
    uint64_t cap = (3ull << J->log2_bs) + 4096;
    uint8_t* sym = J->pass == 1 ? (uint8_t*)malloc(cap) : NULL;
    for (;;) {
        uint64_t i = atomic_fetch_add(&J->next, 64);
        if (i >= J->work_hi) break;
        uint64_t e = i + 64 < J->work_hi ? i + 64 : J->work_hi;
        for (; i < e; i++) {
            if (J->pass == 1) { if (block_pass1(J, i, sym, cap)) atomic_store(&J->err, -1); }
            else block_pass2(J, J->by_level[i]);
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

/* Decodes the whole archive into out (>= N bytes) with `threads` host threads.  Returns 0, or a negative error. */
int acx_mt_decode(const uint8_t* a, uint64_t n, uint8_t* out, uint64_t out_cap, int threads) {
    job_t* J = (job_t*)calloc(1, sizeof(job_t));
    if (!J || n < 160 || memcmp(a, "ACXB200", 8) || g32(a + 8) != 2) { free(J); return -1; }
    J->a = a; J->out = out; J->N = g64(a + 16); J->n_blocks = g64(a + 24); J->log2_bs = g32(a + 32); J->min_match = g32(a + 36);
    J->W = g32(a + 40); J->n_tables = g32(a + 48); J->max_level = g32(a + 52); J->dir_off = g64(a + 72);
    uint64_t tables_off = g64(a + 64), total_cmds = g64(a + 128);
    if (out_cap < J->N || J->n_tables > 11 || threads < 1) { free(J); return -2; }
    for (uint32_t t = 0; t < J->n_tables; t++) {
        const uint8_t* p = a + tables_off + 528ull * t;
        tab_t* T = &J->T[t];
        T->mode = g32(p);
        uint32_t cum = 0;
        for (int s = 0; s < 256; s++) {
            T->freq[s] = (uint16_t)g16(p + 16 + 2 * s); T->cum[s] = (uint16_t)cum;
            for (uint32_t k = 0; k < T->freq[s] && cum + k < 2048; k++) T->slot2sym[cum + k] = (uint8_t)s;
            cum += T->freq[s];
        }
    }
    J->cmds = (cmd_t*)malloc(sizeof(cmd_t) * (total_cmds + 1));
    J->cmd_off = (uint64_t*)malloc(8 * (J->n_blocks + 1));
    J->by_level = (uint32_t*)malloc(4 * (J->n_blocks + 1));
    J->level_off = (uint64_t*)calloc(J->max_level + 3, 8);
    if (!J->cmds || !J->cmd_off || !J->by_level || !J->level_off) return -3;
    uint64_t acc = 0;
    for (uint64_t b = 0; b < J->n_blocks; b++) {
        const uint8_t* d = a + J->dir_off + 32 * b;
        J->cmd_off[b] = acc; acc += g32(d + 8);
        J->level_off[g16(d + 28) + 2]++;
    }
    for (uint32_t l = 2; l < J->max_level + 3; l++) J->level_off[l] += J->level_off[l - 1];
    for (uint64_t b = 0; b < J->n_blocks; b++) J->by_level[J->level_off[g16(a + J->dir_off + 32 * b + 28) + 1]++] = (uint32_t)b;
    run(J, threads, 1, 0, J->n_blocks);                                        /* pass 1: all blocks */
    for (uint32_t l = 0; l <= J->max_level && !atomic_load(&J->err); l++)       /* pass 2: level by level */
        run(J, threads, 2, J->level_off[l], J->level_off[l + 1]);
    int rc = atomic_load(&J->err);
    free(J->cmds); free(J->cmd_off); free(J->by_level); free(J->level_off); free(J);
    return rc;
}
