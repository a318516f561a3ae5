/* ORACLE — test infrastructure, not product code.
 *
 * Plain C rANS ENCODER and decoder for the entropy micro-benchmark (section 6.4: "256 MB
 * exponential, batch 4096 x 64 KB").  A batch is n_rows rows of row_bytes symbols; every row is coded on its own with one
 * static byte table as a rANS section of FORMAT.md 1.7: 32 interleaved states, symbol i on state i mod 32, one word stream
 * per state, [head: 32 x (u32 initial state, u32 word_off)][words].  The encoder is the paragraph of FORMAT.md 1.7 written
 * out: symbols in reverse order from x = 2^16; before coding s on x, emit x & 0xffff and shift x >>= 16 iff
 * x >= freq[s] << (32 - 11); then x = ((x / f) << 11) + (x mod f) + cum[s].
 * It shares nothing with paper_2606_18900_b200/csrc.  Pinned word for word against the pure-Python encoder of
 * tests/acx_build.py and against the oracle's own decoder (tests/test_oracle_rans.py). */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

#define PB 11u

/* Encodes one row.  out must hold 256 + 2 * n bytes.  Returns the encoded size in bytes (256 + 2 * words), or 0 when a
 * symbol has frequency 0. */
static uint64_t encode_row(const uint8_t* in, uint64_t n, const uint16_t* freq, const uint32_t* cum, uint8_t* out, uint16_t* tmp) {
    uint32_t x[32]; uint64_t cnt[32];
    uint64_t per = (n + 31) / 32;                       /* a state emits at most one word per symbol */
    for (int k = 0; k < 32; k++) { x[k] = 1u << 16; cnt[k] = 0; }
    for (uint64_t i = n; i-- > 0;) {
        int k = (int)(i & 31);
        uint32_t f = freq[in[i]], c = cum[in[i]];
        if (f == 0) return 0;
        if ((uint64_t)x[k] >= ((uint64_t)f << (32 - PB))) { tmp[k * per + cnt[k]++] = (uint16_t)(x[k] & 0xffff); x[k] >>= 16; }
        x[k] = ((x[k] / f) << PB) + (x[k] % f) + c;
    }
    uint64_t off = 0;
    for (int k = 0; k < 32; k++) {
        uint32_t h[2] = {x[k], (uint32_t)off};
        memcpy(out + 8 * k, h, 8);
        for (uint64_t j = 0; j < cnt[k]; j++) {         /* the words, reversed: the order the decoder consumes them in */
            uint16_t w = tmp[k * per + cnt[k] - 1 - j];
            memcpy(out + 256 + 2 * (off + j), &w, 2);
        }
        off += cnt[k];
    }
    return 256 + 2 * off;
}

/* freq: 256 frequencies summing to 2^11.  out: n_rows x row_cap bytes (row_cap >= 256 + 2 * row_bytes); row_sizes[r] = encoded
 * bytes of row r.  Returns 0, or -1 on a bad argument / a symbol without frequency. */
int acx_rows_encode(const uint8_t* in, uint64_t n_rows, uint64_t row_bytes, const uint16_t* freq, uint8_t* out, uint64_t row_cap, uint32_t* row_sizes) {
    uint32_t cum[257]; cum[0] = 0;
    for (int s = 0; s < 256; s++) cum[s + 1] = cum[s] + freq[s];
    if (cum[256] != (1u << PB) || row_cap < 256 + 2 * row_bytes) return -1;
    uint16_t* tmp = malloc(2 * 32 * ((row_bytes + 31) / 32 + 1));
    if (!tmp) return -1;
    for (uint64_t r = 0; r < n_rows; r++) {
        uint64_t sz = encode_row(in + r * row_bytes, row_bytes, freq, cum, out + r * row_cap, tmp);
        if (!sz) { free(tmp); return -1; }
        row_sizes[r] = (uint32_t)sz;
    }
    free(tmp);
    return 0;
}

/* The decoder of FORMAT.md 1.7 for one table, row by row.  Returns 0, -1 on a bad table, -2 when a row does not end with
 * every state at 2^16 and every stream consumed exactly (row_sizes gives the encoded sizes). */
int acx_rows_decode(const uint8_t* enc, uint64_t n_rows, uint64_t row_bytes, uint64_t row_cap, const uint32_t* row_sizes, const uint16_t* freq, uint8_t* out) {
    uint32_t cum[257]; uint8_t slot2sym[1u << PB]; cum[0] = 0;
    for (int s = 0; s < 256; s++) { cum[s + 1] = cum[s] + freq[s]; for (uint32_t k = cum[s]; k < cum[s + 1] && k < (1u << PB); k++) slot2sym[k] = (uint8_t)s; }
    if (cum[256] != (1u << PB)) return -1;
    for (uint64_t r = 0; r < n_rows; r++) {
        const uint8_t* p = enc + r * row_cap;
        uint32_t x[32]; uint64_t pos[32], end[32];
        uint64_t n_words = (row_sizes[r] - 256) / 2;
        for (int k = 0; k < 32; k++) { uint32_t h[2]; memcpy(h, p + 8 * k, 8); x[k] = h[0]; pos[k] = h[1]; }
        for (int k = 0; k < 32; k++) end[k] = k < 31 ? pos[k + 1] : n_words;
        for (uint64_t i = 0; i < row_bytes; i++) {
            int k = (int)(i & 31);
            uint32_t slot = x[k] & ((1u << PB) - 1), s = slot2sym[slot];
            x[k] = freq[s] * (x[k] >> PB) + slot - cum[s];
            if (x[k] < (1u << 16)) { uint16_t w; if (pos[k] >= end[k]) return -2; memcpy(&w, p + 256 + 2 * pos[k], 2); pos[k]++; x[k] = (x[k] << 16) | w; }
            out[r * row_bytes + i] = (uint8_t)s;
        }
        for (int k = 0; k < 32; k++) if (x[k] != (1u << 16) || pos[k] != end[k]) return -2;
    }
    return 0;
}
