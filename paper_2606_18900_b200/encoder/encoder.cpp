// ACX-B200 archive writer (FORMAT.md).  CPU only; it exists to produce test inputs (BASELINE.json north_star,
// subsystem 1; the paper's encoder: "global match search", absolute offsets, fixed-size blocks, §2).
// It shares no code with the decoders (oracle/, csrc/): decoders are checked against the ORIGINAL bytes.
//
// Levels (FORMAT.md §3): level(B) >= level(S) for every block S that B reads, > when B reads match bytes of S.
// Parse: greedy LZ77 with (a) a global first-occurrence table of 8-byte keys filled batch by batch and (b) per-chunk
// 4-byte hash chains.  A candidate is accepted only if it keeps the FORMAT.md §3 invariant: seed bytes inside the
// current block must be literal bytes, seed bytes that are match bytes of an earlier block S need
// level(S) + 1 <= max_level.  Chunks of a batch are parsed in parallel and see only their own chunk and earlier
// batches, so the archive does not depend on the thread count.
#include <algorithm>
#include <atomic>
#include <cmath>
#include <cstdint>
#include <cstdlib>
#include <cstring>
#include <thread>
#include <vector>

namespace {

constexpr uint32_t PROB_BITS = 11;
constexpr uint32_t M = 1u << PROB_BITS;
constexpr uint32_t RANS_L = 1u << 16;

struct Opts {
    uint32_t log2_bs, min_match, max_level, threads;
    uint64_t src_window;
    uint32_t chunk_log2, batch_chunks, chain_depth, hash_log2, with_fnv, reserved[3];
};

struct Block {
    std::vector<uint8_t> cmd, mlen, lit;
    std::vector<uint64_t> off;
    std::vector<uint32_t> ext_cmd, ext_mlen;
    uint16_t level = 0;
    uint64_t match_bytes = 0;
};

inline uint64_t ld64(const uint8_t* p) { uint64_t v; memcpy(&v, p, 8); return v; }
inline uint32_t ld32(const uint8_t* p) { uint32_t v; memcpy(&v, p, 4); return v; }
inline uint32_t hash4(uint32_t v, int bits) { return (v * 2654435761u) >> (32 - bits); }
constexpr uint64_t GKEY = 16;   // bytes of the global-table key: long enough to be near-unique in DNA (4^16 keys)
inline uint64_t hash16(const uint8_t* p, int bits) {
    uint64_t a = ld64(p) * 0x9E3779B97F4A7C15ull, b = ld64(p + 8) * 0xC2B2AE3D27D4EB4Full;
    return ((a ^ (b >> 29) ^ (b << 35)) * 0x9E3779B97F4A7C15ull) >> (64 - bits);
}

struct Enc {
    const uint8_t* x; uint64_t N; Opts o;
    uint64_t BS, n_blocks;
    std::vector<uint64_t> litmap;            // bit = 1: literal byte
    std::vector<uint16_t> level;
    std::vector<Block> blocks;
    std::vector<std::atomic<uint64_t>> gtab; // first occurrence of a GKEY-byte key, positions of earlier batches only
    int gbits;
    uint32_t cost[256];                      // literal cost in 1/16 bit
    uint32_t match_cost;

    bool is_lit(uint64_t p) const { return (litmap[p >> 6] >> (p & 63)) & 1; }
    // first non-literal position in [a, b), or b
    uint64_t first_nonlit(uint64_t a, uint64_t b) const {
        while (a < b) {
            uint64_t w = ~litmap[a >> 6] >> (a & 63);
            if (w) { uint64_t q = a + (uint64_t)__builtin_ctzll(w); return q < b ? q : b; }
            a = (a | 63) + 1;
        }
        return b;
    }
    void clear_lit(uint64_t a, uint64_t b) { // caller owns [a, b) (its own block), word-sharing handled by chunk alignment
        for (uint64_t p = a; p < b;) {
            uint64_t w = p >> 6, lo = p & 63, n = std::min<uint64_t>(64 - lo, b - p);
            uint64_t mask = (n == 64 ? ~0ull : ((1ull << n) - 1)) << lo;
            litmap[w] &= ~mask;
            p += n;
        }
    }

    struct Cand { uint64_t p; uint32_t len; uint32_t lvl; int64_t gain; };

    // Longest valid match of source p for destination i (dst limited to bend); returns false if unusable.
    bool evaluate(uint64_t p, uint64_t i, uint64_t bstart, uint64_t bend, uint64_t cs, uint64_t batch_start, Cand& c) const {
        if (p >= i) return false;
        if (i + 4 <= N && ld32(x + p) != ld32(x + i)) return false;   // hash collision
        if (o.src_window && i - p > o.src_window) return false;
        uint64_t maxlen = bend - i, l = 0;
        // sources may only touch [0, batch_start) and [cs, i): other chunks of this batch are being parsed concurrently
        if (p < batch_start && cs > batch_start) maxlen = std::min(maxlen, batch_start - p);
        while (l + 8 <= maxlen && i + l + 8 <= N) {
            uint64_t d = ld64(x + p + l) ^ ld64(x + i + l);
            if (d) { l += (uint64_t)__builtin_ctzll(d) >> 3; goto done; }
            l += 8;
        }
        while (l < maxlen && x[p + l] == x[i + l]) l++;
    done:
        if (l < o.min_match) return false;
        if (p + l > i && p < bstart) l = i - p;                 // FORMAT.md §3 (c): a self-overlapping match starts in its own block
        if (l < o.min_match) return false;
        uint64_t seed_end = std::min(p + l, i);
        uint32_t lvl = 0;
        uint64_t a = p;
        while (a < seed_end) {
            uint64_t S = a / BS, sb_end = std::min(seed_end, (S + 1) * BS);
            uint64_t q = first_nonlit(a, sb_end);
            if (S * BS != bstart) lvl = std::max(lvl, (uint32_t)level[S]);   // literal bytes of S: level(B) >= level(S)
            if (q < sb_end) {
                bool ok = (S * BS != bstart) && (uint32_t)level[S] + 1 <= o.max_level;
                if (!ok) { seed_end = q; l = q - p; break; } // cut the match in front of the offending byte
                lvl = std::max(lvl, (uint32_t)level[S] + 1);                 // match bytes of S: level(B) > level(S)
            }
            a = sb_end;
        }
        if (l < o.min_match) return false;
        int64_t g = -(int64_t)match_cost;
        for (uint64_t k = 0; k < l; k++) g += cost[x[i + k]];
        g -= (int64_t)lvl * 8 * 16;   // prefer shallow sources: 8 bits per level
        c.p = p; c.len = (uint32_t)l; c.lvl = lvl; c.gain = g;
        return true;
    }

    void parse_chunk(uint64_t cs, uint64_t ce, uint64_t batch_start) {
        const int LB = 20;
        std::vector<uint32_t> head(1u << LB, 0xffffffffu), first(1u << LB, 0xffffffffu), prev(ce - cs);
        auto insert = [&](uint64_t i) {
            if (i + 4 > N) return;
            uint32_t h = hash4(ld32(x + i), LB), r = (uint32_t)(i - cs);
            prev[r] = head[h]; head[h] = r;
            if (first[h] == 0xffffffffu) first[h] = r;
        };
        for (uint64_t bstart = cs; bstart < ce; bstart += BS) {
            uint64_t bend = std::min(bstart + BS, N), bi = bstart / BS;
            Block& B = blocks[bi];
            uint64_t i = bstart, lit_start = bstart;
            uint32_t blvl = 0;
            auto put_lit_token = [&](uint64_t n) {
                if (n < 255) B.cmd.push_back((uint8_t)n); else { B.cmd.push_back(255); B.ext_cmd.push_back((uint32_t)(n - 255)); }
                B.lit.insert(B.lit.end(), x + lit_start, x + lit_start + n);
            };
            while (i < bend) {
                Cand best{0, 0, 0, 0}; bool have = false;
                auto consider = [&](uint64_t p) {
                    Cand c;
                    if (!evaluate(p, i, bstart, bend, cs, batch_start, c)) return;
                    if (c.gain <= 0) return;
                    if (!have || c.gain > best.gain || (c.gain == best.gain && (c.lvl < best.lvl || (c.lvl == best.lvl && c.p < best.p)))) { best = c; have = true; }
                };
                if (i + GKEY <= N && batch_start > 0) {
                    uint64_t p = gtab[hash16(x + i, gbits)].load(std::memory_order_relaxed);
                    if (p != ~0ull && p < batch_start) consider(p);
                }
                if (i + 4 <= N) {
                    uint32_t h = hash4(ld32(x + i), LB);
                    if (first[h] != 0xffffffffu) consider(cs + first[h]);
                    uint32_t r = head[h];
                    for (uint32_t d = 0; d < o.chain_depth && r != 0xffffffffu; d++) { consider(cs + r); r = prev[r]; }
                }
                if (!have) { // no match: step faster through incompressible stretches (back-extension recovers match starts)
                    uint64_t step = 1 + (std::min<uint64_t>(i - lit_start, 1024) >> 6);
                    for (uint64_t k = 0; k < step && i < bend; k++) { insert(i); i++; }
                    continue;
                }
                // extend backwards over pending literals while the source byte is a literal byte
                uint64_t p = best.p, len = best.len;
                while (i > lit_start && p > 0 && x[i - 1] == x[p - 1] && (p - 1 >= cs || p - 1 < batch_start) && is_lit(p - 1) &&
                       !(len + 1 > i - p && p - 1 < bstart)) {   // FORMAT.md §3 (c): the extended match (len + 1, same period) would
                    // overlap itself with its source starting outside the block
                    // the new seed byte p-1 is a literal byte: allowed by FORMAT.md §3 (a); its block may raise the level
                    i--; p--; len++;
                    if (p / BS != bi) best.lvl = std::max(best.lvl, (uint32_t)level[p / BS]);
                }
                put_lit_token(i - lit_start);
                uint64_t t = len - o.min_match;
                if (t < 255) B.mlen.push_back((uint8_t)t); else { B.mlen.push_back(255); B.ext_mlen.push_back((uint32_t)(t - 255)); }
                B.off.push_back(p);
                B.match_bytes += len;
                blvl = std::max(blvl, best.lvl);
                clear_lit(i, i + len);
                for (uint64_t k = i + len - best.len; k < i + len; k++) insert(k); // [i, old i) were inserted as literals
                i += len; lit_start = i;
            }
            if (lit_start < bend || B.cmd.empty()) put_lit_token(bend - lit_start);
            B.level = (uint16_t)blvl;
            level[bi] = (uint16_t)blvl;
        }
    }

    void insert_global(uint64_t a, uint64_t b) { // positions [a, b) whose key is made of literal bytes only
        for (uint64_t p = a; p < b && p + GKEY <= N; p++) {
            uint64_t q = first_nonlit(p, p + GKEY);
            if (q != p + GKEY) { p = q; continue; }   // no key starting in [p, q] is all-literal
            std::atomic<uint64_t>& s = gtab[hash16(x + p, gbits)];
            uint64_t cur = s.load(std::memory_order_relaxed);
            while (p < cur && !s.compare_exchange_weak(cur, p, std::memory_order_relaxed)) {}
        }
    }
};

template <class F> void parallel_for(uint64_t n, uint32_t threads, F f) {
    if (threads <= 1 || n <= 1) { for (uint64_t i = 0; i < n; i++) f(i); return; }
    std::atomic<uint64_t> next{0};
    std::vector<std::thread> th;
    for (uint32_t t = 0; t < std::min<uint64_t>(threads, n); t++)
        th.emplace_back([&] { for (;;) { uint64_t i = next.fetch_add(1); if (i >= n) break; f(i); } });
    for (auto& t : th) t.join();
}

// ---- static tables --------------------------------------------------------------------------------------------
struct Table { uint32_t mode = 0; uint16_t freq[256] = {0}; uint16_t cum[257] = {0}; };

void normalise(const uint64_t* h, Table& t) {
    uint64_t total = 0; int present = 0, top = 0;
    for (int s = 0; s < 256; s++) { total += h[s]; if (h[s]) present++; if (h[s] > h[top]) top = s; }
    memset(t.freq, 0, sizeof t.freq);
    if (total == 0) { t.freq[0] = M; }
    else {
        int64_t sum = 0;
        for (int s = 0; s < 256; s++) if (h[s]) {
            uint64_t f = (h[s] * (uint64_t)M + total / 2) / total;
            if (f == 0) f = 1;
            t.freq[s] = (uint16_t)f; sum += (int64_t)f;
        }
        // fix the sum on the symbols that lose least: repeatedly adjust the currently largest frequency
        while (sum != (int64_t)M) {
            int best = -1;
            for (int s = 0; s < 256; s++) if (t.freq[s] > 1 || (sum < (int64_t)M && t.freq[s] >= 1)) if (best < 0 || t.freq[s] > t.freq[best]) best = s;
            int64_t d = (int64_t)M - sum;
            int64_t room = d > 0 ? d : -std::min<int64_t>(-d, (int64_t)t.freq[best] - 1);
            t.freq[best] = (uint16_t)(t.freq[best] + room); sum += room;
        }
    }
    t.cum[0] = 0;
    for (int s = 0; s < 256; s++) t.cum[s + 1] = (uint16_t)(t.cum[s] + t.freq[s]);
}

struct Out {
    std::vector<uint8_t> b;
    void u32(uint32_t v) { for (int i = 0; i < 4; i++) b.push_back((uint8_t)(v >> (8 * i))); }
    void u64(uint64_t v) { for (int i = 0; i < 8; i++) b.push_back((uint8_t)(v >> (8 * i))); }
    void pad(size_t a) { while (b.size() % a) b.push_back(0); }
};

// rANS-encode the block's symbol sequence (FORMAT.md §1.5); returns the 32 initial decoder states and, per state, its
// own word stream in the order the decoder consumes it
void rans_block(const std::vector<uint8_t>& sym, const std::vector<uint8_t>& tid, const std::vector<Table>& T,
                uint32_t X[32], std::vector<uint16_t> words[32]) {
    for (int k = 0; k < 32; k++) { X[k] = RANS_L; words[k].clear(); }
    for (size_t i = sym.size(); i-- > 0;) {
        const Table& t = T[tid[i]];
        uint32_t f = t.freq[sym[i]], c = t.cum[sym[i]];
        uint32_t& xs = X[i & 31];
        uint32_t xv = xs;
        if ((uint64_t)xv >= ((uint64_t)f << (32 - PROB_BITS))) { words[i & 31].push_back((uint16_t)(xv & 0xffff)); xv >>= 16; }
        xs = ((xv / f) << PROB_BITS) + (xv % f) + c;
    }
    for (int k = 0; k < 32; k++) std::reverse(words[k].begin(), words[k].end());
}

} // namespace

extern "C" {

struct acx_enc_opts {
    uint32_t log2_bs, min_match, max_level, threads;
    uint64_t src_window;
    uint32_t chunk_log2, batch_chunks, chain_depth, hash_log2, with_fnv, reserved[3];
};

void acx_enc_default_opts(acx_enc_opts* o) {
    memset(o, 0, sizeof *o);
    o->log2_bs = 14; o->min_match = 4; o->max_level = 3; o->threads = 0; o->src_window = 0;
    o->chunk_log2 = 22; o->batch_chunks = 16; o->chain_depth = 2; o->hash_log2 = 0; o->with_fnv = 1;
}

void acx_enc_free(void* p) { free(p); }

// Returns 0 on success; *out is malloc'ed (free with acx_enc_free).
int acx_encode(const uint8_t* in, uint64_t N, const acx_enc_opts* uo, uint8_t** out, uint64_t* out_bytes) {
    Enc e;
    static_assert(sizeof(Opts) == sizeof(acx_enc_opts), "opts");
    memcpy(&e.o, uo, sizeof(Opts));
    Opts& o = e.o;
    if (o.log2_bs < 3 || o.log2_bs > 20 || o.min_match < 4 || o.max_level > 65534) return -1;
    if (o.chunk_log2 < o.log2_bs) o.chunk_log2 = o.log2_bs;
    if (o.chunk_log2 < 6) o.chunk_log2 = 6; // chunks own whole 64-bit words of the literal bitmap
    if (o.chunk_log2 > 30) return -1;
    if (o.batch_chunks == 0) o.batch_chunks = 1;
    uint32_t threads = o.threads ? o.threads : std::max(1u, std::thread::hardware_concurrency());
    e.x = in; e.N = N; e.BS = 1ull << o.log2_bs; e.n_blocks = (N + e.BS - 1) / e.BS;
    uint32_t W = 4; while (W < 8 && (N >> (8 * W)) > 0 && N != (1ull << (8 * W))) W++;
    e.litmap.assign((N + 63) / 64 + 1, ~0ull);
    e.level.assign(e.n_blocks + 1, 0);
    e.blocks.resize(e.n_blocks);
    int gb = (int)o.hash_log2;
    if (gb == 0) { gb = 16; while (gb < 30 && (1ull << (gb + 1)) < N) gb++; }
    e.gbits = gb;
    { std::vector<std::atomic<uint64_t>> g(1ull << gb); e.gtab.swap(g); }
    parallel_for(threads, threads, [&](uint64_t t) {
        uint64_t n = 1ull << gb, a = n * t / threads, b = n * (t + 1) / threads;
        for (uint64_t i = a; i < b; i++) e.gtab[i].store(~0ull, std::memory_order_relaxed);
    });
    // literal cost model: order-0 entropy of the input (1/16 bit), match cost: offset + tokens
    {
        std::vector<uint64_t> h(256, 0);
        uint64_t step = N > (64ull << 20) ? N / (64ull << 20) : 1;
        uint64_t cnt = 0;
        for (uint64_t i = 0; i < N; i += step) { h[in[i]]++; cnt++; }
        for (int s = 0; s < 256; s++) {
            double pr = (h[s] + 0.5) / (double)(cnt + 128);
            double bits = -std::log2(pr); if (bits > 12) bits = 12;
            e.cost[s] = (uint32_t)(bits * 16 + 0.5);
        }
        double nb = N > 1 ? std::log2((double)N) : 1;
        e.match_cost = (uint32_t)((nb + 14) * 16);
    }
    uint64_t chunk = 1ull << o.chunk_log2, n_chunks = (N + chunk - 1) / chunk;
    for (uint64_t c0 = 0; c0 < n_chunks; c0 += o.batch_chunks) {
        uint64_t c1 = std::min<uint64_t>(n_chunks, c0 + o.batch_chunks), bs = c0 * chunk;
        parallel_for(c1 - c0, threads, [&](uint64_t k) {
            uint64_t cs = (c0 + k) * chunk, ce = std::min(N, cs + chunk);
            e.parse_chunk(cs, ce, bs);
        });
        if (c1 < n_chunks)
            parallel_for(c1 - c0, threads, [&](uint64_t k) {
                uint64_t cs = (c0 + k) * chunk, ce = std::min(N, cs + chunk);
                e.insert_global(cs, ce);
            });
    }
    { std::vector<std::atomic<uint64_t>> g; e.gtab.swap(g); }

    // ---- histograms and tables
    const uint32_t n_tables = 3 + W;
    std::vector<std::vector<uint64_t>> H(n_tables, std::vector<uint64_t>(256, 0));
    uint64_t tot_lit = 0, tot_mb = 0, tot_m = 0, tot_c = 0; uint32_t max_level = 0, max_cmds = 0;
    for (auto& B : e.blocks) {
        for (uint8_t v : B.cmd) H[0][v]++;
        for (uint8_t v : B.mlen) H[1][v]++;
        for (uint64_t v : B.off) for (uint32_t p = 0; p < W; p++) H[2 + p][(v >> (8 * p)) & 0xff]++;
        for (uint8_t v : B.lit) H[2 + W][v]++;
        tot_lit += B.lit.size(); tot_mb += B.match_bytes; tot_m += B.off.size(); tot_c += B.cmd.size();
        max_level = std::max<uint32_t>(max_level, B.level); max_cmds = std::max<uint32_t>(max_cmds, (uint32_t)B.cmd.size());
    }
    std::vector<Table> T(n_tables);
    for (uint32_t t = 0; t < n_tables; t++) {
        normalise(H[t].data(), T[t]);
        if (t >= 2 && t < 2 + W) { // raw if coding would save < 3 %
            double bits = 0; uint64_t n = 0;
            for (int s = 0; s < 256; s++) if (H[t][s]) { bits += (double)H[t][s] * -std::log2(T[t].freq[s] / (double)M); n += H[t][s]; }
            if (n && bits > 0.97 * 8.0 * (double)n) { T[t].mode = 1; memset(T[t].freq, 0, sizeof T[t].freq); }
        }
    }
    // ---- encode payloads
    std::vector<std::vector<uint8_t>> pay(e.n_blocks);
    std::vector<uint32_t> n_words(e.n_blocks);
    std::vector<uint64_t> fnv(e.n_blocks);
    parallel_for(e.n_blocks, threads, [&](uint64_t bi) {
        Block& B = e.blocks[bi];
        std::vector<uint8_t> sym, tid;
        size_t nm = B.off.size();
        sym.reserve(B.cmd.size() + nm * (1 + W) + B.lit.size()); tid.reserve(sym.capacity());
        for (uint8_t v : B.cmd) { sym.push_back(v); tid.push_back(0); }
        for (uint8_t v : B.mlen) { sym.push_back(v); tid.push_back(1); }
        for (int p = (int)W - 1; p >= 0; p--) if (T[2 + p].mode == 0)
            for (uint64_t v : B.off) { sym.push_back((uint8_t)(v >> (8 * p))); tid.push_back((uint8_t)(2 + p)); }
        for (uint8_t v : B.lit) { sym.push_back(v); tid.push_back((uint8_t)(2 + W)); }
        uint32_t X[32]; std::vector<uint16_t> words[32];
        rans_block(sym, tid, T, X, words);
        Out o2;
        uint32_t woff = 0;
        for (int k = 0; k < 32; k++) { o2.u32(X[k]); o2.u32(woff); woff += (uint32_t)words[k].size(); }   // head
        for (int k = 0; k < 32; k++) for (uint16_t w : words[k]) { o2.b.push_back((uint8_t)w); o2.b.push_back((uint8_t)(w >> 8)); }
        o2.pad(4);
        for (uint32_t v : B.ext_cmd) o2.u32(v);
        for (uint32_t v : B.ext_mlen) o2.u32(v);
        for (uint32_t p = 0; p < W; p++) if (T[2 + p].mode == 1) for (uint64_t v : B.off) o2.b.push_back((uint8_t)(v >> (8 * p)));
        o2.pad(16);
        pay[bi].swap(o2.b); n_words[bi] = woff;
        uint64_t h = 0xcbf29ce484222325ull, a = bi * e.BS, b = std::min(N, a + e.BS);
        for (uint64_t q = a; q < b; q++) { h ^= in[q]; h *= 0x100000001b3ull; }
        fnv[bi] = h;
    });
    // ---- layout
    uint64_t tables_off = 160, dir_off = tables_off + 528ull * n_tables, fnv_off = dir_off + 32 * e.n_blocks;
    uint64_t payload_off = fnv_off + (o.with_fnv ? 8 * e.n_blocks : 0);
    payload_off = (payload_off + 15) & ~15ull;
    uint64_t total = payload_off;
    for (auto& p : pay) total += p.size();
    uint8_t* buf = (uint8_t*)calloc(total ? total : 1, 1);
    if (!buf) return -2;
    Out h;
    const uint8_t magic[8] = {0x41, 0x43, 0x58, 0x42, 0x32, 0x30, 0x30, 0x00};
    h.b.insert(h.b.end(), magic, magic + 8);
    h.u32(2); h.u32(160); h.u64(N); h.u64(e.n_blocks); h.u32(o.log2_bs); h.u32(o.min_match); h.u32(W); h.u32(PROB_BITS);
    h.u32(n_tables); h.u32(max_level); h.u32(max_cmds); h.u32(o.with_fnv ? 1 : 0);
    h.u64(tables_off); h.u64(dir_off); h.u64(o.with_fnv ? fnv_off : 0); h.u64(payload_off); h.u64(total);
    h.u64(tot_lit); h.u64(tot_mb); h.u64(tot_m); h.u64(tot_c); h.u64(o.src_window); h.u64(0); h.u64(0);
    memcpy(buf, h.b.data(), 160);
    for (uint32_t t = 0; t < n_tables; t++) {
        uint8_t* p = buf + tables_off + 528ull * t;
        memcpy(p, &T[t].mode, 4);
        memcpy(p + 16, T[t].freq, 512);
    }
    uint64_t po = payload_off;
    for (uint64_t bi = 0; bi < e.n_blocks; bi++) {
        Block& B = e.blocks[bi];
        uint8_t* d = buf + dir_off + 32 * bi;
        uint32_t v32[5] = {(uint32_t)B.cmd.size(), (uint32_t)B.off.size(), (uint32_t)B.lit.size(), n_words[bi],
                           (uint32_t)(B.ext_cmd.size() + B.ext_mlen.size())};
        memcpy(d, &po, 8); memcpy(d + 8, v32, 20); memcpy(d + 28, &B.level, 2);
        if (o.with_fnv) memcpy(buf + fnv_off + 8 * bi, &fnv[bi], 8);
        memcpy(buf + po, pay[bi].data(), pay[bi].size());
        po += pay[bi].size();
    }
    *out = buf; *out_bytes = total;
    return 0;
}

} // extern "C"
