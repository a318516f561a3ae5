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

constexpr uint32_t MQ_BITS = 12;
constexpr uint32_t MAX_SEG_CMDS = 510, MAX_SEG_LITS = 16384;     // FORMAT.md §1.5
constexpr uint64_t TAIL_PAD = 128;

struct Opts {
    uint32_t log2_bs, min_match, max_level, threads;
    uint64_t src_window;
    uint32_t chunk_log2, batch_chunks, chain_depth, hash_log2, with_fnv, log2_seg, q_min, q_mode;
};

struct Cmd { uint32_t lit_len, match_len; uint64_t off; };       // match_len 0: no match

struct Block {
    std::vector<Cmd> cmds;
    std::vector<uint8_t> lit;                                     // the literal runs back to back
    uint16_t level = 0;
    uint64_t match_bytes = 0;
};

// a segment: commands [c0, c1) of its block after cutting (FORMAT.md §1.5)
struct Seg {
    uint64_t block, out_start;
    std::vector<Cmd> cmds;
    std::vector<uint8_t> lit_a, lit_q;
    std::vector<uint16_t> q_sym;                                  // pair mode: LITQ symbols v0 | v1 << 8 (lit_q is released once they exist)
    uint32_t n_lit_q = 0, n_sym_q = 0;                            // LITQ bytes / LITQ symbols of the segment
    std::vector<uint32_t> q_edge;                                 // pair mode: indices into q_sym of the pairs with a filler half
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
    // lit_start: start of the pending literal run of the command this match would close
    bool evaluate(uint64_t p, uint64_t i, uint64_t bstart, uint64_t bend, uint64_t cs, uint64_t batch_start, uint64_t lit_start, Cand& c) const {
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
        // FORMAT.md §3 (c): the seed of a self-overlapping match is the tail of its own literal run (and short enough to stay
        // in one piece when the run is cut at a segment boundary)
        if (p + l > i && (p < lit_start || i - p > 4096)) l = i - p;
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
            auto put_lit = [&](uint64_t n) { B.lit.insert(B.lit.end(), x + lit_start, x + lit_start + n); };
            while (i < bend) {
                Cand best{0, 0, 0, 0}; bool have = false;
                auto consider = [&](uint64_t p) {
                    Cand c;
                    if (!evaluate(p, i, bstart, bend, cs, batch_start, lit_start, c)) return;
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
                       !(len + 1 > i - p) && !(p + len > i)) {   // FORMAT.md §3 (c): an overlapping match keeps its seed inside the
                    // literal run in front of it, so it is never extended backwards, and an extension may not create an overlap
                    // the new seed byte p-1 is a literal byte: allowed by FORMAT.md §3 (a); its block may raise the level
                    i--; p--; len++;
                    if (p / BS != bi) best.lvl = std::max(best.lvl, (uint32_t)level[p / BS]);
                }
                put_lit(i - lit_start);
                B.cmds.push_back(Cmd{(uint32_t)(i - lit_start), (uint32_t)len, p});
                B.match_bytes += len;
                blvl = std::max(blvl, best.lvl);
                clear_lit(i, i + len);
                for (uint64_t k = i + len - best.len; k < i + len; k++) insert(k); // [i, old i) were inserted as literals
                i += len; lit_start = i;
            }
            if (lit_start < bend || B.cmds.empty()) { put_lit(bend - lit_start); B.cmds.push_back(Cmd{(uint32_t)(bend - lit_start), 0, 0}); }
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
struct Table { uint32_t mode = 0; std::vector<uint16_t> freq, cum; };   // cum has one entry more than freq

// counts -> frequencies summing to 2^bits, every present symbol >= 1 (needs at most 2^bits present symbols)
void normalise(const std::vector<uint64_t>& h, uint32_t bits, Table& t) {
    const int64_t m = 1ll << bits;
    const size_t n = h.size();
    uint64_t total = 0;
    for (size_t s = 0; s < n; s++) total += h[s];
    t.freq.assign(n, 0);
    if (total == 0) { t.freq[0] = (uint16_t)m; }
    else {
        int64_t sum = 0;
        for (size_t s = 0; s < n; s++) if (h[s]) {
            uint64_t f = (h[s] * (uint64_t)m + total / 2) / total;
            if (f == 0) f = 1;
            t.freq[s] = (uint16_t)std::min<uint64_t>(f, 65535); sum += (int64_t)t.freq[s];
        }
        // fix the sum on the symbols that lose least: repeatedly adjust the currently largest frequency
        while (sum != m) {
            size_t best = n;
            for (size_t s = 0; s < n; s++) if (t.freq[s] > 1 || (sum < m && t.freq[s] >= 1)) if (best == n || t.freq[s] > t.freq[best]) best = s;
            int64_t d = m - sum;
            int64_t room = d > 0 ? d : -std::min<int64_t>(-d, (int64_t)t.freq[best] - 1);
            t.freq[best] = (uint16_t)(t.freq[best] + room); sum += room;
        }
    }
    t.cum.assign(n + 1, 0);
    for (size_t s = 0; s < n; s++) t.cum[s + 1] = (uint16_t)(t.cum[s] + t.freq[s]);
}

double coded_bits(const std::vector<uint64_t>& h, const Table& t, uint32_t bits) {
    double b = 0;
    for (size_t s = 0; s < h.size(); s++) if (h[s]) b += (double)h[s] * -std::log2(t.freq[s] / (double)(1u << bits));
    return b;
}

struct Out {
    std::vector<uint8_t> b;
    void u16(uint32_t v) { b.push_back((uint8_t)v); b.push_back((uint8_t)(v >> 8)); }
    void u32(uint32_t v) { for (int i = 0; i < 4; i++) b.push_back((uint8_t)(v >> (8 * i))); }
    void u64(uint64_t v) { for (int i = 0; i < 8; i++) b.push_back((uint8_t)(v >> (8 * i))); }
    void pad(size_t a) { while (b.size() % a) b.push_back(0); }
};

struct Sym { uint16_t freq, cum; uint8_t pb; };

// rANS-encode the segment's symbol sequence (FORMAT.md §1.7); returns the 32 initial decoder states and, per state, its
// own word stream in the order the decoder consumes it
void rans_segment(const std::vector<Sym>& sym, uint32_t X[32], std::vector<uint16_t> words[32]) {
    for (int k = 0; k < 32; k++) { X[k] = RANS_L; words[k].clear(); }
    for (size_t i = sym.size(); i-- > 0;) {
        const uint32_t f = sym[i].freq, c = sym[i].cum, pb = sym[i].pb;
        uint32_t& xs = X[i & 31];
        uint32_t xv = xs;
        if ((uint64_t)xv >= ((uint64_t)f << (32 - pb))) { words[i & 31].push_back((uint16_t)(xv & 0xffff)); xv >>= 16; }
        xs = ((xv / f) << pb) + (xv % f) + c;
    }
    for (int k = 0; k < 32; k++) std::reverse(words[k].begin(), words[k].end());
}

// FORMAT.md §1.5: cut the commands of one block into segments.  A command starts only while its segment holds fewer than
// SEG output bytes; at most 510 commands and 16384 literal bytes per segment; a literal run that does not fit is cut (the
// segment ends with a match-less command, the run goes on in the next one).  A self-overlapping match keeps at least
// its period of literal bytes in front of it (FORMAT.md §3 (c)).
void cut_block(const Block& B, uint64_t bi, uint64_t BS, uint64_t SEG, std::vector<Seg>& out) {
    uint64_t pos = bi * BS, lp = 0;
    Seg cur; cur.block = bi; cur.out_start = pos;
    uint64_t seg_lits = 0;
    std::vector<std::pair<uint64_t, uint32_t>> runs;     // (position in B.lit, length) of the literal part of each command of cur
    auto close = [&]() {
        // literal classes are assigned later (they need q_min); keep the raw run list in lit_a for now
        out.push_back(std::move(cur));
        cur = Seg(); cur.block = bi; cur.out_start = pos; seg_lits = 0;
    };
    for (const Cmd& c : B.cmds) {
        if (!cur.cmds.empty() && (pos - cur.out_start >= SEG || cur.cmds.size() == MAX_SEG_CMDS)) close();
        uint64_t R = c.lit_len;
        const uint64_t dst = pos + R;
        const uint64_t period = (c.match_len && c.off + c.match_len > dst) ? dst - c.off : 0;   // self-overlap: keep >= period literals
        while (seg_lits + R > MAX_SEG_LITS) {
            uint64_t t = MAX_SEG_LITS - seg_lits;
            if (R - t < period) t = R > period ? R - period : 0;
            if (t > 0) {
                cur.cmds.push_back(Cmd{(uint32_t)t, 0, 0});
                cur.lit_a.insert(cur.lit_a.end(), B.lit.begin() + lp, B.lit.begin() + lp + t);
                lp += t; pos += t; R -= t;
            }
            close();
        }
        cur.cmds.push_back(Cmd{(uint32_t)R, c.match_len, c.off});
        cur.lit_a.insert(cur.lit_a.end(), B.lit.begin() + lp, B.lit.begin() + lp + R);
        lp += R; pos += R + c.match_len; seg_lits += R;
    }
    if (!cur.cmds.empty()) out.push_back(std::move(cur));
}

} // namespace

extern "C" {

struct acx_enc_opts {
    uint32_t log2_bs, min_match, max_level, threads;
    uint64_t src_window;
    uint32_t chunk_log2, batch_chunks, chain_depth, hash_log2, with_fnv, log2_seg, q_min, q_mode;
};

// q_mode: 0 = LITQ as bytes, 1 = LITQ as aligned pairs (falls back to bytes when the data has more than 4096 distinct
// pairs; the default: pairs halve the decode steps of the long literal runs.  Measured on the 1 GiB FASTQ of configs[1]:
// archive 457.8 MB against 443.4 MB with bytes (ratio 2.346 / 2.422: 12-bit precision over ~1000 distinct pairs), literal
// launch 0.83 ms against 1.00 ms), 2 = whichever is smaller, pairs when they cost at most 2 % more.
// log2_seg 0 = min(log2_bs, 14).  q_min 0 = one literal class.
void acx_enc_default_opts(acx_enc_opts* o) {
    memset(o, 0, sizeof *o);
    o->log2_bs = 14; o->min_match = 4; o->max_level = 2; o->threads = 0; o->src_window = 0;
    o->chunk_log2 = 22; o->batch_chunks = 16; o->chain_depth = 2; o->hash_log2 = 0; o->with_fnv = 1;
    o->log2_seg = 0; o->q_min = 64; o->q_mode = 1;
}

void acx_enc_free(void* p) { free(p); }

// Returns 0 on success; *out is malloc'ed (free with acx_enc_free).
int acx_encode(const uint8_t* in, uint64_t N, const acx_enc_opts* uo, uint8_t** out, uint64_t* out_bytes) {
    Enc e;
    static_assert(sizeof(Opts) == sizeof(acx_enc_opts), "opts");
    memcpy(&e.o, uo, sizeof(Opts));
    Opts& o = e.o;
    if (o.log2_bs < 3 || o.log2_bs > 20 || o.min_match < 4 || o.max_level > 65534) return -1;
    if (o.log2_seg == 0) o.log2_seg = std::min(o.log2_bs, 14u);
    if (o.log2_seg < 3 || o.log2_seg > 14 || o.log2_seg > o.log2_bs || o.q_min == 1 || o.q_mode > 2) return -1;
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
    { std::vector<uint64_t> g; e.litmap.swap(g); }

    // ---- segments (FORMAT.md §1.5): cut block by block, in parallel over groups of blocks, concatenated in block order
    const uint64_t SEG = 1ull << o.log2_seg;
    std::vector<Seg> segs;
    std::vector<uint32_t> first_seg(e.n_blocks + 1, 0);
    {
        const uint64_t G = 256, n_groups = (e.n_blocks + G - 1) / G;
        std::vector<std::vector<Seg>> part(n_groups);
        parallel_for(n_groups, threads, [&](uint64_t g) {
            for (uint64_t bi = g * G; bi < std::min(e.n_blocks, (g + 1) * G); bi++) {
                cut_block(e.blocks[bi], bi, e.BS, SEG, part[g]);
                Block& B = e.blocks[bi];
                std::vector<Cmd>().swap(B.cmds); std::vector<uint8_t>().swap(B.lit);
            }
        });
        uint64_t total = 0;
        for (auto& p : part) total += p.size();
        if (total >= (1ull << 32)) return -3;
        segs.reserve(total);
        for (auto& p : part) { for (auto& s : p) segs.push_back(std::move(s)); std::vector<Seg>().swap(p); }
        uint64_t at = 0;
        for (uint64_t bi = 0; bi < e.n_blocks; bi++) {
            first_seg[bi] = (uint32_t)at;
            while (at < segs.size() && segs[at].block == bi) at++;
        }
        first_seg[e.n_blocks] = (uint32_t)segs.size();
    }
    const uint64_t n_segs = segs.size();

    // ---- literal classes (FORMAT.md §1.6): runs of q_min bytes or more -> LITQ.  cut_block left every run in lit_a.
    const uint32_t q_min = o.q_min;
    parallel_for(n_segs, threads, [&](uint64_t si) {
        Seg& s = segs[si];
        if (q_min == 0) return;
        std::vector<uint8_t> a, q;
        uint64_t lp = 0;
        for (const Cmd& c : s.cmds) {
            std::vector<uint8_t>& dst = c.lit_len >= q_min ? q : a;
            dst.insert(dst.end(), s.lit_a.begin() + lp, s.lit_a.begin() + lp + c.lit_len);
            lp += c.lit_len;
        }
        s.lit_a.swap(a); s.lit_q.swap(q);
    });

    // ---- LITQ model: bytes or aligned pairs (FORMAT.md §1.7)
    // pass 1: histogram of the complete pairs (both halves inside a run) and of the LITQ bytes
    std::vector<uint64_t> pair_h(65536, 0), qbyte_h(256, 0);
    uint64_t tot_litq = 0;
    for (const Seg& s : segs) {
        uint64_t pos = s.out_start, lq = 0;
        for (const Cmd& c : s.cmds) {
            if (q_min && c.lit_len >= q_min) {
                const uint8_t* r = s.lit_q.data() + lq;
                for (uint64_t k = (pos + 1) >> 1; 2 * k + 1 < pos + c.lit_len; k++) pair_h[r[2 * k - pos] | r[2 * k + 1 - pos] << 8]++;
                for (uint32_t i = 0; i < c.lit_len; i++) qbyte_h[r[i]]++;
                lq += c.lit_len; tot_litq += c.lit_len;
            }
            pos += (uint64_t)c.lit_len + c.match_len;
        }
    }
    // pass 2: a pair with one half outside its run gets the filler that makes it the most frequent complete pair
    // (ties: the smaller filler); best_lo[v1] = filler for (?, v1), best_hi[v0] = filler for (v0, ?)
    uint32_t q_mode = (q_min && tot_litq) ? o.q_mode : 0;
    std::vector<uint16_t> qpair_of;            // table order: sorted pair values
    Table TQ;                                   // over qpair_of
    std::vector<uint32_t> qindex(65536, 0);
    std::vector<uint64_t> qh;
    if (q_mode >= 1) {
        uint8_t best_lo[256], best_hi[256];
        for (int v = 0; v < 256; v++) {
            int bl = 0, bh = 0;
            for (int f = 1; f < 256; f++) { if (pair_h[f | v << 8] > pair_h[bl | v << 8]) bl = f; if (pair_h[v | f << 8] > pair_h[v | bh << 8]) bh = f; }
            best_lo[v] = (uint8_t)bl; best_hi[v] = (uint8_t)bh;
        }
        std::vector<uint64_t> edge_h(65536, 0);
        for (const Seg& s : segs) {
            uint64_t pos = s.out_start, lq = 0;
            for (const Cmd& c : s.cmds) {
                if (c.lit_len >= q_min) {
                    const uint8_t* r = s.lit_q.data() + lq;
                    if (pos & 1) edge_h[best_lo[r[0]] | r[0] << 8]++;
                    if ((pos + c.lit_len) & 1) { uint8_t v0 = r[c.lit_len - 1]; if (!(c.lit_len == 1 && (pos & 1))) edge_h[v0 | best_hi[v0] << 8]++; }
                    lq += c.lit_len;
                }
                pos += (uint64_t)c.lit_len + c.match_len;
            }
        }
        uint64_t distinct = 0;
        for (uint32_t v = 0; v < 65536; v++) { pair_h[v] += edge_h[v]; distinct += pair_h[v] != 0; }
        if (distinct > 4096 || distinct == 0) q_mode = 0;
        else {
            for (uint32_t v = 0; v < 65536; v++) if (pair_h[v]) { qindex[v] = (uint32_t)qpair_of.size(); qpair_of.push_back((uint16_t)v); qh.push_back(pair_h[v]); }
            normalise(qh, MQ_BITS, TQ);
            if (q_mode == 2) {                  // smaller of the two, pairs preferred within 2 %
                Table tb; std::vector<uint64_t> hb(qbyte_h.begin(), qbyte_h.end());
                normalise(hb, PROB_BITS, tb);
                q_mode = coded_bits(qh, TQ, MQ_BITS) <= 1.02 * coded_bits(hb, tb, PROB_BITS) ? 1 : 0;
            }
        }
        // pass 3: the LITQ symbols of every segment
        if (q_mode == 1) parallel_for(n_segs, threads, [&](uint64_t si) {
            Seg& s = segs[si];
            uint64_t pos = s.out_start, lq = 0;
            for (const Cmd& c : s.cmds) {
                if (c.lit_len >= q_min) {
                    const uint8_t* r = s.lit_q.data() + lq;
                    const uint64_t end = pos + c.lit_len;
                    for (uint64_t k = pos >> 1; k <= (end - 1) >> 1; k++) {
                        const bool in0 = 2 * k >= pos, in1 = 2 * k + 1 < end;
                        uint8_t v0 = in0 ? r[2 * k - pos] : 0, v1 = in1 ? r[2 * k + 1 - pos] : 0;
                        if (!in0) v0 = best_lo[v1];
                        if (!in1) v1 = best_hi[v0];
                        s.q_sym.push_back((uint16_t)(v0 | v1 << 8));
                    }
                    lq += c.lit_len;
                }
                pos += (uint64_t)c.lit_len + c.match_len;
            }
            s.n_lit_q = (uint32_t)s.lit_q.size(); s.n_sym_q = (uint32_t)s.q_sym.size();
            std::vector<uint8_t>().swap(s.lit_q);           // 50 GiB inputs: the literals are held once, not twice
        });
    }
    if (q_mode == 0) for (Seg& s : segs) s.n_lit_q = s.n_sym_q = (uint32_t)s.lit_q.size();

    // ---- histograms and byte tables
    const uint32_t n_tables = 4 + W;
    std::vector<std::vector<uint64_t>> H(n_tables, std::vector<uint64_t>(256, 0));
    uint64_t tot_lit = 0, tot_mb = 0, tot_m = 0, tot_c = 0; uint32_t max_level = 0, max_cmds = 0;
    for (const Seg& s : segs) {
        for (const Cmd& c : s.cmds) {
            H[0][std::min<uint32_t>(c.lit_len, 255)]++;
            if (c.match_len) {
                H[1][std::min<uint32_t>(c.match_len - o.min_match, 255)]++;
                for (uint32_t p = 0; p < W; p++) H[2 + p][(c.off >> (8 * p)) & 0xff]++;
                tot_m++; tot_mb += c.match_len;
            }
        }
        for (uint8_t v : s.lit_a) H[2 + W][v]++;
        if (q_mode == 0) for (uint8_t v : s.lit_q) H[3 + W][v]++;
        tot_lit += s.lit_a.size() + s.n_lit_q; tot_c += s.cmds.size();
        max_cmds = std::max<uint32_t>(max_cmds, (uint32_t)s.cmds.size());
    }
    for (const Block& B : e.blocks) max_level = std::max<uint32_t>(max_level, B.level);
    std::vector<Table> T(n_tables);
    for (uint32_t t = 0; t < n_tables; t++) {
        normalise(H[t], PROB_BITS, T[t]);
        if (t >= 2 && t < 2 + W) { // raw if coding would save < 3 %
            uint64_t n = 0;
            for (int s = 0; s < 256; s++) n += H[t][s];
            if (n && coded_bits(H[t], T[t], PROB_BITS) > 0.97 * 8.0 * (double)n) { T[t].mode = 1; T[t].freq.assign(256, 0); }
        }
    }
    if (q_min == 0 || q_mode == 1 || tot_litq == 0) { T[3 + W].mode = (q_min == 0 || q_mode == 1) ? 2 : 0; if (T[3 + W].mode == 2) T[3 + W].freq.assign(256, 0); }

    // ---- encode payloads
    std::vector<std::vector<uint8_t>> pay(n_segs);
    std::vector<uint32_t> n_words(n_segs), n_ext(n_segs);
    parallel_for(n_segs, threads, [&](uint64_t si) {
        const Seg& s = segs[si];
        std::vector<Sym> sym;
        std::vector<uint32_t> ext_c, ext_m;
        size_t nm = 0;
        for (const Cmd& c : s.cmds) nm += c.match_len != 0;
        sym.reserve(s.cmds.size() + nm * (1 + W) + s.lit_a.size() + s.n_sym_q);
        auto put = [&](const Table& t, uint32_t v, uint32_t pb) { sym.push_back(Sym{t.freq[v], t.cum[v], (uint8_t)pb}); };
        for (const Cmd& c : s.cmds) { put(T[0], std::min<uint32_t>(c.lit_len, 255), PROB_BITS); if (c.lit_len >= 255) ext_c.push_back(c.lit_len - 255); }
        for (const Cmd& c : s.cmds) if (c.match_len) {
            uint32_t t = c.match_len - o.min_match;
            put(T[1], std::min<uint32_t>(t, 255), PROB_BITS); if (t >= 255) ext_m.push_back(t - 255);
        }
        for (int p = (int)W - 1; p >= 0; p--) if (T[2 + p].mode == 0)
            for (const Cmd& c : s.cmds) if (c.match_len) put(T[2 + p], (uint8_t)(c.off >> (8 * p)), PROB_BITS);
        for (uint8_t v : s.lit_a) put(T[2 + W], v, PROB_BITS);
        if (q_mode == 1) for (uint16_t v : s.q_sym) put(TQ, qindex[v], MQ_BITS);
        else for (uint8_t v : s.lit_q) put(T[3 + W], v, PROB_BITS);
        uint32_t X[32]; std::vector<uint16_t> words[32];
        rans_segment(sym, X, words);
        Out o2;
        uint32_t woff = 0;
        for (int k = 0; k < 32; k++) { o2.u32(X[k]); o2.u32(woff); woff += (uint32_t)words[k].size(); }   // head
        for (int k = 0; k < 32; k++) for (uint16_t w : words[k]) o2.u16(w);
        o2.pad(4);
        for (uint32_t v : ext_c) o2.u32(v);
        for (uint32_t v : ext_m) o2.u32(v);
        for (uint32_t p = 0; p < W; p++) if (T[2 + p].mode == 1) for (const Cmd& c : s.cmds) if (c.match_len) o2.b.push_back((uint8_t)(c.off >> (8 * p)));
        o2.pad(16);
        pay[si].swap(o2.b); n_words[si] = woff; n_ext[si] = (uint32_t)(ext_c.size() + ext_m.size());
    });
    for (uint64_t si = 0; si < n_segs; si++) if (n_words[si] > 65535 || n_ext[si] > 65535) return -4;
    std::vector<uint64_t> fnv(e.n_blocks);
    if (o.with_fnv) parallel_for(e.n_blocks, threads, [&](uint64_t bi) {
        uint64_t h = 0xcbf29ce484222325ull, a = bi * e.BS, b = std::min(N, a + e.BS);
        for (uint64_t q = a; q < b; q++) { h ^= in[q]; h *= 0x100000001b3ull; }
        fnv[bi] = h;
    });
    // ---- layout
    auto al16 = [](uint64_t v) { return (v + 15) & ~15ull; };
    const uint32_t n_qpairs = q_mode == 1 ? (uint32_t)qpair_of.size() : 0;
    uint64_t tables_off = 192, qtab_off = tables_off + 528ull * n_tables, blocktab_off = al16(qtab_off + 4ull * n_qpairs);
    uint64_t dir_off = al16(blocktab_off + 8 * (e.n_blocks + 1)), fnv_off = dir_off + 32 * n_segs;
    uint64_t payload_off = al16(fnv_off + (o.with_fnv ? 8 * e.n_blocks : 0));
    uint64_t total = payload_off;
    for (auto& p : pay) total += p.size();
    total += TAIL_PAD;
    uint8_t* buf = (uint8_t*)calloc(total ? total : 1, 1);
    if (!buf) return -2;
    Out h;
    const uint8_t magic[8] = {0x41, 0x43, 0x58, 0x42, 0x32, 0x30, 0x30, 0x00};
    h.b.insert(h.b.end(), magic, magic + 8);
    h.u32(3); h.u32(192); h.u64(N); h.u64(e.n_blocks); h.u64(n_segs);
    h.u32(o.log2_bs); h.u32(o.min_match); h.u32(W); h.u32(PROB_BITS); h.u32(n_tables); h.u32(max_level); h.u32(max_cmds); h.u32(o.with_fnv ? 1 : 0);
    h.u32(o.log2_seg); h.u32(q_min); h.u32(q_mode); h.u32(n_qpairs);
    h.u64(tables_off); h.u64(qtab_off); h.u64(blocktab_off); h.u64(dir_off); h.u64(o.with_fnv ? fnv_off : 0); h.u64(payload_off); h.u64(total);
    h.u64(tot_lit); h.u64(tot_mb); h.u64(tot_m); h.u64(tot_c); h.u64(tot_litq); h.u64(o.src_window);
    memcpy(buf, h.b.data(), 192);
    for (uint32_t t = 0; t < n_tables; t++) {
        uint8_t* p = buf + tables_off + 528ull * t;
        memcpy(p, &T[t].mode, 4);
        memcpy(p + 16, T[t].freq.data(), 512);
    }
    for (uint32_t i = 0; i < n_qpairs; i++) { uint16_t v[2] = {qpair_of[i], TQ.freq[i]}; memcpy(buf + qtab_off + 4ull * i, v, 4); }
    for (uint64_t bi = 0; bi <= e.n_blocks; bi++) {
        uint8_t* d = buf + blocktab_off + 8 * bi;
        uint16_t lv = bi < e.n_blocks ? e.blocks[bi].level : 0;
        memcpy(d, &first_seg[bi], 4); memcpy(d + 4, &lv, 2);
    }
    uint64_t po = payload_off;
    for (uint64_t si = 0; si < n_segs; si++) {
        const Seg& s = segs[si];
        uint8_t* d = buf + dir_off + 32 * si;
        uint32_t nm = 0;
        for (const Cmd& c : s.cmds) nm += c.match_len != 0;
        uint16_t v16[8] = {(uint16_t)s.cmds.size(), (uint16_t)nm, (uint16_t)s.lit_a.size(), (uint16_t)s.n_lit_q, (uint16_t)s.n_sym_q,
                           (uint16_t)n_words[si], (uint16_t)n_ext[si], e.blocks[s.block].level};
        memcpy(d, &po, 8); memcpy(d + 8, &s.out_start, 8); memcpy(d + 16, v16, 16);
        memcpy(buf + po, pay[si].data(), pay[si].size());
        po += pay[si].size();
    }
    if (o.with_fnv) memcpy(buf + fnv_off, fnv.data(), 8 * e.n_blocks);
    *out = buf; *out_bytes = total;
    return 0;
}

} // extern "C"
