// Decode kernels of the ACX-B200 library (FORMAT.md version 3) for sm_100a.  Included by aceapex.cu only.
//   k_literals   A1 + A2 + A3: rANS decode of a segment's streams, command scan, literal placement
//   k_copy       A4: match resolution from the descriptors k_literals leaves (wait-free per level, or flag-driven)
//   k_fused      the whole wavefront in ONE cooperative launch (literal wave, grid barrier, match waves)
//   k_plan / k_scatter / k_serve / k_rounds / k_seed   A5-A7: demand rounds of range decode and batched reads
//   k_spans      A6: read access by recursion inside one warp
#pragma once
#include "acx_device.cuh"
#include <cooperative_groups.h>

namespace acx {

struct SegCtx {
    uint64_t s, b, sstart, send;    // segment id, its block, absolute byte range
    SegEntry d;
    const uint8_t* payload;
    const uint32_t* ext;            // EXT array
    const uint8_t* raw_planes;      // raw OFF planes, n_match bytes each
    uint32_t n_ext_cmd;             // number of CMD escapes (they come first in EXT)
    // per-warp scratch
    uint8_t *tok_cmd, *tok_mlen, *off_planes, *lit_a, *lit_q;
    uint16_t* side;                 // span service: position of every command's literal run in its stream
    uint8_t* off_scratch;           // the warp's own buffer for the coded offset planes
    uint32_t plane_stride;          // bytes between two coded planes at off_planes
};

__device__ __forceinline__ void report(const Params& P, uint32_t bit) { atomicOr(P.err, bit); }

// Scratch layout per warp: [tok_cmd: 512][tok_mlen: 512][off planes: n_coded x 512][lit_a: 16384 + 64][lit_q: 17536 (bytes, or u16 pairs)]
constexpr uint64_t SCRATCH_LIT_A = MAX_SEG_LITS + 64, SCRATCH_LIT_Q = 2 * (MAX_SEG_LITS / 2 + MAX_SEG_CMDS + 2) + 64, SCRATCH_SIDE = 2 * TOK_STRIDE;
__host__ __device__ inline uint64_t scratch_bytes(uint32_t n_coded_planes) {
    return ((uint64_t)TOK_STRIDE * (2 + n_coded_planes) + SCRATCH_LIT_A + SCRATCH_LIT_Q + SCRATCH_SIDE + 255) & ~255ull;
}
__device__ __forceinline__ void bind_scratch(const Params& P, uint32_t warp_global, SegCtx& c) {
    uint8_t* s = P.scratch + (uint64_t)warp_global * P.scratch_per_warp;
    c.tok_cmd = s; s += TOK_STRIDE;
    c.tok_mlen = s; s += TOK_STRIDE;
    c.off_planes = s; c.off_scratch = s; c.plane_stride = TOK_STRIDE; s += (uint64_t)TOK_STRIDE * P.n_coded_planes;
    c.lit_a = s; s += SCRATCH_LIT_A;
    c.lit_q = s; s += SCRATCH_LIT_Q;
    c.side = reinterpret_cast<uint16_t*>(s);
}

// ---- segment geometry (FORMAT.md §1.4, §1.5) ---------------------------------------------------------------------------
__device__ __forceinline__ uint64_t block_end(const Params& P, uint64_t b) {
    return min((unsigned long long)((b + 1) << P.log2_bs), (unsigned long long)P.N);
}
// end of segment s of block b: the next segment's out_start when it belongs to the same block, else the block end
__device__ __forceinline__ uint64_t seg_end(const Params& P, uint64_t s, uint64_t b) {
    const uint64_t bend = block_end(P, b);
    if (s + 1 < P.n_segs) {
        const uint64_t nx = __ldg(&P.dir[s + 1].out_start);
        if (nx < bend && nx >= (b << P.log2_bs)) return nx;
    }
    return bend;
}
// the segment that holds position pos (pos < N)
__device__ __forceinline__ uint32_t seg_of(const Params& P, uint64_t pos) {
    const uint64_t b = pos >> P.log2_bs;
    uint32_t lo = __ldg(P.first_seg + b), hi = __ldg(P.first_seg + b + 1);
    while (hi - lo > 1) {                       // last segment of the block with out_start <= pos
        const uint32_t mid = (lo + hi) >> 1;
        if (__ldg(&P.dir[mid].out_start) <= pos) lo = mid; else hi = mid;
    }
    return lo;
}

__device__ __forceinline__ bool load_seg(const Params& P, SegCtx& c) {
    const uint4* d4 = reinterpret_cast<const uint4*>(P.dir + c.s);
    const uint4 a = __ldg(d4), q = __ldg(d4 + 1);
    c.d.payload_off = (uint64_t)a.x | ((uint64_t)a.y << 32);
    c.d.out_start = (uint64_t)a.z | ((uint64_t)a.w << 32);
    c.d.n_cmd = (uint16_t)q.x; c.d.n_match = (uint16_t)(q.x >> 16); c.d.n_lit_a = (uint16_t)q.y; c.d.n_lit_q = (uint16_t)(q.y >> 16);
    c.d.n_sym_q = (uint16_t)q.z; c.d.n_words = (uint16_t)(q.z >> 16); c.d.n_ext = (uint16_t)q.w; c.d.level = (uint16_t)(q.w >> 16);
    c.sstart = c.d.out_start;
    c.b = c.sstart >> P.log2_bs;
    c.send = seg_end(P, c.s, c.b);
    c.payload = P.archive + c.d.payload_off;
    const uint64_t rans_bytes = 256 + 2ull * c.d.n_words;
    // the whole payload towards L2 now: a warp that is alone on its SM (a seek, a read) would otherwise meet DRAM latency at
    // every ring refill; in a full launch the lines arrive a little earlier than their first use
    for (uint64_t o = 128ull * lane_id(); o < rans_bytes; o += 4096) asm volatile("prefetch.global.L2 [%0];" ::"l"(c.payload + o));
    c.ext = reinterpret_cast<const uint32_t*>(c.payload + ((rans_bytes + 3) & ~3ull));
    c.raw_planes = reinterpret_cast<const uint8_t*>(c.ext + c.d.n_ext);
    // the host validated the directory at open (counts within FORMAT.md §1.5, payload inside the archive); these are the
    // properties the kernels rely on for memory safety
    const bool ok = c.d.n_cmd >= 1 && c.d.n_cmd <= MAX_SEG_CMDS && c.d.n_match <= c.d.n_cmd && c.sstart < c.send &&
                    (uint32_t)c.d.n_lit_a + c.d.n_lit_q <= MAX_SEG_LITS && c.d.n_sym_q <= MAX_SEG_LITS / 2 + MAX_SEG_CMDS + 1 + (P.q_mode ? 0u : MAX_SEG_LITS);
    if (!ok && lane_id() == 0) report(P, DF_LENGTH);
    return ok;
}

// offset of match j assembled from coded planes (decode order = high plane first) and raw planes (payload)
__device__ __forceinline__ uint64_t match_src(const Params& P, const SegCtx& c, uint32_t j) {
    const uint32_t mc = c.plane_stride;
    const uint8_t* cp = c.off_planes + j;
    const uint8_t* rp = c.raw_planes + j;
    if (P.W <= 4) {                                          // files up to 4 GiB: 32-bit arithmetic
        uint32_t src = 0;
        for (uint32_t k = 0; k < P.n_coded_planes; k++, cp += mc) src |= (uint32_t)*cp << P.coded_shift[k];
        for (uint32_t r = 0; r < P.n_raw_planes; r++, rp += c.d.n_match) src |= (uint32_t)__ldg(rp) << P.raw_shift[r];
        return src;
    }
    uint64_t src = 0;
    for (uint32_t k = 0; k < P.n_coded_planes; k++, cp += mc) src |= (uint64_t)*cp << P.coded_shift[k];
    for (uint32_t r = 0; r < P.n_raw_planes; r++, rp += c.d.n_match) src |= (uint64_t)__ldg(rp) << P.raw_shift[r];
    return src;
}

// A1 for the literal launch: the CMD, MLEN and coded OFF streams and LITA.  Tokens go to the warp's scratch, the coded planes
// straight to the workspace of the match launch, LITA to c.lit_a.  ONE instance of the byte decode loop serves all of them
// (instruction fetch).  Leaves the rANS state at the first LITQ symbol (global symbol index *i_next).
__device__ __forceinline__ void parse_streams(const Params& P, uint32_t s_luts, uint32_t ring, SegCtx& c, Rans& r, uint32_t* i_next) {
    c.off_planes = P.cplanes + (uint64_t)P.n_coded_planes * __ldg(P.match_prefix + c.s);
    c.plane_stride = c.d.n_match;
    r.init(c.payload, c.d.n_words, ring);
    uint32_t i0 = 0;
    const uint32_t n_reg = 3 + P.n_coded_planes;
#pragma unroll 1
    for (uint32_t k = 0; k < n_reg; k++) {
        uint32_t lut, cnt; uint8_t* dst;
        if (k == 0) { lut = P.lut_cmd; cnt = c.d.n_cmd; dst = c.tok_cmd; }
        else if (k == 1) { lut = P.lut_mlen; cnt = c.d.n_match; dst = c.tok_mlen; }
        else if (k + 1 < n_reg) { lut = P.coded_lut[k - 2]; cnt = c.d.n_match; dst = c.off_planes + (k - 2) * c.d.n_match; }
        else { lut = P.lut_lita; cnt = c.d.n_lit_a; dst = c.lit_a; }
        const uint32_t esc = rans_region<false>(r, s_luts + lut * (4 * LUT_SIZE), i0, cnt, dst);
        if (k == 0) c.n_ext_cmd = esc;
        i0 += cnt;
    }
    __syncwarp();
    *i_next = i0;
}

// FORMAT.md §1.7 integrity check once every symbol of the segment has been decoded
__device__ __forceinline__ bool rans_final_ok(const Params& P, const Rans& r) {
    const bool bad = !r.finished();
    if (__any_sync(0xffffffffu, bad)) { if (lane_id() == 0) report(P, DF_RANS); return false; }
    return true;
}

// ---- A2: the command scan -------------------------------------------------------------------------------------------
// 32 commands per step, one per lane: token -> lengths (escapes through ballot ranks into EXT), then two warp prefix sums:
// one over the packed literal counts (LITA bytes in the low half, LITQ symbols in the high half) and one over the output.
struct ScanState { uint32_t lit_base, out_base, ec, em; };      // lit_base: LITA bytes | LITQ symbols << 16
struct CmdLane {
    bool valid, has_match, is_q;
    uint32_t lit_len, match_len;
    uint32_t out_rel;        // segment-relative position of the command's literal run
    uint32_t lit_pos;        // position of the run in its own stream (LITA byte index / LITQ symbol index)
    uint32_t q_syms;         // LITQ symbols of the run (0 for a LITA run)
};
__device__ __forceinline__ void scan_init(ScanState& st, const SegCtx& c) { st.lit_base = 0; st.out_base = 0; st.ec = 0; st.em = c.n_ext_cmd; }

// the tokens of the group of 32 commands that starts at c0 (written by this warp earlier in the kernel: plain loads)
__device__ __forceinline__ uint2 load_tokens(const SegCtx& c, uint32_t c0) {
    const uint32_t ci = c0 + lane_id();
    return make_uint2(ci < c.d.n_cmd ? c.tok_cmd[ci] : 0u, ci < c.d.n_match ? c.tok_mlen[ci] : 0u);
}

__device__ __forceinline__ CmdLane scan_step(const Params& P, const SegCtx& c, ScanState& st, uint32_t c0, uint2 tok) {
    const uint32_t lane = lane_id(), ci = c0 + lane;
    CmdLane L;
    L.valid = ci < c.d.n_cmd; L.has_match = ci < c.d.n_match;
    const uint32_t tl = tok.x, tm = tok.y;
    const uint32_t ml = __ballot_sync(0xffffffffu, L.valid && tl == 255), mm = __ballot_sync(0xffffffffu, L.has_match && tm == 255);
    L.lit_len = tl; L.match_len = L.has_match ? P.min_match + tm : 0;
    if (L.valid && tl == 255) { const uint32_t k = st.ec + __popc(ml & lanemask_lt()); L.lit_len = k < c.d.n_ext ? 255 + __ldg(c.ext + k) : 0xffffffu; }
    if (L.has_match && tm == 255) { const uint32_t k = st.em + __popc(mm & lanemask_lt()); L.match_len = k < c.d.n_ext ? P.min_match + 255 + __ldg(c.ext + k) : 0xffffffu; }
    st.ec += __popc(ml); st.em += __popc(mm);
    L.lit_len = min(L.lit_len, 0xffffffu); L.match_len = min(L.match_len, 0xffffffu);      // sums stay far below 2^32
    uint32_t so = L.lit_len + L.match_len;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, so, o); if (lane >= (uint32_t)o) so += t; }
    L.out_rel = st.out_base + so - L.lit_len - L.match_len;
    st.out_base += __shfl_sync(0xffffffffu, so, 31);
    L.is_q = L.valid && P.q_min && L.lit_len >= P.q_min;
    L.q_syms = 0;
    if (L.is_q) {
        const uint64_t d = c.sstart + L.out_rel;
        L.q_syms = P.q_mode ? (uint32_t)(((d + L.lit_len - 1) >> 1) - (d >> 1) + 1) : L.lit_len;
    }
    // a command whose literals cannot fit a segment fails the validation of every caller; clamp so that the packed sums hold
    const uint32_t la = (L.valid && !L.is_q) ? min(L.lit_len, 0x7fffu) : 0u, lq = min(L.q_syms, 0x7fffu);
    uint32_t sl = la | lq << 16;
#pragma unroll
    for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, sl, o); if (lane >= (uint32_t)o) sl += t; }
    const uint32_t mine = st.lit_base + sl - (la | lq << 16);
    L.lit_pos = L.is_q ? mine >> 16 : mine & 0xffffu;
    st.lit_base += __shfl_sync(0xffffffffu, sl, 31);
    return L;
}
// per-command validation shared by every walker: the run and the match stay inside the segment, the command starts below SEG
__device__ __forceinline__ bool cmd_ok(const Params& P, const SegCtx& c, const CmdLane& L) {
    return !L.valid || ((uint64_t)L.out_rel + L.lit_len + L.match_len <= c.send - c.sstart && L.out_rel < (1u << P.log2_seg) &&
                        (L.is_q ? L.lit_pos + L.q_syms <= c.d.n_sym_q : L.lit_pos + L.lit_len <= c.d.n_lit_a));
}
__device__ __forceinline__ bool scan_totals_ok(const SegCtx& c, const ScanState& st) {
    return (st.lit_base & 0xffffu) == c.d.n_lit_a && (st.lit_base >> 16) == c.d.n_sym_q && c.sstart + st.out_base == c.send;
}

// ---- A2 + A3 fused into the literal decode ("direct placement") --------------------------------------------------
// The command scan runs after LITA has been decoded (into the warp's staging area in shared memory when it fits, else into
// its scratch in global memory) and before LITQ is decoded:
//  * LITA runs are short and many (bases between matches, header digits: 207 runs of 4.7 bytes per 16 KB of FASTQ): the lane
//    that owns the command copies its run to the output (8-byte loads, byte stores: the runs start anywhere);
//  * LITQ runs are long (quality strings): the scan leaves one entry per run in the warp's run table in shared memory,
//    (last symbol index of the run) | (delta + bias) << 16, and the LITQ decode stores every symbol straight to its final
//    position: while a 32-symbol round stays inside one run that is a pointer bump; a round that crosses run boundaries
//    walks the table (one broadcast read per boundary);
//  * the match descriptors (dst_rel, len) go to the workspace for k_copy.
// In pair mode a LITQ symbol is always stored as a whole aligned pair: inside a segment a literal run has a match (or the
// segment's edge) on either side (a command is a run followed by its match, FORMAT.md §1.6), so the filler half of a run's
// first / last pair lands on a match byte, which k_copy writes later.  Only symbol 0 and the last symbol can reach outside
// the segment; q_edge says whether they do.
constexpr uint32_t QDELTA_BIAS = 1024; // pair mode: delta = (even position of the run's first pair) - 2 * (first symbol) >= -2 * runs

__host__ __device__ inline uint32_t runs_bytes_for(uint32_t q_min) {   // run table of a warp: one entry per LITQ run + sentinel
    const uint32_t n = q_min ? (MAX_SEG_LITS / q_min < MAX_SEG_CMDS ? MAX_SEG_LITS / q_min : MAX_SEG_CMDS) : 0;
    return (4 * (n + 2) + 15) & ~15u;
}

// COLLECT (a window of a range decode whose demands fit the lists in one go): the scan also does the collect pass of the
// window, i.e. appends the unknown seed bytes of every match to the demand lists (defined behind resolve_src)
__device__ __forceinline__ void collect_match(const Params& P, const SegCtx& c, uint64_t src, uint64_t dst, uint32_t len);

template <bool COLLECT>
__device__ __forceinline__ bool build_runs(const Params& P, const SegCtx& c, uint32_t runs /* shared address */, uint8_t* out_seg, uint32_t* q_edge_out) {
    ScanState st; scan_init(st, c);
    const uint32_t alist = runs + P.runs_bytes;                // 32 x 8 bytes behind the run table
    uint32_t n_q = 0, q_bytes = 0, q_edge = 0;
    uint2* const pairs = P.pairs ? P.pairs + __ldg(P.match_prefix + c.s) : nullptr;
    const uint32_t lane = lane_id();
    const uint32_t even0 = (uint32_t)(c.sstart & 1);           // pair addressing is relative to the even position sstart - even0
    const uint32_t slen = (uint32_t)(c.send - c.sstart), q_cap = P.runs_bytes / 4 - 1;
    bool good = true;
    uint2 tok = load_tokens(c, 0);
    for (uint32_t c0 = 0; c0 < c.d.n_cmd; c0 += 32) {
        const uint2 tok_next = load_tokens(c, c0 + 32);        // in flight while this group is scanned
        const CmdLane L = scan_step(P, c, st, c0, tok);
        tok = tok_next;
        const uint32_t mq = __ballot_sync(0xffffffffu, L.is_q);
        good = good && cmd_ok(P, c, L) && n_q + __popc(mq) <= q_cap;
        if (__any_sync(0xffffffffu, !good)) break;
        if (pairs && L.has_match) pairs[c0 + lane] = make_uint2(L.out_rel + L.lit_len, L.match_len);
        if (COLLECT && L.has_match) collect_match(P, c, match_src(P, c, c0 + lane), c.sstart + L.out_rel + L.lit_len, L.match_len);
        const bool a_run = L.valid && !L.is_q && L.lit_len;
        {   // LITA runs of this group: up to eight bytes by the lane that owns the command (two aligned 32-bit loads and a
            // funnel shift per four bytes, byte stores: the runs start anywhere); longer ones by the whole warp, coalesced
            const uint8_t* sa = c.lit_a + L.lit_pos; uint8_t* da = out_seg + L.out_rel;
            const uint32_t n = (a_run && L.lit_len <= 8) ? L.lit_len : 0u;
            if (__any_sync(0xffffffffu, n != 0)) {
                const uint32_t sh = 8u * ((uint32_t)reinterpret_cast<uintptr_t>(sa) & 3u);
                const uint32_t* wa = reinterpret_cast<const uint32_t*>(sa - (sh >> 3));
                if (n) {
                    const uint32_t w0 = wa[0], w1 = (sh + 8 * n > 32) ? wa[1] : 0u, w2 = (sh + 8 * n > 64) ? wa[2] : 0u;
                    const uint32_t v0 = __funnelshift_r(w0, w1, sh), v1 = __funnelshift_r(w1, w2, sh);
                    da[0] = (uint8_t)v0;
                    if (n > 1) da[1] = (uint8_t)(v0 >> 8);
                    if (n > 2) da[2] = (uint8_t)(v0 >> 16);
                    if (n > 3) da[3] = (uint8_t)(v0 >> 24);
                    if (n > 4) da[4] = (uint8_t)v1;
                    if (n > 5) da[5] = (uint8_t)(v1 >> 8);
                    if (n > 6) da[6] = (uint8_t)(v1 >> 16);
                    if (n > 7) da[7] = (uint8_t)(v1 >> 24);
                }
            }
            // runs of 9..63 bytes: compacted into a list in shared memory, then four runs at a time, eight lanes per run
            // (lane sub copies bytes sub, sub + 8, ..): one pass of predicated byte copies serves four runs
            const bool a_mid = a_run && L.lit_len > 8 && L.lit_len < 64;
            const uint32_t m_mid = __ballot_sync(0xffffffffu, a_mid);
            if (m_mid) {
                if (a_mid) sts64(alist + 8 * __popc(m_mid & lanemask_lt()), L.lit_pos | L.lit_len << 16, L.out_rel);
                __syncwarp();
                const uint32_t n_mid = __popc(m_mid), sub = lane & 7u;
                for (uint32_t k = lane >> 3; k < ((n_mid + 3u) & ~3u); k += 4) {
                    uint2 e = make_uint2(0u, 0u);
                    if (k < n_mid) e = lds64(alist + 8 * k);
                    const uint32_t m = e.x >> 16;
                    const uint8_t* sp = c.lit_a + (e.x & 0xffffu) + sub; uint8_t* dp = out_seg + e.y + sub;
                    uint32_t v[4];
#pragma unroll
                    for (int j = 0; j < 4; j++) if (sub + 8 * j < m) v[j] = sp[8 * j];
#pragma unroll
                    for (int j = 0; j < 4; j++) if (sub + 8 * j < m) dp[8 * j] = (uint8_t)v[j];
                    if (__any_sync(0xffffffffu, m > 32)) {
#pragma unroll
                        for (int j = 4; j < 8; j++) if (sub + 8 * j < m) v[j - 4] = sp[8 * j];
#pragma unroll
                        for (int j = 4; j < 8; j++) if (sub + 8 * j < m) dp[8 * j] = (uint8_t)v[j - 4];
                    }
                }
                __syncwarp();                                   // the list is rewritten by the next group
            }
            uint32_t a_long = __ballot_sync(0xffffffffu, a_run && L.lit_len >= 64);      // only archives without a LITQ class have them
            while (a_long) {
                const int l = __ffs(a_long) - 1; a_long &= a_long - 1;
                const uint32_t m = __shfl_sync(0xffffffffu, L.lit_len, l), lp = __shfl_sync(0xffffffffu, L.lit_pos, l), orl = __shfl_sync(0xffffffffu, L.out_rel, l);
                warp_copy<false>(out_seg + orl, c.lit_a + lp, m);
            }
        }
        if (L.is_q) {
            uint32_t e;
            if (P.q_mode) {
                const uint32_t d = L.out_rel + even0;          // position relative to the even base
                e = ((L.lit_pos + L.q_syms - 1) & 0x7fffu) | (((d & ~1u) + QDELTA_BIAS - 2 * L.lit_pos) & 0x7fffu) << 16;
                if (L.out_rel == 0 && even0) q_edge |= 1u;
                if (L.out_rel + L.lit_len == slen && ((d + L.lit_len) & 1u)) q_edge |= 2u;
            } else e = ((L.lit_pos + L.lit_len - 1) & 0x7fffu) | ((L.out_rel - L.lit_pos) & 0x7fffu) << 16;
            sts32(runs + 4 * (n_q + __popc(mq & lanemask_lt())), e);
            q_bytes += L.lit_len;
        }
        n_q += __popc(mq);
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) { q_bytes += __shfl_xor_sync(0xffffffffu, q_bytes, o); q_edge |= __shfl_xor_sync(0xffffffffu, q_edge, o); }
    good = !__any_sync(0xffffffffu, !good) && scan_totals_ok(c, st) && q_bytes == c.d.n_lit_q;
    if (!good) { if (lane == 0) report(P, DF_LENGTH); return false; }
    if (lane == 0) sts32(runs + 4 * n_q, 0x7fffu);             // sentinel
    __syncwarp();
    *q_edge_out = q_edge;
    return true;
}

struct RunCursor {
    uint32_t k;          // shared address of the entry of the run that holds the first symbol of the coming round
    uint32_t last;       // last symbol index of that run
    uint32_t delta;      // out position - symbol position (pair mode: biased, in bytes from the even base)
    __device__ __forceinline__ void load(uint32_t e) { last = e & 0x7fffu; delta = (e >> 16) & 0x7fffu; }
    // A round whose symbols [.., j_hi] are not all strictly inside run k: walk the cursor over the runs that end inside the
    // round (one broadcast table read per boundary; the table ends with a sentinel whose `last` is 0x7fff).  Returns the
    // delta of this lane's symbol j and leaves the cursor on the run of symbol j_hi + 1.
    __device__ __forceinline__ uint32_t walk(uint32_t j, uint32_t j_hi) {
        uint32_t mine = delta;
        while (last <= j_hi) {
            const uint32_t prev = last;
            k += 4; load(lds32(k));
            if (j > prev) mine = delta;
        }
        return mine;
    }
};

// LITQ straight to its positions.  PAIR = false: symbol j of the stream is the byte at zero + j + delta(run of j).
// PAIR = true (FORMAT.md §1.7): symbol j is the aligned pair at zero + 2 j + delta(run of j), stored whole (see above)
// except for the halves of symbol 0 / symbol n - 1 that q_edge says lie outside the segment.  ODD: the output address of an
// even position is odd (a range-decode window placed at an odd address): two byte stores instead of one 16-bit store.
// SIMPLE: every run has at least 32 symbols (q_min >= 64), so a full round holds at most one run boundary.
template <bool PAIR, bool ODD, bool SIMPLE>
__device__ __forceinline__ void decode_q(Rans& r, uint32_t lut, uint32_t i0, uint32_t n, uint32_t runs, uint8_t* zero, uint32_t q_edge) {
    if (n == 0) return;
    constexpr uint32_t S = PAIR ? 2 : 1;
    const uint32_t lane = lane_id(), i1 = i0 + n;
    RunCursor rc; rc.k = runs; rc.load(lds32(runs));
    auto put = [&](uint8_t* p, uint32_t e) {
        if (!PAIR) *p = (uint8_t)e;
        else if (ODD) { p[0] = (uint8_t)e; p[1] = (uint8_t)(e >> 8); }
        else *reinterpret_cast<uint16_t*>(p) = (uint16_t)e;
    };
    // a round that may hold a run boundary, an inactive lane, symbol 0 or the last symbol
    auto careful = [&](uint32_t j, uint32_t j_hi, bool active, uint32_t e) {
        uint8_t* p = zero + S * j + rc.walk(j, j_hi);
        if (!active) return;
        if (PAIR && ((j == 0 && (q_edge & 1u)) || (j == n - 1 && (q_edge & 2u)))) { if (j == 0 && (q_edge & 1u)) p[1] = (uint8_t)(e >> 8); else p[0] = (uint8_t)e; }
        else put(p, e);
    };
    uint32_t base = i0 & ~31u;
    uint8_t* pj = zero + (int64_t)S * ((int64_t)base + lane - i0);      // address of symbol (base + lane - i0) if delta were 0
#pragma unroll 1
    while (base < i1) {
        r.prepare8();
        if (base > i0 && base + 256 < i1) {               // eight full rounds, none of them the first or the last of the stream
            // pd = address of this lane's symbol of round 0 under the current run's delta; lim = symbols of the group's
            // first position up to the run's last one: a round q lies strictly inside the run iff 32 q + 31 < lim
            uint8_t* pd = pj + rc.delta;
            uint32_t lim = rc.last - (base - i0);
#pragma unroll 1
            for (int h = 0; h < 2; h++) {                 // two groups of four (code size)
#pragma unroll
                for (int q = 0; q < 4; q++) {
                    const uint32_t e = PAIR ? r.step_pair_full(lut) : r.step_full(lut);
                    if (32u * q + 31u < lim) put(pd + 32 * S * q, e);        // pointer bump
                    else if (SIMPLE) {                                 // run k ends in this round, run k + 1 goes on beyond it
                        const uint32_t old_delta = rc.delta;
                        rc.k += 4; rc.load(lds32(rc.k));
                        const int32_t dd = (int32_t)(rc.delta - old_delta);
                        put(pd + 32 * S * q + (32u * q + lane > lim ? dd : 0), e);
                        pd += dd; lim = rc.last - (base - i0);
                    } else {
                        const uint32_t old_delta = rc.delta, j_hi = base + 32 * q + 31 - i0;
                        put(pj + 32 * S * q + rc.walk(j_hi - 31 + lane, j_hi), e);
                        pd += (int32_t)(rc.delta - old_delta); lim = rc.last - (base - i0);
                    }
                }
                base += 128; pj += 128 * S; pd += 128 * S; lim -= 128;
            }
        } else {
#pragma unroll 1
            for (int k = 0; k < 8 && base < i1 && !(k && base + 256 < i1); k++, base += 32, pj += 32 * S) {
                const uint32_t i = base + lane;
                const bool active = i >= i0 && i < i1;
                const uint32_t e = PAIR ? r.step_pair(lut, active) : r.step(lut, active);
                careful(i - i0, min(base + 31, i1 - 1) - i0, active, e);
            }
        }
    }
}

// A1 + A2 + A3 for one segment: tokens and LITA, scan (LITA placement, LITQ run table, match descriptors), LITQ straight to
// its positions.  QM: 0 = LITQ bytes, 1 = aligned pairs, 2 = pairs at an odd address.  lita_stage: the warp's staging area
// in shared memory (generic pointer); a segment with more LITA bytes than it holds stages them in the global scratch.
template <int QM, bool COLLECT = false>
__device__ __forceinline__ bool literals_of_segment(const Params& P, uint32_t s_luts, uint32_t s_lutq, uint32_t ring, uint32_t runs, uint8_t* lita_stage, SegCtx& c) {
    if (!load_seg(P, c)) return false;
    uint8_t* const out_seg = P.out + (c.sstart - P.out_pos0);
    uint8_t* const lit_a_scratch = c.lit_a;
    if (c.d.n_lit_a <= P.lita_bytes) c.lit_a = lita_stage;
    Rans r; uint32_t i0, q_edge;
    parse_streams(P, s_luts, ring, c, r, &i0);
    const bool ok = build_runs<COLLECT>(P, c, runs, out_seg, &q_edge);
    c.lit_a = lit_a_scratch;
    if (!ok) return false;
    // QM: 0 / 1 / 2 as above with run tables of any shape; 3 = bytes, 4 = pairs when every LITQ run has 32 symbols or more
    if (QM == 0) decode_q<false, false, false>(r, s_luts + P.lut_litq * (4 * LUT_SIZE), i0, c.d.n_sym_q, runs, out_seg, 0);
    else if (QM == 3) decode_q<false, false, true>(r, s_luts + P.lut_litq * (4 * LUT_SIZE), i0, c.d.n_sym_q, runs, out_seg, 0);
    else if (QM == 4) decode_q<true, false, true>(r, s_lutq, i0, c.d.n_sym_q, runs, out_seg - (c.sstart & 1) - QDELTA_BIAS, q_edge);
    else decode_q<true, QM == 2, false>(r, s_lutq, i0, c.d.n_sym_q, runs, out_seg - (c.sstart & 1) - QDELTA_BIAS, q_edge);
    return rans_final_ok(P, r);
}

// ---- dependency flags ------------------------------------------------------------------------------------------------
// done[S] counts the segments of block S completed by the current flag-driven launch (zeroed before it).
__device__ __forceinline__ void wait_block(const Params& P, uint64_t S) {
    const uint32_t* f = P.done + S;
    const uint32_t want = (__ldg(P.first_seg + S + 1) - __ldg(P.first_seg + S)) * P.copy_parts;   // every share of every segment
    uint32_t spins = 0, ns = 128;
    while (ld_flag(f) < want) {
        __nanosleep(ns);
        if (ns < 2048) ns *= 2;          // back off: thousands of lanes polling one L2 line slow everybody down
        if (++spins > (1u << 21)) { report(P, DF_TIMEOUT); break; }
    }
    // The polls are relaxed loads; one acquire-release fence once the count has been seen orders every later read of the
    // guarded bytes after it (the writer: stores, __threadfence, atomic add).  Once per wait, not per poll.
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
}
__device__ __forceinline__ void publish_segment(const Params& P, uint64_t b) {   // the warp's stores happen-before lane 0's fence + add
    __syncwarp();
    if (lane_id() == 0) { __threadfence(); atomicAdd(P.done + b, 1u); }
}

// ---- demands: where unknown source bytes go ---------------------------------------------------------------------------
// A per-warp LIFO (read access: depth-first recursion by the warp itself) or the global per-source-segment lists of a
// range decode (gl != null).  policy: see fetch_source.
struct Stack { Demand* base; uint32_t cap; uint32_t top; /* shared address of the entry count */ const GList* gl; uint32_t policy; };
enum : uint32_t { SKIP_KNOWN = 1, SKIP_UNKNOWN = 2 };

__device__ __forceinline__ uint32_t lds_top(const Stack& st) { return lds32(st.top); }

constexpr uint32_t GL_SPAN_MAX = 96;     // a record of the global lists covers at most this many bytes (= ITEM_LANE_MAX: one lane serves
                                         // it; a work item of GL_ITEM records is bounded in bytes, not only in records)
// append "original bytes [pos, pos + len) -> out2[dst ..)" (inside segment seg)
__device__ __forceinline__ void gl_append(const Params& P, const GList& gl, uint64_t pos, uint32_t len, uint64_t dst, uint32_t seg) {
    const uint32_t idx = atomicAdd(gl.count, 1u);
    if (idx >= gl.cap) { report(P, DF_STACK); return; }
    GDemand d; d.pos = pos; d.dst = dst; d.len = len; d.seg = seg;
    gl.rec[idx] = d;
    if (atomicAdd(gl.cnt + seg, 1u) == 0) {
        const uint32_t t = atomicAdd(gl.count + 1, 1u);
        if (t < gl.touched_cap) gl.touched[t] = seg; else report(P, DF_STACK);
    }
}

__device__ __forceinline__ void push_span(const Params& P, const Stack& st, uint64_t pos, uint64_t len, uint64_t dst) {
    while (len) {                                   // a demand never crosses a segment boundary
        if (pos >= P.N) { report(P, DF_OFFSET); return; }
        const uint64_t pb = pos >> P.log2_bs;
        uint32_t seg = __ldg(P.first_seg + pb);
        uint64_t send = block_end(P, pb);
        if (__ldg(P.first_seg + pb + 1) - seg > 1) { seg = seg_of(P, pos); send = seg_end(P, seg, pb); }   // several segments in the block
        uint64_t n = min((unsigned long long)len, (unsigned long long)(send - pos));
        if (st.gl) n = min((unsigned long long)n, (unsigned long long)GL_SPAN_MAX);   // work items are sized by record count: bound a record's bytes
        if (st.gl) gl_append(P, *st.gl, pos, (uint32_t)n, dst, seg);
        else {
            uint32_t idx;
            asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(idx) : "r"(st.top) : "memory");
            if (idx < st.cap) { st.base[idx].pos = pos; st.base[idx].dst = dst; __threadfence_block(); st.base[idx].len = n; }   // len last: k_spans_cta polls it
            else report(P, DF_STACK);
        }
        pos += n; dst += n; len -= n;
    }
}

// one out-of-line copy routine for the span-service paths (their code must stay small: the kernels that serve spans were
// bound by instruction fetch, 5.3 stalled warps per issue, when everything was inlined)
__device__ __noinline__ void copy_any(uint8_t* dst, const uint8_t* src, uint32_t len) {
#pragma unroll 1
    for (uint32_t i = 0; i < len; i += 32) {                // sources may have been written by other SMs: ld.cg; four loads in flight
        uint64_t v[4];
#pragma unroll
        for (uint32_t q = 0; q < 4; q++) if (i + 8 * q < len) v[q] = ld64u<true>(src + i + 8 * q, min(len - i - 8 * q, 8u));
#pragma unroll
        for (uint32_t q = 0; q < 4; q++) if (i + 8 * q < len) st_small(dst + i + 8 * q, v[q], min(len - i - 8 * q, 8u));
    }
}

// n contiguous original bytes from absolute position sp -> out2 + dst_off.  Window bytes and resident slots are copied
// (unless policy SKIP_KNOWN), the rest becomes demands (unless policy SKIP_UNKNOWN).
template <bool COPY_INLINE>
__device__ __forceinline__ void fetch_source_body(const Params& P, const Stack& st, uint64_t sp, uint64_t n, uint64_t dst_off) {
    while (n) {
        uint64_t m = n;
        const uint8_t* from = nullptr;
        if (sp >= P.out_pos0 && sp < P.win_end) {
            m = min((unsigned long long)n, (unsigned long long)(P.win_end - sp));
            from = P.out + (sp - P.out_pos0);
        } else {
            uint64_t next = sp < P.out_pos0 && P.out_pos0 < P.win_end ? P.out_pos0 : ~0ull;   // start of the next known region
#pragma unroll
            for (int r = 0; r < MAX_RESIDENT; r++) {
                if (P.res[r].lo >= P.res[r].hi) continue;
                if (sp >= P.res[r].lo && sp < P.res[r].hi) { m = min((unsigned long long)n, (unsigned long long)(P.res[r].hi - sp)); from = P.res[r].ptr + (sp - P.res[r].lo); }
                else if (P.res[r].lo > sp && P.res[r].lo < next) next = P.res[r].lo;
            }
            if (!from) m = min((unsigned long long)n, (unsigned long long)(next - sp));
        }
        if (from) {
            if (!(st.policy & SKIP_KNOWN)) {
                uint8_t* d = P.out2 + dst_off;
                uint64_t left = m; const uint8_t* f = from;
                while (left) { uint32_t k = (uint32_t)min((unsigned long long)left, 1ull << 30); if (COPY_INLINE) copy_bytes<true>(d, f, k); else copy_any(d, f, k); d += k; f += k; left -= k; }
            }
        } else if (!(st.policy & SKIP_UNKNOWN)) push_span(P, st, sp, m, dst_off);
        sp += m; dst_off += m; n -= m;
    }
}

// the match kernels inline it (a call in their inner loop costs more than the code), the span-service kernels call it
__device__ __forceinline__ void fetch_source_inl(const Params& P, const Stack& st, uint64_t sp, uint64_t n, uint64_t dst_off) { fetch_source_body<true>(P, st, sp, n, dst_off); }
__device__ __noinline__ void fetch_source(const Params& P, const Stack st, uint64_t sp, uint64_t n, uint64_t dst_off) { fetch_source_body<false>(P, st, sp, n, dst_off); }

// Where the bytes [src, src + n) live if one known buffer holds them all: the window, or a resident slot (range decode).
// *end = end of that buffer.  Null when they are unknown or spread over several buffers.
__device__ __forceinline__ const uint8_t* resolve_src(const Params& P, uint64_t src, uint64_t n, const uint8_t** end) {
    if (src >= P.out_pos0 && src + n <= P.win_end) { *end = P.out + (P.win_end - P.out_pos0); return P.out + (src - P.out_pos0); }
#pragma unroll
    for (int r = 0; r < MAX_RESIDENT; r++)
        if (src >= P.res[r].lo && src + n <= P.res[r].hi) { *end = P.res[r].ptr + (P.res[r].hi - P.res[r].lo); return P.res[r].ptr + (src - P.res[r].lo); }
    return nullptr;
}

// the collect pass for one match (see copy_body<.., COLLECT>): seed bytes that are neither in the window nor in a resident
// slot become records of the demand list P.gl_nxt; bad offsets are reported by the match launch
__device__ __forceinline__ void collect_match(const Params& P, const SegCtx& c, uint64_t src, uint64_t dst, uint32_t len) {
    if (src >= dst || len == 0) return;
    const bool ovl = src + len > dst;
    if (ovl && src >= c.sstart) return;                      // FORMAT.md §3 (c): its own literal run
    const uint32_t seed_len = ovl ? (uint32_t)(dst - src) : len;
    const uint8_t* end;
    if (resolve_src(P, src, seed_len, &end)) return;
    const Stack sk{nullptr, 0, 0, &P.gl_nxt, SKIP_KNOWN};
    fetch_source_inl(P, sk, src, seed_len, dst - P.out_pos0);
}

// ---- A4: match resolution from the descriptors the literal launch left ---------------------------------------------------
// No entropy decode, no scan: per segment the warp walks its descriptors 32 at a time.  The sources of the short
// non-overlapping matches of a group travel global -> shared memory with 16-byte cp.async issued by the lanes that own
// them; the stage is double-buffered, so the sources of round r + 1 are in flight while the warp copies round r to the
// output (lane i moves bytes i, i + 32, ...).  Matches of LONG_MATCH bytes and more use the 16-byte warp copy,
// self-overlapping ones replicate src + (i mod period).  By FORMAT.md §3 no match reads match bytes of its own block, so
// the loads of a segment never depend on its stores.
// WAIT: segments arrive sorted by (level, index) and wait for the completion of lower-level source blocks.
// WIN: a window of a range decode: sources are looked up in the window and the resident slots; source bytes that are in
// neither have been delivered by the demand rounds before this launch and are skipped.  COLLECT (range decode, before the
// demand rounds): nothing is copied, the unknown seed bytes of every match are appended to the demand lists.
constexpr uint32_t LONG_MATCH = 192;
constexpr uint32_t MTAB_BYTES = 36 * 16;   // per warp and buffer: 32 entries (+ 3 empty) {destination pointer, shared address of the staged source, len}
constexpr uint32_t STAGE_CHUNKS = 160;     // per warp and buffer: 2560 bytes of staged source data
constexpr uint32_t COPY_WARP_BYTES = 2 * (MTAB_BYTES + 16 * STAGE_CHUNKS);
static_assert(LONG_MATCH < 256 && (15 + LONG_MATCH + 15) / 16 <= STAGE_CHUNKS, "a short match fits the stage");
static_assert(COPY_WARP_BYTES % 16 == 0, "tables and stages are 16-byte aligned");

// parts: a small launch (a seek) cuts every segment's matches into `parts` interleaved shares of 32-match groups, a work item
// each (no match reads match bytes of its own block, so the shares are independent): a lone warp per segment is all latency
struct Work { unsigned long long* ticket; const uint32_t* seg_list; uint64_t first_work, n_work; uint32_t parts; };

template <bool WAIT, bool WIN, bool COLLECT, bool REVERSE>
__device__ __forceinline__ void copy_body(const Params& P, const Work W, uint32_t smem_warp /* shared address of this warp's COPY_WARP_BYTES */) {
    const uint32_t lane = lane_id();
    const uint32_t sbase = smem_warp;
    const uint8_t* const out_end = P.out + (P.win_end - P.out_pos0);
    for (;;) {
        unsigned long long t = 0;
        if (lane == 0) t = atomicAdd(W.ticket, 1ull);
        t = __shfl_sync(0xffffffffu, t, 0);
        if (t >= W.n_work) break;
        // The wait-free launch of the whole file takes the last segments first: their literals and descriptors are what
        // k_literals wrote last, so the first ~100 MB of the launch's destination sectors and descriptors are still in L2.
        unsigned long long tt = REVERSE ? W.n_work - 1 - t : t;
        uint32_t part = 0;
        if (W.parts > 1) { part = (uint32_t)(tt % W.parts); tt /= W.parts; }
        const uint32_t g_step = 32u * W.parts;
        const uint64_t s = W.seg_list ? (uint64_t)W.seg_list[tt] : W.first_work + tt;
        const uint64_t mp0 = __ldg(P.match_prefix + s);
        const uint4* d4 = reinterpret_cast<const uint4*>(P.dir + s);
        const uint4 da = __ldg(d4), dq = __ldg(d4 + 1);       // FORMAT.md §1.5
        const uint32_t n = dq.x >> 16, n_words = dq.z >> 16, n_ext = dq.w & 0xffffu;
        const uint8_t* const raw = P.archive + ((uint64_t)da.y << 32 | da.x) + ((256 + 2ull * n_words + 3) & ~3ull) + 4ull * n_ext;
        const uint8_t* const cpl = P.cplanes + (uint64_t)P.n_coded_planes * mp0;
        const uint2* const prs = P.pairs + mp0;
        const uint64_t sstart = (uint64_t)da.w << 32 | da.z, b = sstart >> P.log2_bs;
        const uint32_t slen = (uint32_t)(seg_end(P, s, b) - sstart);
        const uint32_t lvl = dq.w >> 16;
        uint8_t* const out_seg = P.out + (sstart - P.out_pos0);
        uint32_t g0 = 32u * part, pending = 0, mis = 0, len = 0, dst_rel = 0;
        uint64_t sp = 0;
        bool done = n == 0;
        // (dst_rel, len) from k_literals, the offset bytes from its decoded coded planes and the raw planes of the payload.
        // The loads of a group are issued one group ahead and their values stay untouched in registers until the group is
        // staged (any arithmetic on them here would wait for the loads): v[i] = byte of the i-th plane in load order
        // (coded planes in decode order, then raw planes) for W <= 4, else the assembled 64-bit offset in v[0], v[1].
        auto load_desc = [&](uint32_t j, uint2& pr, uint32_t (&v)[4]) {
            pr = make_uint2(0, 0); v[0] = v[1] = v[2] = v[3] = 0;
            if (j >= n) return;
            pr = __ldcg(prs + j);
            const uint8_t* cq = cpl + j; const uint8_t* rq = raw + j;
            if (P.W <= 4) {                                   // files up to 4 GiB
#pragma unroll
                for (uint32_t i = 0; i < 4; i++) {
                    if (i < P.n_coded_planes) v[i] = __ldcg(cq + (uint64_t)i * n);
                    else if (i < P.W) v[i] = __ldg(rq + (uint64_t)(i - P.n_coded_planes) * n);
                }
                return;
            }
            uint64_t src = 0;
            for (uint32_t k = 0; k < P.n_coded_planes; k++, cq += n) src |= (uint64_t)__ldcg(cq) << P.coded_shift[k];
            for (uint32_t r = 0; r < P.n_raw_planes; r++, rq += n) src |= (uint64_t)__ldg(rq) << P.raw_shift[r];
            v[0] = (uint32_t)src; v[1] = (uint32_t)(src >> 32);
        };
        auto desc_src = [&](const uint32_t (&v)[4]) -> uint64_t {
            if (P.W > 4) return (uint64_t)v[1] << 32 | v[0];
            uint32_t s32 = 0;
#pragma unroll
            for (uint32_t i = 0; i < 4; i++)
                s32 |= v[i] << (i < P.n_coded_planes ? P.coded_shift[i] : P.raw_shift[(i - P.n_coded_planes) & (MAX_W - 1)]);
            return s32;
        };
        uint2 npr; uint32_t nv[4];
        bool have = false;
        // one staging round into buffer `buf`: returns the number of staged matches; commits exactly one cp.async group
        auto issue = [&](uint32_t buf, uint32_t& more) -> uint32_t {
            const uint32_t mtab = sbase + buf * (MTAB_BYTES + 16 * STAGE_CHUNKS), stage = mtab + MTAB_BYTES;
            for (;;) {
                if (pending == 0) {
                    if (g0 >= n) { done = true; more = 0; cp_async_commit(); return 0; }
                    if (!have) load_desc(g0 + lane, npr, nv);            // head of a segment, or a group that staged nothing
                    have = false;
                    const uint64_t src = desc_src(nv), dst = sstart + npr.x;
                    dst_rel = npr.x; len = npr.y;
                    const bool has = g0 + lane < n;
                    g0 += g_step;
                    const bool good = has && src < dst && (uint64_t)dst_rel + len <= slen && len != 0;
                    if (has && !good) report(P, src < dst ? DF_LENGTH : DF_OFFSET);
                    const bool ovl = good && src + len > dst;
                    if (ovl && src < sstart) report(P, DF_OFFSET);       // FORMAT.md §3 (c): the seed is the literal run in front of the match
                    const uint32_t seed_len = ovl ? (uint32_t)(dst - src) : len;   // source bytes that are not the match's own output
                    const uint8_t* sb = P.out + (src - P.out_pos0);
                    const uint8_t* send = out_end;
                    if (WIN || COLLECT) sb = good ? resolve_src(P, src, seed_len, &send) : nullptr;
                    if (ovl && src >= sstart) { sb = out_seg + (src - sstart); send = out_end; }   // its own literal run: always here
                    if (COLLECT) {                                        // unknown seed bytes -> demand lists; nothing is copied
                        if (g0 < n) { load_desc(g0 + lane, npr, nv); have = true; }
                        if (good && !sb) {
                            const Stack sk{nullptr, 0, 0, &P.gl_nxt, SKIP_KNOWN};
                            fetch_source_inl(P, sk, src, seed_len, dst - P.out_pos0);
                        }
                        continue;
                    }
                    if (WAIT && good && lvl) {                            // completion of lower-level source blocks (of the window)
                        const uint64_t s1 = (min((unsigned long long)(src + len), (unsigned long long)dst) - 1) >> P.log2_bs;
                        for (uint64_t S = src >> P.log2_bs; S <= s1; S++) {
                            if (WIN && ((S << P.log2_bs) < P.out_pos0 || (S << P.log2_bs) >= P.win_end)) continue;   // final already
                            if (S != b && __ldg(P.levels + S) < lvl) wait_block(P, S);
                        }
                    }
                    const bool known = good && sb != nullptr;
                    if (WIN && good && !sb) {                             // seed spread over several buffers or (partly) delivered by the demand rounds
                        const Stack sk{nullptr, 0, 0, nullptr, SKIP_UNKNOWN};
                        fetch_source_inl(P, sk, src, seed_len, dst - P.out_pos0);   // the known pieces of the seed
                    }
                    sp = reinterpret_cast<uint64_t>(sb);
                    mis = (uint32_t)sp & 15u;
                    const bool lng = known && !ovl && len >= LONG_MATCH;
                    const bool sht = known && !ovl && !lng;
                    // a chunk may not reach past the end of the buffer (only possible for sources in its last 16 bytes)
                    const bool stg = sht && ((sp - mis) + 16ull * ((mis + len + 15u) >> 4) <= reinterpret_cast<uint64_t>(send));
                    uint32_t longs = __ballot_sync(0xffffffffu, lng);
                    while (longs) {
                        const int l = __ffs(longs) - 1; longs &= longs - 1;
                        const uint32_t d2 = __shfl_sync(0xffffffffu, dst_rel, l), m = __shfl_sync(0xffffffffu, len, l);
                        warp_copy<true>(out_seg + d2, reinterpret_cast<const uint8_t*>(__shfl_sync(0xffffffffu, sp, l)), m);
                    }
                    uint32_t direct = __ballot_sync(0xffffffffu, (sht && !stg) || (known && ovl));
                    while (direct) {                                     // byte i of the match = seed[i mod period] (FORMAT.md §2)
                        const int l = __ffs(direct) - 1; direct &= direct - 1;
                        const uint32_t d2 = __shfl_sync(0xffffffffu, dst_rel, l), m = __shfl_sync(0xffffffffu, len, l);
                        const uint32_t per = __shfl_sync(0xffffffffu, (uint32_t)min((unsigned long long)(dst - src), 0xffffffffull), l);
                        const uint8_t* sq = reinterpret_cast<const uint8_t*>(__shfl_sync(0xffffffffu, sp, l));
                        uint32_t r = lane % per; const uint32_t stp = 32 % per;
                        for (uint32_t i = lane; i < m; i += 32) { out_seg[d2 + i] = __ldcg(sq + r); r += stp; if (r >= per) r -= per; }
                    }
                    pending = __ballot_sync(0xffffffffu, stg);
                    if (pending == 0) continue;
                }
                const bool mine = (pending >> lane) & 1u;
                const uint32_t need = mine ? (mis + len + 15u) >> 4 : 0u;
                uint32_t ce = need;
#pragma unroll
                for (int o = 1; o < 32; o <<= 1) { uint32_t a = __shfl_up_sync(0xffffffffu, ce, o); if (lane >= (uint32_t)o) ce += a; }
                const bool fits = mine && ce <= STAGE_CHUNKS;
                const uint32_t fmask = __ballot_sync(0xffffffffu, fits);
                const uint32_t ent = __popc(fmask & lanemask_lt());
                more = __reduce_or_sync(0xffffffffu, fits && len > 64 ? 1u << ent : 0u);   // entries that need more than two passes
                if (fits) {
                    const uint32_t so = 16u * (ce - need);
                    const uint8_t* g = reinterpret_cast<const uint8_t*>(sp - mis);
                    for (uint32_t q = 0; q < need; q++) cp_async16s(stage + so + 16 * q, g + 16 * q);
                    const uint64_t dp = reinterpret_cast<uint64_t>(out_seg) + dst_rel;
                    sts128(mtab + 16 * ent, (uint32_t)dp, (uint32_t)(dp >> 32), stage + so + mis, len);
                }
                const uint32_t n_ent = __popc(fmask);
                if (lane < 3) sts128(mtab + 16 * (n_ent + lane), 0, 0, 0, 0);   // empty entries: matches are taken four at a time
                cp_async_commit();
                pending &= ~fmask;
                if (pending == 0 && g0 < n) { load_desc(g0 + lane, npr, nv); have = true; }
                return n_ent;
            }
        };
        auto copy_out = [&](uint32_t buf, uint32_t n_ent, uint32_t more) {
            const uint32_t mtab = sbase + buf * (MTAB_BYTES + 16 * STAGE_CHUNKS);
            // four matches per iteration: their table reads, stage reads and stores are independent of each other, so
            // the two shared-memory round trips of an iteration are shared by four matches
            for (uint32_t k = 0; k < n_ent; k += 4) {
                uint4 e[4];
#pragma unroll
                for (int q = 0; q < 4; q++) e[q] = lds128(mtab + 16 * k + 16 * q);
                uint32_t v0[4], v1[4];
#pragma unroll
                for (int q = 0; q < 4; q++) { const uint32_t a = e[q].z + lane; v0[q] = lds8(a); v1[q] = lds8(a + 32); }
#pragma unroll
                for (int q = 0; q < 4; q++) {
                    uint8_t* d = reinterpret_cast<uint8_t*>((uint64_t)e[q].y << 32 | e[q].x) + lane;
                    if (lane < e[q].w) d[0] = (uint8_t)v0[q];
                    if (lane + 32 < e[q].w) d[32] = (uint8_t)v1[q];
                }
            }
            while (more) {                                   // bytes 64.. of the longer ones (about one match in nine on FASTQ)
                const int k = __ffs(more) - 1; more &= more - 1;
                const uint4 e = lds128(mtab + 16 * k);
                const uint32_t ln = e.w, sa = e.z + lane;
                uint8_t* dp = reinterpret_cast<uint8_t*>((uint64_t)e.y << 32 | e.x) + lane;
                for (uint32_t o = 64; o + lane < ln; o += 32) dp[o] = (uint8_t)lds8(sa + o);
            }
        };
        if (!done) {
            uint32_t cur = 0, more_cur = 0, n_cur = issue(0, more_cur);
            for (;;) {
                uint32_t n_nxt = 0, more_nxt = 0;
                if (done) cp_async_commit(); else n_nxt = issue(cur ^ 1, more_nxt);
                cp_async_wait_group<1>();                    // everything but the round just issued has landed
                __syncwarp();
                copy_out(cur, n_cur, more_cur);
                __syncwarp();                                // this buffer is refilled by the next round
                if (done && n_nxt == 0) break;
                n_cur = n_nxt; more_cur = more_nxt; cur ^= 1;
            }
            cp_async_wait_group<0>();
        }
        if (WAIT) publish_segment(P, b);
    }
}

// shared memory of the entropy kernels: [byte tables: n_coded_tables x 8 KB][pair table: 32 KB when q_mode = 1]
// [rings: warps x 2 KB][per warp: run table | list of 32 runs | LITA staging][stack tops: warps x 4]   (absolute shared addresses).
// The span-service kernels use the per-warp area as one command table (2 KB at least).
struct CtaSmem { uint32_t luts, lutq, ring, runs, top; uint8_t* lita; uint8_t* area; };   // area: generic pointer of `runs`
constexpr uint32_t ALIST_BYTES = 256;       // k_literals: list of the mid-length LITA runs of a command group, behind the run table

__host__ __device__ inline size_t entropy_smem(uint32_t n_coded_tables, uint32_t q_mode, uint32_t warp_area, int threads) {
    return (size_t)n_coded_tables * LUT_SIZE * 4 + (q_mode ? (size_t)QLUT_SIZE * 8 : 0) + (size_t)(threads / 32) * (RING_BYTES + warp_area + 4) + 128;
}

__device__ __forceinline__ CtaSmem setup_cta(const Params& P, uint8_t* smem_raw) {
    const uint32_t raw0 = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t smem0 = (raw0 + 15u) & ~15u;
    uint8_t* base_ptr = smem_raw + (smem0 - raw0);
    const uint32_t n_lut_words = P.n_coded_tables * LUT_SIZE;
    {
        uint4* dstv = reinterpret_cast<uint4*>(base_ptr);
        for (uint32_t i = threadIdx.x; i < n_lut_words / 4; i += blockDim.x) dstv[i] = __ldg(reinterpret_cast<const uint4*>(P.luts) + i);
        if (P.q_mode) {
            uint4* dq = reinterpret_cast<uint4*>(base_ptr + 4ull * n_lut_words);
            for (uint32_t i = threadIdx.x; i < QLUT_SIZE / 2; i += blockDim.x) dq[i] = __ldg(reinterpret_cast<const uint4*>(P.lutq) + i);
        }
    }
    __syncthreads();
    const uint32_t warp = threadIdx.x >> 5, warps = blockDim.x >> 5, area = P.runs_bytes + ALIST_BYTES + P.lita_bytes;
    CtaSmem m;
    m.luts = smem0;
    m.lutq = smem0 + n_lut_words * 4;
    uint32_t base = m.lutq + (P.q_mode ? QLUT_SIZE * 8 : 0);
    base = (base + 63u) & ~63u;                                // rings are 64-byte aligned (ring | slot)
    m.ring = base + warp * RING_BYTES; base += warps * RING_BYTES;
    m.runs = base + warp * area;
    m.area = smem_raw + (m.runs - raw0);
    m.lita = m.area + P.runs_bytes + ALIST_BYTES;
    base += warps * area;
    m.top = base + 4 * warp;
    return m;
}

// ---- A5-A7: serving spans of a parsed segment ------------------------------------------------------------------------------
// Command table of a parsed segment: word ci = segment-relative output position of command ci (15 bits) | lit_len << 15
// (15 bits) | LITQ class << 30; c.side[ci] = position of the run in its stream.  Word n_cmd is a sentinel (position 0x7fff).
// The words live in the warp's area in shared memory (tab), the side table behind them when it fits, else in the scratch.
__device__ __forceinline__ bool build_cmd_table(const Params& P, SegCtx& c, uint32_t tab, uint8_t* area, uint32_t area_bytes) {
    const uint32_t words = 4 * (c.d.n_cmd + 1);
    if (words + 2 * c.d.n_cmd <= area_bytes) c.side = reinterpret_cast<uint16_t*>(area + words);
    ScanState st; scan_init(st, c);
    bool good = true;
    for (uint32_t c0 = 0; c0 < c.d.n_cmd; c0 += 32) {
        const CmdLane L = scan_step(P, c, st, c0, load_tokens(c, c0));
        good = good && cmd_ok(P, c, L) && L.lit_len <= MAX_SEG_LITS;
        if (__any_sync(0xffffffffu, !good)) { if (lane_id() == 0) report(P, DF_LENGTH); return false; }
        if (L.valid) {
            sts32(tab + 4 * (c0 + lane_id()), L.out_rel | L.lit_len << 15 | (L.is_q ? 1u << 30 : 0u));
            c.side[c0 + lane_id()] = (uint16_t)L.lit_pos;
        }
    }
    if (!scan_totals_ok(c, st)) { if (lane_id() == 0) report(P, DF_LENGTH); return false; }
    if (lane_id() == 0) sts32(tab + 4 * c.d.n_cmd, 0x7fffu);
    __syncwarp();
    return true;
}

// LITA bytes / LITQ symbols in front of segment-relative output position `pend_rel`, from the command table (counting the
// whole literal run of a command that starts before it): the literal streams are decoded only that far.
__device__ __forceinline__ void literals_before(const Params& P, const SegCtx& c, uint32_t tab, uint32_t pend_rel, uint32_t* n_a, uint32_t* n_q) {
    uint32_t a = 0, q = 0;
    for (uint32_t ci = lane_id(); ci < c.d.n_cmd; ci += 32) {
        const uint32_t e = lds32(tab + 4 * ci), o0 = e & 0x7fffu, ll = (e >> 15) & 0x7fffu;
        if (o0 < pend_rel) {
            if ((e >> 30) & 1u) { const uint64_t d = c.sstart + o0; q += P.q_mode ? (uint32_t)(((d + ll - 1) >> 1) - (d >> 1) + 1) : ll; }
            else a += ll;
        }
    }
#pragma unroll
    for (int o = 16; o >= 1; o >>= 1) { a += __shfl_xor_sync(0xffffffffu, a, o); q += __shfl_xor_sync(0xffffffffu, q, o); }
    *n_a = min(a, (uint32_t)c.d.n_lit_a); *n_q = min(q, (uint32_t)c.d.n_sym_q);
}

// A1 + A2 for span service: tokens, the command table, then the literals in front of `pend` into the warp's scratch (LITA
// bytes at lit_a; LITQ bytes, or 16-bit pairs, at lit_q).  LITQ follows LITA in the symbol sequence, so needing any of it
// means decoding all of LITA.  One instance of the byte decode loop.
__device__ __forceinline__ bool parse_for_spans(const Params& P, uint32_t s_luts, uint32_t s_lutq, uint32_t ring, uint32_t tab, uint8_t* area, SegCtx& c, uint64_t pend) {
    if (!load_seg(P, c)) return false;
    c.off_planes = c.off_scratch; c.plane_stride = TOK_STRIDE;
    Rans r;
    r.init(c.payload, c.d.n_words, ring);
    uint32_t i0 = 0, na = c.d.n_lit_a, nq = c.d.n_sym_q;
    const uint32_t n_tok = 2 + P.n_coded_planes, n_reg = n_tok + 1 + (P.q_mode ? 0u : 1u);
    bool ok = true;
#pragma unroll 1
    for (uint32_t k = 0; k < n_reg; k++) {
        uint32_t lut, cnt, adv; uint8_t* dst;
        if (k == 0) { lut = P.lut_cmd; cnt = c.d.n_cmd; dst = c.tok_cmd; }
        else if (k == 1) { lut = P.lut_mlen; cnt = c.d.n_match; dst = c.tok_mlen; }
        else if (k < n_tok) { lut = P.coded_lut[k - 2]; cnt = c.d.n_match; dst = c.off_planes + (k - 2) * TOK_STRIDE; }
        else if (k == n_tok) {
            __syncwarp();                                       // the tokens are complete: the scan reads them
            ok = build_cmd_table(P, c, tab, area, P.runs_bytes + ALIST_BYTES + P.lita_bytes);
            if (!ok) break;
            if (pend < c.send) { literals_before(P, c, tab, (uint32_t)(pend - c.sstart), &na, &nq); if (nq) na = c.d.n_lit_a; }
            lut = P.lut_lita; cnt = na; dst = c.lit_a;
        } else { lut = P.lut_litq; cnt = nq; dst = c.lit_q; }
        adv = k == n_tok ? c.d.n_lit_a : cnt;
        const uint32_t esc = rans_region<false>(r, s_luts + lut * (4 * LUT_SIZE), i0, cnt, dst);
        if (k == 0) c.n_ext_cmd = esc;
        i0 += adv;
        if (k == n_tok && nq == 0) break;                       // nothing of LITQ is wanted
    }
    if (ok && P.q_mode && nq) rans_region<true>(r, s_lutq, i0, nq, c.lit_q);
    if (ok && na == c.d.n_lit_a && nq == c.d.n_sym_q) ok = rans_final_ok(P, r);
    cp_async_wait_group<0>();
    __syncwarp();
    return ok;
}

// byte at absolute position p of a literal run of the parsed segment (run at absolute position d, lit_pos in its stream)
__device__ __forceinline__ uint32_t lit_byte(const Params& P, const SegCtx& c, bool is_q, uint32_t lit_pos, uint64_t d, uint64_t p) {
    if (!is_q) return c.lit_a[lit_pos + (p - d)];
    if (!P.q_mode) return c.lit_q[lit_pos + (p - d)];
    const uint32_t sym = lit_pos + (uint32_t)((p >> 1) - (d >> 1));
    return c.lit_q[2ull * sym + (p & 1)];
}

// the piece [pos, pend) (absolute positions) of a command (literal run at absolute position o0) -> out2[dst + (x - pos)]
__device__ __forceinline__ void emit_cmd_piece(const Params& P, const SegCtx& c, const Stack& st, bool is_q, uint32_t lit_pos, uint64_t o0,
                                            uint32_t lit_len, uint32_t match_len, bool has_match, uint32_t ci,
                                            uint64_t pos, uint64_t pend, uint64_t dst) {
    uint64_t a = max((unsigned long long)o0, (unsigned long long)pos), b = min((unsigned long long)(o0 + lit_len), (unsigned long long)pend);
    if (a < b) {
        // bytes [a, b) of the run; pairs in the scratch sit at even positions of the OUTPUT: byte p of the run is byte
        // (p - (o0 & ~1)) of the pair array that starts at symbol lit_pos
        const uint8_t* src = !is_q ? c.lit_a + lit_pos + (a - o0) : !P.q_mode ? c.lit_q + lit_pos + (a - o0) : c.lit_q + 2ull * lit_pos + (a - (o0 & ~1ull));
        copy_any(P.out2 + dst + (a - pos), src, (uint32_t)(b - a));
    }
    const uint64_t md = o0 + lit_len;
    a = max((unsigned long long)md, (unsigned long long)pos); b = min((unsigned long long)(md + match_len), (unsigned long long)pend);
    if (has_match && a < b) {
        const uint64_t src = match_src(P, c, ci);
        const uint64_t period = md - src;
        if (src >= md) report(P, DF_OFFSET);
        else if (period >= match_len) fetch_source(P, st, src + (a - md), b - a, dst + (a - pos));
        else if (period > lit_len) report(P, DF_OFFSET);      // FORMAT.md §3 (c): the seed is the tail of this literal run
        else {                                                // byte i of the match = seed[i mod period]
            uint8_t* d = P.out2 + dst + (a - pos);
            uint32_t r = (uint32_t)((a - md) % period);
            const uint32_t n = (uint32_t)(b - a);
            // the seed [src, md) lies in this command's literal run, contiguous in the warp's scratch: copy it piecewise,
            // wrapping at the period (a FASTA N-run with its newlines has period 61; a byte loop here made one hot source
            // segment cost milliseconds)
            const uint8_t* seed = !is_q ? c.lit_a + lit_pos + (src - o0) : !P.q_mode ? c.lit_q + lit_pos + (src - o0) : c.lit_q + 2ull * lit_pos + (src - (o0 & ~1ull));
            if (period < 8) {                                  // short periods: one byte at a time is as good as it gets per piece
                for (uint32_t k = 0; k < n; k++) { d[k] = seed[r]; if (++r == (uint32_t)period) r = 0; }
            } else {
                for (uint32_t k = 0; k < n;) {
                    const uint32_t m = min(n - k, (uint32_t)period - r);
                    copy_any(d + k, seed + r, m);
                    k += m; r = 0;
                }
            }
        }
    }
}

constexpr uint32_t ITEM_LANE_MAX = 96;   // spans up to this many bytes are served by one lane each
constexpr uint32_t WIDE_PIECE = 64;      // longer ones are cut into pieces of this size, a lane per piece

// Records of the parsed segment c, one per lane (have == false: none): lane l emits bytes [pos, pos + len) to out2[dst ..).
// A binary search in the command table finds the first command of the span; the lane then walks its commands (one to
// three for a 32-byte span): literal bytes come from the warp's scratch, match pieces are forwarded to their sources.
// A record longer than ITEM_LANE_MAX is cut into pieces that all lanes serve together, 32 pieces at a time.  The loop is
// written so that the body exists once in the code (the kernels that serve spans are sensitive to instruction fetch).
__device__ __forceinline__ void emit_records(const Params& P, const SegCtx& c, const Stack& st, uint32_t tab, bool have,
                                             uint64_t pos, uint32_t len, uint64_t dst) {
    const uint32_t lane = lane_id(), slen = (uint32_t)(c.send - c.sstart);
    have = have && len != 0;
    uint32_t wides = __ballot_sync(0xffffffffu, have && len > ITEM_LANE_MAX);
    uint64_t wpos = 0, wdst = 0; uint32_t wlen = 0, q = 0;
    for (uint32_t pass = 0;; pass++) {
        bool mine; uint64_t mpos, mdst; uint32_t mlen;
        if (pass == 0) { mine = have && len <= ITEM_LANE_MAX; mpos = pos; mlen = len; mdst = dst; }
        else {
            if (q == 0) {
                if (!wides) break;
                const int l = __ffs(wides) - 1; wides &= wides - 1;
                wpos = __shfl_sync(0xffffffffu, pos, l); wlen = __shfl_sync(0xffffffffu, len, l); wdst = __shfl_sync(0xffffffffu, dst, l);
            }
            const uint32_t off = WIDE_PIECE * (lane + 32u * q);
            mine = off < wlen; mpos = wpos + off; mlen = mine ? min(WIDE_PIECE, wlen - off) : 0u; mdst = wdst + off;
            q = (WIDE_PIECE * 32u * (q + 1) < wlen) ? q + 1 : 0u;
        }
        if (mine) {
            const uint32_t pr = (uint32_t)(mpos - c.sstart), pe = pr + mlen;
            uint32_t lo = 0, hi = c.d.n_cmd;
            while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if ((lds32(tab + 4 * mid) & 0x7fffu) <= pr) lo = mid; else hi = mid; }
            for (uint32_t k = lo; k < c.d.n_cmd; k++) {
                const uint32_t e = lds32(tab + 4 * k);
                const uint32_t o0 = e & 0x7fffu, lit_len = (e >> 15) & 0x7fffu;
                if (o0 >= pe) break;
                const uint32_t nx = k + 1 < c.d.n_cmd ? lds32(tab + 4 * k + 4) & 0x7fffu : slen;
                emit_cmd_piece(P, c, st, (e >> 30) & 1u, c.side[k], c.sstart + o0, lit_len, nx - o0 - lit_len, k < c.d.n_match, k, mpos, mpos + mlen, mdst);
            }
        }
        __syncwarp();
    }
}

// Serve every pending demand of the warp's stack (depth-first; all demands of one segment from one parse).
__device__ __forceinline__ void process_demands(const Params& P, const CtaSmem& m, SegCtx& c, const Stack& st) {
    const uint32_t lane = lane_id();
    for (;;) {
        __syncwarp();
        uint32_t top = min(lds_top(st), st.cap);
        while (top > 0 && st.base[top - 1].len == 0) top--;  // drop served entries
        __syncwarp();
        if (lane == 0) sts32(st.top, top);
        __syncwarp();
        if (top == 0) return;
        const uint64_t p0 = st.base[top - 1].pos;
        if (p0 >= P.N) { if (lane == 0) { report(P, DF_OFFSET); st.base[top - 1].len = 0; } continue; }
        c.s = seg_of(P, p0);
        const uint64_t b0 = p0 >> P.log2_bs, lo = __ldg(&P.dir[c.s].out_start), hi = seg_end(P, c.s, b0);
        uint64_t pend = 0;                                   // the literals are needed up to the last pending span of this segment
        for (uint32_t i0 = 0; i0 < top; i0 += 32) {
            const uint32_t idx = i0 + lane;
            if (idx < top && st.base[idx].len != 0 && st.base[idx].pos >= lo && st.base[idx].pos < hi)
                pend = max((unsigned long long)pend, (unsigned long long)(st.base[idx].pos + st.base[idx].len));
        }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) pend = max((unsigned long long)pend, (unsigned long long)__shfl_xor_sync(0xffffffffu, pend, o));
        uint16_t* const side0 = c.side;
        const bool ok = parse_for_spans(P, m.luts, m.lutq, m.ring, m.runs, m.area, c, pend);
        bool found = true;
        while (found) {                                      // serving may push more demands for this same segment
            found = false;
            const uint32_t n = min(lds_top(st), st.cap);
            for (uint32_t i0 = 0; i0 < n; i0 += 32) {
                const uint32_t idx = i0 + lane;
                const bool mine = idx < n && st.base[idx].len != 0 && st.base[idx].pos >= lo && st.base[idx].pos < hi;
                uint64_t pos = 0, len = 0, dst = 0;
                if (mine) { pos = st.base[idx].pos; len = st.base[idx].len; dst = st.base[idx].dst; st.base[idx].len = 0; }
                if (!__any_sync(0xffffffffu, mine)) continue;
                __syncwarp();
                emit_records(P, c, st, m.runs, ok && mine && pos + len <= hi, pos, (uint32_t)len, dst);
                found = true;
            }
            __syncwarp();
        }
        c.side = side0;
    }
}

// Two ticket slots alternate between consecutive launches of a handle: a kernel draws from its own slot and clears the
// other one, so no memset has to be queued between launches.
__device__ __forceinline__ void clear_next_ticket(const Params& P) {
    if (blockIdx.x == 0 && threadIdx.x == 0) *P.ticket_next = 0ull;
}

__device__ __forceinline__ bool next_ticket(const Params& P, unsigned long long& t) {
    t = 0;
    if (lane_id() == 0) t = atomicAdd(P.ticket, 1ull);
    t = __shfl_sync(0xffffffffu, t, 0);
    return t < P.n_work;
}

// The literal launch: A1 + A2 + A3 for every segment of the work list, no dependencies.
template <int QM, bool COLLECT = false>
__global__ void __launch_bounds__(1024, 1) k_literals(const __grid_constant__ Params P) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    const CtaSmem m = setup_cta(P, smem_raw);
    SegCtx c;
    bind_scratch(P, blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), c);
    unsigned long long t;
    while (next_ticket(P, t)) {
        c.s = P.seg_list ? (uint64_t)P.seg_list[t] : P.first_work + t;
        literals_of_segment<QM, COLLECT>(P, m.luts, m.lutq, m.ring, m.runs, m.lita, c);
    }
}

template <bool WAIT, bool WIN, bool COLLECT, bool REVERSE>
__global__ void __launch_bounds__(1024, 1) k_copy(const __grid_constant__ Params P) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    const uint32_t smem0 = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 15u) & ~15u;
    copy_body<WAIT, WIN, COLLECT, REVERSE>(P, Work{P.ticket, P.seg_list, P.first_work, P.n_work, P.copy_parts}, smem0 + (threadIdx.x >> 5) * COPY_WARP_BYTES);
}

// The whole wavefront in ONE cooperative launch (a single persistent kernel): the literal wave over
// every segment, a grid-wide barrier, then the match waves: one flag-driven pass over the segments below the top level
// (when there are any) and one wait-free pass over the top level.  tickets[0..2] are zero at launch.
struct FusedArgs { uint64_t n_low, n_top; const uint32_t* low_list; const uint32_t* top_list; unsigned long long* tickets; };
template <int QM>
__global__ void __launch_bounds__(1024, 1) k_fused(const __grid_constant__ Params P, const FusedArgs F) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    {
        const CtaSmem m = setup_cta(P, smem_raw);
        SegCtx c;
        bind_scratch(P, blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), c);
        for (;;) {
            unsigned long long t = 0;
            if (lane_id() == 0) t = atomicAdd(F.tickets, 1ull);
            t = __shfl_sync(0xffffffffu, t, 0);
            if (t >= P.n_segs) break;
            c.s = t;
            literals_of_segment<QM>(P, m.luts, m.lutq, m.ring, m.runs, m.lita, c);
        }
    }
    __threadfence();
    grid.sync();
    const uint32_t smem0 = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 15u) & ~15u;
    const uint32_t mine = smem0 + (threadIdx.x >> 5) * COPY_WARP_BYTES;
    if (F.n_low) {
        copy_body<true, false, false, false>(P, Work{F.tickets + 1, F.low_list, 0, F.n_low, 1u}, mine);
        __threadfence();
        grid.sync();
    }
    copy_body<false, false, false, true>(P, Work{F.tickets + 2, F.top_list, 0, F.n_top, 1u}, mine);
}

// ---- demand rounds ---------------------------------------------------------------------------------------------------
// The list arrays are written by other CTAs, possibly earlier in the SAME launch (k_rounds): they are read at L2.
__device__ __forceinline__ GDemand ld_demand(const GDemand* p) {
    const unsigned long long* q = reinterpret_cast<const unsigned long long*>(p);
    GDemand d; d.pos = __ldcg(q); d.dst = __ldcg(q + 1);
    const unsigned long long w = __ldcg(q + 2); d.len = (uint32_t)w; d.seg = (uint32_t)(w >> 32);
    return d;
}

// Bucket offsets and work items of the list g: every warp of the launch takes 32 touched segments at a time; the bucket
// offsets and the work-item slots come from two global counters (count[3]: records placed, count[2]: work items), one
// atomicAdd per warp each (the order of the buckets in the sorted array is irrelevant); cnt[segment] becomes the fill
// pointer of the segment's bucket.  Both counters are zero when a list becomes the current one.
__device__ __forceinline__ void plan_body(const GList& g, uint32_t warp_global, uint32_t n_warps_global) {
    const uint32_t n = min(__ldcg(g.count + 1), g.touched_cap), lane = threadIdx.x & 31;
    for (uint32_t t0 = 32 * warp_global; t0 < n; t0 += 32 * n_warps_global) {
        const uint32_t t = t0 + lane;
        uint32_t sg = 0, c = 0;
        if (t < n) { sg = __ldcg(g.touched + t); c = __ldcg(g.cnt + sg); }
        uint32_t it = (c + GL_ITEM - 1) / GL_ITEM, ps = c, pi = it;      // inclusive warp scans of records and items
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t a = __shfl_up_sync(0xffffffffu, ps, o), b2 = __shfl_up_sync(0xffffffffu, pi, o);
            if (lane >= (uint32_t)o) { ps += a; pi += b2; }
        }
        uint32_t rb = 0, ib = 0;
        if (lane == 31) { rb = atomicAdd(g.count + 3, ps); ib = atomicAdd(g.count + 2, pi); }
        rb = __shfl_sync(0xffffffffu, rb, 31); ib = __shfl_sync(0xffffffffu, ib, 31);
        const uint32_t r0 = rb + ps - c, i0 = ib + pi - it;
        if (t < n) {
            g.cnt[sg] = r0;
            for (uint32_t j = 0; j < it; j++) if (i0 + j < g.work_cap) {
                g.work[i0 + j] = (unsigned long long)sg << 32 | (r0 + j * GL_ITEM);
                g.work_n[i0 + j] = min(GL_ITEM, c - j * GL_ITEM);
            }
        }
    }
}

__global__ void __launch_bounds__(1024, 1) k_plan(const __grid_constant__ Params P) {
    plan_body(P.gl_cur, blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), gridDim.x * (blockDim.x >> 5));
}

__device__ __forceinline__ void scatter_body(const GList& g, uint32_t tid, uint32_t n_threads) {
    const uint32_t n = min(__ldcg(g.count), g.cap);
    for (uint32_t i = tid; i < n; i += n_threads) {
        const GDemand d = ld_demand(g.rec + i);
        const uint32_t p = atomicAdd(g.cnt + d.seg, 1u);
        if (p < g.cap) g.sorted[p] = d;
    }
}

__global__ void __launch_bounds__(256) k_scatter(const __grid_constant__ Params P) {
    scatter_body(P.gl_cur, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}

// One round of the demand lists: a work item = up to GL_ITEM records of one source segment; the segment is parsed once
// (tokens + the literals in front of the last wanted span into the warp's scratch) and serves them, one record per lane;
// match pieces whose sources are unknown go to the lists of the next round (recursion depth <= max_level + 1, FORMAT.md §3).
__device__ __forceinline__ void serve_body(const Params& P, const CtaSmem& m, SegCtx& c, const GList& cur, const GList& nxt,
                                           unsigned long long* ticket) {
    const Stack sk{nullptr, 0, m.top, &nxt, 0};
    const unsigned long long n = min(__ldcg(cur.count + 2), cur.work_cap);
    const uint32_t lane = lane_id();
    for (;;) {
        unsigned long long t = 0;
        if (lane == 0) t = atomicAdd(ticket, 1ull);
        t = __shfl_sync(0xffffffffu, t, 0);
        if (t >= n) break;
        const unsigned long long item = __ldcg(cur.work + t);
        const uint32_t first = (uint32_t)item, cnt = __ldcg(cur.work_n + t);
        c.s = item >> 32;
        if (c.s >= P.n_segs) { if (lane == 0) report(P, DF_OFFSET); continue; }
        if (lane == 0) cur.cnt[c.s] = 0;                      // every item of the segment writes the same value: the array is idle again
        uint64_t pend = 0;                                    // the literals are needed up to the last span of the item
        for (uint32_t r0 = 0; r0 < cnt; r0 += 32)
            if (r0 + lane < cnt && first + r0 + lane < cur.cap) { const GDemand d = ld_demand(cur.sorted + first + r0 + lane); pend = max((unsigned long long)pend, (unsigned long long)(d.pos + d.len)); }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) pend = max((unsigned long long)pend, (unsigned long long)__shfl_xor_sync(0xffffffffu, pend, o));
        uint16_t* const side0 = c.side;
        if (parse_for_spans(P, m.luts, m.lutq, m.ring, m.runs, m.area, c, pend)) {
            for (uint32_t r0 = 0; r0 < cnt; r0 += 32) {
                const bool have = r0 + lane < cnt && first + r0 + lane < cur.cap;
                GDemand d; d.pos = 0; d.len = 0; d.dst = 0; d.seg = 0;
                if (have) d = ld_demand(cur.sorted + first + r0 + lane);
                const bool inside = have && d.pos >= c.sstart && d.pos + d.len <= c.send;
                if (have && !inside) report(P, DF_LENGTH);
                emit_records(P, c, sk, m.runs, inside, d.pos, d.len, d.dst);
            }
        }
        c.side = side0;
        __syncwarp();
    }
}

__global__ void __launch_bounds__(1024, 1) k_serve(const __grid_constant__ Params P) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    const CtaSmem m = setup_cta(P, smem_raw);
    SegCtx c;
    bind_scratch(P, blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), c);
    serve_body(P, m, c, P.gl_cur, P.gl_nxt, P.ticket);
}

// All rounds of a demand list in ONE cooperative launch (every CTA resident, grid-wide barriers between plan, scatter and
// serve): a seek or the ragged ends of a range need a handful of records per round, and one launch instead of three per
// round, with an exit as soon as a round leaves nothing, is what their latency is made of.  P.gl_cur = the filled list,
// P.gl_nxt = the other one; round_tickets = one zeroed counter per round.
__global__ void __launch_bounds__(1024, 1) k_rounds(const __grid_constant__ Params P, unsigned long long* round_tickets, uint32_t rounds) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const CtaSmem m = setup_cta(P, smem_raw);
    SegCtx c;
    bind_scratch(P, blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), c);
    for (uint32_t r = 0;; r++) {
        const GList& cur = (r & 1) ? P.gl_nxt : P.gl_cur;
        const GList& nxt = (r & 1) ? P.gl_cur : P.gl_nxt;
        const uint32_t n_rec = *reinterpret_cast<volatile uint32_t*>(cur.count);
        if (n_rec == 0) break;                                // uniform over the grid: read after a grid-wide barrier
        if (r == rounds) { if (blockIdx.x == 0 && threadIdx.x == 0) report(P, DF_STACK); break; }
        if (blockIdx.x == 0 && threadIdx.x < 4) nxt.count[threadIdx.x] = 0;
        plan_body(cur, blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), gridDim.x * (blockDim.x >> 5));
        __threadfence();
        grid.sync();
        scatter_body(cur, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
        __threadfence();
        grid.sync();
        serve_body(P, m, c, cur, nxt, round_tickets + r);
        __threadfence();
        grid.sync();
    }
}

// top-level spans (ragged ends of a range, reads of a batch) enter the demand lists like any other record
__global__ void k_seed(const __grid_constant__ Params P, uint32_t n) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const Demand d = P.n_inline ? P.inline_dem[i] : P.demands[i];
        const Stack sk{nullptr, 0, 0, &P.gl_nxt, 0};
        push_span(P, sk, d.pos, d.len, d.dst);
    }
}

__global__ void k_assert_empty(const uint32_t* count, uint32_t* err) { if (*count) atomicOr(err, (uint32_t)DF_STACK); }

// Read access by recursion inside one warp: one top-level span per ticket; the warp parses the segment that holds it,
// emits the span, and serves the source spans it pushed on its own stack until the stack is empty.
__global__ void __launch_bounds__(1024, 1) k_spans(const __grid_constant__ Params P) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    const CtaSmem m = setup_cta(P, smem_raw);
    const uint32_t gw = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    SegCtx c;
    bind_scratch(P, gw, c);
    Stack st;
    st.base = P.stacks + (uint64_t)gw * P.stack_cap; st.cap = P.stack_cap; st.top = m.top; st.gl = nullptr; st.policy = 0;
    if (lane_id() == 0) sts32(st.top, 0u);
    __syncwarp();
    unsigned long long t;
    while (next_ticket(P, t)) {
        if (lane_id() == 0) {
            const Demand d = P.n_inline ? P.inline_dem[t] : P.demands[t];
            push_span(P, st, d.pos, d.len, d.dst);
        }
        process_demands(P, m, c, st);
    }
}

// A single read (at most four top-level spans): ONE CTA whose warps share a queue of spans in place of the per-warp stack of
// k_spans, so that the source segments of a span (five or so for a FASTQ record, then theirs) are parsed side by side by
// different warps instead of one after the other by one warp: the latency of a read is its recursion depth
// (<= max_level + 2 parses), not its number of source segments.  Queue = the CTA's first stack area in the workspace;
// shared counters: tail (entries pushed; push_span adds), head (entries claimed), done (entries served).  An entry is
// published by its `len` (written last, zero before); a warp leaves when everything pushed so far has been served (then
// nobody can push any more).  Every demand is served from its own parse of its segment and written straight to its
// destination: there are no data dependencies between entries.  All waits are bounded (DF_TIMEOUT).
__global__ void __launch_bounds__(1024, 1) k_spans_cta(const __grid_constant__ Params P) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    const CtaSmem m = setup_cta(P, smem_raw);
    const uint32_t lane = lane_id(), warps = blockDim.x >> 5;
    // tail, head, done: the stack-top words of the CTA's first three warps (the CTA has at least four; no static shared
    // memory: the kernel uses the whole opt-in maximum of dynamic shared memory like the others)
    const uint32_t a_tail = m.top - 4u * (threadIdx.x >> 5);
    uint32_t* const s_q = reinterpret_cast<uint32_t*>(smem_raw + (a_tail - (uint32_t)__cvta_generic_to_shared(smem_raw)));
    Demand* const queue = P.stacks + (uint64_t)blockIdx.x * warps * P.stack_cap;
    const uint32_t cap = P.stack_cap;
    for (uint32_t i = threadIdx.x; i < cap; i += blockDim.x) queue[i].len = 0;
    if (threadIdx.x < 3) s_q[threadIdx.x] = 0;
    __threadfence_block();
    __syncthreads();
    SegCtx c;
    bind_scratch(P, blockIdx.x * warps + (threadIdx.x >> 5), c);
    Stack st;
    st.base = queue; st.cap = cap; st.top = a_tail; st.gl = nullptr; st.policy = 0;
    if (threadIdx.x == 0)
        for (uint32_t i = 0; i < P.n_inline; i++) push_span(P, st, P.inline_dem[i].pos, P.inline_dem[i].len, P.inline_dem[i].dst);
    __syncthreads();                                         // nobody looks at the counters before the read's own spans are in
    volatile uint32_t* const q = s_q;
    constexpr uint32_t LEAVE = 0xffffffffu;
    for (;;) {
        uint32_t h = LEAVE;
        if (lane == 0) {
            for (uint32_t spins = 0;; spins++) {
                const uint32_t done = q[2];                  // read BEFORE tail: done == tail then means that nothing is in flight
                const uint32_t tail = min(q[0], cap), head = q[1];
                if (head < tail) { if (atomicCAS(&s_q[1], head, head + 1) == head) { h = head; break; } continue; }
                if (done >= tail) break;
                if (spins > (1u << 22)) { report(P, DF_TIMEOUT); break; }
                __nanosleep(64);
            }
        }
        h = __shfl_sync(0xffffffffu, h, 0);
        if (h == LEAVE) break;
        Demand d; d.pos = 0; d.dst = 0; d.len = 0;
        {
            volatile Demand* const e = queue + h;
            for (uint32_t spins = 0; (d.len = e->len) == 0 && spins < (1u << 22); spins++) __nanosleep(32);
            __threadfence_block();
            d.pos = e->pos; d.dst = e->dst;
        }
        if (d.len == 0) { if (lane == 0) report(P, DF_TIMEOUT); }
        else if (d.pos >= P.N) { if (lane == 0) report(P, DF_OFFSET); }
        else {
            c.s = seg_of(P, d.pos);
            uint16_t* const side0 = c.side;
            const bool ok = parse_for_spans(P, m.luts, m.lutq, m.ring, m.runs, m.area, c, d.pos + d.len);
            const bool inside = d.pos >= c.sstart && d.pos + d.len <= c.send;
            if (ok && !inside && lane == 0) report(P, DF_LENGTH);
            emit_records(P, c, st, m.runs, ok && inside && lane == 0, d.pos, (uint32_t)d.len, d.dst);
            c.side = side0;
        }
        __syncwarp();
        if (lane == 0) { __threadfence_block(); atomicAdd(&s_q[2], 1u); }
    }
}

// FNV-1a 64 of each block of d_data, compared with the archive's table; one thread per block, 16 bytes per load (the hash is
// a serial chain over the block's bytes: a check, not a hot path)
__global__ void k_fnv(const uint8_t* data, uint64_t n_bytes, uint32_t log2_bs, const uint64_t* expect, unsigned long long* n_bad) {
    uint64_t b = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    uint64_t lo = b << log2_bs;
    if (lo >= n_bytes) return;
    uint64_t hi = min((unsigned long long)(lo + (1ull << log2_bs)), (unsigned long long)n_bytes), f = 0xcbf29ce484222325ull;
    uint64_t q = lo;
    if ((reinterpret_cast<uintptr_t>(data + q) & 15) == 0)
        for (; q + 16 <= hi; q += 16) {
            const uint4 v = __ldg(reinterpret_cast<const uint4*>(data + q));
            const uint32_t w[4] = {v.x, v.y, v.z, v.w};
#pragma unroll
            for (int k = 0; k < 4; k++)
#pragma unroll
                for (int j = 0; j < 4; j++) { f ^= (w[k] >> (8 * j)) & 0xffu; f *= 0x100000001b3ull; }
        }
    for (; q < hi; q++) { f ^= data[q]; f *= 0x100000001b3ull; }
    if (f != expect[b]) atomicAdd(n_bad, 1ull);
}

} // namespace acx
