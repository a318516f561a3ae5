// Host side of the C ABI (include/aceapex.h) and the decode kernels for sm_100a.
#include "aceapex.h"
#include "acx_device.cuh"
#include <cooperative_groups.h>

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace acx;

// =================================================================================================== kernels =====

namespace {

struct BlockCtx {
    uint64_t b, bstart, bend;       // block id, absolute byte range
    DirEntry d;
    const uint8_t* payload;
    const uint32_t* ext;            // EXT array
    const uint8_t* raw_planes;      // raw OFF planes, n_match bytes each
    uint32_t n_ext_cmd;             // number of CMD escapes (they come first in EXT)
    // per-warp scratch
    uint8_t *tok_cmd, *tok_mlen, *off_planes, *lit;
    uint8_t* off_scratch;           // the warp's own buffer for the coded offset planes
    uint32_t plane_stride;          // bytes between two coded planes at off_planes
};

__device__ __forceinline__ void report(const Params& P, uint32_t bit) { atomicOr(P.err, bit); }

// Scratch layout per warp: [lit: BS + 32][tok_cmd: max_cmds][tok_mlen: max_cmds][off planes: n_coded x max_cmds]
__device__ __forceinline__ void bind_scratch(const Params& P, uint32_t warp_global, BlockCtx& c) {
    uint8_t* s = P.scratch + (uint64_t)warp_global * P.scratch_per_warp;
    uint64_t mc = (P.max_cmds + 15u) & ~15u;
    c.lit = s; s += (1ull << P.log2_bs) + 32;
    c.tok_cmd = s; s += mc;
    c.tok_mlen = s; s += mc;
    c.off_planes = s; c.off_scratch = s; c.plane_stride = (uint32_t)mc;
}

// offset of match j assembled from coded planes (scratch, decode order = high plane first) and raw planes (payload)
__device__ __forceinline__ uint64_t match_src(const Params& P, const BlockCtx& c, uint32_t j) {
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

// Warm L2 with the source sectors of every match of the block (issued before the copies, so the HBM latency of the
// scattered sources is paid once per block, not once per match).  Only sectors the match really touches are requested.
__device__ __forceinline__ void prefetch_sources(const Params& P, const BlockCtx& c) {
    for (uint32_t j = lane_id(); j < c.d.n_match; j += 32) {
        uint64_t src = match_src(P, c, j);
        if (src >= P.out_pos0 && src < c.bstart && src < P.win_end) {
            const uint8_t* p = P.out + (src - P.out_pos0);
            uint32_t len = P.min_match + c.tok_mlen[j];                  // escapes (>= 259 bytes) are served by the copy itself
            uint32_t span = (uint32_t)(reinterpret_cast<uintptr_t>(p) & 31) + len;
            prefetch_l2(p);
            if (span > 32) prefetch_l2(p + 32);
            if (span > 64) prefetch_l2(p + 64);
            if (span > 96) prefetch_l2(p + len - 1);
        }
    }
}

// A1 (first part): directory entry, then the CMD, MLEN and coded OFF streams into the warp's scratch.  Leaves the rANS
// state positioned at the first literal symbol (global symbol index *lit_i0).
__device__ __forceinline__ bool parse_tokens(const Params& P, uint32_t s_luts, uint32_t ring, BlockCtx& c, Rans& r, uint32_t* lit_i0) {
    const DirEntry* dp = P.dir + c.b;
    const uint4* d4 = reinterpret_cast<const uint4*>(dp);
    uint4 a = __ldg(d4), q = __ldg(d4 + 1);
    c.d.payload_off = (uint64_t)a.x | ((uint64_t)a.y << 32);
    c.d.n_cmd = a.z; c.d.n_match = a.w; c.d.n_lit = q.x; c.d.n_words = q.y; c.d.n_ext = q.z; c.d.level = (uint16_t)(q.w & 0xffff);
    c.bstart = c.b << P.log2_bs;
    c.bend = min((unsigned long long)(c.bstart + (1ull << P.log2_bs)), (unsigned long long)P.N);
    c.payload = P.archive + c.d.payload_off;
    uint64_t rans_bytes = 256 + 2ull * c.d.n_words;
    c.ext = reinterpret_cast<const uint32_t*>(c.payload + ((rans_bytes + 3) & ~3ull));
    c.raw_planes = reinterpret_cast<const uint8_t*>(c.ext + c.d.n_ext);
    uint64_t mc = (P.max_cmds + 15u) & ~15u;
    c.off_planes = c.off_scratch; c.plane_stride = (uint32_t)mc;
    if (P.cplanes) {                                     // whole-file decode: the coded planes are decoded straight into k_copy's input
        c.off_planes = P.cplanes + (uint64_t)P.n_coded_planes * __ldg(P.match_prefix + c.b);
        c.plane_stride = c.d.n_match; mc = c.d.n_match;
    }
    if (c.d.n_cmd > P.max_cmds || c.d.n_match > c.d.n_cmd || c.d.n_lit > (1u << P.log2_bs)) { if (lane_id() == 0) report(P, DF_LENGTH); return false; }
    r.init(c.payload, c.d.n_words, P.archive + P.archive_bytes, ring);
    uint32_t i0 = 0;
    c.n_ext_cmd = rans_region<true>(r, s_luts + P.lut_cmd * (4 * LUT_SIZE), i0, c.d.n_cmd, c.tok_cmd); i0 += c.d.n_cmd;
    rans_region<false>(r, s_luts + P.lut_mlen * (4 * LUT_SIZE), i0, c.d.n_match, c.tok_mlen); i0 += c.d.n_match;
    for (int p = (int)P.W - 1; p >= 0; p--) {
        int li = P.plane_lut[p];
        if (li < 0) continue;
        // coded planes are stored in decode order: slot k = number of coded planes above p
        uint32_t k = 0;
        for (int t = (int)P.W - 1; t > p; t--) k += P.plane_lut[t] >= 0;
        rans_region<false>(r, s_luts + li * (4 * LUT_SIZE), i0, c.d.n_match, c.off_planes + k * mc); i0 += c.d.n_match;
    }
    __syncwarp();
    *lit_i0 = i0;
    return true;
}

// FORMAT.md §1.5 integrity check once every symbol of the block has been decoded
__device__ __forceinline__ bool rans_final_ok(const Params& P, const BlockCtx& c, const Rans& r) {
    bool bad = !r.finished();
    if (__any_sync(0xffffffffu, bad)) { if (lane_id() == 0) report(P, DF_RANS); return false; }
    return true;
}

// A1, whole block: tokens, then the first min(lit_limit, n_lit) literal symbols into the scratch staging buffer.
__device__ __forceinline__ bool parse_block(const Params& P, uint32_t s_luts, uint32_t ring, BlockCtx& c, uint32_t lit_limit, bool prefetch = true) {
    Rans r; uint32_t i0;
    if (!parse_tokens(P, s_luts, ring, c, r, &i0)) return false;
    if (prefetch) prefetch_sources(P, c);
    uint32_t nl = min(lit_limit, c.d.n_lit);
    rans_region<false>(r, s_luts + P.lut_lit * (4 * LUT_SIZE), i0, nl, c.lit);
    if (nl == c.d.n_lit && !rans_final_ok(P, c, r)) return false;
    __syncwarp();
    return true;
}

// Number of literal bytes of the parsed block that lie in front of output position `pend` (counting the whole literal
// run of a command that starts before pend): the LIT stream has to be decoded only that far to serve spans ending at pend.
__device__ __forceinline__ uint32_t literals_before(const Params& P, const BlockCtx& c, uint64_t pend) {
    uint32_t out_base = 0, ec = 0, em = c.n_ext_cmd, lits = 0;
    const uint32_t lane = lane_id();
    for (uint32_t c0 = 0; c0 < c.d.n_cmd && c.bstart + out_base < pend; c0 += 32) {
        uint32_t ci = c0 + lane;
        bool valid = ci < c.d.n_cmd, has_match = ci < c.d.n_match;
        uint32_t tl = valid ? c.tok_cmd[ci] : 0, tm = has_match ? c.tok_mlen[ci] : 0;
        uint32_t ml = __ballot_sync(0xffffffffu, valid && tl == 255), mm = __ballot_sync(0xffffffffu, has_match && tm == 255);
        uint32_t lit_len = tl, match_len = has_match ? P.min_match + tm : 0;
        if (valid && tl == 255) lit_len = 255 + __ldg(c.ext + ec + __popc(ml & lanemask_lt()));
        if (has_match && tm == 255) match_len = P.min_match + 255 + __ldg(c.ext + em + __popc(mm & lanemask_lt()));
        ec += __popc(ml); em += __popc(mm);
        uint32_t st = lit_len + match_len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { uint32_t t = __shfl_up_sync(0xffffffffu, st, o); if (lane >= (uint32_t)o) st += t; }
        const uint64_t out_pos = c.bstart + out_base + (st - lit_len - match_len);
        uint32_t mine = (valid && out_pos < pend) ? lit_len : 0;
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) mine += __shfl_xor_sync(0xffffffffu, mine, o);
        lits += mine;
        out_base += __shfl_sync(0xffffffffu, st, 31);
    }
    return min(lits, c.d.n_lit);
}

// A1 for span service: tokens, then only the literals in front of `pend` (all of them when pend is past the block)
__device__ __forceinline__ bool parse_block_upto(const Params& P, uint32_t s_luts, uint32_t ring, BlockCtx& c, uint64_t pend) {
    Rans r; uint32_t i0;
    if (!parse_tokens(P, s_luts, ring, c, r, &i0)) return false;
    const uint32_t nl = pend >= c.bend ? c.d.n_lit : literals_before(P, c, pend);
    rans_region<false>(r, s_luts + P.lut_lit * (4 * LUT_SIZE), i0, nl, c.lit);
    if (nl == c.d.n_lit && !rans_final_ok(P, c, r)) return false;
    __syncwarp();
    return true;
}

// ---- A2 + A3 fused into the literal decode ("direct placement") --------------------------------------------------
// The command scan runs BEFORE the literal stream is decoded and leaves, in shared memory, one entry per non-empty
// literal run: (last literal index of the run) | (out_start - lit_start) << 16.  The literal decode then stores every
// decoded byte straight to its final position: while a 32-symbol round stays inside one run that is a pointer bump;
// a round that crosses run boundaries looks its runs up with a 5-step shuffle search over the next 32 entries.
constexpr uint32_t RUNS_CAP = 512;     // entries per warp (2 KB); blocks with more runs, or > 64 KB, use the staged path

// returns the number of runs, or 0xffffffff when the block does not fit the table / fails validation
__device__ __forceinline__ uint32_t build_runs(const Params& P, const BlockCtx& c, uint32_t runs /* shared address */) {
    uint32_t lit_base = 0, out_base = 0, ec = 0, em = c.n_ext_cmd, n_runs = 0;
    uint2* const pairs = P.pairs ? P.pairs + __ldg(P.match_prefix + c.b) : nullptr;   // whole-file decode: matches for k_copy
    const uint32_t lane = lane_id();
    bool fits = true;
    for (uint32_t c0 = 0; c0 < c.d.n_cmd; c0 += 32) {
        uint32_t ci = c0 + lane;
        bool valid = ci < c.d.n_cmd, has_match = ci < c.d.n_match;
        uint32_t tl = valid ? c.tok_cmd[ci] : 0, tm = has_match ? c.tok_mlen[ci] : 0;
        uint32_t ml = __ballot_sync(0xffffffffu, valid && tl == 255), mm = __ballot_sync(0xffffffffu, has_match && tm == 255);
        uint32_t lit_len = tl, match_len = has_match ? P.min_match + tm : 0;
        if (valid && tl == 255) lit_len = 255 + __ldg(c.ext + ec + __popc(ml & lanemask_lt()));
        if (has_match && tm == 255) match_len = P.min_match + 255 + __ldg(c.ext + em + __popc(mm & lanemask_lt()));
        ec += __popc(ml); em += __popc(mm);
        uint32_t sl = lit_len, st = lit_len + match_len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t a = __shfl_up_sync(0xffffffffu, sl, o), t = __shfl_up_sync(0xffffffffu, st, o);
            if (lane >= (uint32_t)o) { sl += a; st += t; }
        }
        uint32_t lit_pos = lit_base + sl - lit_len, out_rel = out_base + (st - lit_len - match_len);
        lit_base += __shfl_sync(0xffffffffu, sl, 31);
        out_base += __shfl_sync(0xffffffffu, st, 31);
        if (pairs && has_match) pairs[ci] = make_uint2(out_rel + lit_len, match_len);
        uint32_t ne = __ballot_sync(0xffffffffu, valid && lit_len > 0);
        uint32_t k = n_runs + __popc(ne & lanemask_lt());
        if (valid && lit_len > 0 && k < RUNS_CAP) {
            uint32_t e = ((lit_pos + lit_len - 1) & 0xffff) | ((out_rel - lit_pos) << 16);
            asm volatile("st.shared.u32 [%0], %1;" ::"r"(runs + 4 * k), "r"(e) : "memory");
        }
        n_runs += __popc(ne);
    }
    fits = n_runs < RUNS_CAP && c.d.n_lit < 0xffffu && lit_base == c.d.n_lit && c.bstart + out_base == c.bend;
    if (fits && lane == 0) asm volatile("st.shared.u32 [%0], %1;" ::"r"(runs + 4 * n_runs), "r"(0xffffu) : "memory");   // sentinel
    __syncwarp();
    return fits ? n_runs : 0xffffffffu;
}

// Literal decode with direct placement.  out_blk = address of the block's first output byte.
struct RunCursor {
    uint32_t k;          // run that holds the first literal of the coming round
    uint32_t last;       // last literal index of run k
    uint32_t delta;      // out_start - lit_start of run k
};

// A round whose literals [.., j_hi] are not all strictly inside run k: walk the cursor over the runs that end inside
// the round (one broadcast table read per boundary; the table ends with a sentinel whose `last` is 0xffff).  Returns the
// delta of this lane's literal j and leaves the cursor on the run of literal j_hi + 1.
__device__ __forceinline__ uint32_t walk_runs(RunCursor& rc, uint32_t runs, uint32_t j, uint32_t j_hi) {
    uint32_t mine = rc.delta;
    while (rc.last <= j_hi) {
        const uint32_t prev = rc.last;
        rc.k++;
        const uint32_t e = lds32(runs + 4 * rc.k);
        rc.last = e & 0xffff; rc.delta = e >> 16;
        if (j > prev) mine = rc.delta;
    }
    return mine;
}

__device__ __forceinline__ void decode_lit_direct(Rans& r, uint32_t lut, uint32_t i0, uint32_t n_lit, uint32_t runs, uint8_t* out_blk) {
    if (n_lit == 0) return;
    const uint32_t lane = lane_id(), i1 = i0 + n_lit;
    RunCursor rc;
    { uint32_t e0 = lds32(runs); rc.k = 0; rc.last = e0 & 0xffff; rc.delta = e0 >> 16; }
    uint32_t base = i0 & ~31u;
    if (base != i0) {                                     // ragged first round
        uint32_t i = base + lane;
        bool active = i >= i0 && i < i1;
        r.prepare8();
        uint32_t e = r.step(lut, active);
        uint32_t j_hi = min(base + 31, i1 - 1) - i0;
        uint32_t d = walk_runs(rc, runs, i - i0, j_hi);
        if (active) out_blk[d + (i - i0)] = (uint8_t)e;
        base += 32;
    }
    uint8_t* pj = out_blk + (base + lane - i0);           // address of literal (base + lane - i0) if delta were 0
    while (base + 256 <= i1) {                            // eight full rounds per ring check
        r.prepare8();
        uint8_t* pd = pj + rc.delta;
#pragma unroll
        for (int q = 0; q < 8; q++) {
            uint32_t e = r.step_full(lut);
            uint32_t j_hi = base + 32 * q + 31 - i0;
            if (j_hi < rc.last) pd[32 * q] = (uint8_t)e;   // the whole round lies strictly inside run k: pointer bump
            else { uint32_t d = walk_runs(rc, runs, j_hi - 31 + lane, j_hi); pj[32 * q + d] = (uint8_t)e; pd = pj + rc.delta; }
        }
        base += 256; pj += 256;
    }
    if (base < i1) {                                      // fewer than eight rounds left, the last may be ragged
        r.prepare8();
        for (; base < i1; base += 32) {
            bool active = base + lane < i1;
            uint32_t e = r.step(lut, active);
            uint32_t j_hi = min(base + 31, i1 - 1) - i0;
            uint32_t d = walk_runs(rc, runs, base + lane - i0, j_hi);
            if (active) out_blk[d + (base + lane - i0)] = (uint8_t)e;
        }
    }
}

// flag[S] = 2 * epoch once block S has placed its literal bytes, 2 * epoch + 1 once it is complete
__device__ __forceinline__ void wait_block(const Params& P, uint64_t S, bool need_full) {
    const uint32_t* f = P.flags + S;
    const uint32_t want = 2 * P.epoch + (need_full ? 1u : 0u);
    uint32_t spins = 0, ns = 128;
    while (ld_flag(f) < want) {
        __nanosleep(ns);
        if (ns < 2048) ns *= 2;          // back off: thousands of lanes polling one L2 line slow everybody down
        if (++spins > (1u << 21)) { report(P, DF_TIMEOUT); break; }
    }
    // The polls are relaxed loads; one acquire-release fence once the flag has been seen orders every later read of the
    // guarded bytes after it (the writer: stores, __threadfence, st.release).  Once per wait, not per poll.
    asm volatile("fence.acq_rel.gpu;" ::: "memory");
#ifdef ACX_WAIT_STATS
    if (spins) { atomicAdd(P.err + 4 + (need_full ? 2 : 0), 1u); atomicAdd(P.err + 5 + (need_full ? 2 : 0), spins); }
#endif
}

// Flag-driven schedule: wait for the blocks that hold the seed of a match (other than the own block).
// By FORMAT.md §3 a source block S with level(S) >= level(B) can only contribute literal bytes, so B waits for S's
// literal phase only; S with level(S) < level(B) may contribute match bytes, so B waits for S to complete.  Waits for
// completion therefore go to strictly lower levels and chain at most max_level deep, whatever the distance.
// LIT_WAITS = false: all literals were placed by an earlier launch, only completion waits remain.
template <bool LIT_WAITS>
__device__ __forceinline__ void wait_sources(const Params& P, const BlockCtx& c, uint64_t dst, uint64_t src, uint32_t len) {
    uint64_t seed_end = min((unsigned long long)(src + len), (unsigned long long)dst);
    uint64_t s0 = src >> P.log2_bs, s1 = (seed_end - 1) >> P.log2_bs;
    for (uint64_t S = s0; S <= s1; S++) if (S != c.b) {
        if ((S << P.log2_bs) < P.out_pos0 || (S << P.log2_bs) >= P.win_end) continue;   // outside the window: final already
        bool full = __ldg(P.levels + S) < c.d.level;
        if (full || LIT_WAITS) wait_block(P, S, full);
    }
}

constexpr uint32_t LONG_RUN = 64;   // runs at least this long are copied by the whole warp

// Where source bytes that are neither in the window nor resident go: a per-warp LIFO (read access: depth-first recursion
// by the warp itself) or the global per-source-block lists of a range decode (gl != null).  policy: see fetch_source.
struct Stack { Demand* base; uint32_t cap; uint32_t top; /* shared address of the entry count */ const GList* gl; uint32_t policy; };
enum : uint32_t { SKIP_KNOWN = 1, SKIP_UNKNOWN = 2 };

__device__ __forceinline__ uint32_t lds_top(const Stack& st) { return lds32(st.top); }

// append "original bytes [pos, pos + len) -> out2[dst ..)" (inside one block)
__device__ __forceinline__ void gl_append(const Params& P, const GList& gl, uint64_t pos, uint32_t len, uint64_t dst) {
    const uint32_t idx = atomicAdd(gl.count, 1u);
    if (idx >= gl.cap) { report(P, DF_STACK); return; }
    gl.rec[idx].pos = pos; gl.rec[idx].dst = dst; gl.rec[idx].len = len;
    const uint64_t blk = pos >> P.log2_bs;
    if (atomicAdd(gl.cnt + blk, 1u) == 0) {
        const uint32_t t = atomicAdd(gl.count + 1, 1u);
        if (t < gl.touched_cap) gl.touched[t] = (uint32_t)blk; else report(P, DF_STACK);
    }
}

__device__ __forceinline__ void push_span(const Params& P, const Stack& st, uint64_t pos, uint64_t len, uint64_t dst) {
    while (len) {                                   // a demand never crosses a block boundary
        uint64_t bend = ((pos >> P.log2_bs) + 1) << P.log2_bs;
        uint64_t n = min((unsigned long long)len, (unsigned long long)(bend - pos));
        if (st.gl) gl_append(P, *st.gl, pos, (uint32_t)n, dst);
        else {
            uint32_t idx;
            asm volatile("atom.shared.add.u32 %0, [%1], 1;" : "=r"(idx) : "r"(st.top) : "memory");
            if (idx < st.cap) { st.base[idx].pos = pos; st.base[idx].dst = dst; st.base[idx].len = n; }
            else report(P, DF_STACK);
        }
        pos += n; dst += n; len -= n;
    }
}

// n contiguous original bytes from absolute position sp -> dptr (= out2 + dst_off).  Window bytes and resident slots
// are copied (unless policy SKIP_KNOWN), the rest becomes demands (unless policy SKIP_UNKNOWN).  WAIT: window sources of
// a block being decoded in the same launch need flags.
template <bool WAIT>
__device__ __forceinline__ void fetch_source(const Params& P, const BlockCtx& c, const Stack& st, uint64_t sp, uint64_t n, uint64_t dst_off) {
    while (n) {
        uint64_t m = n;
        const uint8_t* from = nullptr;
        if (sp >= P.out_pos0 && sp < P.win_end) {
            m = min((unsigned long long)n, (unsigned long long)(P.win_end - sp));
            if (WAIT) for (uint64_t S = sp >> P.log2_bs; S <= (sp + m - 1) >> P.log2_bs; S++) if (S != c.b) wait_block(P, S, __ldg(P.levels + S) < c.d.level);
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
                while (left) { uint32_t k = (uint32_t)min((unsigned long long)left, 1ull << 30); copy_bytes<true>(d, f, k, ~0ull); d += k; f += k; left -= k; }
            }
        } else if (!(st.policy & SKIP_UNKNOWN)) push_span(P, st, sp, m, dst_off);
        sp += m; dst_off += m; n -= m;
    }
}

// source of a match piece: bytes [i, i + n) of the match (dst position md, source src, length mlen) -> out2[dst_off ..)
template <bool WAIT>
__device__ __forceinline__ void fetch_match_piece(const Params& P, const BlockCtx& c, const Stack& st, uint64_t md, uint64_t src, uint32_t mlen,
                                                  uint32_t i, uint32_t n, uint64_t dst_off) {
    uint64_t period = md - src;
    if (period >= mlen) { fetch_source<WAIT>(P, c, st, src + i, n, dst_off); return; }
    uint64_t r = i % period;                       // self-overlap: byte i of the match = seed[i mod period] (FORMAT.md §2)
    while (n) {
        uint64_t m = min((unsigned long long)n, (unsigned long long)(period - r));
        fetch_source<WAIT>(P, c, st, src + r, m, dst_off);
        dst_off += m; n -= (uint32_t)m; r = 0;
    }
}

// A2 + A3 + A4 for a whole block: scan the commands 32 at a time, place literal runs, then resolve the matches.
// MODE 2: literals only; MODE 0: matches, waiting on literal and completion flags; MODE 4: matches, waiting on
// completion flags only; MODE 3: matches only, no waits.
template <int MODE, bool DEMANDS = false>
__device__ __forceinline__ void emit_block(const Params& P, const BlockCtx& c, const Stack& stk) {
    uint32_t lit_base = 0, out_base = 0, ec = 0, em = c.n_ext_cmd;
    const uint32_t lane = lane_id();
    for (uint32_t c0 = 0; c0 < c.d.n_cmd; c0 += 32) {
        uint32_t ci = c0 + lane;
        bool valid = ci < c.d.n_cmd, has_match = ci < c.d.n_match;
        uint32_t tl = valid ? c.tok_cmd[ci] : 0, tm = has_match ? c.tok_mlen[ci] : 0;
        uint32_t ml = __ballot_sync(0xffffffffu, valid && tl == 255), mm = __ballot_sync(0xffffffffu, has_match && tm == 255);
        uint32_t lit_len = tl, match_len = has_match ? P.min_match + tm : 0;
        if (valid && tl == 255) lit_len = 255 + __ldg(c.ext + ec + __popc(ml & lanemask_lt()));
        if (has_match && tm == 255) match_len = P.min_match + 255 + __ldg(c.ext + em + __popc(mm & lanemask_lt()));
        ec += __popc(ml); em += __popc(mm);
        // inclusive warp scans of lit_len and lit_len + match_len
        uint32_t sl = lit_len, st = lit_len + match_len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t a = __shfl_up_sync(0xffffffffu, sl, o), t = __shfl_up_sync(0xffffffffu, st, o);
            if (lane >= (uint32_t)o) { sl += a; st += t; }
        }
        uint32_t lit_pos = lit_base + sl - lit_len;          // position of the run in LIT
        uint64_t out_pos = c.bstart + out_base + (st - lit_len - match_len);   // absolute position of the run
        lit_base += __shfl_sync(0xffffffffu, sl, 31);
        out_base += __shfl_sync(0xffffffffu, st, 31);
        bool ok = valid && (uint64_t)lit_pos + lit_len <= c.d.n_lit && out_pos + lit_len + match_len <= c.bend;
        if (__any_sync(0xffffffffu, valid && !ok)) { if (lane == 0) report(P, DF_LENGTH); return; }
        if (MODE == 2) {   // A3: literal runs.  Long runs (quality strings) are copied by the whole warp, short ones per lane.
            uint32_t longs = __ballot_sync(0xffffffffu, ok && lit_len >= LONG_RUN);
            if (ok && lit_len && lit_len < LONG_RUN) copy_bytes<false>(P.out + (out_pos - P.out_pos0), c.lit + lit_pos, lit_len, ~0ull);
            while (longs) {
                int l = __ffs(longs) - 1; longs &= longs - 1;
                uint64_t op = __shfl_sync(0xffffffffu, out_pos, l);
                uint32_t lp = __shfl_sync(0xffffffffu, lit_pos, l), n = __shfl_sync(0xffffffffu, lit_len, l);
                warp_copy<false>(P.out + (op - P.out_pos0), c.lit + lp, n);
            }
            continue;
        }
        // A4: matches.  Non-overlapping long matches by the whole warp, the rest per lane.
        uint64_t dst = out_pos + lit_len, src = (ok && has_match) ? match_src(P, c, ci) : 0;
        bool good = ok && has_match && src < dst;
        if (ok && has_match && !good) report(P, DF_OFFSET);
        if (MODE == 0 && DEMANDS && good && src < P.out_pos0) {          // the source starts below the window: copy what is here,
            fetch_match_piece<true>(P, c, stk, dst, src, match_len, 0u, match_len, dst - P.out_pos0);   // demand the rest
            good = false;
        }
        if (good && MODE == 0) wait_sources<true>(P, c, dst, src, match_len);
        if (good && MODE == 4) wait_sources<false>(P, c, dst, src, match_len);
        bool is_long = good && match_len >= LONG_RUN && src + match_len <= dst;
        uint32_t longs = __ballot_sync(0xffffffffu, is_long);
        if (good && !is_long) copy_bytes<true>(P.out + (dst - P.out_pos0), P.out + (src - P.out_pos0), match_len, dst - src);
        while (longs) {
            int l = __ffs(longs) - 1; longs &= longs - 1;
            uint64_t d2 = __shfl_sync(0xffffffffu, dst, l), s2 = __shfl_sync(0xffffffffu, src, l);
            uint32_t n = __shfl_sync(0xffffffffu, match_len, l);
            warp_copy<true>(P.out + (d2 - P.out_pos0), P.out + (s2 - P.out_pos0), n);
        }
    }
    if (out_base != (uint32_t)(c.bend - c.bstart) || lit_base != c.d.n_lit) { if (lane == 0) report(P, DF_LENGTH); }
}

// ---- A4 for the whole-file schedules: matches of one block, 32 commands at a time ---------------------------------------
// Short non-overlapping matches are staged through shared memory (see below); matches of LONG_MATCH bytes and more use
// the 16-byte warp copy; self-overlapping ones read src + (i mod period).  By FORMAT.md §3 no match reads match bytes of
// its own block, so the loads of a block never depend on its stores.
constexpr uint32_t LONG_MATCH = 192;
constexpr uint32_t MTAB_BYTES = 36 * 16;   // per warp: 32 entries (+ 1 empty; a multiple of 64 bytes keeps the rings aligned) {destination pointer | len << 56, shared address of the staged source}
constexpr uint32_t STAGE_CHUNKS = 160;     // per warp: 2560 bytes of staged source data
static_assert((RING_BYTES + MTAB_BYTES + 16 * STAGE_CHUNKS) % 64 == 0, "per-warp shared memory must keep 64-byte ring alignment");
static_assert(LONG_MATCH < 256 && (15 + LONG_MATCH + 15) / 16 <= STAGE_CHUNKS, "a short match has an 8-bit length and fits the stage");

__device__ __forceinline__ void sts128(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ uint2 lds64(uint32_t a) {
    uint2 v; asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a)); return v;
}
__device__ __forceinline__ uint4 lds128(uint32_t a) {
    uint4 v; asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a)); return v;
}

// MODE 3: no waits (one launch per level); MODE 4: completion waits for lower-level source blocks
// Where the bytes [src, src + n) live if one known buffer holds them all: the window, or a resident slot (range decode).
// *end = end of that buffer.  Null when they are unknown or spread over several buffers.
__device__ __forceinline__ const uint8_t* resolve_src(const Params& P, uint64_t src, uint64_t n, const uint8_t** end) {
    if (src >= P.out_pos0 && src + n <= P.win_end) { *end = P.out + (P.win_end - P.out_pos0); return P.out + (src - P.out_pos0); }
#pragma unroll
    for (int r = 0; r < MAX_RESIDENT; r++)
        if (src >= P.res[r].lo && src + n <= P.res[r].hi) { *end = P.res[r].ptr + (P.res[r].hi - P.res[r].lo); return P.res[r].ptr + (src - P.res[r].lo); }
    return nullptr;
}

// WIN = false: whole file (every source is in P.out).  WIN = true: a window of a range decode: sources are looked up in
// the window and the resident slots; source bytes that are in neither have been delivered by the demand rounds before
// this launch and are skipped.  COLLECT = true (range decode, before the demand rounds): nothing is copied, the unknown
// seed bytes of every match are appended to the demand lists.
template <int MODE, bool WIN = false, bool COLLECT = false>
__device__ __forceinline__ void emit_matches(const Params& P, const BlockCtx& c, uint32_t mtab, uint32_t stage) {
    uint32_t lit_base = 0, out_base = 0, ec = 0, em = c.n_ext_cmd;
    const uint32_t lane = lane_id();
    uint8_t* const out_blk = P.out + (c.bstart - P.out_pos0);
    // tokens and offsets of a group are loaded one group ahead, so that their latency overlaps the copies
    uint32_t n_tl = 0, n_tm = 0; uint64_t n_src = 0;
    { uint32_t ci = lane; if (ci < c.d.n_cmd) n_tl = c.tok_cmd[ci]; if (ci < c.d.n_match) { n_tm = c.tok_mlen[ci]; n_src = match_src(P, c, ci); } }
    for (uint32_t c0 = 0; c0 < c.d.n_cmd; c0 += 32) {
        uint32_t ci = c0 + lane;
        bool valid = ci < c.d.n_cmd, has_match = ci < c.d.n_match;
        const uint32_t tl = n_tl, tm = n_tm; const uint64_t src = n_src;
        { uint32_t cn = ci + 32; n_tl = 0; n_tm = 0; n_src = 0;
          if (cn < c.d.n_cmd) n_tl = c.tok_cmd[cn]; if (cn < c.d.n_match) { n_tm = c.tok_mlen[cn]; n_src = match_src(P, c, cn); } }
        uint32_t ml = __ballot_sync(0xffffffffu, valid && tl == 255), mm = __ballot_sync(0xffffffffu, has_match && tm == 255);
        uint32_t lit_len = tl, match_len = has_match ? P.min_match + tm : 0;
        if (valid && tl == 255) lit_len = 255 + __ldg(c.ext + ec + __popc(ml & lanemask_lt()));
        if (has_match && tm == 255) match_len = P.min_match + 255 + __ldg(c.ext + em + __popc(mm & lanemask_lt()));
        ec += __popc(ml); em += __popc(mm);
        uint32_t sl = lit_len, st = lit_len + match_len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t a = __shfl_up_sync(0xffffffffu, sl, o), t = __shfl_up_sync(0xffffffffu, st, o);
            if (lane >= (uint32_t)o) { sl += a; st += t; }
        }
        uint32_t lit_pos = lit_base + sl - lit_len;
        uint32_t dst_rel = out_base + (st - match_len);      // block-relative position of the match
        lit_base += __shfl_sync(0xffffffffu, sl, 31);
        out_base += __shfl_sync(0xffffffffu, st, 31);
        bool ok = valid && (uint64_t)lit_pos + lit_len <= c.d.n_lit && c.bstart + dst_rel + match_len <= c.bend;
        if (__any_sync(0xffffffffu, valid && !ok)) { if (lane == 0) report(P, DF_LENGTH); return; }
        uint64_t dst = c.bstart + dst_rel;
        bool good = ok && has_match && src < dst;
        if (ok && has_match && !good) report(P, DF_OFFSET);
        if (MODE == 4 && good && c.d.level) wait_sources<false>(P, c, dst, src, match_len);
        const bool ovl = good && src + match_len > dst;
        if (ovl && src < c.bstart) report(P, DF_OFFSET);     // FORMAT.md §3 (c)
        const uint32_t seed_len = ovl ? (uint32_t)(dst - src) : match_len;     // source bytes that are not the match's own output
        const uint8_t* sbase = P.out + (src - P.out_pos0);
        const uint8_t* send = P.out + (P.win_end - P.out_pos0);
        if (WIN || COLLECT) sbase = good ? resolve_src(P, src, seed_len, &send) : nullptr;
        if (COLLECT) {                                       // unknown seed bytes -> demands; nothing else happens here
            if (good && !sbase) {
                Stack sk{nullptr, 0, 0, &P.gl_nxt, SKIP_KNOWN};
                fetch_source<false>(P, c, sk, src, seed_len, dst - P.out_pos0);
            }
            continue;
        }
        const bool known = good && sbase != nullptr;
        const bool lng = known && !ovl && match_len >= LONG_MATCH;
        const bool sht = known && !ovl && !lng;
        // Short matches: their source bytes travel global -> shared memory with 16-byte cp.async (issued by the lane that
        // owns the match, all matches of the group at once: one exposed memory latency per group instead of one per
        // match), then the warp copies match after match from the stage to the output: lane i moves bytes i, i + 32, ...
        // A group whose sources do not fit the stage is served in several rounds.
        const uint64_t sp = reinterpret_cast<uint64_t>(sbase);
        const uint32_t mis = (uint32_t)sp & 15u;
        // a chunk may not reach past the end of the buffer (only possible for sources in its last 16 bytes)
        const bool stg = sht && ((sp - mis) + 16ull * ((mis + match_len + 15u) >> 4) <= reinterpret_cast<uint64_t>(send));
        const bool direct = (sht && !stg) || (known && ovl);
        if (WIN && good && !sbase) {                         // seed spread over several buffers or (partly) delivered by demands
            Stack sk{nullptr, 0, 0, nullptr, SKIP_UNKNOWN};
            fetch_source<false>(P, c, sk, src, seed_len, dst - P.out_pos0);     // the known pieces of the seed
            uint8_t* d = P.out + (dst - P.out_pos0);
            for (uint32_t i = seed_len; i < match_len; i++) d[i] = d[i - seed_len];   // the rest repeats it (FORMAT.md §2)
        }
        uint32_t pending = __ballot_sync(0xffffffffu, stg);
        while (pending) {
            const bool mine = (pending >> lane) & 1u;
            const uint32_t need = mine ? (mis + match_len + 15u) >> 4 : 0u;
            uint32_t ce = need;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) { uint32_t a = __shfl_up_sync(0xffffffffu, ce, o); if (lane >= (uint32_t)o) ce += a; }
            const bool fits = mine && ce <= STAGE_CHUNKS;
            const uint32_t fmask = __ballot_sync(0xffffffffu, fits);
            if (fits) {
                const uint32_t so = 16u * (ce - need);
                const uint8_t* g = reinterpret_cast<const uint8_t*>(sp - mis);
                for (uint32_t q = 0; q < need; q++) cp_async16s(stage + so + 16 * q, g + 16 * q);
                const uint64_t dp = reinterpret_cast<uint64_t>(out_blk) + dst_rel;
                sts128(mtab + 16 * __popc(fmask & lanemask_lt()), (uint32_t)dp, (uint32_t)(dp >> 32) | (match_len << 24), stage + so + mis, 0);
            }
            const uint32_t n_ent = __popc(fmask);
            if (lane == 0) sts128(mtab + 16 * n_ent, 0, 0, 0, 0);       // empty entry: matches are taken two at a time
            cp_async_commit();
            cp_async_wait_group<0>();
            __syncwarp();
            uint32_t more = 0;
            for (uint32_t k = 0; k < n_ent; k += 2) {
                const uint4 e0 = lds128(mtab + 16 * k), e1 = lds128(mtab + 16 * k + 16);
                const uint32_t l0 = e0.y >> 24, l1 = e1.y >> 24;
                const uint32_t a0 = e0.z + lane, a1 = e1.z + lane;
                const uint32_t v00 = lds8(a0), v01 = lds8(a0 + 32), v10 = lds8(a1), v11 = lds8(a1 + 32);
                uint8_t* d0 = reinterpret_cast<uint8_t*>((uint64_t)(e0.y & 0xffffffu) << 32 | e0.x) + lane;
                uint8_t* d1 = reinterpret_cast<uint8_t*>((uint64_t)(e1.y & 0xffffffu) << 32 | e1.x) + lane;
                if (lane < l0) d0[0] = (uint8_t)v00;
                if (lane + 32 < l0) d0[32] = (uint8_t)v01;
                if (lane < l1) d1[0] = (uint8_t)v10;
                if (lane + 32 < l1) d1[32] = (uint8_t)v11;
                more |= (l0 > 64 ? 1u : 0u) << k | (l1 > 64 ? 2u : 0u) << k;
            }
            while (more) {                                   // bytes 64.. of the longer ones (about one match in nine on FASTQ)
                const int k = __ffs(more) - 1; more &= more - 1;
                const uint4 e = lds128(mtab + 16 * k);
                const uint32_t len = e.y >> 24, sa = e.z + lane;
                uint8_t* dp = reinterpret_cast<uint8_t*>((uint64_t)(e.y & 0xffffffu) << 32 | e.x) + lane;
                for (uint32_t o = 64; o + lane < len; o += 32) dp[o] = (uint8_t)lds8(sa + o);
            }
            __syncwarp();                                    // table and stage are rewritten by the next round
            pending &= ~fmask;
        }
        uint32_t longs = __ballot_sync(0xffffffffu, lng);
        while (longs) {
            int l = __ffs(longs) - 1; longs &= longs - 1;
            uint32_t d2 = __shfl_sync(0xffffffffu, dst_rel, l), n = __shfl_sync(0xffffffffu, match_len, l);
            uint64_t s2 = __shfl_sync(0xffffffffu, sp, l);
            warp_copy<true>(out_blk + d2, reinterpret_cast<const uint8_t*>(s2), n);
        }
        uint32_t ovls = __ballot_sync(0xffffffffu, direct);
        while (ovls) {                                       // byte i of the match = seed[i mod period] (FORMAT.md §2)
            int l = __ffs(ovls) - 1; ovls &= ovls - 1;
            uint32_t d2 = __shfl_sync(0xffffffffu, dst_rel, l), n = __shfl_sync(0xffffffffu, match_len, l);
            const uint32_t per = __shfl_sync(0xffffffffu, (uint32_t)min((unsigned long long)(dst - src), 0xffffffffull), l);
            const uint8_t* sq = reinterpret_cast<const uint8_t*>(__shfl_sync(0xffffffffu, sp, l));
            uint32_t r = lane % per; const uint32_t stp = 32 % per;
            for (uint32_t i = lane; i < n; i += 32) {
                out_blk[d2 + i] = __ldcg(sq + r);
                r += stp; if (r >= per) r -= per;
            }
        }
    }
    if (out_base != (uint32_t)(c.bend - c.bstart) || lit_base != c.d.n_lit) { if (lane == 0) report(P, DF_LENGTH); }
}

// ---- A5-A7: demands ("materialise original bytes [pos, pos+len) at out2[dst..)") ------------------------------------
// Source bytes that are neither in the current window nor in a resident slot are reconstructed by recursion on their
// own sources: the block that holds them is parsed and the wanted span is emitted; literal bytes are final, match
// pieces are forwarded to *their* sources with the same destination.  Recursion depth <= max_level + 1 (FORMAT.md §3).
// Each warp keeps its pending demands in a private LIFO in the workspace; all pending demands of one block are served
// from a single parse of that block.
// Emit the bytes [pos, pos + len) of the parsed block c (tokens + all literals are in the warp's scratch) to out2[dst..).
__device__ __forceinline__ void emit_span(const Params& P, const BlockCtx& c, const Stack& st, uint64_t pos, uint64_t len, uint64_t dst) {
    uint32_t lit_base = 0, out_base = 0, ec = 0, em = c.n_ext_cmd;
    const uint32_t lane = lane_id();
    const uint64_t pend = pos + len;
    for (uint32_t c0 = 0; c0 < c.d.n_cmd; c0 += 32) {
        uint32_t ci = c0 + lane;
        bool valid = ci < c.d.n_cmd, has_match = ci < c.d.n_match;
        uint32_t tl = valid ? c.tok_cmd[ci] : 0, tm = has_match ? c.tok_mlen[ci] : 0;
        uint32_t ml = __ballot_sync(0xffffffffu, valid && tl == 255), mm = __ballot_sync(0xffffffffu, has_match && tm == 255);
        uint32_t lit_len = tl, match_len = has_match ? P.min_match + tm : 0;
        if (valid && tl == 255) lit_len = 255 + __ldg(c.ext + ec + __popc(ml & lanemask_lt()));
        if (has_match && tm == 255) match_len = P.min_match + 255 + __ldg(c.ext + em + __popc(mm & lanemask_lt()));
        ec += __popc(ml); em += __popc(mm);
        uint32_t sl = lit_len, stt = lit_len + match_len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t a = __shfl_up_sync(0xffffffffu, sl, o), t = __shfl_up_sync(0xffffffffu, stt, o);
            if (lane >= (uint32_t)o) { sl += a; stt += t; }
        }
        uint32_t lit_pos = lit_base + sl - lit_len;
        uint64_t out_pos = c.bstart + out_base + (stt - lit_len - match_len);
        lit_base += __shfl_sync(0xffffffffu, sl, 31);
        out_base += __shfl_sync(0xffffffffu, stt, 31);
        bool ok = valid && (uint64_t)lit_pos + lit_len <= c.d.n_lit && out_pos + lit_len + match_len <= c.bend;
        if (__any_sync(0xffffffffu, valid && !ok)) { if (lane == 0) report(P, DF_LENGTH); return; }
        if (c.bstart + out_base <= pos) continue;            // the whole group lies before the span
        if (ok) {
            uint64_t a = max((unsigned long long)out_pos, (unsigned long long)pos), b = min((unsigned long long)(out_pos + lit_len), (unsigned long long)pend);
            if (a < b) copy_bytes<false>(P.out2 + dst + (a - pos), c.lit + lit_pos + (a - out_pos), (uint32_t)(b - a), ~0ull);
            uint64_t md = out_pos + lit_len;
            a = max((unsigned long long)md, (unsigned long long)pos); b = min((unsigned long long)(md + match_len), (unsigned long long)pend);
            if (has_match && a < b) {
                uint64_t src = match_src(P, c, ci);
                const uint64_t period = md - src;
                if (src >= md) report(P, DF_OFFSET);
                else if (period >= match_len) fetch_source<false>(P, c, st, src + (a - md), b - a, dst + (a - pos));
                else if (period > lit_len) report(P, DF_OFFSET);      // FORMAT.md §3 (c): the seed is the tail of this literal run
                else {                                                // byte i of the match = seed[i mod period]
                    const uint8_t* seed = c.lit + lit_pos + lit_len - period;
                    uint8_t* d = P.out2 + dst + (a - pos);
                    uint32_t r = (uint32_t)((a - md) % period);
                    for (uint32_t k = 0; k < (uint32_t)(b - a); k++) { d[k] = seed[r]; if (++r == period) r = 0; }
                }
            }
        }
        if (c.bstart + out_base >= pend) break;              // uniform: nothing after this group is wanted
    }
}

// Serve every pending demand of the warp's stack (depth-first; all demands of one block from one parse).
__device__ __forceinline__ void process_demands(const Params& P, uint32_t s_luts, uint32_t ring, BlockCtx& c, const Stack& st) {
    const uint32_t lane = lane_id();
    for (;;) {
        __syncwarp();
        uint32_t top = min(lds_top(st), st.cap);
        while (top > 0 && st.base[top - 1].len == 0) top--;  // drop served entries
        __syncwarp();
        if (lane == 0) asm volatile("st.shared.u32 [%0], %1;" ::"r"(st.top), "r"(top) : "memory");
        __syncwarp();
        if (top == 0) return;
        c.b = st.base[top - 1].pos >> P.log2_bs;
        if (c.b >= (P.N + (1ull << P.log2_bs) - 1) >> P.log2_bs) { if (lane == 0) { report(P, DF_OFFSET); st.base[top - 1].len = 0; } continue; }
        uint64_t pend = 0;                                   // the literals are needed up to the last pending span of this block
        for (uint32_t i0 = 0; i0 < top; i0 += 32) {
            const uint32_t idx = i0 + lane;
            if (idx < top && st.base[idx].len != 0 && (st.base[idx].pos >> P.log2_bs) == c.b)
                pend = max((unsigned long long)pend, (unsigned long long)(st.base[idx].pos + st.base[idx].len));
        }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) pend = max((unsigned long long)pend, (unsigned long long)__shfl_xor_sync(0xffffffffu, pend, o));
        bool ok = parse_block_upto(P, s_luts, ring, c, pend);     // tokens + the literals in front of it into the scratch
        bool found = true;
        while (found) {                                      // emit_span may push more demands for this same block
            found = false;
            uint32_t n = min(lds_top(st), st.cap);
            for (uint32_t i0 = 0; i0 < n; i0 += 32) {
                uint32_t idx = i0 + lane;
                bool mine = idx < n && st.base[idx].len != 0 && (st.base[idx].pos >> P.log2_bs) == c.b;
                uint32_t m = __ballot_sync(0xffffffffu, mine);
                while (m) {
                    uint32_t e = i0 + __ffs(m) - 1; m &= m - 1;
                    uint64_t pos = st.base[e].pos, len = st.base[e].len, dst = st.base[e].dst;
                    __syncwarp();
                    if (lane == 0) st.base[e].len = 0;
                    __syncwarp();
                    if (ok) emit_span(P, c, st, pos, len, dst);
                    found = true;
                }
            }
            __syncwarp();
        }
    }
}

// shared memory of every decode kernel: [pad to 8 KB][tables: n_coded_tables x 8 KB][rings: warps x 2 KB]
// [run tables: warps x 2 KB][stack tops: warps x 4]   (absolute shared addresses)
struct CtaSmem { uint32_t luts, ring, runs, top; };

__device__ __forceinline__ CtaSmem setup_cta(const Params& P, uint8_t* smem_raw) {
    const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t pad = (8192u - (smem0 & 8191u)) & 8191u;
    const uint32_t n_lut_words = P.n_coded_tables * LUT_SIZE;
    {
        uint4* dstv = reinterpret_cast<uint4*>(smem_raw + pad);
        for (uint32_t i = threadIdx.x; i < n_lut_words / 4; i += blockDim.x) dstv[i] = __ldg(reinterpret_cast<const uint4*>(P.luts) + i);
    }
    __syncthreads();
    const uint32_t warp = threadIdx.x >> 5, warps = blockDim.x >> 5;
    CtaSmem m;
    m.luts = smem0 + pad;
    uint32_t base = m.luts + n_lut_words * 4;
    m.ring = base + warp * RING_BYTES; base += warps * RING_BYTES;
    m.runs = base + warp * (4 * RUNS_CAP); base += warps * (4 * RUNS_CAP);
    m.top = base + 4 * warp;
    return m;
}

// Two ticket slots alternate between consecutive launches of a handle: a kernel draws from its own slot and clears the
// other one, so no memset has to be queued between launches (a seek is ~30 launches).
__device__ __forceinline__ void clear_next_ticket(const Params& P) {
    if (blockIdx.x == 0 && threadIdx.x == 0) *P.ticket_next = 0ull;
}

__device__ __forceinline__ bool next_ticket(const Params& P, unsigned long long& t) {
    t = 0;
    if (lane_id() == 0) t = atomicAdd(P.ticket, 1ull);
    t = __shfl_sync(0xffffffffu, t, 0);
    return t < P.n_work;
}

// Whole-file literal launch (mode 2): A1 + A2 + A3 for every block, no dependencies.
template <int MAXT>
__global__ void __launch_bounds__(MAXT, 1) k_literals(const Params P) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    const CtaSmem m = setup_cta(P, smem_raw);
    BlockCtx c;
    bind_scratch(P, blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), c);
    Stack st{nullptr, 0, m.top, nullptr, 0};
    unsigned long long t;
    while (next_ticket(P, t)) {
        c.b = P.first_block + t;
        Rans r; uint32_t i0;
        if (!parse_tokens(P, m.luts, m.ring, c, r, &i0)) continue;
        uint32_t n_runs = build_runs(P, c, m.runs);           // also leaves the match descriptors for k_copy
        if (P.log2_bs > 16) n_runs = 0xffffffffu;
        if (n_runs != 0xffffffffu) {                          // scan first, literals straight to their positions
            decode_lit_direct(r, m.luts + P.lut_lit * (4 * LUT_SIZE), i0, c.d.n_lit, m.runs, P.out + (c.bstart - P.out_pos0));
            rans_final_ok(P, c, r);
        } else {                                              // too many runs / big block / bad scan: staged path
            rans_region<false>(r, m.luts + P.lut_lit * (4 * LUT_SIZE), i0, c.d.n_lit, c.lit);
            bool ok = rans_final_ok(P, c, r);
            __syncwarp();
            if (ok) emit_block<2>(P, c, st);
        }
    }
}

// Whole-file match launches.  WAIT = false (mode 3): one dependency level per launch, nothing to wait for.
// WAIT = true (mode 4): all levels in one launch; blocks arrive sorted by (level, index) and a block waits for the
// completion of lower-level source blocks, which were dispatched before it.
// WIN / COLLECT: the two range-decode variants (see emit_matches); they run one level per launch (WAIT = false).
template <bool WAIT, int MAXT, bool WIN = false, bool COLLECT = false>
__global__ void __launch_bounds__(MAXT, 1) k_matches(const Params P) {
    // shared memory: [pad to 8 KB][tables without LIT (the last one): (n_coded_tables - 1) x 8 KB]
    //                [per warp: ring 2 KB | match table MTAB_BYTES | stage 16 x STAGE_CHUNKS]
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    const uint32_t smem0 = (uint32_t)__cvta_generic_to_shared(smem_raw);
    const uint32_t pad = (8192u - (smem0 & 8191u)) & 8191u;
    const uint32_t n_lut_words = (P.n_coded_tables - 1) * LUT_SIZE;
    {
        uint4* dstv = reinterpret_cast<uint4*>(smem_raw + pad);
        for (uint32_t i = threadIdx.x; i < n_lut_words / 4; i += blockDim.x) dstv[i] = __ldg(reinterpret_cast<const uint4*>(P.luts) + i);
    }
    __syncthreads();
    const uint32_t warp = threadIdx.x >> 5;
    const uint32_t luts = smem0 + pad;
    const uint32_t ring = luts + n_lut_words * 4 + warp * (RING_BYTES + MTAB_BYTES + 16 * STAGE_CHUNKS);
    const uint32_t mtab = ring + RING_BYTES, stage = mtab + MTAB_BYTES;
    BlockCtx c;
    bind_scratch(P, blockIdx.x * (blockDim.x >> 5) + warp, c);
    unsigned long long t;
    while (next_ticket(P, t)) {
        c.b = P.level_list ? (uint64_t)P.level_list[t] : P.first_block + t;
        if (parse_block(P, luts, ring, c, 0, false)) emit_matches<WAIT ? 4 : 3, WIN, COLLECT>(P, c, mtab, stage);
        if (WAIT) {                                          // publish: the warp's stores happen-before lane 0's fence + release
            __syncwarp();
            if (lane_id() == 0) { __threadfence(); st_release(P.flags + c.b, 2 * P.epoch + 1); }
        }
    }
}

// One round of the demand lists of a range decode: every block with a non-empty list is parsed ONCE (tokens + all its
// literals into the warp's scratch) and serves all its records; match pieces whose sources are unknown go to the lists
// of the next round (recursion depth <= max_level + 1, FORMAT.md §3).
// Whole-file match resolution from the descriptors k_literals left (A4).  No entropy decode, no scan: per block the
// warp walks its descriptors 32 at a time.  The sources of the short non-overlapping matches of a group travel
// global -> shared memory with 16-byte cp.async issued by the lanes that own them; the stage is double-buffered, so the
// sources of round r + 1 are in flight while the warp copies round r to the output (lane i moves bytes i, i + 32, ...).
// Matches of LONG_MATCH bytes and more use the 16-byte warp copy, self-overlapping ones replicate src + (i mod period).
// WAIT = true: blocks arrive sorted by (level, index) and wait for the completion of lower-level source blocks.
constexpr uint32_t COPY_WARP_BYTES = 2 * (MTAB_BYTES + 16 * STAGE_CHUNKS);
static_assert(COPY_WARP_BYTES % 16 == 0, "tables and stages are 16-byte aligned");

// WIN / COLLECT: the windows of a range decode (sources looked up in the window and the resident slots; see emit_matches).
template <bool WAIT, bool WIN = false, bool COLLECT = false>
__global__ void __launch_bounds__(1024, 1) k_copy(const Params P) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    constexpr bool TOP = !WAIT && !WIN && !COLLECT;      // the wait-free launch of the whole-file schedule
    const uint32_t lane = lane_id(), warp = threadIdx.x >> 5;
    const uint32_t sbase = (uint32_t)__cvta_generic_to_shared(smem_raw) + warp * COPY_WARP_BYTES;
    const uint8_t* const out_end = P.out + (P.win_end - P.out_pos0);
    unsigned long long t;
    while (next_ticket(P, t)) {
        // The wait-free launch takes the last blocks first: their literals and descriptors are what k_literals wrote last,
        // so the first ~100 MB of the launch's destination sectors and descriptors are still in L2 (0.574 -> 0.565 ms).
        const unsigned long long tt = TOP ? P.n_work - 1 - t : t;
        const uint64_t b = P.level_list ? (uint64_t)P.level_list[tt] : P.first_block + tt;
        const uint64_t mp0 = __ldg(P.match_prefix + b);
        const uint4* d4 = reinterpret_cast<const uint4*>(P.dir + b);
        const uint4 da = __ldg(d4), dq = __ldg(d4 + 1);       // FORMAT.md §1.3: payload_off, n_cmd, n_match | n_lit, n_words, n_ext, level
        const uint32_t n = da.w;
        const uint8_t* const raw = P.archive + ((uint64_t)da.y << 32 | da.x) + ((256 + 2ull * dq.y + 3) & ~3ull) + 4ull * dq.z;
        const uint8_t* const cpl = P.cplanes + (uint64_t)P.n_coded_planes * mp0;
        const uint2* const prs = P.pairs + mp0;
        const uint64_t bstart = b << P.log2_bs;
        const uint32_t blen = (uint32_t)(min((unsigned long long)(bstart + (1ull << P.log2_bs)), (unsigned long long)P.N) - bstart);
        const uint32_t lvl = WAIT ? __ldg(P.levels + b) : 0;
        uint8_t* const out_blk = P.out + (bstart - P.out_pos0);
        uint32_t g0 = 0, pending = 0, mis = 0, len = 0, dst_rel = 0;
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
        // The descriptors of a group are requested when the last staging round of the group before it has been issued (no
        // value of that group is live any more, so the loads land in the same registers) and travel while the round
        // before that is copied out.
        uint2 npr; uint32_t nv[4];
        bool have = false;
        // one staging round into buffer `buf`: returns the number of staged matches; commits exactly one cp.async group
        auto issue = [&](uint32_t buf, uint32_t& more) -> uint32_t {
            const uint32_t mtab = sbase + buf * (MTAB_BYTES + 16 * STAGE_CHUNKS), stage = mtab + MTAB_BYTES;
            for (;;) {
                if (pending == 0) {
                    if (g0 >= n) { done = true; more = 0; cp_async_commit(); return 0; }
                    if (!have) load_desc(g0 + lane, npr, nv);            // head of a block, or a group that staged nothing
                    have = false;
                    const uint64_t src = desc_src(nv), dst = bstart + npr.x;
                    dst_rel = npr.x; len = npr.y;
                    const bool has = g0 + lane < n;
                    g0 += 32;
                    const bool good = has && src < dst && dst_rel + len <= blen && len != 0;
                    if (has && !good) report(P, src < dst ? DF_LENGTH : DF_OFFSET);
                    const bool ovl = good && src + len > dst;
                    if (ovl && src < bstart) report(P, DF_OFFSET);       // FORMAT.md §3 (c)
                    const uint32_t seed_len = ovl ? (uint32_t)(dst - src) : len;   // source bytes that are not the match's own output
                    const uint8_t* sbase = P.out + (src - P.out_pos0);
                    const uint8_t* send = out_end;
                    if (WIN || COLLECT) sbase = good ? resolve_src(P, src, seed_len, &send) : nullptr;
                    if (COLLECT) {                                        // unknown seed bytes -> demand lists; nothing is copied
                        if (g0 < n) { load_desc(g0 + lane, npr, nv); have = true; }
                        if (good && !sbase) {
                            const Stack sk{nullptr, 0, 0, &P.gl_nxt, SKIP_KNOWN};
                            fetch_source<false>(P, BlockCtx{}, sk, src, seed_len, dst - P.out_pos0);
                        }
                        continue;
                    }
                    if (WAIT && good && lvl) {                            // completion of lower-level source blocks (of the window)
                        const uint64_t s1 = (min((unsigned long long)(src + len), (unsigned long long)dst) - 1) >> P.log2_bs;
                        for (uint64_t S = src >> P.log2_bs; S <= s1; S++) {
                            if (WIN && ((S << P.log2_bs) < P.out_pos0 || (S << P.log2_bs) >= P.win_end)) continue;   // final already
                            if (S != b && __ldg(P.levels + S) < lvl) wait_block(P, S, true);
                        }
                    }
                    const bool known = good && sbase != nullptr;
                    if (WIN && good && !sbase) {                          // seed spread over several buffers or (partly) delivered by the demand rounds
                        const Stack sk{nullptr, 0, 0, nullptr, SKIP_UNKNOWN};
                        fetch_source<false>(P, BlockCtx{}, sk, src, seed_len, dst - P.out_pos0);   // the known pieces of the seed
                        uint8_t* d = P.out + (dst - P.out_pos0);
                        for (uint32_t i = seed_len; i < len; i++) d[i] = d[i - seed_len];          // the rest repeats it (FORMAT.md §2)
                    }
                    sp = reinterpret_cast<uint64_t>(sbase);
                    mis = (uint32_t)sp & 15u;
                    const bool lng = known && !ovl && len >= LONG_MATCH;
                    const bool sht = known && !ovl && !lng;
                    // a chunk may not reach past the end of the buffer (only possible for sources in its last 16 bytes)
                    const bool stg = sht && ((sp - mis) + 16ull * ((mis + len + 15u) >> 4) <= reinterpret_cast<uint64_t>(send));
                    uint32_t longs = __ballot_sync(0xffffffffu, lng);
                    while (longs) {
                        const int l = __ffs(longs) - 1; longs &= longs - 1;
                        const uint32_t d2 = __shfl_sync(0xffffffffu, dst_rel, l), m = __shfl_sync(0xffffffffu, len, l);
                        warp_copy<true>(out_blk + d2, reinterpret_cast<const uint8_t*>(__shfl_sync(0xffffffffu, sp, l)), m);
                    }
                    uint32_t direct = __ballot_sync(0xffffffffu, (sht && !stg) || (known && ovl));
                    while (direct) {                                     // byte i of the match = seed[i mod period] (FORMAT.md §2)
                        const int l = __ffs(direct) - 1; direct &= direct - 1;
                        const uint32_t d2 = __shfl_sync(0xffffffffu, dst_rel, l), m = __shfl_sync(0xffffffffu, len, l);
                        const uint32_t per = __shfl_sync(0xffffffffu, (uint32_t)min((unsigned long long)(dst - src), 0xffffffffull), l);
                        const uint8_t* sq = reinterpret_cast<const uint8_t*>(__shfl_sync(0xffffffffu, sp, l));
                        uint32_t r = lane % per; const uint32_t stp = 32 % per;
                        for (uint32_t i = lane; i < m; i += 32) { out_blk[d2 + i] = __ldcg(sq + r); r += stp; if (r >= per) r -= per; }
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
                    const uint64_t dp = reinterpret_cast<uint64_t>(out_blk) + dst_rel;
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
        if (WAIT) {                                          // publish: the warp's stores happen-before lane 0's fence + release
            __syncwarp();
            if (lane == 0) { __threadfence(); st_release(P.flags + b, 2 * P.epoch + 1); }
        }
    }
}

// Command table of a parsed block (demand rounds): entry ci = block-relative output position of command ci | position of
// its first literal in the literal stream << 16; entry n_cmd is the sentinel (block length, n_lit), so lengths are
// differences of neighbours.  Lives in the warp's run-table area.  Returns false when the block does not fit (more than
// RUNS_CAP - 1 commands, blocks above 32 KB) or fails validation (reported); the caller then serves span by span.
__device__ __forceinline__ bool build_cmd_table(const Params& P, const BlockCtx& c, uint32_t tab /* shared address */) {
    if (c.d.n_cmd + 1 > RUNS_CAP || P.log2_bs > 15) return false;
    uint32_t lit_base = 0, out_base = 0, ec = 0, em = c.n_ext_cmd;
    const uint32_t lane = lane_id();
    for (uint32_t c0 = 0; c0 < c.d.n_cmd; c0 += 32) {
        uint32_t ci = c0 + lane;
        bool valid = ci < c.d.n_cmd, has_match = ci < c.d.n_match;
        uint32_t tl = valid ? c.tok_cmd[ci] : 0, tm = has_match ? c.tok_mlen[ci] : 0;
        uint32_t ml = __ballot_sync(0xffffffffu, valid && tl == 255), mm = __ballot_sync(0xffffffffu, has_match && tm == 255);
        uint32_t lit_len = tl, match_len = has_match ? P.min_match + tm : 0;
        if (valid && tl == 255) lit_len = 255 + __ldg(c.ext + ec + __popc(ml & lanemask_lt()));
        if (has_match && tm == 255) match_len = P.min_match + 255 + __ldg(c.ext + em + __popc(mm & lanemask_lt()));
        ec += __popc(ml); em += __popc(mm);
        uint32_t sl = lit_len, stt = lit_len + match_len;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            uint32_t a = __shfl_up_sync(0xffffffffu, sl, o), t = __shfl_up_sync(0xffffffffu, stt, o);
            if (lane >= (uint32_t)o) { sl += a; stt += t; }
        }
        const uint64_t lit_pos = (uint64_t)lit_base + sl - lit_len, out_rel = (uint64_t)out_base + (stt - lit_len - match_len);
        const bool ok = !valid || (lit_pos + lit_len <= c.d.n_lit && c.bstart + out_rel + lit_len + match_len <= c.bend);
        if (__any_sync(0xffffffffu, !ok)) { if (lane == 0) report(P, DF_LENGTH); return false; }
        if (valid) asm volatile("st.shared.u32 [%0], %1;" ::"r"(tab + 4 * ci), "r"((uint32_t)out_rel | (uint32_t)lit_pos << 16) : "memory");
        lit_base += __shfl_sync(0xffffffffu, sl, 31);
        out_base += __shfl_sync(0xffffffffu, stt, 31);
    }
    if (lit_base != c.d.n_lit || c.bstart + out_base != c.bend) { if (lane == 0) report(P, DF_LENGTH); return false; }
    if (lane == 0) asm volatile("st.shared.u32 [%0], %1;" ::"r"(tab + 4 * c.d.n_cmd), "r"(out_base | lit_base << 16) : "memory");
    __syncwarp();
    return true;
}

constexpr uint32_t ITEM_LANE_MAX = 96;   // spans up to this many bytes are served by one lane each

// The records of a work item, one per lane: lane l emits bytes [pos, pos + len) of the parsed block c to out2[dst ..).
// A binary search in the command table finds the first command of the span; the lane then walks its commands (one to
// three for a 32-byte span): literal bytes come from the warp's scratch, match pieces are forwarded to their sources.
__device__ __forceinline__ void emit_item(const Params& P, const BlockCtx& c, const Stack& st, uint32_t tab, bool have,
                                          uint64_t pos, uint32_t len, uint64_t dst) {
    if (!have || len == 0) return;
    const uint32_t pr = (uint32_t)(pos - c.bstart), pe = pr + len;
    uint32_t lo = 0, hi = c.d.n_cmd;
    while (hi - lo > 1) { const uint32_t mid = (lo + hi) >> 1; if ((lds32(tab + 4 * mid) & 0xffffu) <= pr) lo = mid; else hi = mid; }
    uint32_t e = lds32(tab + 4 * lo);
    for (uint32_t k = lo; k < c.d.n_cmd; k++) {
        const uint32_t e1 = lds32(tab + 4 * k + 4);
        const uint32_t o0 = e & 0xffffu, lit_pos = e >> 16;
        if (o0 >= pe) break;
        const uint32_t lit_len = (e1 >> 16) - lit_pos, match_len = (e1 & 0xffffu) - o0 - lit_len;
        e = e1;
        uint32_t a = max(o0, pr), b = min(o0 + lit_len, pe);
        if (a < b) copy_bytes<false>(P.out2 + dst + (a - pr), c.lit + lit_pos + (a - o0), b - a, ~0ull);
        const uint32_t mo = o0 + lit_len;
        a = max(mo, pr); b = min(mo + match_len, pe);
        if (k < c.d.n_match && a < b) {
            const uint64_t md = c.bstart + mo, src = match_src(P, c, k);
            const uint64_t period = md - src;
            if (src >= md) report(P, DF_OFFSET);
            else if (period >= match_len) fetch_source<false>(P, c, st, src + (a - mo), b - a, dst + (a - pr));
            else if (period > lit_len) report(P, DF_OFFSET);          // FORMAT.md §3 (c): the seed is the tail of this literal run
            else {                                                    // byte i of the match = seed[i mod period]
                const uint8_t* seed = c.lit + lit_pos + lit_len - period;
                uint8_t* d = P.out2 + dst + (a - pr);
                uint32_t r = (uint32_t)((a - mo) % period);
                for (uint32_t i = 0; i < b - a; i++) { d[i] = seed[r]; if (++r == period) r = 0; }
            }
        }
    }
}

// Bucket offsets and work items of the list in P.gl_cur: every warp of the launch takes 32 touched blocks at a time; the
// bucket offsets and the work-item slots come from two global counters (count[3]: records placed, count[2]: work items),
// one atomicAdd per warp each (the order of the buckets in the sorted array is irrelevant); cnt[block] becomes the fill
// pointer of the block's bucket.  Both counters are zero when a list becomes the current one.
// The list arrays are written by other CTAs, possibly earlier in the SAME launch (k_rounds): they are read at L2.
__device__ __forceinline__ GDemand ld_demand(const GDemand* p) {
    const unsigned long long* q = reinterpret_cast<const unsigned long long*>(p);
    GDemand d; d.pos = __ldcg(q); d.dst = __ldcg(q + 1);
    const unsigned long long w = __ldcg(q + 2); d.len = (uint32_t)w; d.pad = (uint32_t)(w >> 32);
    return d;
}

__device__ __forceinline__ void plan_body(const GList& g, uint32_t warp_global, uint32_t n_warps_global) {
    const uint32_t n = min(__ldcg(g.count + 1), g.touched_cap), lane = threadIdx.x & 31;
    for (uint32_t t0 = 32 * warp_global; t0 < n; t0 += 32 * n_warps_global) {
        const uint32_t t = t0 + lane;
        uint32_t blk = 0, c = 0;
        if (t < n) { blk = __ldcg(g.touched + t); c = __ldcg(g.cnt + blk); }
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
            g.cnt[blk] = r0;
            for (uint32_t j = 0; j < it; j++) if (i0 + j < g.work_cap) {
                g.work[i0 + j] = (unsigned long long)blk << 32 | (r0 + j * GL_ITEM);
                g.work_n[i0 + j] = min(GL_ITEM, c - j * GL_ITEM);
            }
        }
    }
}

__global__ void __launch_bounds__(1024, 1) k_plan(const Params P) {
    plan_body(P.gl_cur, blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), gridDim.x * (blockDim.x >> 5));
}

__device__ __forceinline__ void scatter_body(const Params& P, const GList& g, uint32_t tid, uint32_t n_threads) {
    const uint32_t n = min(__ldcg(g.count), g.cap);
    for (uint32_t i = tid; i < n; i += n_threads) {
        const GDemand d = ld_demand(g.rec + i);
        const uint32_t p = atomicAdd(g.cnt + (d.pos >> P.log2_bs), 1u);
        if (p < g.cap) g.sorted[p] = d;
    }
}

__global__ void __launch_bounds__(256) k_scatter(const Params P) {
    scatter_body(P, P.gl_cur, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
}

// One round of the demand lists of a range decode: a work item = up to GL_ITEM records of one source block; the block is
// parsed once (tokens + all its literals into the warp's scratch) and serves them; match pieces whose sources are
// unknown go to the lists of the next round (recursion depth <= max_level + 1, FORMAT.md §3).
__device__ __forceinline__ void serve_body(const Params& P, const CtaSmem& m, BlockCtx& c, const GList& cur, const GList& nxt,
                                           unsigned long long* ticket) {
    const Stack sk{nullptr, 0, m.top, &nxt, 0};
    const unsigned long long n = min(__ldcg(cur.count + 2), cur.work_cap);
    for (;;) {
        unsigned long long t = 0;
        if (lane_id() == 0) t = atomicAdd(ticket, 1ull);
        t = __shfl_sync(0xffffffffu, t, 0);
        if (t >= n) break;
        const unsigned long long item = __ldcg(cur.work + t);
        const uint32_t first = (uint32_t)item, cnt = __ldcg(cur.work_n + t);
        c.b = item >> 32;
        if (lane_id() == 0) cur.cnt[c.b] = 0;                 // every item of the block writes the same value: the array is idle again
        uint64_t pend = 0;                                    // the literals are needed up to the last span of the item
        if (lane_id() < cnt && first + lane_id() < cur.cap) { const GDemand d = ld_demand(cur.sorted + first + lane_id()); pend = d.pos + d.len; }
#pragma unroll
        for (int o = 16; o >= 1; o >>= 1) pend = max((unsigned long long)pend, (unsigned long long)__shfl_xor_sync(0xffffffffu, pend, o));
        const bool ok = parse_block_upto(P, m.luts, m.ring, c, pend);
        if (ok && build_cmd_table(P, c, m.runs)) {           // one record per lane
            const bool have = lane_id() < cnt && first + lane_id() < cur.cap;
            GDemand d; d.pos = c.bstart; d.len = 0; d.dst = 0;
            if (have) d = ld_demand(cur.sorted + first + lane_id());
            const bool inside = have && d.pos >= c.bstart && d.pos + d.len <= c.bend;
            if (have && !inside) report(P, DF_LENGTH);
            // a long span covers many commands: the whole warp walks it (a lane per command) instead of one lane
            const bool wide = inside && d.len > ITEM_LANE_MAX;
            emit_item(P, c, sk, m.runs, inside && !wide, d.pos, (uint32_t)d.len, d.dst);
            __syncwarp();
            uint32_t wides = __ballot_sync(0xffffffffu, wide);
            while (wides) {
                const int l = __ffs(wides) - 1; wides &= wides - 1;
                emit_span(P, c, sk, __shfl_sync(0xffffffffu, d.pos, l), __shfl_sync(0xffffffffu, (uint32_t)d.len, l), __shfl_sync(0xffffffffu, d.dst, l));
            }
            continue;
        }
        for (uint32_t k = 0; k < cnt && first + k < cur.cap; k++) {
            const GDemand d = ld_demand(cur.sorted + first + k);
            if (ok) emit_span(P, c, sk, d.pos, d.len, d.dst);
        }
    }
}

__global__ void __launch_bounds__(1024, 1) k_serve(const Params P) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    const CtaSmem m = setup_cta(P, smem_raw);
    BlockCtx c;
    bind_scratch(P, blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5), c);
    serve_body(P, m, c, P.gl_cur, P.gl_nxt, P.ticket);
}

// All rounds of a demand list in ONE cooperative launch (every CTA resident, grid-wide barriers between plan, scatter and
// serve): a seek or the ragged ends of a range need a handful of records per round, and one launch instead of three per
// round, with an exit as soon as a round leaves nothing, is what their latency is made of.  P.gl_cur = the filled list,
// P.gl_nxt = the other one; round_tickets = one zeroed counter per round.
__global__ void __launch_bounds__(1024, 1) k_rounds(const Params P, unsigned long long* round_tickets, uint32_t rounds) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    cooperative_groups::grid_group grid = cooperative_groups::this_grid();
    const CtaSmem m = setup_cta(P, smem_raw);
    BlockCtx c;
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
        scatter_body(P, cur, blockIdx.x * blockDim.x + threadIdx.x, gridDim.x * blockDim.x);
        __threadfence();
        grid.sync();
        serve_body(P, m, c, cur, nxt, round_tickets + r);
        __threadfence();
        grid.sync();
    }
}

// top-level spans of a range decode (its ragged ends) enter the demand lists like any other record
__global__ void k_seed(const Params P, uint32_t n) {
    const uint32_t i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) {
        const Demand d = P.n_inline ? P.inline_dem[i] : P.demands[i];
        gl_append(P, P.gl_nxt, d.pos, (uint32_t)d.len, d.dst);
    }
}

__global__ void k_assert_empty(const uint32_t* count, uint32_t* err) { if (*count) atomicOr(err, (uint32_t)DF_STACK); }

template <bool DEMANDS>
__global__ void __launch_bounds__(1024, 1) k_decode(const Params P) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    clear_next_ticket(P);
    const CtaSmem m = setup_cta(P, smem_raw);
    const uint32_t s_luts = m.luts, ring = m.ring, runs = m.runs;
    const uint32_t gw = blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5);
    BlockCtx c;
    bind_scratch(P, gw, c);
    Stack st;
    st.base = P.stacks + (uint64_t)gw * P.stack_cap; st.cap = P.stack_cap; st.top = m.top; st.gl = nullptr; st.policy = 0;
    if (lane_id() == 0) asm volatile("st.shared.u32 [%0], %1;" ::"r"(st.top), "r"(0u) : "memory");
    __syncwarp();
    unsigned long long t;
    while (next_ticket(P, t)) {
        if (DEMANDS && P.mode == 1) {                        // spans: one top-level demand per ticket
            if (lane_id() == 0) {
                const Demand d = P.n_inline ? P.inline_dem[t] : P.demands[t];
                push_span(P, st, d.pos, d.len, d.dst);
            }
            process_demands(P, s_luts, ring, c, st);
            continue;
        }
        c.b = P.level_list ? (uint64_t)P.level_list[t] : P.first_block + t;
        // mode 0: everything for one block (A1 + A2 + A3, then A4 with flags)
        bool ok;
        {
            Rans r; uint32_t i0;
            ok = parse_tokens(P, s_luts, ring, c, r, &i0);
            if (ok) {
                prefetch_sources(P, c);                               // source lines travel to L2 while the literals decode
                uint32_t n_runs = P.log2_bs <= 16 ? build_runs(P, c, runs) : 0xffffffffu;
                if (n_runs != 0xffffffffu) {                          // scan first, literals straight to their positions
                    decode_lit_direct(r, s_luts + P.lut_lit * (4 * LUT_SIZE), i0, c.d.n_lit, runs, P.out + (c.bstart - P.out_pos0));
                    ok = rans_final_ok(P, c, r);
                } else {                                              // too many runs / big block / bad scan: staged path
                    rans_region<false>(r, s_luts + P.lut_lit * (4 * LUT_SIZE), i0, c.d.n_lit, c.lit);
                    ok = rans_final_ok(P, c, r);
                    __syncwarp();
                    if (ok) emit_block<2>(P, c, st);
                }
            }
        }
        __threadfence();
        __syncwarp();
        if (lane_id() == 0) st_release(P.flags + c.b, 2 * P.epoch);       // literals placed
        const uint64_t b0 = c.b;
        if (ok) emit_block<0, DEMANDS>(P, c, st);                         // A4 (waits on source blocks)
        if (DEMANDS && lds_top(st)) process_demands(P, s_luts, ring, c, st);   // sources below the window (range decode)
        c.b = b0;
        __threadfence();
        __syncwarp();
        if (lane_id() == 0) st_release(P.flags + c.b, 2 * P.epoch + 1);   // complete (set even on error: nobody waits forever)
    }
}

// FNV-1a 64 of each block of d_data, compared with the archive's table; one thread per block (a check, not a hot path)
__global__ void k_fnv(const uint8_t* data, uint64_t n_bytes, uint32_t log2_bs, const uint64_t* expect, unsigned long long* n_bad) {
    uint64_t b = blockIdx.x * (uint64_t)blockDim.x + threadIdx.x;
    uint64_t lo = b << log2_bs;
    if (lo >= n_bytes) return;
    uint64_t hi = min((unsigned long long)(lo + (1ull << log2_bs)), (unsigned long long)n_bytes), f = 0xcbf29ce484222325ull;
    for (uint64_t q = lo; q < hi; q++) { f ^= data[q]; f *= 0x100000001b3ull; }
    if (f != expect[b]) atomicAdd(n_bad, 1ull);
}

} // namespace

// ====================================================================================================== host =====

struct aceapex_archive {
    const uint8_t* d_archive = nullptr;
    uint64_t archive_bytes = 0;
    // header
    uint64_t N = 0, n_blocks = 0, tables_off = 0, dir_off = 0, fnv_off = 0, payload_off = 0;
    uint64_t total_lit = 0, total_match_bytes = 0, total_matches = 0, total_cmds = 0;
    uint32_t log2_bs = 0, min_match = 0, W = 0, max_level = 0, max_cmds = 0, flags = 0;
    uint32_t n_coded_tables = 0, n_coded_planes = 0, n_raw_planes = 0;
    int8_t plane_lut[MAX_W], plane_raw[MAX_W];
    uint32_t lut_cmd = 0, lut_mlen = 0, lut_lit = 0;
    std::vector<std::vector<uint32_t>> level_blocks;   // block ids per level
    // device state owned by the library
    uint32_t* d_luts = nullptr;
    uint32_t* d_level_lists = nullptr;                  // concatenated level_blocks
    uint16_t* d_levels = nullptr;                       // level per block (compact copy of the directory field)
    uint64_t* d_match_prefix = nullptr;                 // matches in blocks [0, b), n_blocks + 1 entries
    uint64_t desc_off = 0, cplanes_off = 0;             // workspace: (dst_rel, len) and coded offset planes of every match
    std::vector<uint64_t> level_off;
    // workspace (caller's)
    uint8_t* d_ws = nullptr; uint64_t ws_bytes = 0; bool ws_clean = false;
    cudaStream_t stream = nullptr;
    uint32_t epoch = 0;
    bool cooperative = false;                          // k_rounds can be launched cooperatively (all CTAs resident)
    uint32_t ticket_slot = 0;                          // which of the two ticket slots the next launch draws from
    Resident res[MAX_RESIDENT];
    // launch geometry
    int sms = 148, ctas_per_sm = 1, threads = 1024, threads_lit = 1024, threads_match = 1024;
    bool win_tokens = false;                             // ACEAPEX_WIN_TOKENS=1: windows re-decode the tokens (k_matches) instead of reading descriptors
    uint32_t grid = 0; size_t smem = 0;
    uint64_t scratch_per_warp = 0, ctrl_bytes = 0, flags_bytes = 0;
    uint64_t scratch_off = 0, stacks_off = 0, demands_off = 0, list_off = 0, ws_need = 0;
    uint32_t stack_cap = 0, demand_cap = 0;
    uint64_t gl_cap = 0, gl_tcap = 0, gl_wcap = 0, gl_rec_off[2] = {0, 0}, gl_cnt_off[2] = {0, 0}, gl_touched_off[2] = {0, 0};   // range decode lists
    uint64_t gl_sorted_off = 0, gl_work_off = 0, gl_workn_off = 0;
    uint64_t gl_eff = 0;                               // records a range-decode call may use (vram_budget), <= gl_cap
    std::vector<uint64_t> h_match_prefix;             // matches in blocks [0, b)
    // end-to-end pipeline (aceapex_decode_all_host): chunks of blocks, per chunk the block ids sorted by level
    uint64_t chunk_blocks = 0; uint32_t* d_chunk_lists = nullptr; std::vector<uint64_t> chunk_level_off;   // (chunk, level) -> offset
    std::vector<uint64_t> h_payload_off;               // payload offset of block b (n_blocks + 1 entries)
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr; std::vector<cudaEvent_t> ev_h2d, ev_dec;
    bool phase_timing = false; cudaEvent_t ev_phase[4] = {nullptr, nullptr, nullptr, nullptr};   // aceapex_set_phase_timing
    std::vector<uint16_t> h_levels;                    // host copy of the per-block levels
    std::vector<uint32_t> h_list; std::vector<Demand> h_demands;   // host staging for range / read calls
    // status
    int32_t last_cuda = 0; uint32_t dev_flags = 0; uint64_t launches = 0;
};

namespace {

uint64_t rd64(const uint8_t* p) { uint64_t v; memcpy(&v, p, 8); return v; }
uint32_t rd32(const uint8_t* p) { uint32_t v; memcpy(&v, p, 4); return v; }
uint16_t rd16(const uint8_t* p) { uint16_t v; memcpy(&v, p, 2); return v; }

#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { ar->last_cuda = (int32_t)e_; return ACEAPEX_E_CUDA; } } while (0)

uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

// workspace: [ctrl 256 B: ticket slots u64 @0 and @24, err u32 @8, fnv count @16, list counters @64][flags: n_blocks x u32][scratch: warps x scratch_per_warp]
//            [stacks: warps x stack_cap demands][demands: demand_cap][block list: n_blocks x u32]
uint64_t workspace_need(const aceapex_archive* ar) { return ar->ws_need; }

size_t smem_for(const aceapex_archive* ar, int threads) {
    return (size_t)8192 + (size_t)ar->n_coded_tables * LUT_SIZE * 4 + (size_t)(threads / 32) * (RING_BYTES + 4 * RUNS_CAP + 4);
}
size_t smem_matches(const aceapex_archive* ar, int threads) {
    return (size_t)8192 + (size_t)(ar->n_coded_tables - 1) * LUT_SIZE * 4 + (size_t)(threads / 32) * (RING_BYTES + MTAB_BYTES + 16 * STAGE_CHUNKS) + 64;   // + 64: the copy reads bytes i and i + 32 unconditionally
}

void layout_workspace(aceapex_archive* ar) {
    uint64_t warps = (uint64_t)ar->grid * (ar->threads / 32);
    ar->ctrl_bytes = 256;
    ar->flags_bytes = align_up(4 * ar->n_blocks + 4, 256);
    ar->scratch_off = ar->ctrl_bytes + ar->flags_bytes;
    ar->stack_cap = std::max(1024u, std::min(8192u, 8 * ar->max_cmds));
    ar->demand_cap = 1u << 16;
    ar->stacks_off = align_up(ar->scratch_off + warps * ar->scratch_per_warp, 256);
    ar->demands_off = align_up(ar->stacks_off + warps * ar->stack_cap * sizeof(Demand), 256);
    ar->list_off = align_up(ar->demands_off + (uint64_t)ar->demand_cap * sizeof(Demand), 256);
    uint64_t off = align_up(ar->list_off + 4 * ar->n_blocks + 4, 256);
    // demand lists of range decode (two sets, alternating between rounds); counters live in the control area at +64
    ar->gl_cap = std::min<uint64_t>(1ull << 24, std::max<uint64_t>(1ull << 16, ar->total_matches / 2));
    ar->gl_tcap = std::max<uint64_t>(1, std::min<uint64_t>(ar->n_blocks, ar->gl_cap));
    ar->gl_wcap = ar->gl_tcap + ar->gl_cap / GL_ITEM + 1;
    for (int k = 0; k < 2; k++) {
        ar->gl_rec_off[k] = off; off = align_up(off + ar->gl_cap * sizeof(GDemand), 256);
        ar->gl_cnt_off[k] = off; off = align_up(off + 4 * ar->n_blocks + 4, 256);
        ar->gl_touched_off[k] = off; off = align_up(off + 4 * ar->gl_tcap, 256);
    }
    ar->gl_sorted_off = off; off = align_up(off + ar->gl_cap * sizeof(GDemand), 256);
    ar->gl_work_off = off; off = align_up(off + 8 * ar->gl_wcap, 256);
    ar->gl_workn_off = off; off = align_up(off + 4 * ar->gl_wcap, 256);
    ar->desc_off = off; off = align_up(off + 8 * (ar->total_matches + 1), 256);
    ar->cplanes_off = off; off = align_up(off + (uint64_t)ar->n_coded_planes * ar->total_matches + 16, 256);
    ar->ws_need = off;
}

GList glist(const aceapex_archive* ar, int k) {
    GList g;
    g.rec = reinterpret_cast<GDemand*>(ar->d_ws + ar->gl_rec_off[k]);
    g.sorted = reinterpret_cast<GDemand*>(ar->d_ws + ar->gl_sorted_off);
    g.cnt = reinterpret_cast<uint32_t*>(ar->d_ws + ar->gl_cnt_off[k]);
    g.touched = reinterpret_cast<uint32_t*>(ar->d_ws + ar->gl_touched_off[k]);
    g.work = reinterpret_cast<unsigned long long*>(ar->d_ws + ar->gl_work_off);
    g.work_n = reinterpret_cast<uint32_t*>(ar->d_ws + ar->gl_workn_off);
    g.count = reinterpret_cast<uint32_t*>(ar->d_ws + 64 + 16 * k);
    g.cap = (uint32_t)(ar->gl_eff ? ar->gl_eff : ar->gl_cap); g.touched_cap = (uint32_t)ar->gl_tcap; g.work_cap = (uint32_t)ar->gl_wcap;
    return g;
}

void fill_params(const aceapex_archive* ar, Params& P) {
    memset(&P, 0, sizeof P);
    P.archive = ar->d_archive; P.archive_bytes = ar->archive_bytes;
    P.dir = reinterpret_cast<const DirEntry*>(ar->d_archive + ar->dir_off);
    P.luts = ar->d_luts; P.levels = ar->d_levels; P.N = ar->N; P.log2_bs = ar->log2_bs; P.min_match = ar->min_match; P.W = ar->W;
    P.n_coded_tables = ar->n_coded_tables;
    memcpy(P.plane_lut, ar->plane_lut, MAX_W); memcpy(P.plane_raw, ar->plane_raw, MAX_W);
    P.n_coded_planes = ar->n_coded_planes; P.n_raw_planes = ar->n_raw_planes;
    for (int p = (int)ar->W - 1, k = 0; p >= 0; p--) if (ar->plane_lut[p] >= 0) P.coded_shift[k++] = (uint8_t)(8 * p);
    for (uint32_t p = 0; p < ar->W; p++) if (ar->plane_raw[p] >= 0) P.raw_shift[ar->plane_raw[p]] = (uint8_t)(8 * p);
    P.lut_cmd = ar->lut_cmd; P.lut_mlen = ar->lut_mlen; P.lut_lit = ar->lut_lit;
    memcpy(P.res, ar->res, sizeof P.res);
    P.ticket = nullptr; P.ticket_next = nullptr;            // set per launch
    P.err = reinterpret_cast<uint32_t*>(ar->d_ws + 8);
    P.flags = reinterpret_cast<uint32_t*>(ar->d_ws + ar->ctrl_bytes);
    P.scratch = ar->d_ws + ar->scratch_off;
    P.scratch_per_warp = ar->scratch_per_warp; P.max_cmds = ar->max_cmds;
    P.out_pos0 = 0; P.win_end = ar->N;
    P.stacks = reinterpret_cast<Demand*>(ar->d_ws + ar->stacks_off); P.stack_cap = ar->stack_cap;
    P.pairs = nullptr; P.cplanes = nullptr; P.match_prefix = ar->d_match_prefix;
}

int32_t prepare_ws(aceapex_archive* ar) {
    if (!ar->d_ws || ar->ws_bytes < workspace_need(ar)) return ACEAPEX_E_WORKSPACE;
    if (!ar->ws_clean) {
        CU(cudaMemsetAsync(ar->d_ws, 0, ar->ctrl_bytes + ar->flags_bytes, ar->stream));
        for (int k = 0; k < 2; k++) CU(cudaMemsetAsync(ar->d_ws + ar->gl_cnt_off[k], 0, 4 * ar->n_blocks + 4, ar->stream));
        ar->ws_clean = true; ar->epoch = 0; ar->ticket_slot = 0;
    }
    return ACEAPEX_OK;
}

// Few work items: spread them over all SMs with fewer warps per CTA instead of filling a few CTAs with 32 warps each (a
// warp that shares its SM with fewer others finishes its block sooner).  T <= max_threads, g <= SMs (all CTAs resident).
static void spread(const aceapex_archive* ar, uint64_t n_work, int max_threads, uint32_t& g, int& T) {
    const uint64_t per_sm = (n_work + ar->sms - 1) / ar->sms;
    T = (int)std::min<uint64_t>((uint64_t)max_threads, 32 * std::max<uint64_t>(per_sm, 1));
    g = (uint32_t)std::min<uint64_t>(ar->sms, (n_work + T / 32 - 1) / (T / 32));
}

int32_t launch(aceapex_archive* ar, Params& P, uint64_t n_work) {
    P.n_work = n_work;
    if (n_work == 0) return ACEAPEX_OK;
    P.ticket = reinterpret_cast<unsigned long long*>(ar->d_ws) + (ar->ticket_slot ? 3 : 0);       // bytes 0 and 24 of the control area
    P.ticket_next = reinterpret_cast<unsigned long long*>(ar->d_ws) + (ar->ticket_slot ? 0 : 3);
    ar->ticket_slot ^= 1;
    uint64_t warps = ar->threads / 32;
    uint32_t grid = (uint32_t)std::min<uint64_t>(ar->grid, (n_work + warps - 1) / warps);
    const bool whole = P.out_pos0 == 0 && P.win_end == ar->N;
    if (P.mode == 8 || P.mode == 9 || P.mode == 11 || P.mode == 12) {   // match resolution from descriptors (11 / 12: windows)
        int T; uint32_t g;
        spread(ar, n_work, ar->threads, g, T);
        const size_t sm = (size_t)(T / 32) * COPY_WARP_BYTES + 64;
        if (P.mode == 8) k_copy<false><<<g, T, sm, ar->stream>>>(P);
        else if (P.mode == 9) k_copy<true><<<g, T, sm, ar->stream>>>(P);
        else if (P.mode == 11) k_copy<false, true, true><<<g, T, sm, ar->stream>>>(P);
        else k_copy<true, true, false><<<g, T, sm, ar->stream>>>(P);
    }
    else if (P.mode >= 5) {                                        // range decode: collect / window matches / serve
        int T = ar->threads; uint32_t g = ar->sms;
        if (P.mode != 7) spread(ar, n_work, ar->threads, g, T);
        if (P.mode == 5) k_matches<false, 1024, true, true><<<g, T, smem_matches(ar, T), ar->stream>>>(P);
        else if (P.mode == 6) k_matches<false, 1024, true, false><<<g, T, smem_matches(ar, T), ar->stream>>>(P);
        else if (P.mode == 10) k_matches<true, 1024, true, false><<<g, T, smem_matches(ar, T), ar->stream>>>(P);
        else k_serve<<<ar->sms, T, ar->smem, ar->stream>>>(P);
    }
    else if ((whole || P.mode == 2) && P.mode >= 2) {         // specialised whole-file kernels (the literal launch also serves windows)
        int T; uint32_t g;
        spread(ar, n_work, P.mode == 2 ? ar->threads_lit : ar->threads_match, g, T);
        const size_t sm = P.mode == 2 ? smem_for(ar, T) : smem_matches(ar, T);
        if (P.mode == 2) k_literals<1024><<<g, T, sm, ar->stream>>>(P);
        else if (P.mode == 3) k_matches<false, 1024><<<g, T, sm, ar->stream>>>(P);
        else k_matches<true, 1024><<<g, T, sm, ar->stream>>>(P);
    }
    else if (P.mode == 1 || !whole) k_decode<true><<<grid, ar->threads, ar->smem, ar->stream>>>(P);
    else k_decode<false><<<grid, ar->threads, ar->smem, ar->stream>>>(P);
    CU(cudaGetLastError());
    ar->launches++;
    return ACEAPEX_OK;
}

} // namespace

extern "C" {

int32_t aceapex_open(const void* d_archive, uint64_t archive_bytes, const void* h_archive, aceapex_archive** out) {
    if (!d_archive || !out || (reinterpret_cast<uintptr_t>(d_archive) & 15)) return ACEAPEX_E_ARG;
    *out = nullptr;
    aceapex_archive* ar = new (std::nothrow) aceapex_archive();
    if (!ar) return ACEAPEX_E_ARG;
    struct Guard { aceapex_archive* a; ~Guard() { if (a) aceapex_close(a); } } guard{ar};
    ar->d_archive = static_cast<const uint8_t*>(d_archive); ar->archive_bytes = archive_bytes;
    memset(ar->res, 0, sizeof ar->res);
    if (archive_bytes < 160) return ACEAPEX_E_TRUNCATED;
    uint8_t hdr[160];
    if (h_archive) memcpy(hdr, h_archive, 160); else CU(cudaMemcpy(hdr, d_archive, 160, cudaMemcpyDeviceToHost));
    static const uint8_t magic[8] = {0x41, 0x43, 0x58, 0x42, 0x32, 0x30, 0x30, 0x00};
    if (memcmp(hdr, magic, 8)) return ACEAPEX_E_MAGIC;
    if (rd32(hdr + 8) != 2 || rd32(hdr + 44) != (uint32_t)PROB_BITS) return ACEAPEX_E_VERSION;
    if (rd32(hdr + 12) != 160) return ACEAPEX_E_CORRUPT;
    ar->N = rd64(hdr + 16); ar->n_blocks = rd64(hdr + 24); ar->log2_bs = rd32(hdr + 32); ar->min_match = rd32(hdr + 36);
    ar->W = rd32(hdr + 40); uint32_t n_tables = rd32(hdr + 48); ar->max_level = rd32(hdr + 52); ar->max_cmds = rd32(hdr + 56);
    ar->flags = rd32(hdr + 60); ar->tables_off = rd64(hdr + 64); ar->dir_off = rd64(hdr + 72); ar->fnv_off = rd64(hdr + 80);
    ar->payload_off = rd64(hdr + 88); uint64_t abytes = rd64(hdr + 96);
    ar->total_lit = rd64(hdr + 104); ar->total_match_bytes = rd64(hdr + 112); ar->total_matches = rd64(hdr + 120); ar->total_cmds = rd64(hdr + 128);
    if (ar->log2_bs < 3 || ar->log2_bs > 20 || ar->min_match < 1 || ar->W < 4 || ar->W > 8 || n_tables != 3 + ar->W) return ACEAPEX_E_CORRUPT;
    if (ar->W < 8 && ar->N > (1ull << (8 * ar->W))) return ACEAPEX_E_CORRUPT;
    if (ar->n_blocks != (ar->N + (1ull << ar->log2_bs) - 1) >> ar->log2_bs) return ACEAPEX_E_CORRUPT;
    if (abytes > archive_bytes) return ACEAPEX_E_TRUNCATED;
    if (abytes % 16 || ar->tables_off < 160 || ar->tables_off % 16 || ar->dir_off % 16 || ar->dir_off < ar->tables_off + 528ull * n_tables) return ACEAPEX_E_CORRUPT;
    uint64_t meta_end = ar->dir_off + 32 * ar->n_blocks;
    if (ar->flags & 1) { if (ar->fnv_off < meta_end || ar->fnv_off % 8) return ACEAPEX_E_CORRUPT; meta_end = ar->fnv_off + 8 * ar->n_blocks; }
    if (ar->payload_off < meta_end || ar->payload_off % 16 || ar->payload_off > abytes) return ACEAPEX_E_CORRUPT;
    if (ar->total_lit + ar->total_match_bytes != ar->N) return ACEAPEX_E_CORRUPT;
    ar->archive_bytes = abytes;
    // tables + directory
    std::vector<uint8_t> meta_own;
    const uint8_t* meta;   // bytes [0, meta_end)
    if (h_archive) meta = static_cast<const uint8_t*>(h_archive);
    else { meta_own.resize(meta_end); CU(cudaMemcpy(meta_own.data(), d_archive, meta_end, cudaMemcpyDeviceToHost)); meta = meta_own.data(); }
    std::vector<uint32_t> luts;
    auto add_lut = [&](uint32_t t, uint32_t& idx) -> bool {
        const uint8_t* p = meta + ar->tables_off + 528ull * t;
        uint32_t cum = 0;
        idx = (uint32_t)(luts.size() / LUT_SIZE);
        luts.resize(luts.size() + LUT_SIZE);
        uint32_t* L = luts.data() + (size_t)idx * LUT_SIZE;
        for (uint32_t s = 0; s < 256; s++) {
            uint32_t f = rd16(p + 16 + 2 * s);
            if (cum + f > (uint32_t)LUT_SIZE) return false;
            for (uint32_t k = 0; k < f; k++) L[cum + k] = s | (k << 8) | (f << 20);
            cum += f;
        }
        return cum == (uint32_t)LUT_SIZE;
    };
    for (uint32_t t = 0; t < n_tables; t++) {
        uint32_t mode = rd32(meta + ar->tables_off + 528ull * t);
        bool is_plane = t >= 2 && t < 2 + ar->W;
        if (mode > 1 || (mode == 1 && !is_plane)) return ACEAPEX_E_CORRUPT;
        uint32_t idx = 0;
        if (mode == 0 && !add_lut(t, idx)) return ACEAPEX_E_CORRUPT;
        if (t == 0) ar->lut_cmd = idx; else if (t == 1) ar->lut_mlen = idx; else if (t == 2 + ar->W) ar->lut_lit = idx;
        else {
            uint32_t p = t - 2;
            ar->plane_lut[p] = mode == 0 ? (int8_t)idx : -1;
            ar->plane_raw[p] = mode == 1 ? (int8_t)ar->n_raw_planes : -1;
            if (mode == 0) ar->n_coded_planes++; else ar->n_raw_planes++;
        }
    }
    for (uint32_t p = ar->W; p < MAX_W; p++) { ar->plane_lut[p] = -1; ar->plane_raw[p] = -1; }
    ar->n_coded_tables = (uint32_t)(luts.size() / LUT_SIZE);
    // directory validation + level lists
    ar->level_blocks.assign(ar->max_level + 1, {});
    ar->h_match_prefix.assign(ar->n_blocks + 1, 0);
    ar->h_payload_off.assign(ar->n_blocks + 1, abytes);
    uint64_t prev = ar->payload_off;
    uint32_t seen_max_cmds = 0;
    for (uint64_t b = 0; b < ar->n_blocks; b++) {
        const uint8_t* p = meta + ar->dir_off + 32 * b;
        uint64_t po = rd64(p), end = b + 1 < ar->n_blocks ? rd64(p + 32) : abytes;
        uint32_t n_cmd = rd32(p + 8), n_match = rd32(p + 12), n_lit = rd32(p + 16), n_words = rd32(p + 20), n_ext = rd32(p + 24), lvl = rd16(p + 28);
        if (po % 16 || po < prev || end <= po || end > abytes) return ACEAPEX_E_CORRUPT;
        if (n_cmd < 1 || n_cmd > ar->max_cmds || !(n_match == n_cmd || n_match + 1 == n_cmd) || lvl > ar->max_level) return ACEAPEX_E_CORRUPT;
        uint64_t need = ((256 + 2ull * n_words + 3) & ~3ull) + 4ull * n_ext + (uint64_t)ar->n_raw_planes * n_match;
        if (po + need > end || n_lit > (1u << ar->log2_bs)) return ACEAPEX_E_CORRUPT;
        prev = po; seen_max_cmds = std::max(seen_max_cmds, n_cmd);
        ar->level_blocks[lvl].push_back((uint32_t)b);
        ar->h_match_prefix[b + 1] = ar->h_match_prefix[b] + n_match;
        ar->h_payload_off[b] = po;
    }
    if (ar->h_match_prefix[ar->n_blocks] != ar->total_matches) return ACEAPEX_E_CORRUPT;
    // device tables
    if (!luts.empty()) {
        CU(cudaMalloc(&ar->d_luts, luts.size() * 4));
        CU(cudaMemcpy(ar->d_luts, luts.data(), luts.size() * 4, cudaMemcpyHostToDevice));
    }
    if (ar->n_blocks) {
        std::vector<uint16_t>& lv = ar->h_levels;
        lv.resize(ar->n_blocks);
        for (uint64_t b = 0; b < ar->n_blocks; b++) lv[b] = rd16(meta + ar->dir_off + 32 * b + 28);
        CU(cudaMalloc(&ar->d_levels, lv.size() * 2));
        CU(cudaMemcpy(ar->d_levels, lv.data(), lv.size() * 2, cudaMemcpyHostToDevice));
        CU(cudaMalloc(&ar->d_match_prefix, ar->h_match_prefix.size() * 8));
        CU(cudaMemcpy(ar->d_match_prefix, ar->h_match_prefix.data(), ar->h_match_prefix.size() * 8, cudaMemcpyHostToDevice));
    }
    if (ar->n_blocks && ar->n_blocks < (1ull << 32)) {
        std::vector<uint32_t> cat;
        for (auto& v : ar->level_blocks) { ar->level_off.push_back(cat.size()); cat.insert(cat.end(), v.begin(), v.end()); }
        CU(cudaMalloc(&ar->d_level_lists, cat.size() * 4));
        CU(cudaMemcpy(ar->d_level_lists, cat.data(), cat.size() * 4, cudaMemcpyHostToDevice));
    }
    // launch geometry
    int dev = 0; cudaDeviceProp prop;
    CU(cudaGetDevice(&dev)); CU(cudaGetDeviceProperties(&prop, dev));
    ar->sms = prop.multiProcessorCount;
    // one CTA per SM: the decode tables are staged once per SM and shared by all its warps (fewer warps when many
    // offset planes are coded and the tables leave less room)
    ar->threads = 1024;
    while (ar->threads > 128 && std::max(smem_for(ar, ar->threads), smem_matches(ar, ar->threads)) > (size_t)prop.sharedMemPerBlockOptin) ar->threads -= 128;
    ar->smem = smem_for(ar, ar->threads);
    ar->threads_lit = ar->threads_match = ar->threads;
    {
        const void* fns[] = {(const void*)k_decode<false>, (const void*)k_decode<true>, (const void*)k_literals<1024>,
                             (const void*)k_matches<false, 1024>, (const void*)k_matches<true, 1024>, (const void*)k_matches<false, 1024, true, true>,
                             (const void*)k_matches<false, 1024, true, false>, (const void*)k_matches<true, 1024, true, false>, (const void*)k_serve, (const void*)k_copy<false>,
                             (const void*)k_copy<true>, (const void*)k_copy<false, true, true>, (const void*)k_copy<true, true, false>, (const void*)k_rounds};
        for (const void* f : fns) {
            CU(cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)std::max(std::max(ar->smem, smem_matches(ar, ar->threads)), (size_t)(ar->threads / 32) * COPY_WARP_BYTES + 64)));
            CU(cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        }
    }
    {
        int coop = 0, occ_r = 0;
        CU(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_r, k_rounds, ar->threads, ar->smem));
        ar->cooperative = coop && occ_r >= 1 && !getenv("ACEAPEX_NO_COOPERATIVE");
        ar->win_tokens = getenv("ACEAPEX_WIN_TOKENS") && atoi(getenv("ACEAPEX_WIN_TOKENS")) != 0;
    }
    int occ = 0;
    CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ, k_decode<true>, ar->threads, ar->smem));
    if (occ < 1) return ACEAPEX_E_CUDA;
    if (const char* e = getenv("ACEAPEX_CTAS_PER_SM")) occ = std::max(1, std::min(occ, atoi(e)));
    ar->ctas_per_sm = occ;
    ar->grid = (uint32_t)(ar->sms * occ);
    uint64_t mc = align_up(ar->max_cmds, 16);
    ar->scratch_per_warp = align_up((1ull << ar->log2_bs) + 32 + mc * (2 + ar->n_coded_planes), 256);
    layout_workspace(ar);
    guard.a = nullptr;
    *out = ar;
    return ACEAPEX_OK;
}

int32_t aceapex_close(aceapex_archive* ar) {
    if (!ar) return ACEAPEX_E_ARG;
    cudaDeviceSynchronize();
    if (ar->d_luts) cudaFree(ar->d_luts);
    if (ar->d_level_lists) cudaFree(ar->d_level_lists);
    if (ar->d_levels) cudaFree(ar->d_levels);
    if (ar->d_match_prefix) cudaFree(ar->d_match_prefix);
    if (ar->d_chunk_lists) cudaFree(ar->d_chunk_lists);
    for (cudaEvent_t e : ar->ev_h2d) cudaEventDestroy(e);
    for (cudaEvent_t e : ar->ev_dec) cudaEventDestroy(e);
    for (cudaEvent_t e : ar->ev_phase) if (e) cudaEventDestroy(e);
    if (ar->s_h2d) cudaStreamDestroy(ar->s_h2d);
    if (ar->s_d2h) cudaStreamDestroy(ar->s_d2h);
    delete ar;
    return ACEAPEX_OK;
}

int32_t aceapex_info(const aceapex_archive* ar, aceapex_info_t* o) {
    if (!ar || !o) return ACEAPEX_E_ARG;
    memset(o, 0, sizeof *o);
    o->raw_bytes = ar->N; o->archive_bytes = ar->archive_bytes; o->n_blocks = ar->n_blocks; o->block_size = 1ull << ar->log2_bs;
    o->total_lit_bytes = ar->total_lit; o->total_match_bytes = ar->total_match_bytes; o->total_matches = ar->total_matches;
    o->total_cmds = ar->total_cmds; o->workspace_bytes = workspace_need(ar); o->max_level = ar->max_level; o->offset_width = ar->W;
    o->min_match = ar->min_match; o->max_cmds = ar->max_cmds; o->n_coded_planes = ar->n_coded_planes; o->has_fnv = ar->flags & 1;
    o->resident_warps = ar->grid * (ar->threads / 32);
    return ACEAPEX_OK;
}

int32_t aceapex_set_workspace(aceapex_archive* ar, void* d_ws, uint64_t bytes) {
    if (!ar || (reinterpret_cast<uintptr_t>(d_ws) & 255)) return ACEAPEX_E_ARG;
    ar->d_ws = static_cast<uint8_t*>(d_ws); ar->ws_bytes = bytes; ar->ws_clean = false;
    return (d_ws && bytes >= workspace_need(ar)) ? ACEAPEX_OK : ACEAPEX_E_WORKSPACE;
}

int32_t aceapex_set_stream(aceapex_archive* ar, void* s) {
    if (!ar) return ACEAPEX_E_ARG;
    ar->stream = static_cast<cudaStream_t>(s);
    return ACEAPEX_OK;
}

// literal launch, one flag-driven match launch for the blocks below the top dependency level, one wait-free match launch
// for the top level (FORMAT.md §3)
int32_t aceapex_decode_all(aceapex_archive* ar, void* d_out) {
    if (!ar || (!d_out && ar->N) || (reinterpret_cast<uintptr_t>(d_out) & 15)) return ACEAPEX_E_ARG;
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    Params P; fill_params(ar, P);
    P.out = static_cast<uint8_t*>(d_out); P.out_pos0 = 0; P.first_block = 0;
    P.pairs = reinterpret_cast<uint2*>(ar->d_ws + ar->desc_off);          // k_literals leaves (dst_rel, len) and the coded offset
    P.cplanes = ar->d_ws + ar->cplanes_off;                               // planes of every match for k_copy
    const bool tm = ar->phase_timing;
    if (tm) CU(cudaEventRecord(ar->ev_phase[0], ar->stream));
    P.mode = 2; P.level_list = nullptr;
    if ((rc = launch(ar, P, ar->n_blocks))) return rc;
    if (tm) CU(cudaEventRecord(ar->ev_phase[1], ar->stream));
    if (!ar->d_level_lists) return ACEAPEX_OK;
    // the top level (on FASTQ 97 % of the blocks sit at the level cap) runs without waits in a launch of its own: every
    // source is a literal byte (placed by the launch above) or a match byte of a lower level (FORMAT.md §3); the few
    // blocks of all lower levels share one flag-driven launch instead of one small latency-bound launch per level
    const uint32_t top = ar->max_level;
    if (top > 0 && ar->level_off[top] > 0) {
        P.mode = 9; P.level_list = ar->d_level_lists; P.epoch = ++ar->epoch;
        if ((rc = launch(ar, P, ar->level_off[top]))) return rc;
    }
    if (tm) CU(cudaEventRecord(ar->ev_phase[2], ar->stream));
    P.mode = 8; P.level_list = ar->d_level_lists + ar->level_off[top];
    rc = launch(ar, P, ar->level_blocks[top].size());
    if (tm && !rc) CU(cudaEventRecord(ar->ev_phase[3], ar->stream));
    return rc;
}

int32_t aceapex_set_phase_timing(aceapex_archive* ar, int32_t on) {
    if (!ar) return ACEAPEX_E_ARG;
    if (on && !ar->ev_phase[0]) for (int k = 0; k < 4; k++) CU(cudaEventCreate(&ar->ev_phase[k]));
    ar->phase_timing = on != 0;
    return ACEAPEX_OK;
}

int32_t aceapex_phase_times(aceapex_archive* ar, float* ms3) {
    if (!ar || !ms3 || !ar->phase_timing || !ar->ev_phase[0]) return ACEAPEX_E_ARG;
    CU(cudaEventSynchronize(ar->ev_phase[3]));
    for (int k = 0; k < 3; k++) CU(cudaEventElapsedTime(ms3 + k, ar->ev_phase[k], ar->ev_phase[k + 1]));
    return ACEAPEX_OK;
}

// literal launch + ONE match launch over the blocks sorted by (level, index) with completion flags
int32_t aceapex_decode_all_flags(aceapex_archive* ar, void* d_out) {
    if (!ar || (!d_out && ar->N) || (reinterpret_cast<uintptr_t>(d_out) & 15)) return ACEAPEX_E_ARG;
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    Params P; fill_params(ar, P);
    P.out = static_cast<uint8_t*>(d_out); P.out_pos0 = 0; P.first_block = 0; P.epoch = ++ar->epoch;
    if (!ar->d_level_lists) return ACEAPEX_OK;      // no blocks
    P.mode = 2; P.level_list = nullptr;             // launch 1: entropy decode + literal placement, every block
    if ((rc = launch(ar, P, ar->n_blocks))) return rc;
    P.mode = 4; P.level_list = ar->d_level_lists;   // launch 2: matches, blocks sorted by (level, index)
    return launch(ar, P, ar->n_blocks);
}

int32_t aceapex_decode_all_fused(aceapex_archive* ar, void* d_out) {
    if (!ar || (!d_out && ar->N)) return ACEAPEX_E_ARG;
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    Params P; fill_params(ar, P);
    P.mode = 0; P.out = static_cast<uint8_t*>(d_out); P.out_pos0 = 0; P.first_block = 0; P.epoch = ++ar->epoch;
    P.level_list = ar->d_level_lists;   // blocks sorted by (level, index): everything a block reads from precedes it
    return launch(ar, P, ar->n_blocks);
}

// launches span-mode work for the demands staged in ar->h_demands (in batches of demand_cap)
static int32_t run_demands(aceapex_archive* ar, Params& P) {
    Demand* d_dem = reinterpret_cast<Demand*>(ar->d_ws + ar->demands_off);
    P.mode = 1; P.level_list = nullptr; P.demands = d_dem; P.n_inline = 0;
    if (ar->h_demands.size() <= 4) {                   // a single read: the items travel in the kernel arguments, no copy
        P.n_inline = (uint32_t)ar->h_demands.size();
        for (uint32_t i = 0; i < P.n_inline; i++) P.inline_dem[i] = ar->h_demands[i];
        return launch(ar, P, P.n_inline);
    }
    for (size_t i = 0; i < ar->h_demands.size(); i += ar->demand_cap) {
        size_t n = std::min<size_t>(ar->demand_cap, ar->h_demands.size() - i);
        CU(cudaMemcpyAsync(d_dem, ar->h_demands.data() + i, n * sizeof(Demand), cudaMemcpyHostToDevice, ar->stream));
        int32_t rc = launch(ar, P, n);
        if (rc) return rc;
        if (i + n < ar->h_demands.size()) CU(cudaStreamSynchronize(ar->stream));   // the staging area is reused
    }
    return ACEAPEX_OK;
}

static void add_demands(aceapex_archive* ar, uint64_t pos, uint64_t len, uint64_t dst) {
    while (len) {
        uint64_t bend = ((pos >> ar->log2_bs) + 1) << ar->log2_bs, n = std::min(len, bend - pos);
        ar->h_demands.push_back(Demand{pos, dst, n});
        pos += n; dst += n; len -= n;
    }
}

// Serves the demand list g[0] (filled by the caller) in at most `rounds` rounds; the list left by the last round must be
// empty.  One cooperative launch (k_rounds) where the device supports it, else three launches per round.
static int32_t serve_rounds(aceapex_archive* ar, Params Q, const GList g[2], uint32_t rounds) {
    Q.mode = 7;
    if (ar->cooperative && rounds <= 16) {
        unsigned long long* tickets = reinterpret_cast<unsigned long long*>(ar->d_ws + 128);     // 16 counters in the control area
        CU(cudaMemsetAsync(tickets, 0, 128, ar->stream));
        Q.gl_cur = g[0]; Q.gl_nxt = g[1];
        void* args[] = {&Q, &tickets, &rounds};
        CU(cudaLaunchCooperativeKernel((const void*)k_rounds, dim3(ar->sms), dim3(ar->threads), args, ar->smem, ar->stream));
        ar->launches++;
        return ACEAPEX_OK;
    }
    for (uint32_t r = 0; r < rounds; r++) {
        Q.gl_cur = g[r & 1]; Q.gl_nxt = g[(r + 1) & 1];
        CU(cudaMemsetAsync(Q.gl_nxt.count, 0, 16, ar->stream));
        k_plan<<<ar->sms, 256, 0, ar->stream>>>(Q);          // bucket offsets + work items
        k_scatter<<<4 * ar->sms, 256, 0, ar->stream>>>(Q);
        ar->launches += 2;
        int32_t rc = launch(ar, Q, 1);
        if (rc) return rc;
    }
    k_assert_empty<<<1, 1, 0, ar->stream>>>(g[rounds & 1].count, Q.err);
    CU(cudaGetLastError());
    ar->launches++;
    return ACEAPEX_OK;
}

int32_t aceapex_decode_range(aceapex_archive* ar, uint64_t lo, uint64_t hi, void* d_out, uint64_t budget) {
    if (!ar) return ACEAPEX_E_ARG;
    if (lo > hi || hi > ar->N) return ACEAPEX_E_RANGE;
    if (lo == hi) return ACEAPEX_OK;
    if (!d_out) return ACEAPEX_E_ARG;
    // vram_budget bounds the workspace bytes this call touches: everything but the demand lists is fixed, the lists use
    // 3 x 24 bytes per record (two arrival arrays, one bucketed copy) plus their work items; fewer records mean more
    // sub-windows, not failure, down to a floor of 4096 records
    ar->gl_eff = ar->gl_cap;
    if (budget && budget < workspace_need(ar)) {
        const uint64_t per_rec = 3 * sizeof(GDemand) + 8, fixed = workspace_need(ar) - std::min<uint64_t>(workspace_need(ar), per_rec * ar->gl_cap);
        if (budget < fixed + per_rec * 4096) return ACEAPEX_E_BUDGET;
        ar->gl_eff = std::min<uint64_t>(ar->gl_cap, (budget - fixed) / per_rec);
    }
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    const uint64_t BS = 1ull << ar->log2_bs;
    // whole blocks [alo, ahi) are decoded as a window (flag-driven schedule); the ragged ends are spans
    uint64_t alo = (lo + BS - 1) & ~(BS - 1), ahi = hi == ar->N ? hi : hi & ~(BS - 1);
    Params P; fill_params(ar, P);
    uint8_t* out = static_cast<uint8_t*>(d_out);
    P.out2 = out; P.out_pos0 = 0; P.win_end = 0; P.out = out;
    if (alo < ahi) {
        uint64_t b0 = alo >> ar->log2_bs, b1 = (ahi + BS - 1) >> ar->log2_bs, nb = b1 - b0;
        // blocks of the window sorted by (level, index): counting sort on the host copy of the levels
        std::vector<uint32_t>& L = ar->h_list;
        L.resize(nb);
        std::vector<uint64_t> cnt(ar->max_level + 2, 0);
        for (uint64_t b = b0; b < b1; b++) cnt[ar->h_levels[b] + 1]++;
        for (size_t l = 1; l < cnt.size(); l++) cnt[l] += cnt[l - 1];
        for (uint64_t b = b0; b < b1; b++) L[cnt[ar->h_levels[b]]++] = (uint32_t)b;
        uint32_t* d_list = reinterpret_cast<uint32_t*>(ar->d_ws + ar->list_off);
        CU(cudaMemcpyAsync(d_list, L.data(), nb * 4, cudaMemcpyHostToDevice, ar->stream));
        P.out = out + (alo - lo); P.out2 = P.out; P.out_pos0 = alo; P.win_end = ahi;
        if (reinterpret_cast<uintptr_t>(P.out) & 15) {
            // window not 16-byte aligned in d_out: one launch, every warp reconstructs the foreign sources of its block by recursion
            P.mode = 0; P.level_list = d_list; P.epoch = ++ar->epoch;
            if ((rc = launch(ar, P, nb))) return rc;
        } else {
            // (1) literals of the window; (2) foreign seed bytes of its matches -> demand lists, served in rounds, every
            // source block parsed once per round; (3) matches of the window, one launch per dependency level
            // the literal launch leaves (dst_rel, len) and the decoded offset planes of the window's matches for (2) and (3)
            P.pairs = reinterpret_cast<uint2*>(ar->d_ws + ar->desc_off); P.cplanes = ar->d_ws + ar->cplanes_off;
            P.mode = 2; P.level_list = nullptr; P.first_block = b0;
            if ((rc = launch(ar, P, nb))) return rc;
            const GList g[2] = {glist(ar, 0), glist(ar, 1)};
            for (uint64_t s0 = b0; s0 < b1;) {                // sub-windows whose demands fit the lists
                uint64_t s1 = s0 + 1;
                while (s1 < b1 && ar->h_match_prefix[s1 + 1] - ar->h_match_prefix[s0] <= ar->gl_eff / 3) s1++;
                CU(cudaMemsetAsync(g[0].count, 0, 32, ar->stream));
                P.mode = ar->win_tokens ? 5 : 11; P.level_list = nullptr; P.first_block = s0; P.gl_nxt = g[0];
                if ((rc = launch(ar, P, s1 - s0))) return rc;
                Params Q = P;                                   // serving knows no window: sources of foreign bytes precede it
                Q.out_pos0 = 0; Q.win_end = 0; Q.pairs = nullptr; Q.cplanes = nullptr;
                // a seed byte is found after at most max_level + 1 source blocks (FORMAT.md §3): one round each
                if ((rc = serve_rounds(ar, Q, g, ar->max_level + 2))) return rc;
                s0 = s1;
            }
            // matches of the window: its blocks sorted by (level, index) in one flag-driven launch (a block waits for
            // lower-level source blocks of the window only; everything outside the window is final)
            P.mode = ar->win_tokens ? 10 : 12; P.level_list = d_list; P.first_block = 0; P.epoch = ++ar->epoch;
            if ((rc = launch(ar, P, nb))) return rc;
            P.pairs = nullptr; P.cplanes = nullptr;
        }
    }
    // the ragged ends: spans that enter the demand lists as top-level records; the finished window is a plain source
    ar->h_demands.clear();
    if (alo >= ahi) add_demands(ar, lo, hi - lo, 0);
    else {
        if (lo < alo) add_demands(ar, lo, alo - lo, 0);
        if (ahi < hi) add_demands(ar, ahi, hi - ahi, ahi - lo);
    }
    if (!ar->h_demands.empty()) {
        const GList g[2] = {glist(ar, 0), glist(ar, 1)};
        Demand* d_dem = reinterpret_cast<Demand*>(ar->d_ws + ar->demands_off);
        const uint32_t n = (uint32_t)ar->h_demands.size();      // at most a handful: two spans cut at block boundaries
        CU(cudaMemcpyAsync(d_dem, ar->h_demands.data(), n * sizeof(Demand), cudaMemcpyHostToDevice, ar->stream));
        CU(cudaMemsetAsync(g[0].count, 0, 32, ar->stream));
        Params Q = P;
        if (alo >= ahi) { Q.out_pos0 = 0; Q.win_end = 0; }
        Q.out2 = out; Q.demands = d_dem; Q.gl_nxt = g[0];
        k_seed<<<(n + 127) / 128, 128, 0, ar->stream>>>(Q, n);
        CU(cudaGetLastError());
        ar->launches++;
        if ((rc = serve_rounds(ar, Q, g, ar->max_level + 3))) return rc;   // one more round: the span's own block comes first
    }
    return ACEAPEX_OK;
}

int32_t aceapex_reads_bytes(const uint64_t* idx, uint64_t n_index, const uint64_t* ids, uint64_t n, uint64_t* total, uint64_t* offs) {
    if ((!idx && n_index) || (!ids && n) || !total) return ACEAPEX_E_ARG;
    uint64_t t = 0;
    for (uint64_t i = 0; i < n; i++) {
        if (ids[i] >= n_index) return ACEAPEX_E_RANGE;
        if (offs) offs[i] = t;
        t += idx[ids[i]] >> 40;
    }
    if (offs) offs[n] = t;
    *total = t;
    return ACEAPEX_OK;
}

int32_t aceapex_decode_reads(aceapex_archive* ar, const uint64_t* idx, uint64_t n_index, const uint64_t* ids, uint64_t n, void* d_out) {
    if (!ar || (!idx && n_index) || (!ids && n)) return ACEAPEX_E_ARG;
    if (n == 0) return ACEAPEX_OK;
    if (!d_out) return ACEAPEX_E_ARG;
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    ar->h_demands.clear();
    uint64_t off = 0;
    for (uint64_t i = 0; i < n; i++) {               // index lookup: O(1) per read
        if (ids[i] >= n_index) return ACEAPEX_E_RANGE;
        uint64_t e = idx[ids[i]], pos = e & ((1ull << 40) - 1), len = e >> 40;
        if (pos + len > ar->N) return ACEAPEX_E_RANGE;
        add_demands(ar, pos, len, off);
        off += len;
    }
    Params P; fill_params(ar, P);
    P.out = static_cast<uint8_t*>(d_out); P.out2 = P.out; P.out_pos0 = 0; P.win_end = 0;
    static const int force_rounds = getenv("ACEAPEX_READS_ROUNDS") ? atoi(getenv("ACEAPEX_READS_ROUNDS")) : -1;
    // Medium batches go through the demand lists as top-level records: their blocks, then the source blocks of every
    // round, are parsed in parallel by different warps.  A single read is served faster by one warp that recurses on its
    // sources itself (one launch); a batch that fills the machine gains nothing from the extra passes.
    const bool by_rounds = ar->cooperative && (force_rounds >= 0 ? force_rounds != 0 : (n >= 2 && n <= 1024));
    if (by_rounds) {
        const GList g[2] = {glist(ar, 0), glist(ar, 1)};
        Demand* d_dem = reinterpret_cast<Demand*>(ar->d_ws + ar->demands_off);
        ar->gl_eff = ar->gl_cap;
        const size_t chunk = std::max<size_t>(1, std::min<size_t>(ar->demand_cap, ar->gl_cap / 8));
        for (size_t i = 0; i < ar->h_demands.size(); i += chunk) {
            const uint32_t m = (uint32_t)std::min<size_t>(chunk, ar->h_demands.size() - i);
            CU(cudaMemsetAsync(g[0].count, 0, 32, ar->stream));
            Params Q = P;
            Q.gl_nxt = g[0]; Q.demands = d_dem; Q.n_inline = 0;
            if (m <= 4) { Q.n_inline = m; for (uint32_t k = 0; k < m; k++) Q.inline_dem[k] = ar->h_demands[i + k]; }
            else CU(cudaMemcpyAsync(d_dem, ar->h_demands.data() + i, m * sizeof(Demand), cudaMemcpyHostToDevice, ar->stream));
            k_seed<<<(m + 127) / 128, 128, 0, ar->stream>>>(Q, m);
            CU(cudaGetLastError());
            ar->launches++;
            if ((rc = serve_rounds(ar, Q, g, ar->max_level + 3))) return rc;
            if (i + chunk < ar->h_demands.size()) CU(cudaStreamSynchronize(ar->stream));   // the staging area is reused
        }
    } else if ((rc = run_demands(ar, P))) return rc;
    CU(cudaStreamSynchronize(ar->stream));           // h_demands is host staging; the call returns the reads
    return ACEAPEX_OK;
}

int32_t aceapex_set_resident(aceapex_archive* ar, uint32_t slot, uint64_t lo, uint64_t hi, const void* p) {
    if (!ar || slot >= MAX_RESIDENT || lo > hi || hi > ar->N) return ACEAPEX_E_ARG;
    ar->res[slot].lo = lo; ar->res[slot].hi = hi; ar->res[slot].ptr = static_cast<const uint8_t*>(p);
    return ACEAPEX_OK;
}

int32_t aceapex_verify_fnv(aceapex_archive* ar, const void* d_data, uint64_t lo, uint64_t hi, uint64_t* n_bad) {
    if (!ar || !n_bad || !(ar->flags & 1) || (lo & ((1ull << ar->log2_bs) - 1)) || lo > hi || hi > ar->N) return ACEAPEX_E_ARG;
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    unsigned long long* cnt = reinterpret_cast<unsigned long long*>(ar->d_ws + 16);
    CU(cudaMemsetAsync(cnt, 0, 8, ar->stream));
    uint64_t nb = ((hi - lo) + (1ull << ar->log2_bs) - 1) >> ar->log2_bs;
    if (nb) {
        const uint64_t* expect = reinterpret_cast<const uint64_t*>(ar->d_archive + ar->fnv_off) + (lo >> ar->log2_bs);
        k_fnv<<<(unsigned)((nb + 127) / 128), 128, 0, ar->stream>>>(static_cast<const uint8_t*>(d_data), hi - lo, ar->log2_bs, expect, cnt);
        CU(cudaGetLastError());
        ar->launches++;
    }
    unsigned long long h = 0;
    CU(cudaMemcpyAsync(&h, cnt, 8, cudaMemcpyDeviceToHost, ar->stream));
    CU(cudaStreamSynchronize(ar->stream));
    *n_bad = h;
    return ACEAPEX_OK;
}

// End to end with host buffers, pipelined over chunks of blocks: the payload of chunk k+1 travels host -> device while
// chunk k decodes and the output of chunk k-1 travels device -> host (a chunk only reads output bytes of lower positions,
// and inside a chunk the levels are launched in order, FORMAT.md §3).
int32_t aceapex_decode_all_host(aceapex_archive* ar, const void* h_archive, void* d_stage, void* h_out) {
    if (!ar || !h_archive || (!d_stage && ar->N) || (!h_out && ar->N) || (reinterpret_cast<uintptr_t>(d_stage) & 15)) return ACEAPEX_E_ARG;
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    const uint8_t* h_a = static_cast<const uint8_t*>(h_archive);
    uint8_t* d_a = const_cast<uint8_t*>(ar->d_archive);
    if (ar->n_blocks == 0) {
        CU(cudaMemcpyAsync(d_a, h_a, ar->archive_bytes, cudaMemcpyHostToDevice, ar->stream));
        CU(cudaStreamSynchronize(ar->stream));
        return ACEAPEX_OK;
    }
    const uint32_t n_lv = ar->max_level + 1;
    if (!ar->s_h2d) {                                      // first use: streams, events, per-chunk level lists
        CU(cudaStreamCreateWithFlags(&ar->s_h2d, cudaStreamNonBlocking));
        CU(cudaStreamCreateWithFlags(&ar->s_d2h, cudaStreamNonBlocking));
        ar->chunk_blocks = std::max<uint64_t>(256, (ar->n_blocks + 15) / 16);
        const uint64_t n_chunks = (ar->n_blocks + ar->chunk_blocks - 1) / ar->chunk_blocks;
        std::vector<uint32_t> list(ar->n_blocks);
        ar->chunk_level_off.assign(n_chunks * n_lv + 1, 0);
        uint64_t at = 0;
        for (uint64_t k = 0; k < n_chunks; k++) {
            const uint64_t b0 = k * ar->chunk_blocks, b1 = std::min(ar->n_blocks, b0 + ar->chunk_blocks);
            for (uint32_t l = 0; l < n_lv; l++) {
                ar->chunk_level_off[k * n_lv + l] = at;
                for (uint64_t b = b0; b < b1; b++) if (ar->h_levels[b] == l) list[at++] = (uint32_t)b;
            }
        }
        ar->chunk_level_off[n_chunks * n_lv] = at;
        CU(cudaMalloc(&ar->d_chunk_lists, list.size() * 4));
        CU(cudaMemcpy(ar->d_chunk_lists, list.data(), list.size() * 4, cudaMemcpyHostToDevice));
        ar->ev_h2d.resize(n_chunks); ar->ev_dec.resize(n_chunks);
        for (uint64_t k = 0; k < n_chunks; k++) {
            CU(cudaEventCreateWithFlags(&ar->ev_h2d[k], cudaEventDisableTiming));
            CU(cudaEventCreateWithFlags(&ar->ev_dec[k], cudaEventDisableTiming));
        }
    }
    const uint64_t n_chunks = ar->ev_h2d.size();
    // everything queued on the handle's stream so far must be done before the archive bytes are replaced
    CU(cudaEventRecord(ar->ev_dec[0], ar->stream));
    CU(cudaStreamWaitEvent(ar->s_h2d, ar->ev_dec[0], 0));
    CU(cudaStreamWaitEvent(ar->s_d2h, ar->ev_dec[0], 0));
    CU(cudaMemcpyAsync(d_a, h_a, ar->payload_off, cudaMemcpyHostToDevice, ar->s_h2d));     // header, tables, directory, fnv
    Params P; fill_params(ar, P);
    P.out = static_cast<uint8_t*>(d_stage); P.out_pos0 = 0;
    P.pairs = reinterpret_cast<uint2*>(ar->d_ws + ar->desc_off); P.cplanes = ar->d_ws + ar->cplanes_off;
    for (uint64_t k = 0; k < n_chunks; k++) {
        const uint64_t b0 = k * ar->chunk_blocks, b1 = std::min(ar->n_blocks, b0 + ar->chunk_blocks);
        const uint64_t p0 = ar->h_payload_off[b0], p1 = b1 < ar->n_blocks ? ar->h_payload_off[b1] : ar->archive_bytes;
        CU(cudaMemcpyAsync(d_a + p0, h_a + p0, p1 - p0, cudaMemcpyHostToDevice, ar->s_h2d));
        CU(cudaEventRecord(ar->ev_h2d[k], ar->s_h2d));
        CU(cudaStreamWaitEvent(ar->stream, ar->ev_h2d[k], 0));
        P.mode = 2; P.level_list = nullptr; P.first_block = b0;
        if ((rc = launch(ar, P, b1 - b0))) return rc;
        for (uint32_t l = 0; l < n_lv; l++) {
            const uint64_t l0 = ar->chunk_level_off[k * n_lv + l], l1 = ar->chunk_level_off[k * n_lv + l + 1];
            P.mode = 8; P.level_list = ar->d_chunk_lists + l0; P.first_block = 0;
            if ((rc = launch(ar, P, l1 - l0))) return rc;
        }
        CU(cudaEventRecord(ar->ev_dec[k], ar->stream));
        CU(cudaStreamWaitEvent(ar->s_d2h, ar->ev_dec[k], 0));
        const uint64_t o0 = b0 << ar->log2_bs, o1 = std::min(ar->N, b1 << ar->log2_bs);
        CU(cudaMemcpyAsync(static_cast<uint8_t*>(h_out) + o0, static_cast<uint8_t*>(d_stage) + o0, o1 - o0, cudaMemcpyDeviceToHost, ar->s_d2h));
    }
    CU(cudaStreamSynchronize(ar->s_d2h));
    CU(cudaStreamSynchronize(ar->stream));
    return ACEAPEX_OK;
}

int32_t aceapex_check(aceapex_archive* ar) {
    if (!ar) return ACEAPEX_E_ARG;
    CU(cudaStreamSynchronize(ar->stream));
    ar->dev_flags = 0;
    if (ar->d_ws && ar->ws_clean) {
        uint32_t f = 0;
        CU(cudaMemcpy(&f, ar->d_ws + 8, 4, cudaMemcpyDeviceToHost));
        ar->dev_flags = f;
        if (f) { CU(cudaMemset(ar->d_ws + 8, 0, 4)); return ACEAPEX_E_CORRUPT; }
    }
    return ACEAPEX_OK;
}

uint32_t aceapex_device_flags(const aceapex_archive* ar) { return ar ? ar->dev_flags : 0; }
int32_t aceapex_last_cuda_error(const aceapex_archive* ar) { return ar ? ar->last_cuda : 0; }
uint64_t aceapex_launch_count(const aceapex_archive* ar) { return ar ? ar->launches : 0; }

const char* aceapex_strerror(int32_t c) {
    switch (c) {
        case ACEAPEX_OK: return "ok";
        case ACEAPEX_E_MAGIC: return "not an ACX-B200 archive";
        case ACEAPEX_E_VERSION: return "unsupported archive version";
        case ACEAPEX_E_TRUNCATED: return "archive truncated";
        case ACEAPEX_E_CORRUPT: return "archive corrupt";
        case ACEAPEX_E_RANGE: return "range or read id out of bounds";
        case ACEAPEX_E_BUDGET: return "vram budget too small";
        case ACEAPEX_E_WORKSPACE: return "workspace missing or too small";
        case ACEAPEX_E_CUDA: return "CUDA runtime error";
        case ACEAPEX_E_ARG: return "bad argument";
    }
    return "unknown error";
}

} // extern "C"
