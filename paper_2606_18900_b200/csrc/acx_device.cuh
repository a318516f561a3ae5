// Device side of the ACX-B200 decoder (FORMAT.md version 3): shared declarations, the rANS step (A1) and the byte copies
// (A3/A4) — SURVEY §8(a).  One warp owns one segment at a time.
#pragma once
#include <cstdint>
#include <cuda_runtime.h>

namespace acx {

constexpr int PROB_BITS = 11;
constexpr int LUT_SIZE = 1 << PROB_BITS;          // u32 entries per byte table: sym | bias << 8 | freq << 20
constexpr int QPROB_BITS = 12;
constexpr int QLUT_SIZE = 1 << QPROB_BITS;        // uint2 entries of the pair table: {pair | freq << 16, bias}
constexpr int RING_BYTES = 2048;                  // per warp: 32 lanes x 64-byte ring of rANS words in shared memory
constexpr int MAX_W = 8;
constexpr int MAX_RESIDENT = 8;
constexpr uint32_t MAX_SEG_CMDS = 510;            // FORMAT.md §1.5
constexpr uint32_t MAX_SEG_LITS = 16384;
constexpr uint32_t TOK_STRIDE = 512;              // per-warp token arrays hold one segment's commands

enum : uint32_t { DF_RANS = 1, DF_OFFSET = 2, DF_LENGTH = 4, DF_TIMEOUT = 8, DF_STACK = 16 };

struct SegEntry {            // FORMAT.md §1.5, 32 bytes
    uint64_t payload_off, out_start;
    uint16_t n_cmd, n_match, n_lit_a, n_lit_q, n_sym_q, n_words, n_ext, level;
};

struct Resident { uint64_t lo, hi; const uint8_t* ptr; };

// "materialise original bytes [pos, pos + len) at out2[dst ..)"; never crosses a segment boundary; len == 0: served
struct Demand { uint64_t pos; uint64_t dst; uint64_t len; };

// Aggregated demands (range decode).  Records are appended unsorted while a per-segment counter counts them; before they
// are served they are bucketed by SOURCE segment (plan + scatter), so one parse of a segment serves its whole bucket and a
// hot segment (thousands of records) is cut into work items of GL_ITEM records that different warps take.
struct GDemand { uint64_t pos; uint64_t dst; uint32_t len; uint32_t seg; };
constexpr uint32_t GL_ITEM = 128;                 // records per work item: one parse of the source segment, then 32 records at a time
struct GList {
    GDemand* rec;            // cap records, in order of arrival
    GDemand* sorted;         // the same records bucketed by segment (written by the scatter phase)
    uint32_t* cnt;           // per segment: records appended; after the plan phase: fill pointer of its bucket; 0 when idle
    uint32_t* touched;       // segments with at least one record, in order of first touch
    unsigned long long* work;// work items written by the plan phase: segment << 32 | first record, the record count in work_n
    uint32_t* work_n;
    uint32_t* count;         // [0] = records appended, [1] = segments touched, [2] = work items, [3] = records given a bucket
    uint32_t cap, touched_cap, work_cap;
};

struct Params {
    const uint8_t* archive;      // device archive
    const SegEntry* dir;         // = archive + dir_off
    const uint32_t* luts;        // n_coded_tables x LUT_SIZE
    const uint2* lutq;           // QLUT_SIZE entries (pair mode)
    const uint16_t* levels;      // level per block
    const uint32_t* first_seg;   // n_blocks + 1 entries (FORMAT.md §1.4)
    uint64_t N, n_segs;
    uint32_t log2_bs, log2_seg, min_match, W, n_coded_tables, q_min, q_mode;
    int8_t plane_lut[MAX_W];     // coded OFF plane p -> lut index, -1 if raw
    uint32_t n_coded_planes, n_raw_planes;
    uint8_t coded_shift[MAX_W];  // bit position of the k-th coded plane in decode order (high plane first)
    uint8_t coded_lut[MAX_W];    // lut index of the k-th coded plane in decode order
    uint8_t raw_shift[MAX_W];    // bit position of the r-th raw plane (ascending p)
    uint32_t lut_cmd, lut_mlen, lut_lita, lut_litq;
    uint32_t runs_bytes, lita_bytes;     // per-warp shared memory: LITQ run table / LITA staging (multiples of 16)
    // work
    uint64_t first_work, n_work;         // work items: segments first_work + i, or seg_list[i]
    uint32_t copy_parts;                 // k_copy: shares per segment (n_work = segments x copy_parts); 1 in every other kernel
    const uint32_t* seg_list;
    uint8_t* out;                        // byte at absolute position p is out[p - out_pos0]
    uint64_t out_pos0, win_end;          // out holds the original bytes [out_pos0, win_end) (the window; block aligned start)
    uint32_t out_odd;                    // (out - out_pos0) is an odd address: pair stores fall back to byte stores
    const Demand* demands; uint8_t* out2; // span mode: top-level work items, destination buffer of every demand
    Demand inline_dem[4]; uint32_t n_inline; // span mode with at most four items: they travel in the kernel arguments
    Resident res[MAX_RESIDENT];
    // workspace
    uint32_t* done;                      // per block: segments completed by the current flag-driven launch
    unsigned long long* ticket;          // work counter of this launch (zero when the kernel starts)
    unsigned long long* ticket_next;     // the other slot: every kernel clears it for the launch that follows
    uint32_t* err;
    uint8_t* scratch; uint64_t scratch_per_warp;
    Demand* stacks; uint32_t stack_cap;  // per-warp LIFO of pending demands
    GList gl_cur, gl_nxt;                // range decode: demands being served / being collected
    uint2* pairs;                        // left by the literal launch for the match launch: (dst_rel, len) of every match,
                                         // segment s at pairs[match_prefix[s] ..]
    uint8_t* cplanes;                    // ... and its decoded coded offset planes: n_coded_planes x n_match bytes per segment
    const uint64_t* match_prefix;        // n_segs + 1 entries
};

__device__ __forceinline__ uint32_t lane_id() { return threadIdx.x & 31; }
__device__ __forceinline__ uint32_t lanemask_lt() { uint32_t m; asm("mov.u32 %0, %%lanemask_lt;" : "=r"(m)); return m; }

// Flag poll.  Relaxed on purpose: an acquire load makes ptxas invalidate the whole L1 (CCTL.IVALL) on every poll.
// wait_block issues ONE fence.acq_rel.gpu after the loop has seen the value (PTX memory model: the relaxed load that
// observed the release, followed by the fence, synchronises with the writer); the guarded data is read with
// ld.cg / cp.async.cg (L2, the coherence point) after that fence.
__device__ __forceinline__ uint32_t ld_flag(const uint32_t* p) {
    uint32_t v; asm volatile("ld.relaxed.gpu.global.u32 %0, [%1];" : "=r"(v) : "l"(p) : "memory"); return v;
}
// data that other SMs may have written during this kernel: read at L2, never from a stale L1 line
__device__ __forceinline__ uint8_t ldcg8(const uint8_t* p) { return __ldcg(p); }
__device__ __forceinline__ uint64_t ldcg64(const uint8_t* p) { return __ldcg(reinterpret_cast<const unsigned long long*>(p)); }

// ------------------------------------------------------------------------------------------------ rANS ----------
// FORMAT.md §1.7.  32 states, one per lane; symbol i lives on lane i & 31; every state renormalises from its OWN word
// stream, so the decode step needs no ballot, no prefix and no shared cursor.  Each lane stages its stream through a
// private 64-byte ring in shared memory (four 16-byte chunks, filled with cp.async two chunks ahead of their use).
// The archive ends with a 128-byte pad (FORMAT.md §1), so the refill never tests the archive end.
__device__ __forceinline__ uint32_t lds32(uint32_t a) { uint32_t v; asm volatile("ld.shared.u32 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ uint32_t lds8(uint32_t a) { uint32_t v; asm volatile("ld.shared.u8 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ uint32_t lds16(uint32_t a) { uint32_t v; asm volatile("ld.shared.u16 %0, [%1];" : "=r"(v) : "r"(a)); return v; }
__device__ __forceinline__ uint2 lds64(uint32_t a) {
    uint2 v; asm volatile("ld.shared.v2.u32 {%0, %1}, [%2];" : "=r"(v.x), "=r"(v.y) : "r"(a)); return v;
}
__device__ __forceinline__ uint4 lds128(uint32_t a) {
    uint4 v; asm volatile("ld.shared.v4.u32 {%0, %1, %2, %3}, [%4];" : "=r"(v.x), "=r"(v.y), "=r"(v.z), "=r"(v.w) : "r"(a)); return v;
}
__device__ __forceinline__ void sts32(uint32_t a, uint32_t v) { asm volatile("st.shared.u32 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts64(uint32_t a, uint32_t x, uint32_t y) { asm volatile("st.shared.v2.u32 [%0], {%1, %2};" ::"r"(a), "r"(x), "r"(y) : "memory"); }
__device__ __forceinline__ void sts16(uint32_t a, uint32_t v) { asm volatile("st.shared.u16 [%0], %1;" ::"r"(a), "r"(v) : "memory"); }
__device__ __forceinline__ void sts128(uint32_t a, uint32_t x, uint32_t y, uint32_t z, uint32_t w) {
    asm volatile("st.shared.v4.u32 [%0], {%1, %2, %3, %4};" ::"r"(a), "r"(x), "r"(y), "r"(z), "r"(w) : "memory");
}
__device__ __forceinline__ void cp_async16s(uint32_t saddr, const void* gmem) {
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(saddr), "l"(gmem) : "memory");
}
__device__ __forceinline__ void cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
template <int N> __device__ __forceinline__ void cp_async_wait_group() { asm volatile("cp.async.wait_group %0;" ::"n"(N) : "memory"); }

struct Rans {
    uint32_t x;              // this lane's state
    uint32_t rp;             // byte offset of this lane's next word, relative to gbase; ring slot = rp & 63
    uint32_t fp;             // bytes of the stream requested into the ring so far (relative to gbase, multiple of 16)
    uint32_t ring;           // shared address of this lane's ring, 64-byte aligned
    uint32_t end;            // rp after the lane's last word (integrity check)
    uint32_t w;              // the word at rp, read ahead: a renormalisation does not wait for shared memory
    const uint8_t* gbase;    // 16-byte aligned global address that offsets are relative to

    __device__ __forceinline__ void fetch() { cp_async16s(ring | (fp & 63), gbase + fp); fp += 16; }
    // payload: [32 x (u32 state, u32 word_off)][words]; n_words = total words of the segment
    __device__ __forceinline__ void init(const uint8_t* payload, uint32_t n_words, uint32_t ring_warp) {
        const uint32_t lane = lane_id();
        uint2 h = __ldg(reinterpret_cast<const uint2*>(payload) + lane);
        x = h.x;
        uint32_t next = __shfl_down_sync(0xffffffffu, h.y, 1);
        if (lane == 31) next = n_words;
        const uint8_t* start = payload + 256 + 2ull * h.y;
        // bias the base by a lane-dependent multiple of 16 so that lanes in lockstep sit in different ring slots (banks)
        const uint32_t bias = 16u * ((lane >> 1) & 3u);
        gbase = start - (reinterpret_cast<uintptr_t>(start) & 15) - bias;
        rp = (uint32_t)(start - gbase);
        end = rp + 2u * (next - h.y);
        fp = bias;
        ring = ring_warp + 64u * lane;
        cp_async_wait_group<0>();            // chunks still in flight from the previous segment must not land after ours
        fetch(); cp_async_commit(); fetch(); cp_async_commit(); fetch(); cp_async_commit(); fetch(); cp_async_commit();
        cp_async_wait_group<2>();            // the first two chunks: at least 16 bytes from rp on
        w = lds16(ring | (rp & 63));
    }
    // Call before every group of <= 8 symbols per lane (<= 16 B of words).  Invariant after the call: fp - rp >= 50 and
    // everything but the two most recent chunks has landed, so the next 18 bytes are readable: 8 words and the one read
    // ahead (a read past the lane's last word sees the next lane's stream or the archive's tail pad, and is never used).
    __device__ __forceinline__ void prepare8() {
        if (fp - rp <= 48) fetch();          // the slot being refilled holds bytes below rp
        cp_async_commit();
        cp_async_wait_group<2>();
    }
    __device__ __forceinline__ void renorm() {
        if (x < 65536u) { x = (x << 16) + w; rp += 2; w = lds16(ring | (rp & 63)); }      // + : one IMAD
    }
    // one symbol on this lane.  lut = shared address of a byte table.  Returns the table entry (sym | bias << 8 |
    // freq << 20).  The ring is read only by the lanes that renormalise (a predicated load).
    __device__ __forceinline__ uint32_t step_full(uint32_t lut) {
        uint32_t e = lds32(lut + 4u * (x & (LUT_SIZE - 1)));
        x = (e >> 20) * (x >> PROB_BITS) + ((e >> 8) & 0xfff);
        renorm();
        return e;
    }
    // one symbol on the lanes with active == true
    __device__ __forceinline__ uint32_t step(uint32_t lut, bool active) {
        uint32_t e = lds32(lut + 4u * (x & (LUT_SIZE - 1)));
        uint32_t nx = (e >> 20) * (x >> PROB_BITS) + ((e >> 8) & 0xfff);
        if (active) { x = nx; renorm(); }
        return e;
    }
    // one PAIR symbol (FORMAT.md §1.7, pb = 12): entry = {pair | freq << 16, bias}; returns the low word
    __device__ __forceinline__ uint32_t step_pair_full(uint32_t lutq) {
        uint2 e = lds64(lutq + 8u * (x & (QLUT_SIZE - 1)));
        x = (e.x >> 16) * (x >> QPROB_BITS) + e.y;
        renorm();
        return e.x;
    }
    __device__ __forceinline__ uint32_t step_pair(uint32_t lutq, bool active) {
        uint2 e = lds64(lutq + 8u * (x & (QLUT_SIZE - 1)));
        uint32_t nx = (e.x >> 16) * (x >> QPROB_BITS) + e.y;
        if (active) { x = nx; renorm(); }
        return e.x;
    }
    __device__ __forceinline__ bool finished() const { return x == 65536u && rp == end; }
};

// Decodes `count` symbols whose global symbol indices start at i0, storing them to dst[0..count) (byte stores,
// consecutive lanes -> consecutive bytes; PAIR: 16-bit stores to a 2-byte aligned dst).  Returns the number of byte symbols
// equal to 255 (the escape count of a token stream; two instructions per round, ignored by the other streams, so that ONE
// instance of this loop serves every byte stream of a segment: the kernels are bound by instruction fetch as much as by
// issue).  dst == nullptr: decode without storing.
template <bool PAIR>
__device__ __forceinline__ uint32_t rans_region(Rans& r, uint32_t lut, uint32_t i0, uint32_t count, uint8_t* dst) {
    uint32_t esc = 0;
    if (count == 0) return 0;
    const uint32_t i1 = i0 + count, lane = lane_id();
    const bool store = dst != nullptr;
    constexpr uint32_t S = PAIR ? 2 : 1;
    uint32_t base = i0 & ~31u;
    uint8_t* p = dst + (int64_t)S * ((int64_t)lane - (int64_t)(i0 - base));     // address of symbol base + lane
    auto put = [&](uint8_t* q, uint32_t e) { if (PAIR) *reinterpret_cast<uint16_t*>(q) = (uint16_t)e; else *q = (uint8_t)e; };
    auto ragged = [&]() {                                // one round in which some lanes have no symbol
        const uint32_t i = base + lane;
        const bool active = i >= i0 && i < i1;
        r.prepare8();
        const uint32_t e = PAIR ? r.step_pair(lut, active) : r.step(lut, active);
        if (active && store) put(p, e);
        if (!PAIR && active && (~e & 0xffu) == 0) esc++;
        base += 32; p += 32 * S;
    };
    if (base != i0) ragged();
    uint32_t full = i1 > base ? (i1 - base) >> 5 : 0;     // complete rounds
    base += 32 * full;
    for (; full >= 8; full -= 8) {                       // eight rounds per ring check
        r.prepare8();
#pragma unroll
        for (int k = 0; k < 8; k++) {
            const uint32_t e = PAIR ? r.step_pair_full(lut) : r.step_full(lut);
            if (store) put(p + 32 * S * k, e);
            if (!PAIR && (~e & 0xffu) == 0) esc++;
        }
        p += 256 * S;
    }
    if (full) {
        r.prepare8();
#pragma unroll 1
        for (; full; full--, p += 32 * S) {
            const uint32_t e = PAIR ? r.step_pair_full(lut) : r.step_full(lut);
            if (store) put(p, e);
            if (!PAIR && (~e & 0xffu) == 0) esc++;
        }
    }
    if (base < i1) ragged();
    return PAIR ? 0u : __reduce_add_sync(0xffffffffu, esc);    // per-lane counts, one REDUX per region
}

// ------------------------------------------------------------------------------------------------ copies --------
// SRC_CG: the source may have been written by other SMs during this kernel -> read at L2 (ld.cg), never from L1.
template <bool SRC_CG> __device__ __forceinline__ uint64_t ld64a(const uint8_t* p) {   // p is 8-byte aligned
    return SRC_CG ? ldcg64(p) : *reinterpret_cast<const uint64_t*>(p);
}
// 8 bytes starting at any address: the aligned word(s) that hold them (never touches a word without a wanted byte
// when n_valid bytes are wanted)
template <bool SRC_CG> __device__ __forceinline__ uint64_t ld64u(const uint8_t* p, uint32_t n_valid) {
    uint32_t sh = (uint32_t)(reinterpret_cast<uintptr_t>(p) & 7);
    const uint8_t* a = p - sh;
    uint64_t lo = ld64a<SRC_CG>(a);
    if (sh == 0) return lo;
    uint64_t hi = (sh + n_valid > 8) ? ld64a<SRC_CG>(a + 8) : 0;
    return (lo >> (8 * sh)) | (hi << (64 - 8 * sh));
}
// store the low n (<= 8) bytes of v at any address, using the widest naturally aligned stores
__device__ __forceinline__ void st_small(uint8_t* d, uint64_t v, uint32_t n) {
    if (n >= 8 && (reinterpret_cast<uintptr_t>(d) & 7) == 0) { *reinterpret_cast<uint64_t*>(d) = v; return; }
    if (n && (reinterpret_cast<uintptr_t>(d) & 1)) { *d = (uint8_t)v; v >>= 8; d++; n--; }
    if (n >= 2 && (reinterpret_cast<uintptr_t>(d) & 2)) { *reinterpret_cast<uint16_t*>(d) = (uint16_t)v; v >>= 16; d += 2; n -= 2; }
    if (n >= 4) { *reinterpret_cast<uint32_t*>(d) = (uint32_t)v; v >>= 32; d += 4; n -= 4; }   // d is 4-aligned here or n < 2
    if (n >= 4) { *reinterpret_cast<uint32_t*>(d) = (uint32_t)v; d += 4; n -= 4; v = 0; }
    if (n >= 2) { *reinterpret_cast<uint16_t*>(d) = (uint16_t)v; v >>= 16; d += 2; n -= 2; }
    if (n) *d = (uint8_t)v;
}

// dst/src may have any alignment and must not overlap: loads are issued ahead of the stores that depend on them,
// 8 bytes at a time.
template <bool SRC_CG>
__device__ __forceinline__ void copy_bytes(uint8_t* dst, const uint8_t* src, uint32_t len) {
    if (len <= 16) {
        uint64_t lo = ld64u<SRC_CG>(src, len < 8 ? len : 8);
        uint64_t hi = len > 8 ? ld64u<SRC_CG>(src + 8, len - 8) : 0;
        st_small(dst, lo, len < 8 ? len : 8);
        if (len > 8) st_small(dst + 8, hi, len - 8);
        return;
    }
    // head: bring dst to 8-byte alignment; tail: the last (< 8) bytes.  Both are loaded before any store.
    uint32_t head = (uint32_t)(-reinterpret_cast<intptr_t>(dst)) & 7;
    uint64_t hv = head ? ld64u<SRC_CG>(src, head) : 0;
    uint32_t body = (len - head) & ~7u, tail = len - head - body;
    uint64_t tv = tail ? ld64u<SRC_CG>(src + head + body, tail) : 0;
    const uint8_t* s = src + head;
    uint8_t* d = dst + head;
    uint32_t sh = (uint32_t)(reinterpret_cast<uintptr_t>(s) & 7) * 8;
    if (sh == 0) {
        uint32_t i = 0;
        for (; i + 16 <= body; i += 16) {
            uint64_t a = ld64a<SRC_CG>(s + i), b = ld64a<SRC_CG>(s + i + 8);
            *reinterpret_cast<uint64_t*>(d + i) = a; *reinterpret_cast<uint64_t*>(d + i + 8) = b;
        }
        if (i < body) *reinterpret_cast<uint64_t*>(d + i) = ld64a<SRC_CG>(s + i);
    } else {
        const uint8_t* sa = s - (sh >> 3);
        uint64_t lo = ld64a<SRC_CG>(sa);
        uint32_t i = 0;
        for (; i + 16 <= body; i += 16) {   // words sa+8 .. sa+16 hold wanted bytes: i + 16 <= body <= len - head
            uint64_t m = ld64a<SRC_CG>(sa + i + 8), h2 = ld64a<SRC_CG>(sa + i + 16);
            *reinterpret_cast<uint64_t*>(d + i) = (lo >> sh) | (m << (64 - sh));
            *reinterpret_cast<uint64_t*>(d + i + 8) = (m >> sh) | (h2 << (64 - sh));
            lo = h2;
        }
        if (i < body) {
            uint64_t m = ld64a<SRC_CG>(sa + i + 8);
            *reinterpret_cast<uint64_t*>(d + i) = (lo >> sh) | (m << (64 - sh));
        }
    }
    if (head) st_small(dst, hv, head);
    if (tail) st_small(d + body, tv, tail);
}

// Warp-cooperative copy of a long non-overlapping run: every lane moves 16 bytes per iteration, destination-aligned
// 16-byte stores (512 B per warp instruction), byte lanes for the unaligned head and tail.  All 32 lanes must call.
template <bool SRC_CG>
__device__ __forceinline__ void warp_copy(uint8_t* dst, const uint8_t* src, uint32_t len) {
    const uint32_t lane = lane_id();
    uint32_t head = (uint32_t)(-reinterpret_cast<intptr_t>(dst)) & 15;
    if (head > len) head = len;
    if (lane < head) dst[lane] = SRC_CG ? ldcg8(src + lane) : src[lane];
    uint32_t body = (len - head) & ~15u;
    for (uint32_t off = head + 16 * lane; off < head + body; off += 512) {
        const uint8_t* s = src + off;
        uint32_t sh = (uint32_t)(reinterpret_cast<uintptr_t>(s) & 7) * 8;
        const uint8_t* sa = s - (sh >> 3);
        uint64_t w0 = ld64a<SRC_CG>(sa), w1 = ld64a<SRC_CG>(sa + 8), lo, hi;
        if (sh == 0) { lo = w0; hi = w1; }
        else { uint64_t w2 = ld64a<SRC_CG>(sa + 16); lo = (w0 >> sh) | (w1 << (64 - sh)); hi = (w1 >> sh) | (w2 << (64 - sh)); }
        uint2 a = make_uint2((uint32_t)lo, (uint32_t)(lo >> 32)), b2 = make_uint2((uint32_t)hi, (uint32_t)(hi >> 32));
        *reinterpret_cast<uint4*>(dst + off) = make_uint4(a.x, a.y, b2.x, b2.y);
    }
    uint32_t done = head + body;
    if (done + lane < len) dst[done + lane] = SRC_CG ? ldcg8(src + done + lane) : src[done + lane];
}

} // namespace acx
