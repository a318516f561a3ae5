// Host side of the C ABI (include/aceapex.h): archive validation, workspace layout, launch schedules.
// The kernels are in acx_kernels.cuh.
#include "aceapex.h"
#include "acx_kernels.cuh"

#include <algorithm>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>
#include <vector>

using namespace acx;

// ====================================================================================================== host =====

// A launch sequence kept as a CUDA graph (seek latency "dominated by fixed kernel-launch
// overhead").  A seek issues the same kernels in the same order every time, only their arguments differ: the calls are
// recorded instead of launched, the node parameters of the instantiated graph are updated in place, and one
// cudaGraphLaunch replaces six to ten launches and memsets.
struct GNode {
    const void* func = nullptr;                         // null: a memset node
    dim3 grid, block; size_t smem = 0; bool coop = false;
    std::vector<uint8_t> blob; std::vector<size_t> arg_off;   // kernel arguments, copied
    void* ptr = nullptr; size_t bytes = 0;              // memset
};
struct SeekGraph {
    cudaGraph_t graph = nullptr; cudaGraphExec_t exec = nullptr;
    std::vector<cudaGraphNode_t> nodes; std::vector<const void*> sig;
};

struct aceapex_archive {
    const uint8_t* d_archive = nullptr;
    uint64_t archive_bytes = 0;
    // header
    uint64_t N = 0, n_blocks = 0, n_segs = 0, tables_off = 0, qtab_off = 0, blocktab_off = 0, dir_off = 0, fnv_off = 0, payload_off = 0;
    uint64_t total_lit = 0, total_match_bytes = 0, total_matches = 0, total_cmds = 0, total_litq = 0;
    uint32_t log2_bs = 0, log2_seg = 0, min_match = 0, W = 0, max_level = 0, max_cmds = 0, flags = 0, q_min = 0, q_mode = 0, n_qpairs = 0;
    uint32_t n_coded_tables = 0, n_coded_planes = 0, n_raw_planes = 0;
    int8_t plane_lut[MAX_W];
    uint32_t lut_cmd = 0, lut_mlen = 0, lut_lita = 0, lut_litq = 0;
    // device state owned by the library
    uint32_t* d_luts = nullptr; uint2* d_lutq = nullptr;
    uint32_t* d_seg_lists = nullptr;                    // segment ids sorted by (level, index); null when max_level = 0
    std::vector<uint64_t> level_off;                    // level l: d_seg_lists[level_off[l] .. level_off[l + 1])
    uint16_t* d_levels = nullptr;                       // level per block
    uint32_t* d_first_seg = nullptr;                    // n_blocks + 1
    uint64_t* d_match_prefix = nullptr;                 // matches in segments [0, s), n_segs + 1 entries
    // host copies
    std::vector<uint16_t> h_levels; std::vector<uint32_t> h_first_seg; std::vector<uint64_t> h_match_prefix, h_payload_off;
    // workspace (caller's)
    uint8_t* d_ws = nullptr; uint64_t ws_bytes = 0; bool ws_clean = false;
    cudaStream_t stream = nullptr;
    bool cooperative = false;                           // cooperative launches are possible (all CTAs resident)
    uint32_t ticket_slot = 0;                           // which of the two ticket slots the next launch draws from
    Resident res[MAX_RESIDENT];
    // launch geometry
    int sms = 148, threads = 1024;
    size_t smem_entropy = 0, smem_copy = 0, smem_fused = 0;
    uint32_t runs_bytes = 0, lita_bytes = 0;              // per-warp shared memory of the entropy kernels (acx_kernels.cuh setup_cta)
    uint64_t scratch_per_warp = 0, ctrl_bytes = 0;
    uint64_t done_off = 0, scratch_off = 0, stacks_off = 0, demands_off = 0, list_off = 0, ws_need = 0;
    uint32_t stack_cap = 0, demand_cap = 0;
    uint64_t gl_cap = 0, gl_tcap = 0, gl_wcap = 0, gl_rec_off[2] = {0, 0}, gl_cnt_off[2] = {0, 0}, gl_touched_off[2] = {0, 0};   // range decode lists
    uint64_t gl_sorted_off = 0, gl_work_off = 0, gl_workn_off = 0, desc_off = 0, cplanes_off = 0;
    uint64_t gl_eff = 0;                                // records a range-decode call may use (vram_budget), <= gl_cap
    // end-to-end pipeline (aceapex_decode_all_host): chunks of blocks, per chunk the segment ids sorted by level
    uint64_t chunk_blocks = 0; uint32_t* d_chunk_lists = nullptr; std::vector<uint64_t> chunk_level_off;   // (chunk, level) -> offset
    cudaStream_t s_h2d = nullptr, s_d2h = nullptr; std::vector<cudaEvent_t> ev_h2d, ev_dec;
    bool phase_timing = false; cudaEvent_t ev_phase[4] = {nullptr, nullptr, nullptr, nullptr};   // aceapex_set_phase_timing
    std::vector<uint32_t> h_list; std::vector<Demand> h_demands;   // host staging for range / read calls
    // CUDA graphs of the seek / single-read paths
    bool use_graphs = true; bool capturing = false;     // capturing: launches are recorded into `rec` instead of issued
    std::vector<GNode> rec;
    SeekGraph g_seek;
    uint64_t graph_launches = 0, graph_rebuilds = 0;
    // status
    int32_t last_cuda = 0; uint32_t dev_flags = 0; uint64_t launches = 0;
};

namespace {

uint64_t rd64(const uint8_t* p) { uint64_t v; memcpy(&v, p, 8); return v; }
uint32_t rd32(const uint8_t* p) { uint32_t v; memcpy(&v, p, 4); return v; }
uint16_t rd16(const uint8_t* p) { uint16_t v; memcpy(&v, p, 2); return v; }

#define CU(call) do { cudaError_t e_ = (call); if (e_ != cudaSuccess) { ar->last_cuda = (int32_t)e_; return ACEAPEX_E_CUDA; } } while (0)

constexpr uint64_t TAIL_PAD = 128;
uint64_t align_up(uint64_t v, uint64_t a) { return (v + a - 1) / a * a; }

// workspace: [ctrl 512 B: ticket slots u64 @0 and @24, err u32 @8, fnv count @16, list counters @64, round / fused tickets @128]
//            [done: n_blocks x u32][scratch: warps x scratch_per_warp][stacks: warps x stack_cap demands][demands: demand_cap]
//            [segment list of a window: n_segs x u32][demand lists][match descriptors][decoded coded offset planes]
void layout_workspace(aceapex_archive* ar) {
    const uint64_t warps = (uint64_t)ar->sms * (ar->threads / 32);
    ar->ctrl_bytes = 512;
    ar->done_off = ar->ctrl_bytes;
    ar->scratch_off = align_up(ar->done_off + 4 * ar->n_blocks + 4, 256);
    ar->stack_cap = 2048;
    ar->demand_cap = 1u << 16;
    ar->stacks_off = align_up(ar->scratch_off + warps * ar->scratch_per_warp, 256);
    ar->demands_off = align_up(ar->stacks_off + warps * ar->stack_cap * sizeof(Demand), 256);
    ar->list_off = align_up(ar->demands_off + (uint64_t)ar->demand_cap * sizeof(Demand), 256);
    uint64_t off = align_up(ar->list_off + 4 * ar->n_segs + 4, 256);
    // demand lists of range decode (two sets, alternating between rounds); counters live in the control area at +64
    ar->gl_cap = std::min<uint64_t>(1ull << 24, std::max<uint64_t>(1ull << 16, ar->total_matches / 2));
    ar->gl_tcap = std::max<uint64_t>(1, std::min<uint64_t>(ar->n_segs, ar->gl_cap));
    ar->gl_wcap = ar->gl_tcap + ar->gl_cap / GL_ITEM + 1;
    for (int k = 0; k < 2; k++) {
        ar->gl_rec_off[k] = off; off = align_up(off + ar->gl_cap * sizeof(GDemand), 256);
        ar->gl_cnt_off[k] = off; off = align_up(off + 4 * ar->n_segs + 4, 256);
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
    P.archive = ar->d_archive;
    P.dir = reinterpret_cast<const SegEntry*>(ar->d_archive + ar->dir_off);
    P.luts = ar->d_luts; P.lutq = ar->d_lutq; P.levels = ar->d_levels; P.first_seg = ar->d_first_seg;
    P.N = ar->N; P.n_segs = ar->n_segs; P.log2_bs = ar->log2_bs; P.log2_seg = ar->log2_seg; P.min_match = ar->min_match; P.W = ar->W;
    P.n_coded_tables = ar->n_coded_tables; P.q_min = ar->q_min; P.q_mode = ar->q_mode;
    memcpy(P.plane_lut, ar->plane_lut, MAX_W);
    P.n_coded_planes = ar->n_coded_planes; P.n_raw_planes = ar->n_raw_planes;
    for (int p = (int)ar->W - 1, k = 0; p >= 0; p--) if (ar->plane_lut[p] >= 0) P.coded_shift[k++] = (uint8_t)(8 * p);
    for (int p = (int)ar->W - 1, k = 0; p >= 0; p--) if (ar->plane_lut[p] >= 0) P.coded_lut[k++] = (uint8_t)ar->plane_lut[p];
    for (uint32_t p = 0, r = 0; p < ar->W; p++) if (ar->plane_lut[p] < 0) P.raw_shift[r++] = (uint8_t)(8 * p);
    P.lut_cmd = ar->lut_cmd; P.lut_mlen = ar->lut_mlen; P.lut_lita = ar->lut_lita; P.lut_litq = ar->lut_litq;
    P.runs_bytes = ar->runs_bytes; P.lita_bytes = ar->lita_bytes;
    memcpy(P.res, ar->res, sizeof P.res);
    P.err = reinterpret_cast<uint32_t*>(ar->d_ws + 8);
    P.done = reinterpret_cast<uint32_t*>(ar->d_ws + ar->done_off);
    P.scratch = ar->d_ws + ar->scratch_off;
    P.scratch_per_warp = ar->scratch_per_warp;
    P.out_pos0 = 0; P.win_end = ar->N; P.copy_parts = 1;
    P.stacks = reinterpret_cast<Demand*>(ar->d_ws + ar->stacks_off); P.stack_cap = ar->stack_cap;
    P.pairs = reinterpret_cast<uint2*>(ar->d_ws + ar->desc_off);
    P.cplanes = ar->d_ws + ar->cplanes_off;
    P.match_prefix = ar->d_match_prefix;
}

void set_out(Params& P, uint8_t* out, uint64_t pos0, uint64_t end) {
    P.out = out; P.out_pos0 = pos0; P.win_end = end;
    P.out_odd = (uint32_t)((reinterpret_cast<uintptr_t>(out) - pos0) & 1);
}

int32_t prepare_ws(aceapex_archive* ar) {
    if (!ar->d_ws || ar->ws_bytes < ar->ws_need) return ACEAPEX_E_WORKSPACE;
    if (!ar->ws_clean) {
        CU(cudaMemsetAsync(ar->d_ws, 0, ar->scratch_off, ar->stream));
        for (int k = 0; k < 2; k++) CU(cudaMemsetAsync(ar->d_ws + ar->gl_cnt_off[k], 0, 4 * ar->n_segs + 4, ar->stream));
        ar->ws_clean = true; ar->ticket_slot = 0;
    }
    return ACEAPEX_OK;
}

// Few work items: spread them over all SMs with fewer warps per CTA instead of filling a few CTAs with 32 warps each (a
// warp that shares its SM with fewer others finishes its segment sooner).  T <= max_threads, g <= SMs (all CTAs resident).
void spread(const aceapex_archive* ar, uint64_t n_work, int max_threads, uint32_t& g, int& T) {
    const uint64_t per_sm = (n_work + ar->sms - 1) / ar->sms;
    T = (int)std::min<uint64_t>((uint64_t)max_threads, 32 * std::max<uint64_t>(per_sm, 1));
    g = (uint32_t)std::min<uint64_t>(ar->sms, (n_work + T / 32 - 1) / (T / 32));
}

void take_ticket(aceapex_archive* ar, Params& P) {
    P.ticket = reinterpret_cast<unsigned long long*>(ar->d_ws) + (ar->ticket_slot ? 3 : 0);       // bytes 0 and 24 of the control area
    P.ticket_next = reinterpret_cast<unsigned long long*>(ar->d_ws) + (ar->ticket_slot ? 0 : 3);
    ar->ticket_slot ^= 1;
}

constexpr int32_t NOT_GRAPHABLE = 1;                    // internal: the call needs something a recorded sequence cannot hold

struct KArg { const void* p; size_t n; };
int32_t submit_kernel(aceapex_archive* ar, const void* func, dim3 grid, dim3 block, size_t smem, bool coop, std::initializer_list<KArg> args) {
    if (ar->capturing) {
        GNode nd; nd.func = func; nd.grid = grid; nd.block = block; nd.smem = smem; nd.coop = coop;
        for (const KArg& a : args) {
            const size_t off = (nd.blob.size() + 15) & ~(size_t)15;
            nd.blob.resize(off + a.n); memcpy(nd.blob.data() + off, a.p, a.n); nd.arg_off.push_back(off);
        }
        ar->rec.push_back(std::move(nd));
        ar->launches++;
        return ACEAPEX_OK;
    }
    void* argv[4]; int k = 0;
    for (const KArg& a : args) argv[k++] = const_cast<void*>(a.p);
    if (coop) CU(cudaLaunchCooperativeKernel(func, grid, block, argv, smem, ar->stream));
    else CU(cudaLaunchKernel(func, grid, block, argv, smem, ar->stream));
    ar->launches++;
    return ACEAPEX_OK;
}
int32_t submit_memset(aceapex_archive* ar, void* ptr, size_t bytes) {
    if (ar->capturing) { GNode nd; nd.ptr = ptr; nd.bytes = bytes; ar->rec.push_back(std::move(nd)); return ACEAPEX_OK; }
    CU(cudaMemsetAsync(ptr, 0, bytes, ar->stream));
    return ACEAPEX_OK;
}

// launches the recorded sequence as a graph: same sequence of kernels as the instantiated one -> parameters updated in place
int32_t replay(aceapex_archive* ar) {
    SeekGraph& G = ar->g_seek;
    std::vector<const void*> sig;
    for (const GNode& n : ar->rec) sig.push_back(n.func);
    std::vector<std::vector<void*>> argv(ar->rec.size());
    auto kparams = [&](size_t i) {
        GNode& n = ar->rec[i];
        cudaKernelNodeParams kp; memset(&kp, 0, sizeof kp);
        for (size_t off : n.arg_off) argv[i].push_back(n.blob.data() + off);
        kp.func = const_cast<void*>(n.func); kp.gridDim = n.grid; kp.blockDim = n.block; kp.sharedMemBytes = (unsigned)n.smem; kp.kernelParams = argv[i].data();
        return kp;
    };
    auto mparams = [&](size_t i) {
        cudaMemsetParams mp; memset(&mp, 0, sizeof mp);
        mp.dst = ar->rec[i].ptr; mp.value = 0; mp.elementSize = 1; mp.width = ar->rec[i].bytes; mp.height = 1; mp.pitch = ar->rec[i].bytes;
        return mp;
    };
    bool ok = G.exec && sig == G.sig;
    if (ok) {
        for (size_t i = 0; i < ar->rec.size() && ok; i++) {
            if (ar->rec[i].func) { cudaKernelNodeParams kp = kparams(i); ok = cudaGraphExecKernelNodeSetParams(G.exec, G.nodes[i], &kp) == cudaSuccess; }
            else { cudaMemsetParams mp = mparams(i); ok = cudaGraphExecMemsetNodeSetParams(G.exec, G.nodes[i], &mp) == cudaSuccess; }
        }
        if (!ok) cudaGetLastError();
    }
    if (!ok) {                                           // first use, or another sequence: build and instantiate
        if (G.exec) { cudaGraphExecDestroy(G.exec); G.exec = nullptr; }
        if (G.graph) { cudaGraphDestroy(G.graph); G.graph = nullptr; }
        for (auto& v : argv) v.clear();
        CU(cudaGraphCreate(&G.graph, 0));
        G.nodes.assign(ar->rec.size(), nullptr);
        for (size_t i = 0; i < ar->rec.size(); i++) {
            const cudaGraphNode_t* dep = i ? &G.nodes[i - 1] : nullptr;
            if (ar->rec[i].func) {
                cudaKernelNodeParams kp = kparams(i);
                CU(cudaGraphAddKernelNode(&G.nodes[i], G.graph, dep, i ? 1 : 0, &kp));
                if (ar->rec[i].coop) {
                    cudaKernelNodeAttrValue v; memset(&v, 0, sizeof v); v.cooperative = 1;
                    CU(cudaGraphKernelNodeSetAttribute(G.nodes[i], cudaKernelNodeAttributeCooperative, &v));
                }
            } else { cudaMemsetParams mp = mparams(i); CU(cudaGraphAddMemsetNode(&G.nodes[i], G.graph, dep, i ? 1 : 0, &mp)); }
        }
        CU(cudaGraphInstantiate(&G.exec, G.graph, 0));
        G.sig = sig;
        ar->graph_rebuilds++;
    }
    CU(cudaGraphLaunch(G.exec, ar->stream));
    ar->graph_launches++;
    return ACEAPEX_OK;
}

enum Kind { K_LIT, K_LIT_COLLECT, K_COPY_TOP, K_COPY_WAIT, K_COPY_WIN, K_COPY_WIN_WAIT, K_COLLECT, K_SERVE, K_SPANS, K_SPANS_CTA };

int32_t launch(aceapex_archive* ar, Params& P, Kind kind, uint64_t n_work) {
    P.n_work = n_work; P.copy_parts = 1;
    if (n_work == 0) return ACEAPEX_OK;
    take_ticket(ar, P);
    if (kind == K_COPY_TOP || kind == K_COPY_WAIT || kind == K_COPY_WIN || kind == K_COPY_WIN_WAIT || kind == K_COLLECT) {
        // a seek: far fewer segments than resident warps; every segment's matches are shared out among up to eight warps
        static const uint32_t max_parts = getenv("ACEAPEX_COPY_PARTS") ? (uint32_t)atoi(getenv("ACEAPEX_COPY_PARTS")) : 8;
        const uint64_t resident = (uint64_t)ar->sms * (ar->threads / 32);
        uint32_t parts = 1;
        while (parts < max_parts && n_work * parts * 2 <= resident / 2) parts *= 2;
        P.copy_parts = parts; P.n_work = n_work * parts; n_work = P.n_work;
    }
    int T; uint32_t g;
    spread(ar, n_work, ar->threads, g, T);
    // kernels that stage the decode tables (40-70 KB per CTA): a CTA of one or two warps would spend tens of microseconds
    // loading them; at least eight warps load (the ones without work find no ticket and leave)
    static const int min_t = getenv("ACEAPEX_MIN_THREADS") ? atoi(getenv("ACEAPEX_MIN_THREADS")) : 256;
    if ((kind == K_LIT || kind == K_LIT_COLLECT || kind == K_SPANS) && T < min_t) T = std::min(ar->threads, std::max(T, min_t / 32 * 32));
    const size_t sm_e = entropy_smem(ar->n_coded_tables, ar->q_mode, ar->runs_bytes + ALIST_BYTES + ar->lita_bytes, T), sm_c = (size_t)(T / 32) * COPY_WARP_BYTES + 64;
    const void* f = nullptr; size_t sm = sm_c; dim3 gd(g), bd(T);
    switch (kind) {
        case K_LIT:
            sm = sm_e;
            if (!ar->q_mode) f = ar->q_min >= 64 ? (const void*)k_literals<3> : (const void*)k_literals<0>;
            else if (P.out_odd) f = (const void*)k_literals<2>;
            else f = ar->q_min >= 64 ? (const void*)k_literals<4> : (const void*)k_literals<1>;
            break;
        case K_LIT_COLLECT:                                    // a window: literal pass and collect pass in one launch
            sm = sm_e;
            if (!ar->q_mode) f = ar->q_min >= 64 ? (const void*)k_literals<3, true> : (const void*)k_literals<0, true>;
            else if (P.out_odd) f = (const void*)k_literals<2, true>;
            else f = ar->q_min >= 64 ? (const void*)k_literals<4, true> : (const void*)k_literals<1, true>;
            break;
        case K_COPY_TOP: f = (const void*)k_copy<false, false, false, true>; break;
        case K_COPY_WAIT: f = (const void*)k_copy<true, false, false, false>; break;
        case K_COPY_WIN: f = (const void*)k_copy<false, true, false, false>; break;
        case K_COPY_WIN_WAIT: f = (const void*)k_copy<true, true, false, false>; break;
        case K_COLLECT: f = (const void*)k_copy<false, true, true, false>; break;
        case K_SERVE: f = (const void*)k_serve; sm = ar->smem_entropy; gd = dim3(ar->sms); bd = dim3(ar->threads); break;
        case K_SPANS: f = (const void*)k_spans; sm = sm_e; break;
        case K_SPANS_CTA: {                                    // one CTA of up to 16 warps that share the read's queue of spans
            const int Tc = std::max(128, std::min(ar->threads, 512));
            f = (const void*)k_spans_cta; gd = dim3(1); bd = dim3(Tc);
            sm = entropy_smem(ar->n_coded_tables, ar->q_mode, ar->runs_bytes + ALIST_BYTES + ar->lita_bytes, Tc);
            break;
        }
    }
    return submit_kernel(ar, f, gd, bd, sm, false, {{&P, sizeof P}});
}

int32_t zero_done(aceapex_archive* ar, uint64_t b0, uint64_t nb) { return submit_memset(ar, ar->d_ws + ar->done_off + 4 * b0, 4 * nb); }

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
    if (archive_bytes < 192) return ACEAPEX_E_TRUNCATED;
    uint8_t hdr[192];
    if (h_archive) memcpy(hdr, h_archive, 192); else CU(cudaMemcpy(hdr, d_archive, 192, cudaMemcpyDeviceToHost));
    static const uint8_t magic[8] = {0x41, 0x43, 0x58, 0x42, 0x32, 0x30, 0x30, 0x00};
    if (memcmp(hdr, magic, 8)) return ACEAPEX_E_MAGIC;
    if (rd32(hdr + 8) != 3 || rd32(hdr + 52) != (uint32_t)PROB_BITS) return ACEAPEX_E_VERSION;
    if (rd32(hdr + 12) != 192) return ACEAPEX_E_CORRUPT;
    ar->N = rd64(hdr + 16); ar->n_blocks = rd64(hdr + 24); ar->n_segs = rd64(hdr + 32); ar->log2_bs = rd32(hdr + 40); ar->min_match = rd32(hdr + 44);
    ar->W = rd32(hdr + 48); uint32_t n_tables = rd32(hdr + 56); ar->max_level = rd32(hdr + 60); ar->max_cmds = rd32(hdr + 64);
    ar->flags = rd32(hdr + 68); ar->log2_seg = rd32(hdr + 72); ar->q_min = rd32(hdr + 76); ar->q_mode = rd32(hdr + 80); ar->n_qpairs = rd32(hdr + 84);
    ar->tables_off = rd64(hdr + 88); ar->qtab_off = rd64(hdr + 96); ar->blocktab_off = rd64(hdr + 104); ar->dir_off = rd64(hdr + 112);
    ar->fnv_off = rd64(hdr + 120); ar->payload_off = rd64(hdr + 128); uint64_t abytes = rd64(hdr + 136);
    ar->total_lit = rd64(hdr + 144); ar->total_match_bytes = rd64(hdr + 152); ar->total_matches = rd64(hdr + 160); ar->total_cmds = rd64(hdr + 168);
    ar->total_litq = rd64(hdr + 176);
    if (ar->log2_bs < 3 || ar->log2_bs > 20 || ar->min_match < 1 || ar->W < 4 || ar->W > 8 || n_tables != 4 + ar->W) return ACEAPEX_E_CORRUPT;
    if (ar->W < 8 && ar->N > (1ull << (8 * ar->W))) return ACEAPEX_E_CORRUPT;
    if (ar->log2_seg < 3 || ar->log2_seg > 14 || ar->log2_seg > ar->log2_bs) return ACEAPEX_E_CORRUPT;
    if (ar->q_min == 1 || ar->q_mode > 1 || (ar->q_min == 0 && ar->q_mode)) return ACEAPEX_E_CORRUPT;
    if (ar->q_mode == 1 ? (ar->n_qpairs < 1 || ar->n_qpairs > 4096) : ar->n_qpairs != 0) return ACEAPEX_E_CORRUPT;
    if (ar->max_cmds > MAX_SEG_CMDS || ar->max_level > 65535) return ACEAPEX_E_CORRUPT;
    if (ar->n_blocks != (ar->N + (1ull << ar->log2_bs) - 1) >> ar->log2_bs) return ACEAPEX_E_CORRUPT;
    if (ar->n_segs < ar->n_blocks || ar->n_segs >= (1ull << 32)) return ACEAPEX_E_CORRUPT;
    if (abytes > archive_bytes) return ACEAPEX_E_TRUNCATED;
    if (abytes % 16 || abytes < 192 + TAIL_PAD) return ACEAPEX_E_CORRUPT;
    uint64_t at = 192;
    if (ar->tables_off < at || ar->tables_off % 16) return ACEAPEX_E_CORRUPT;
    at = ar->tables_off + 528ull * n_tables;
    if (ar->qtab_off < at || ar->qtab_off % 16) return ACEAPEX_E_CORRUPT;
    at = ar->qtab_off + 4ull * ar->n_qpairs;
    if (ar->blocktab_off < at || ar->blocktab_off % 16) return ACEAPEX_E_CORRUPT;
    at = ar->blocktab_off + 8 * (ar->n_blocks + 1);
    if (ar->dir_off < at || ar->dir_off % 16) return ACEAPEX_E_CORRUPT;
    at = ar->dir_off + 32 * ar->n_segs;
    if (ar->flags & 1) { if (ar->fnv_off < at || ar->fnv_off % 8) return ACEAPEX_E_CORRUPT; at = ar->fnv_off + 8 * ar->n_blocks; }
    const uint64_t meta_end = at;
    if (meta_end > abytes || ar->payload_off < meta_end || ar->payload_off % 16 || ar->payload_off > abytes - TAIL_PAD) return ACEAPEX_E_CORRUPT;
    if (ar->total_lit + ar->total_match_bytes != ar->N || ar->total_litq > ar->total_lit) return ACEAPEX_E_CORRUPT;
    ar->archive_bytes = abytes;
    // tables, block table, directory
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
    for (uint32_t p = 0; p < MAX_W; p++) ar->plane_lut[p] = -1;
    for (uint32_t t = 0; t < n_tables; t++) {
        const uint32_t mode = rd32(meta + ar->tables_off + 528ull * t);
        const bool is_plane = t >= 2 && t < 2 + ar->W, litq_unused = t == 3 + ar->W && (ar->q_min == 0 || ar->q_mode == 1);
        if (mode > 2 || (mode == 1 && !is_plane) || ((mode == 2) != litq_unused)) return ACEAPEX_E_CORRUPT;
        uint32_t idx = 0;
        if (mode == 0 && !add_lut(t, idx)) return ACEAPEX_E_CORRUPT;
        if (t == 0) ar->lut_cmd = idx; else if (t == 1) ar->lut_mlen = idx; else if (t == 2 + ar->W) ar->lut_lita = idx;
        else if (t == 3 + ar->W) ar->lut_litq = idx;
        else {
            ar->plane_lut[t - 2] = mode == 0 ? (int8_t)idx : -1;
            if (mode == 0) ar->n_coded_planes++; else ar->n_raw_planes++;
        }
    }
    ar->n_coded_tables = (uint32_t)(luts.size() / LUT_SIZE);
    std::vector<uint2> lutq;
    if (ar->q_mode == 1) {
        lutq.resize(QLUT_SIZE);
        uint32_t cum = 0, prev = 0;
        for (uint32_t i = 0; i < ar->n_qpairs; i++) {
            const uint32_t pair = rd16(meta + ar->qtab_off + 4ull * i), f = rd16(meta + ar->qtab_off + 4ull * i + 2);
            if (f < 1 || cum + f > (uint32_t)QLUT_SIZE || (i > 0 && pair <= prev)) return ACEAPEX_E_CORRUPT;
            for (uint32_t k = 0; k < f; k++) lutq[cum + k] = make_uint2(pair | f << 16, k);
            cum += f; prev = pair;
        }
        if (cum != (uint32_t)QLUT_SIZE) return ACEAPEX_E_CORRUPT;
    }
    // block table + segment directory validation, level lists
    ar->h_levels.resize(ar->n_blocks); ar->h_first_seg.resize(ar->n_blocks + 1);
    ar->h_match_prefix.assign(ar->n_segs + 1, 0);
    ar->h_payload_off.assign(ar->n_segs + 1, abytes - TAIL_PAD);
    std::vector<uint64_t> level_cnt(ar->max_level + 2, 0);
    uint64_t prev_po = ar->payload_off;
    uint32_t seen_max_cmds = 0, seen_max_level = 0;
    for (uint64_t b = 0; b <= ar->n_blocks; b++) {
        const uint8_t* p = meta + ar->blocktab_off + 8 * b;
        ar->h_first_seg[b] = rd32(p);
        if (b < ar->n_blocks) {
            ar->h_levels[b] = rd16(p + 4);
            if (ar->h_levels[b] > ar->max_level || rd16(p + 6)) return ACEAPEX_E_CORRUPT;
            seen_max_level = std::max<uint32_t>(seen_max_level, ar->h_levels[b]);
        } else if (rd32(p) != ar->n_segs || rd32(p + 4)) return ACEAPEX_E_CORRUPT;
        if (b == 0 ? ar->h_first_seg[0] != 0 : ar->h_first_seg[b] <= ar->h_first_seg[b - 1]) return ACEAPEX_E_CORRUPT;
    }
    if (seen_max_level != ar->max_level) return ACEAPEX_E_CORRUPT;
    for (uint64_t b = 0; b < ar->n_blocks; b++) {
        const uint64_t bstart = b << ar->log2_bs, bend = std::min<uint64_t>(ar->N, bstart + (1ull << ar->log2_bs));
        uint64_t prev_out = 0;
        for (uint64_t s = ar->h_first_seg[b]; s < ar->h_first_seg[b + 1]; s++) {
            const uint8_t* p = meta + ar->dir_off + 32 * s;
            const uint64_t po = rd64(p), os = rd64(p + 8), end = s + 1 < ar->n_segs ? rd64(p + 32) : abytes - TAIL_PAD;
            const uint32_t n_cmd = rd16(p + 16), n_match = rd16(p + 18), n_lit_a = rd16(p + 20), n_lit_q = rd16(p + 22), n_sym_q = rd16(p + 24),
                           n_words = rd16(p + 26), n_ext = rd16(p + 28), lvl = rd16(p + 30);
            if (po % 16 || po < prev_po || end <= po || end > abytes - TAIL_PAD) return ACEAPEX_E_CORRUPT;
            if (n_cmd < 1 || n_cmd > ar->max_cmds || !(n_match == n_cmd || n_match + 1 == n_cmd) || lvl != ar->h_levels[b]) return ACEAPEX_E_CORRUPT;
            if (n_lit_a + n_lit_q > MAX_SEG_LITS || (ar->q_min == 0 && (n_lit_q || n_sym_q)) || (ar->q_mode == 0 && n_sym_q != n_lit_q) ||
                n_sym_q > MAX_SEG_LITS / 2 + MAX_SEG_CMDS + 1 + (ar->q_mode ? 0u : MAX_SEG_LITS)) return ACEAPEX_E_CORRUPT;
            if (s == ar->h_first_seg[b] ? os != bstart : !(os > prev_out && os < bend)) return ACEAPEX_E_CORRUPT;
            const uint64_t need = ((256 + 2ull * n_words + 3) & ~3ull) + 4ull * n_ext + (uint64_t)ar->n_raw_planes * n_match;
            if (po + need > end) return ACEAPEX_E_CORRUPT;
            prev_po = po; prev_out = os; seen_max_cmds = std::max(seen_max_cmds, n_cmd);
            ar->h_match_prefix[s + 1] = ar->h_match_prefix[s] + n_match;
            ar->h_payload_off[s] = po;
            level_cnt[lvl + 1]++;
        }
    }
    if (ar->h_match_prefix[ar->n_segs] != ar->total_matches) return ACEAPEX_E_CORRUPT;
    // device tables
    if (!luts.empty()) {
        CU(cudaMalloc(&ar->d_luts, luts.size() * 4));
        CU(cudaMemcpy(ar->d_luts, luts.data(), luts.size() * 4, cudaMemcpyHostToDevice));
    }
    if (!lutq.empty()) {
        CU(cudaMalloc(&ar->d_lutq, lutq.size() * 8));
        CU(cudaMemcpy(ar->d_lutq, lutq.data(), lutq.size() * 8, cudaMemcpyHostToDevice));
    }
    {
        CU(cudaMalloc(&ar->d_levels, std::max<size_t>(ar->h_levels.size(), 1) * 2));
        if (ar->n_blocks) CU(cudaMemcpy(ar->d_levels, ar->h_levels.data(), ar->h_levels.size() * 2, cudaMemcpyHostToDevice));
        CU(cudaMalloc(&ar->d_first_seg, ar->h_first_seg.size() * 4));
        CU(cudaMemcpy(ar->d_first_seg, ar->h_first_seg.data(), ar->h_first_seg.size() * 4, cudaMemcpyHostToDevice));
        CU(cudaMalloc(&ar->d_match_prefix, ar->h_match_prefix.size() * 8));
        CU(cudaMemcpy(ar->d_match_prefix, ar->h_match_prefix.data(), ar->h_match_prefix.size() * 8, cudaMemcpyHostToDevice));
    }
    // segment ids sorted by (level, index)
    ar->level_off.assign(ar->max_level + 2, 0);
    for (size_t l = 1; l < level_cnt.size(); l++) { level_cnt[l] += level_cnt[l - 1]; ar->level_off[l] = level_cnt[l]; }
    if (ar->n_segs && ar->max_level > 0) {
        std::vector<uint32_t> cat(ar->n_segs);
        std::vector<uint64_t> fill(level_cnt.begin(), level_cnt.end() - 1);
        for (uint64_t b = 0; b < ar->n_blocks; b++)
            for (uint64_t s = ar->h_first_seg[b]; s < ar->h_first_seg[b + 1]; s++) cat[fill[ar->h_levels[b]]++] = (uint32_t)s;
        CU(cudaMalloc(&ar->d_seg_lists, cat.size() * 4));
        CU(cudaMemcpy(ar->d_seg_lists, cat.data(), cat.size() * 4, cudaMemcpyHostToDevice));
    }
    // launch geometry: one CTA per SM, the decode tables are staged once per SM and shared by all its warps (fewer warps
    // when many offset planes are coded and the tables leave less room)
    int dev = 0; cudaDeviceProp prop;
    CU(cudaGetDevice(&dev)); CU(cudaGetDeviceProperties(&prop, dev));
    ar->sms = prop.multiProcessorCount;
    // per-warp shared memory besides the word ring: the LITQ run table (a command table of 2 KB in the span-service kernels)
    // and, with what the tables leave free, a staging area for LITA (up to 4 KB; larger segments stage in global memory)
    ar->threads = 1024;
    if (const char* e = getenv("ACEAPEX_THREADS")) {      // tests: other CTA sizes (other interleavings of the flag-driven launches)
        const int t = atoi(e);
        if (t >= 128 && t <= 1024) ar->threads = t / 64 * 64;
    }
    ar->runs_bytes = runs_bytes_for(ar->q_min);
    const uint32_t min_area = std::max<uint32_t>(4 * (MAX_SEG_CMDS + 2), ar->runs_bytes + ALIST_BYTES);
    auto smem_max = [&](int T, uint32_t area) { return std::max(entropy_smem(ar->n_coded_tables, ar->q_mode, area, T), (size_t)(T / 32) * COPY_WARP_BYTES + 64); };
    while (ar->threads > 128 && smem_max(ar->threads, min_area) > (size_t)prop.sharedMemPerBlockOptin) ar->threads -= 64;
    {
        const size_t fixed = entropy_smem(ar->n_coded_tables, ar->q_mode, 0, ar->threads);
        const size_t room = (size_t)prop.sharedMemPerBlockOptin > fixed ? ((size_t)prop.sharedMemPerBlockOptin - fixed) / (ar->threads / 32) : 0;
        uint32_t area = (uint32_t)std::min<size_t>(room & ~(size_t)15, ar->runs_bytes + ALIST_BYTES + 4096);
        area = std::max(area, min_area);
        ar->lita_bytes = area - ar->runs_bytes - ALIST_BYTES;
    }
    ar->smem_entropy = entropy_smem(ar->n_coded_tables, ar->q_mode, ar->runs_bytes + ALIST_BYTES + ar->lita_bytes, ar->threads);
    ar->smem_copy = (size_t)(ar->threads / 32) * COPY_WARP_BYTES + 64;
    ar->smem_fused = std::max(ar->smem_entropy, ar->smem_copy);
    {
        const void* fns[] = {(const void*)k_literals<0, true>, (const void*)k_literals<1, true>, (const void*)k_literals<2, true>, (const void*)k_literals<3, true>, (const void*)k_literals<4, true>,
                             (const void*)k_literals<0>, (const void*)k_literals<1>, (const void*)k_literals<2>, (const void*)k_literals<3>, (const void*)k_literals<4>,
                             (const void*)k_fused<0>, (const void*)k_fused<1>, (const void*)k_fused<3>, (const void*)k_fused<4>,
                             (const void*)k_copy<false, false, false, true>, (const void*)k_copy<true, false, false, false>,
                             (const void*)k_copy<false, true, false, false>, (const void*)k_copy<true, true, false, false>, (const void*)k_copy<false, true, true, false>,
                             (const void*)k_serve, (const void*)k_spans, (const void*)k_spans_cta, (const void*)k_rounds};
        for (const void* f : fns) {
            // the attribute belongs to the function, not to the handle: always the device maximum, so that handles with
            // different table counts do not lower each other's limit
            CU(cudaFuncSetAttribute(f, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)prop.sharedMemPerBlockOptin));
            CU(cudaFuncSetAttribute(f, cudaFuncAttributePreferredSharedMemoryCarveout, cudaSharedmemCarveoutMaxShared));
        }
    }
    {
        int coop = 0, occ_r = 0, occ_f = 0;
        CU(cudaDeviceGetAttribute(&coop, cudaDevAttrCooperativeLaunch, dev));
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_r, k_rounds, ar->threads, ar->smem_entropy));
        CU(cudaOccupancyMaxActiveBlocksPerMultiprocessor(&occ_f, k_fused<1>, ar->threads, ar->smem_fused));
        ar->cooperative = coop && occ_r >= 1 && occ_f >= 1 && !getenv("ACEAPEX_NO_COOPERATIVE");
        ar->use_graphs = !getenv("ACEAPEX_NO_GRAPHS");
        if (occ_r < 1) return ACEAPEX_E_CUDA;
    }
    ar->scratch_per_warp = scratch_bytes(ar->n_coded_planes);
    layout_workspace(ar);
    guard.a = nullptr;
    *out = ar;
    return ACEAPEX_OK;
}

int32_t aceapex_close(aceapex_archive* ar) {
    if (!ar) return ACEAPEX_E_ARG;
    cudaDeviceSynchronize();
    if (ar->d_luts) cudaFree(ar->d_luts);
    if (ar->d_lutq) cudaFree(ar->d_lutq);
    if (ar->d_seg_lists) cudaFree(ar->d_seg_lists);
    if (ar->d_levels) cudaFree(ar->d_levels);
    if (ar->d_first_seg) cudaFree(ar->d_first_seg);
    if (ar->d_match_prefix) cudaFree(ar->d_match_prefix);
    if (ar->d_chunk_lists) cudaFree(ar->d_chunk_lists);
    for (cudaEvent_t e : ar->ev_h2d) cudaEventDestroy(e);
    for (cudaEvent_t e : ar->ev_dec) cudaEventDestroy(e);
    for (cudaEvent_t e : ar->ev_phase) if (e) cudaEventDestroy(e);
    if (ar->g_seek.exec) cudaGraphExecDestroy(ar->g_seek.exec);
    if (ar->g_seek.graph) cudaGraphDestroy(ar->g_seek.graph);
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
    o->total_cmds = ar->total_cmds; o->workspace_bytes = ar->ws_need; o->max_level = ar->max_level; o->offset_width = ar->W;
    o->min_match = ar->min_match; o->max_cmds = ar->max_cmds; o->n_coded_planes = ar->n_coded_planes; o->has_fnv = ar->flags & 1;
    o->resident_warps = ar->sms * (ar->threads / 32);
    o->n_segments = ar->n_segs; o->total_litq_bytes = ar->total_litq; o->segment_size = 1u << ar->log2_seg; o->q_min = ar->q_min; o->q_mode = ar->q_mode;
    return ACEAPEX_OK;
}

int32_t aceapex_set_workspace(aceapex_archive* ar, void* d_ws, uint64_t bytes) {
    if (!ar || (reinterpret_cast<uintptr_t>(d_ws) & 255)) return ACEAPEX_E_ARG;
    ar->d_ws = static_cast<uint8_t*>(d_ws); ar->ws_bytes = bytes; ar->ws_clean = false;
    return (d_ws && bytes >= ar->ws_need) ? ACEAPEX_OK : ACEAPEX_E_WORKSPACE;
}

int32_t aceapex_set_stream(aceapex_archive* ar, void* s) {
    if (!ar) return ACEAPEX_E_ARG;
    ar->stream = static_cast<cudaStream_t>(s);
    return ACEAPEX_OK;
}

// the match waves of the whole file from the descriptors the literal launch left: one flag-driven launch over the segments
// below the top dependency level (when there are any), one wait-free launch for the top level (FORMAT.md §3)
static int32_t match_waves(aceapex_archive* ar, Params& P, bool timing) {
    const uint32_t top = ar->max_level;
    int32_t rc;
    if (top > 0 && ar->level_off[top] > 0) {
        if ((rc = zero_done(ar, 0, ar->n_blocks))) return rc;
        P.seg_list = ar->d_seg_lists;
        if ((rc = launch(ar, P, K_COPY_WAIT, ar->level_off[top]))) return rc;
    }
    if (timing) CU(cudaEventRecord(ar->ev_phase[2], ar->stream));
    P.seg_list = top > 0 ? ar->d_seg_lists + ar->level_off[top] : nullptr; P.first_work = 0;
    return launch(ar, P, K_COPY_TOP, ar->level_off[top + 1] - ar->level_off[top]);
}

int32_t aceapex_decode_all(aceapex_archive* ar, void* d_out) {
    if (!ar || (!d_out && ar->N) || (reinterpret_cast<uintptr_t>(d_out) & 15)) return ACEAPEX_E_ARG;
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    if (!ar->n_segs) return ACEAPEX_OK;
    Params P; fill_params(ar, P);
    set_out(P, static_cast<uint8_t*>(d_out), 0, ar->N);
    const bool tm = ar->phase_timing;
    if (tm) CU(cudaEventRecord(ar->ev_phase[0], ar->stream));
    P.seg_list = nullptr; P.first_work = 0;
    if ((rc = launch(ar, P, K_LIT, ar->n_segs))) return rc;
    if (tm) CU(cudaEventRecord(ar->ev_phase[1], ar->stream));
    rc = match_waves(ar, P, tm);
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

// literal launch + ONE match launch over the segments sorted by (level, index) with completion counters
int32_t aceapex_decode_all_flags(aceapex_archive* ar, void* d_out) {
    if (!ar || (!d_out && ar->N) || (reinterpret_cast<uintptr_t>(d_out) & 15)) return ACEAPEX_E_ARG;
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    if (!ar->n_segs) return ACEAPEX_OK;
    Params P; fill_params(ar, P);
    set_out(P, static_cast<uint8_t*>(d_out), 0, ar->N);
    P.seg_list = nullptr; P.first_work = 0;
    if ((rc = launch(ar, P, K_LIT, ar->n_segs))) return rc;
    if ((rc = zero_done(ar, 0, ar->n_blocks))) return rc;
    P.seg_list = ar->d_seg_lists;                       // null when every block is at level 0: index order
    return launch(ar, P, K_COPY_WAIT, ar->n_segs);
}

// the whole wavefront in one cooperative launch
int32_t aceapex_decode_all_fused(aceapex_archive* ar, void* d_out) {
    if (!ar || (!d_out && ar->N) || (reinterpret_cast<uintptr_t>(d_out) & 15)) return ACEAPEX_E_ARG;
    if (!ar->cooperative) return aceapex_decode_all(ar, d_out);
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    if (!ar->n_segs) return ACEAPEX_OK;
    Params P; fill_params(ar, P);
    set_out(P, static_cast<uint8_t*>(d_out), 0, ar->N);
    const uint32_t top = ar->max_level;
    FusedArgs F;
    F.tickets = reinterpret_cast<unsigned long long*>(ar->d_ws + 128);
    F.n_low = top > 0 ? ar->level_off[top] : 0; F.low_list = ar->d_seg_lists;
    F.n_top = ar->level_off[top + 1] - ar->level_off[top]; F.top_list = top > 0 ? ar->d_seg_lists + ar->level_off[top] : nullptr;
    CU(cudaMemsetAsync(F.tickets, 0, 32, ar->stream));
    if (F.n_low && (rc = zero_done(ar, 0, ar->n_blocks))) return rc;
    void* args[] = {&P, &F};
    const void* kf = ar->q_mode ? (ar->q_min >= 64 ? (const void*)k_fused<4> : (const void*)k_fused<1>) : (ar->q_min >= 64 ? (const void*)k_fused<3> : (const void*)k_fused<0>);
    CU(cudaLaunchCooperativeKernel(kf, dim3(ar->sms), dim3(ar->threads), args, ar->smem_fused, ar->stream));
    ar->launches++;
    return ACEAPEX_OK;
}

static void add_demands(aceapex_archive* ar, uint64_t pos, uint64_t len, uint64_t dst) {
    while (len) {                                      // cut at block boundaries here; k_seed / push_span cut at segment boundaries
        uint64_t bend = ((pos >> ar->log2_bs) + 1) << ar->log2_bs, n = std::min<uint64_t>(len, bend - pos);
        ar->h_demands.push_back(Demand{pos, dst, n});
        pos += n; dst += n; len -= n;
    }
}

// Serves the demand list g[0] (filled by the caller) in at most `rounds` rounds; the list left by the last round must be
// empty.  One cooperative launch (k_rounds) where the device supports it, else three launches per round.
static int32_t serve_rounds(aceapex_archive* ar, Params Q, const GList g[2], uint32_t rounds) {
    int32_t rc;
    if (ar->cooperative && rounds <= 16) {
        unsigned long long* tickets = reinterpret_cast<unsigned long long*>(ar->d_ws + 128);     // 16 counters in the control area
        if ((rc = submit_memset(ar, tickets, 128))) return rc;
        Q.gl_cur = g[0]; Q.gl_nxt = g[1];
        return submit_kernel(ar, (const void*)k_rounds, dim3(ar->sms), dim3(ar->threads), ar->smem_entropy, true,
                             {{&Q, sizeof Q}, {&tickets, sizeof tickets}, {&rounds, sizeof rounds}});
    }
    if (ar->capturing) return NOT_GRAPHABLE;
    for (uint32_t r = 0; r < rounds; r++) {
        Q.gl_cur = g[r & 1]; Q.gl_nxt = g[(r + 1) & 1];
        CU(cudaMemsetAsync(Q.gl_nxt.count, 0, 16, ar->stream));
        k_plan<<<ar->sms, 256, 0, ar->stream>>>(Q);          // bucket offsets + work items
        k_scatter<<<4 * ar->sms, 256, 0, ar->stream>>>(Q);
        ar->launches += 2;
        if ((rc = launch(ar, Q, K_SERVE, 1))) return rc;
    }
    k_assert_empty<<<1, 1, 0, ar->stream>>>(g[rounds & 1].count, Q.err);
    CU(cudaGetLastError());
    ar->launches++;
    return ACEAPEX_OK;
}

// the launch sequence of a range decode
static int32_t range_launches(aceapex_archive* ar, uint64_t lo, uint64_t hi, uint8_t* out) {
    int32_t rc;
    const uint64_t BS = 1ull << ar->log2_bs;
    // whole blocks [alo, ahi) are decoded as a window; the ragged ends are spans
    const uint64_t alo = (lo + BS - 1) & ~(BS - 1), ahi = hi == ar->N ? hi : hi & ~(BS - 1);
    Params P; fill_params(ar, P);
    P.out2 = out; set_out(P, out, 0, 0);
    if (alo < ahi) {
        const uint64_t b0 = alo >> ar->log2_bs, b1 = (ahi + BS - 1) >> ar->log2_bs;
        const uint64_t s0 = ar->h_first_seg[b0], s1 = ar->h_first_seg[b1], ns = s1 - s0;
        set_out(P, out + (alo - lo), alo, ahi); P.out2 = P.out;
        // (1) literals of the window; (2) foreign seed bytes of its matches -> demand lists, served in rounds, every
        // source segment parsed once per round; (3) matches of the window
        const GList g[2] = {glist(ar, 0), glist(ar, 1)};
        // the demands of the whole window fit the lists: its literal launch does the collect pass too
        static const bool no_merge = getenv("ACEAPEX_NO_COLLECT_MERGE") != nullptr;
        // (not for a seek: there the separate collect launch shares every segment's matches out among eight warps)
        const bool merged = !no_merge && ns >= 1024 && ar->h_match_prefix[s1] - ar->h_match_prefix[s0] <= ar->gl_eff / 3;
        P.seg_list = nullptr; P.first_work = s0;
        if (merged) {
            if ((rc = submit_memset(ar, g[0].count, 32))) return rc;
            P.gl_nxt = g[0];
        }
        if ((rc = launch(ar, P, merged ? K_LIT_COLLECT : K_LIT, ns))) return rc;
        for (uint64_t w0 = s0; w0 < s1;) {                  // sub-windows whose demands fit the lists
            uint64_t w1 = w0 + 1;
            while (w1 < s1 && ar->h_match_prefix[w1 + 1] - ar->h_match_prefix[w0] <= ar->gl_eff / 3) w1++;
            if (merged) w1 = s1;
            else {
                if ((rc = submit_memset(ar, g[0].count, 32))) return rc;
                P.seg_list = nullptr; P.first_work = w0; P.gl_nxt = g[0];
                if ((rc = launch(ar, P, K_COLLECT, w1 - w0))) return rc;
            }
            Params Q = P;                                   // serving knows no window: sources of foreign bytes precede it
            Q.out_pos0 = 0; Q.win_end = 0;
            // a seed byte is found after at most max_level + 1 source blocks (FORMAT.md §3): one round each
            if ((rc = serve_rounds(ar, Q, g, ar->max_level + 2))) return rc;
            w0 = w1;
        }
        if (ar->max_level == 0) {                           // every source is a literal byte: no order among the window's segments
            P.seg_list = nullptr; P.first_work = s0;
            if ((rc = launch(ar, P, K_COPY_WIN, ns))) return rc;
        } else if (ar->capturing || ns <= 1024) {
            // A seek: one flag-driven launch over the window's segments in INDEX order.  A segment waits for lower-level
            // source blocks of the window only, and sources precede their destinations (src < dst), so it only ever waits
            // for segments whose tickets were drawn before its own: no deadlock, no list to build or upload, and the
            // sequence can be replayed as a graph.
            if ((rc = zero_done(ar, b0, b1 - b0))) return rc;
            P.seg_list = nullptr; P.first_work = s0;
            if ((rc = launch(ar, P, K_COPY_WIN_WAIT, ns))) return rc;
        } else {
            // its segments sorted by (level, index) in one flag-driven launch (a segment waits for lower-level source
            // blocks of the window only; everything outside the window is final): sorted, almost nobody waits
            std::vector<uint32_t>& L = ar->h_list;
            L.resize(ns);
            std::vector<uint64_t> cnt(ar->max_level + 2, 0);
            for (uint64_t b = b0; b < b1; b++) cnt[ar->h_levels[b] + 1] += ar->h_first_seg[b + 1] - ar->h_first_seg[b];
            for (size_t l = 1; l < cnt.size(); l++) cnt[l] += cnt[l - 1];
            for (uint64_t b = b0; b < b1; b++) for (uint64_t s = ar->h_first_seg[b]; s < ar->h_first_seg[b + 1]; s++) L[cnt[ar->h_levels[b]]++] = (uint32_t)s;
            uint32_t* d_list = reinterpret_cast<uint32_t*>(ar->d_ws + ar->list_off);
            CU(cudaMemcpyAsync(d_list, L.data(), ns * 4, cudaMemcpyHostToDevice, ar->stream));
            if ((rc = zero_done(ar, b0, b1 - b0))) return rc;
            P.seg_list = d_list; P.first_work = 0;
            if ((rc = launch(ar, P, K_COPY_WIN_WAIT, ns))) return rc;
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
        const uint32_t n = (uint32_t)ar->h_demands.size();      // at most a handful: two spans cut at block boundaries
        if ((rc = submit_memset(ar, g[0].count, 32))) return rc;
        Params Q = P;
        if (alo >= ahi) { Q.out_pos0 = 0; Q.win_end = 0; }
        Q.out2 = out; Q.gl_nxt = g[0];
        Demand* d_dem = reinterpret_cast<Demand*>(ar->d_ws + ar->demands_off);
        Q.demands = d_dem; Q.n_inline = 0;
        if (n <= 4) { Q.n_inline = n; for (uint32_t i = 0; i < n; i++) Q.inline_dem[i] = ar->h_demands[i]; }
        else {
            if (ar->capturing) return NOT_GRAPHABLE;
            CU(cudaMemcpyAsync(d_dem, ar->h_demands.data(), n * sizeof(Demand), cudaMemcpyHostToDevice, ar->stream));
        }
        if ((rc = submit_kernel(ar, (const void*)k_seed, dim3((n + 127) / 128), dim3(128), 0, false, {{&Q, sizeof Q}, {&n, sizeof n}}))) return rc;
        if ((rc = serve_rounds(ar, Q, g, ar->max_level + 3))) return rc;   // one more round: the span's own segment comes first
    }
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
    if (budget && budget < ar->ws_need) {
        const uint64_t per_rec = 3 * sizeof(GDemand) + 8, fixed = ar->ws_need - std::min<uint64_t>(ar->ws_need, per_rec * ar->gl_cap);
        if (budget < fixed + per_rec * 4096) return ACEAPEX_E_BUDGET;
        ar->gl_eff = std::min<uint64_t>(ar->gl_cap, (budget - fixed) / per_rec);
    }
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    // a seek (up to a few hundred blocks): the launch sequence is replayed as a CUDA graph
    if (ar->use_graphs && ar->cooperative && hi - lo <= (8ull << 20)) {
        const uint64_t l0 = ar->launches; const uint32_t slot0 = ar->ticket_slot;
        ar->capturing = true; ar->rec.clear();
        rc = range_launches(ar, lo, hi, static_cast<uint8_t*>(d_out));
        ar->capturing = false;
        if (rc == ACEAPEX_OK) return ar->rec.empty() ? ACEAPEX_OK : replay(ar);
        if (rc != NOT_GRAPHABLE) return rc;
        ar->launches = l0; ar->ticket_slot = slot0;       // nothing was issued: do it again with plain launches
    }
    return range_launches(ar, lo, hi, static_cast<uint8_t*>(d_out));
}

uint64_t aceapex_graph_launch_count(const aceapex_archive* ar) { return ar ? ar->graph_launches : 0; }

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

// launches span-mode work (one warp per span, recursion inside the warp) for the demands staged in ar->h_demands
static int32_t run_spans(aceapex_archive* ar, Params& P) {
    Demand* d_dem = reinterpret_cast<Demand*>(ar->d_ws + ar->demands_off);
    P.seg_list = nullptr; P.demands = d_dem; P.n_inline = 0;
    if (ar->h_demands.size() <= 4) {                   // a single read: the items travel in the kernel arguments, no copy
        P.n_inline = (uint32_t)ar->h_demands.size();
        for (uint32_t i = 0; i < P.n_inline; i++) P.inline_dem[i] = ar->h_demands[i];
        static const bool one_warp = getenv("ACEAPEX_READ_ONE_WARP") != nullptr;      // the earlier path, for comparison
        return launch(ar, P, one_warp ? K_SPANS : K_SPANS_CTA, P.n_inline);
    }
    for (size_t i = 0; i < ar->h_demands.size(); i += ar->demand_cap) {
        size_t n = std::min<size_t>(ar->demand_cap, ar->h_demands.size() - i);
        CU(cudaMemcpyAsync(d_dem, ar->h_demands.data() + i, n * sizeof(Demand), cudaMemcpyHostToDevice, ar->stream));
        int32_t rc = launch(ar, P, K_SPANS, n);
        if (rc) return rc;
        if (i + n < ar->h_demands.size()) CU(cudaStreamSynchronize(ar->stream));   // the staging area is reused
    }
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
    set_out(P, static_cast<uint8_t*>(d_out), 0, 0); P.out2 = P.out;
    static const int force_rounds = getenv("ACEAPEX_READS_ROUNDS") ? atoi(getenv("ACEAPEX_READS_ROUNDS")) : -1;
    // Medium batches go through the demand lists as top-level records: their segments, then the source segments of every
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
            if ((rc = submit_memset(ar, g[0].count, 32))) return rc;
            Params Q = P;
            Q.gl_nxt = g[0]; Q.demands = d_dem; Q.n_inline = 0;
            if (m <= 4) { Q.n_inline = m; for (uint32_t k = 0; k < m; k++) Q.inline_dem[k] = ar->h_demands[i + k]; }
            else CU(cudaMemcpyAsync(d_dem, ar->h_demands.data() + i, m * sizeof(Demand), cudaMemcpyHostToDevice, ar->stream));
            if ((rc = submit_kernel(ar, (const void*)k_seed, dim3((m + 127) / 128), dim3(128), 0, false, {{&Q, sizeof Q}, {&m, sizeof m}}))) return rc;
            if ((rc = serve_rounds(ar, Q, g, ar->max_level + 3))) return rc;
            if (i + chunk < ar->h_demands.size()) CU(cudaStreamSynchronize(ar->stream));   // the staging area is reused
        }
    } else if ((rc = run_spans(ar, P))) return rc;
    CU(cudaStreamSynchronize(ar->stream));           // h_demands is host staging; the call returns the reads
    return ACEAPEX_OK;
}

int32_t aceapex_set_resident(aceapex_archive* ar, uint32_t slot, uint64_t lo, uint64_t hi, const void* p) {
    if (!ar || slot >= MAX_RESIDENT || lo > hi || hi > ar->N) return ACEAPEX_E_ARG;
    ar->res[slot].lo = lo; ar->res[slot].hi = hi; ar->res[slot].ptr = static_cast<const uint8_t*>(p);
    return ACEAPEX_OK;
}

int32_t aceapex_decode_stream(aceapex_archive* ar, uint64_t lo, uint64_t hi, void* d_ring, uint64_t ring_bytes, uint64_t window,
                              aceapex_window_fn consumer, void* user, uint64_t budget, aceapex_stream_stats_t* stats) {
    if (!ar) return ACEAPEX_E_ARG;
    if (lo > hi || hi > ar->N) return ACEAPEX_E_RANGE;
    const uint64_t BS = 1ull << ar->log2_bs;
    if (!d_ring || (reinterpret_cast<uintptr_t>(d_ring) & 15) || window == 0 || window % BS || lo % window || ring_bytes < window) return ACEAPEX_E_ARG;
    const uint64_t n_slots = std::min<uint64_t>(MAX_RESIDENT, ring_bytes / window), n_win = (hi - lo + window - 1) / window;
    aceapex_stream_stats_t st; memset(&st, 0, sizeof st);
    st.n_slots = n_slots; st.peak_device_bytes = ar->archive_bytes + n_slots * window + ar->ws_need;
    int32_t rc = prepare_ws(ar);
    if (rc) return rc;
    for (uint32_t s = 0; s < MAX_RESIDENT; s++) ar->res[s].lo = ar->res[s].hi = 0;
    const bool own_check = !consumer && (ar->flags & 1);
    unsigned long long* bad = reinterpret_cast<unsigned long long*>(ar->d_ws + 16);
    if (own_check) CU(cudaMemsetAsync(bad, 0, 8, ar->stream));
    std::vector<cudaEvent_t> ev(n_win + 1);
    for (auto& e : ev) CU(cudaEventCreate(&e));
    CU(cudaEventRecord(ev[0], ar->stream));
    for (uint64_t w = 0; w < n_win && !rc; w++) {
        const uint64_t wlo = lo + w * window, whi = std::min<uint64_t>(hi, wlo + window);
        const uint32_t slot = (uint32_t)(w % n_slots);
        uint8_t* d_win = static_cast<uint8_t*>(d_ring) + slot * window;
        ar->res[slot].lo = ar->res[slot].hi = 0;               // cleared BEFORE its buffer is overwritten
        rc = aceapex_decode_range(ar, wlo, whi, d_win, budget);
        if (rc) break;
        ar->res[slot].lo = wlo; ar->res[slot].hi = whi; ar->res[slot].ptr = d_win;
        if (own_check) {
            const uint64_t nb = (whi - wlo + BS - 1) >> ar->log2_bs;
            const uint64_t* expect = reinterpret_cast<const uint64_t*>(ar->d_archive + ar->fnv_off) + (wlo >> ar->log2_bs);
            k_fnv<<<(unsigned)((nb + 127) / 128), 128, 0, ar->stream>>>(d_win, whi - wlo, ar->log2_bs, expect, bad);
            ar->launches++;
        } else if (consumer && consumer(user, w, wlo, whi, d_win, ar->stream)) rc = ACEAPEX_E_ARG;
        cudaEventRecord(ev[w + 1], ar->stream);
        st.n_windows++; st.bytes += whi - wlo;
    }
    cudaError_t ce = cudaStreamSynchronize(ar->stream);
    for (uint32_t s = 0; s < MAX_RESIDENT; s++) ar->res[s].lo = ar->res[s].hi = 0;
    if (!rc && ce == cudaSuccess && st.n_windows) {
        cudaEventElapsedTime(&st.device_ms, ev[0], ev[st.n_windows]);
        st.min_window_gbs = 1e30f;
        for (uint64_t w = 0; w < st.n_windows; w++) {
            float ms = 0; cudaEventElapsedTime(&ms, ev[w], ev[w + 1]);
            const uint64_t wlo = lo + w * window, whi = std::min<uint64_t>(hi, wlo + window);
            const float g = ms > 0 ? (float)((whi - wlo) / (ms * 1e6)) : 0.f;
            st.min_window_gbs = std::min(st.min_window_gbs, g); st.max_window_gbs = std::max(st.max_window_gbs, g);
        }
        if (own_check) { unsigned long long h = 0; ce = cudaMemcpy(&h, bad, 8, cudaMemcpyDeviceToHost); st.bad_blocks = h; }
    }
    for (auto& e : ev) cudaEventDestroy(e);
    if (stats) *stats = st;
    if (rc) return rc;
    CU(ce);
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
        ar->chunk_blocks = std::max<uint64_t>(1, std::max<uint64_t>((4ull << 20) >> ar->log2_bs, (ar->n_blocks + 15) / 16));
        const uint64_t n_chunks = (ar->n_blocks + ar->chunk_blocks - 1) / ar->chunk_blocks;
        std::vector<uint32_t> list(ar->n_segs);
        ar->chunk_level_off.assign(n_chunks * n_lv + 1, 0);
        uint64_t at = 0;
        for (uint64_t k = 0; k < n_chunks; k++) {
            const uint64_t b0 = k * ar->chunk_blocks, b1 = std::min<uint64_t>(ar->n_blocks, b0 + ar->chunk_blocks);
            for (uint32_t l = 0; l < n_lv; l++) {
                ar->chunk_level_off[k * n_lv + l] = at;
                for (uint64_t b = b0; b < b1; b++) if (ar->h_levels[b] == l)
                    for (uint64_t s = ar->h_first_seg[b]; s < ar->h_first_seg[b + 1]; s++) list[at++] = (uint32_t)s;
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
    set_out(P, static_cast<uint8_t*>(d_stage), 0, ar->N);
    for (uint64_t k = 0; k < n_chunks; k++) {
        const uint64_t b0 = k * ar->chunk_blocks, b1 = std::min<uint64_t>(ar->n_blocks, b0 + ar->chunk_blocks);
        const uint64_t s0 = ar->h_first_seg[b0], s1 = ar->h_first_seg[b1];
        const uint64_t p0 = ar->h_payload_off[s0], p1 = s1 < ar->n_segs ? ar->h_payload_off[s1] : ar->archive_bytes;
        CU(cudaMemcpyAsync(d_a + p0, h_a + p0, p1 - p0, cudaMemcpyHostToDevice, ar->s_h2d));
        CU(cudaEventRecord(ar->ev_h2d[k], ar->s_h2d));
        CU(cudaStreamWaitEvent(ar->stream, ar->ev_h2d[k], 0));
        P.seg_list = nullptr; P.first_work = s0;
        if ((rc = launch(ar, P, K_LIT, s1 - s0))) return rc;
        for (uint32_t l = 0; l < n_lv; l++) {
            const uint64_t l0 = ar->chunk_level_off[k * n_lv + l], l1 = ar->chunk_level_off[k * n_lv + l + 1];
            P.seg_list = ar->d_chunk_lists + l0; P.first_work = 0;
            if ((rc = launch(ar, P, K_COPY_TOP, l1 - l0))) return rc;
        }
        CU(cudaEventRecord(ar->ev_dec[k], ar->stream));
        CU(cudaStreamWaitEvent(ar->s_d2h, ar->ev_dec[k], 0));
        const uint64_t o0 = b0 << ar->log2_bs, o1 = std::min<uint64_t>(ar->N, b1 << ar->log2_bs);
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
        case ACEAPEX_E_TOO_LARGE: return "size beyond the fixed maximum of the no-allocation entry point";
    }
    return "unknown error";
}

} // extern "C"
