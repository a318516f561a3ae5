// The entropy stage alone (section 6.4: DietGPU on "256 MB exponential, batch 4096 x 64 KB",
// encode 364.9 / decode 592.5 GB/s on an H100): a batch of rows, every row coded on its own with one static byte table as a
// rANS section of FORMAT.md 1.7 (32 interleaved states, one word stream per state, [head 32 x (state, word_off)][words]).
// One warp per row, persistent grid.  The decoder is the decode loop of the archive kernels (acx_device.cuh).
#include "aceapex.h"
#include "acx_device.cuh"

#include <algorithm>
#include <cstring>
#include <mutex>
#include <vector>

using namespace acx;

// Scratch of aceapex_rans_encode_static (include/aceapex.h): the row encoder for callers that may not allocate.  Every GPU
// that loads this library holds these 32 MiB + 256 bytes until the process exits.  Layout: [work ticket u64 @0, pad to 256]
// [word staging of the resident warps].  In HOST code the name below is a host-side stand-in, not a device address: the
// host gets the address once per device with cudaGetSymbolAddress (static_scratch_of) and passes that to the kernel.
static __device__ __align__(256) uint8_t g_static_scratch[ACEAPEX_RANS_STATIC_SCRATCH_BYTES + 256];

namespace {

// encode table entry of symbol s: x_max = freq << 21 (a state at or above it emits a word first), rcp = floor(2^32 / freq),
// freq, cum.  The step is FORMAT.md 1.7: x' = ((x / f) << 11) + (x mod f) + cum, with x / f from one multiply-high by the
// reciprocal and one correction (floor(2^32 / f) underestimates the quotient by at most one for 32-bit x).
struct EncSym { uint32_t x_max, rcp, freq, cum; };

constexpr uint32_t ENC_TABLE_BYTES = 256 * sizeof(EncSym), DEC_TABLE_BYTES = LUT_SIZE * 4;

__global__ void __launch_bounds__(1024, 1) k_rans_encode(const uint8_t* __restrict__ in, uint64_t n_rows, uint32_t row_bytes, const EncSym* __restrict__ table,
                                                          uint8_t* __restrict__ out, uint64_t row_cap, uint32_t* __restrict__ row_sizes, uint16_t* __restrict__ stage,
                                                          unsigned long long* ticket) {
    __shared__ EncSym s_tab[256];
    __shared__ __align__(16) uint16_t s_grp[32][32][8];          // per warp and lane: the eight words being collected
    for (uint32_t i = threadIdx.x; i < 256; i += blockDim.x) s_tab[i] = table[i];
    __syncthreads();
    const uint32_t lane = threadIdx.x & 31;
    const uint32_t per = ((row_bytes + 31) / 32 + 7) & ~7u;   // a state emits at most one word per symbol; whole groups of eight
    // this lane's words, written from the end in groups of eight (one 16-byte store per group instead of eight 2-byte stores
    // to eight different sectors per warp: the scattered stores, not the arithmetic, set the pace of this kernel)
    uint16_t* const my = stage + ((uint64_t)(blockIdx.x * (blockDim.x >> 5) + (threadIdx.x >> 5)) * 32 + lane) * per;
    const uint32_t grp = (uint32_t)__cvta_generic_to_shared(&s_grp[threadIdx.x >> 5][lane][0]);
    for (;;) {
        unsigned long long row = 0;
        if (lane == 0) row = atomicAdd(ticket, 1ull);
        row = __shfl_sync(0xffffffffu, row, 0);
        if (row >= n_rows) break;
        const uint8_t* src = in + row * row_bytes;
        uint32_t x = 1u << 16, cnt = 0;
        // symbols in reverse order: round r holds symbols 32 r + lane.  Eight rounds at a time: their symbol loads are issued
        // together, ahead of the eight dependent coding steps
        auto load8 = [&](int64_t r0, uint32_t (&sym)[8]) {
#pragma unroll
            for (int k = 0; k < 8; k++) {
                const int64_t r = r0 - k;
                const uint32_t i = 32u * (uint32_t)r + lane;
                sym[k] = (r >= 0 && i < row_bytes) ? (uint32_t)__ldg(src + i) : 0xffffffffu;
            }
        };
        uint32_t nxt[8];
        load8((int64_t)((row_bytes + 31) / 32) - 1, nxt);
        for (int64_t r0 = (int64_t)((row_bytes + 31) / 32) - 1; r0 >= 0; r0 -= 8) {
            uint32_t sym[8];
#pragma unroll
            for (int k = 0; k < 8; k++) sym[k] = nxt[k];
            load8(r0 - 8, nxt);                                // the next eight rounds' symbols travel while these are coded
#pragma unroll
            for (int k = 0; k < 8; k++) {
                if (sym[k] == 0xffffffffu) continue;
                const EncSym e = s_tab[sym[k]];
                if (x >= e.x_max && e.x_max) {                 // x_max = 0 stands for 2^32 (freq = 2^11): never
                    sts16(grp + 2u * (7u - (cnt & 7u)), x);    // word c of the lane lands at my[per - 1 - c]
                    x >>= 16; cnt++;
                    if ((cnt & 7u) == 0) *reinterpret_cast<uint4*>(my + (per - cnt)) = lds128(grp);
                }
                uint32_t q = __umulhi(x, e.rcp), rem = x - q * e.freq;
                if (rem >= e.freq) { q++; rem -= e.freq; }
                if (e.freq == 1) { q = x; rem = 0; }
                x = (q << PROB_BITS) + rem + e.cum;
            }
        }
        if (cnt & 7u) *reinterpret_cast<uint4*>(my + (per - ((cnt + 7u) & ~7u))) = lds128(grp);     // the open group: its low slots are not read
        // head: (state, word_off); then every state's words in the order the decoder consumes them (the reverse of emission)
        uint32_t off = cnt;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) { const uint32_t t = __shfl_up_sync(0xffffffffu, off, o); if (lane >= (uint32_t)o) off += t; }
        const uint32_t total = __shfl_sync(0xffffffffu, off, 31);
        off -= cnt;
        uint8_t* dst = out + row * row_cap;
        reinterpret_cast<uint2*>(dst)[lane] = make_uint2(x, off);
        if (lane == 0) row_sizes[row] = 256 + 2 * total;
        __syncwarp();
        uint16_t* words = reinterpret_cast<uint16_t*>(dst + 256);
        for (int k = 0; k < 32; k++) {                       // the whole warp copies state k's stream: coalesced on both sides
            const uint32_t n = __shfl_sync(0xffffffffu, cnt, k), o = __shfl_sync(0xffffffffu, off, k);
            const uint16_t* from = reinterpret_cast<const uint16_t*>(__shfl_sync(0xffffffffu, reinterpret_cast<unsigned long long>(my), k)) + (per - n);
            uint32_t j = lane;
            for (; j + 224 < n; j += 256) {                    // eight loads in flight per lane
                uint16_t v[8];
#pragma unroll
                for (int q = 0; q < 8; q++) v[q] = from[j + 32 * q];
#pragma unroll
                for (int q = 0; q < 8; q++) words[o + j + 32 * q] = v[q];
            }
            for (; j < n; j += 32) words[o + j] = from[j];
        }
        __syncwarp();
    }
}

__global__ void __launch_bounds__(1024, 1) k_rans_decode(const uint8_t* __restrict__ enc, uint64_t n_rows, uint32_t row_bytes, uint64_t row_cap,
                                                          const uint32_t* __restrict__ row_sizes, const uint32_t* __restrict__ lut_g, uint8_t* __restrict__ out, uint32_t* status, unsigned long long* ticket) {
    extern __shared__ __align__(16) uint8_t smem_raw[];
    const uint32_t smem0 = ((uint32_t)__cvta_generic_to_shared(smem_raw) + 63u) & ~63u;
    uint8_t* base = smem_raw + (smem0 - (uint32_t)__cvta_generic_to_shared(smem_raw));
    for (uint32_t i = threadIdx.x; i < LUT_SIZE / 4; i += blockDim.x) reinterpret_cast<uint4*>(base)[i] = __ldg(reinterpret_cast<const uint4*>(lut_g) + i);
    __syncthreads();
    const uint32_t lut = smem0, ring = smem0 + DEC_TABLE_BYTES + (threadIdx.x >> 5) * RING_BYTES, lane = threadIdx.x & 31;
    for (;;) {
        unsigned long long row = 0;
        if (lane == 0) row = atomicAdd(ticket, 1ull);
        row = __shfl_sync(0xffffffffu, row, 0);
        if (row >= n_rows) break;
        const uint8_t* p = enc + row * row_cap;
        Rans r;
        r.init(p, (__ldg(row_sizes + row) - 256u) / 2u, ring);
        rans_region<false>(r, lut, 0, row_bytes, out + row * row_bytes);
        if (__any_sync(0xffffffffu, !r.finished()) && lane == 0) atomicOr(status, 1u);   // every state at 2^16, every stream consumed exactly
    }
}

} // namespace

extern "C" {

uint64_t aceapex_rans_row_capacity(uint64_t row_bytes) { return (256 + 2 * row_bytes + 15) / 16 * 16; }
uint64_t aceapex_rans_table_bytes(void) { return ENC_TABLE_BYTES + DEC_TABLE_BYTES + 64; }

static int rans_geometry(int* sms) {                     // one attribute query per process (cudaGetDeviceProperties takes milliseconds)
    static int cached = 0;
    if (!cached) {
        int dev = 0, n = 0;
        if (cudaGetDevice(&dev) != cudaSuccess || cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return -1;
        cached = n;
    }
    *sms = cached;
    return 0;
}

uint64_t aceapex_rans_scratch_bytes(uint64_t row_bytes) {
    int sms = 148;
    rans_geometry(&sms);
    return (uint64_t)sms * 32 * 32 * (((row_bytes + 31) / 32 + 7) & ~7ull) * 2 + 64;      // per resident warp: 32 states x one word per symbol at most, in groups of eight
}

int32_t aceapex_rans_tables(const uint16_t* h_freq, void* d_tables, void* stream) {
    if (!h_freq || !d_tables || (reinterpret_cast<uintptr_t>(d_tables) & 15)) return ACEAPEX_E_ARG;
    std::vector<uint8_t> buf(ENC_TABLE_BYTES + DEC_TABLE_BYTES);
    EncSym* e = reinterpret_cast<EncSym*>(buf.data());
    uint32_t* lut = reinterpret_cast<uint32_t*>(buf.data() + ENC_TABLE_BYTES);
    uint32_t cum = 0;
    for (uint32_t s = 0; s < 256; s++) {
        const uint32_t f = h_freq[s];
        if (cum + f > (uint32_t)LUT_SIZE) return ACEAPEX_E_ARG;
        e[s].freq = f; e[s].cum = cum;
        e[s].x_max = f >= (uint32_t)LUT_SIZE ? 0u : f << (32 - PROB_BITS);
        e[s].rcp = f ? (uint32_t)((1ull << 32) / f) : 0u;           // f = 1: 2^32 does not fit; the kernel takes q = x
        for (uint32_t k = 0; k < f; k++) lut[cum + k] = s | (k << 8) | (f << 20);
        cum += f;
    }
    if (cum != (uint32_t)LUT_SIZE) return ACEAPEX_E_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (cudaMemcpyAsync(d_tables, buf.data(), buf.size(), cudaMemcpyHostToDevice, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    if (cudaStreamSynchronize(st) != cudaSuccess) return ACEAPEX_E_CUDA;     // buf is host staging
    return ACEAPEX_OK;
}

int32_t aceapex_rans_encode(const void* d_in, uint64_t n_rows, uint64_t row_bytes, const void* d_tables, void* d_out, uint64_t row_cap,
                            uint32_t* d_row_sizes, void* d_scratch, uint64_t scratch_bytes, void* stream) {
    if (!d_in || !d_tables || !d_out || !d_row_sizes || !d_scratch || row_bytes == 0 || row_bytes > (1u << 24) || row_cap < 256 + 2 * row_bytes || (row_cap & 15) ||
        (reinterpret_cast<uintptr_t>(d_out) & 15) || (reinterpret_cast<uintptr_t>(d_scratch) & 15)) return ACEAPEX_E_ARG;
    if (scratch_bytes < aceapex_rans_scratch_bytes(row_bytes)) return ACEAPEX_E_WORKSPACE;
    if (n_rows == 0) return ACEAPEX_OK;
    int sms = 148;
    if (rans_geometry(&sms)) return ACEAPEX_E_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint8_t* sc = static_cast<uint8_t*>(d_scratch);
    unsigned long long* ticket = reinterpret_cast<unsigned long long*>(sc);
    if (cudaMemsetAsync(ticket, 0, 8, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    const uint64_t warps = std::min<uint64_t>((uint64_t)sms * 32, n_rows);
    const int T = (int)std::min<uint64_t>(1024, 32 * ((warps + sms - 1) / sms));
    const unsigned g = (unsigned)std::min<uint64_t>(sms, (warps + T / 32 - 1) / (T / 32));
    k_rans_encode<<<g, T, 0, st>>>(static_cast<const uint8_t*>(d_in), n_rows, (uint32_t)row_bytes, static_cast<const EncSym*>(d_tables), static_cast<uint8_t*>(d_out),
                                   row_cap, d_row_sizes, reinterpret_cast<uint16_t*>(sc + 64), ticket);
    return cudaGetLastError() == cudaSuccess ? ACEAPEX_OK : ACEAPEX_E_CUDA;
}

int32_t aceapex_rans_decode(const void* d_enc, uint64_t n_rows, uint64_t row_bytes, uint64_t row_cap, const uint32_t* d_row_sizes, const void* d_tables, void* d_out,
                            void* d_scratch, uint64_t scratch_bytes, void* stream) {
    if (!d_enc || !d_tables || !d_out || !d_scratch || !d_row_sizes || row_bytes == 0 || row_bytes > (1u << 24) || (reinterpret_cast<uintptr_t>(d_enc) & 15) || (row_cap & 15) || scratch_bytes < 64)
        return ACEAPEX_E_ARG;
    if (n_rows == 0) return ACEAPEX_OK;
    int sms = 148;
    if (rans_geometry(&sms)) return ACEAPEX_E_CUDA;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    uint8_t* sc = static_cast<uint8_t*>(d_scratch);
    if (cudaMemsetAsync(sc, 0, 16, st) != cudaSuccess) return ACEAPEX_E_CUDA;       // ticket @0, status @8
    const uint64_t warps = std::min<uint64_t>((uint64_t)sms * 32, n_rows);
    const int T = (int)std::min<uint64_t>(1024, 32 * ((warps + sms - 1) / sms));
    const unsigned g = (unsigned)std::min<uint64_t>(sms, (warps + T / 32 - 1) / (T / 32));
    const size_t smem = DEC_TABLE_BYTES + (size_t)(T / 32) * RING_BYTES + 64;
    static bool attr = false;
    if (!attr) { cudaFuncSetAttribute(k_rans_decode, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)(DEC_TABLE_BYTES + 32 * RING_BYTES + 64)); attr = true; }
    k_rans_decode<<<g, T, smem, st>>>(static_cast<const uint8_t*>(d_enc), n_rows, (uint32_t)row_bytes, row_cap, d_row_sizes,
                                      reinterpret_cast<const uint32_t*>(static_cast<const uint8_t*>(d_tables) + ENC_TABLE_BYTES), static_cast<uint8_t*>(d_out),
                                      reinterpret_cast<uint32_t*>(sc + 8), reinterpret_cast<unsigned long long*>(sc));
    return cudaGetLastError() == cudaSuccess ? ACEAPEX_OK : ACEAPEX_E_CUDA;
}

// device address of g_static_scratch and SM count of the current device, looked up once per device
static int32_t static_scratch_of(uint8_t** ptr, int* sms) {
    static std::mutex mu;
    static struct { uint8_t* ptr; int sms; } devs[64];
    int dev = -1;
    if (cudaGetDevice(&dev) != cudaSuccess || dev < 0 || dev >= 64) return ACEAPEX_E_CUDA;
    std::lock_guard<std::mutex> lk(mu);
    if (!devs[dev].ptr) {
        uint8_t* p = nullptr; int n = 0;
        if (cudaGetSymbolAddress((void**)&p, g_static_scratch) != cudaSuccess || !p) { cudaGetLastError(); return ACEAPEX_E_CUDA; }
        if (cudaDeviceGetAttribute(&n, cudaDevAttrMultiProcessorCount, dev) != cudaSuccess || n <= 0) return ACEAPEX_E_CUDA;
        devs[dev].sms = n; devs[dev].ptr = p;
    }
    *ptr = devs[dev].ptr; *sms = devs[dev].sms;
    return ACEAPEX_OK;
}

int32_t aceapex_rans_static_setup(void) {
    uint8_t* p; int sms;
    return static_scratch_of(&p, &sms);
}

int32_t aceapex_rans_encode_static(const void* d_in, uint64_t n_rows, uint64_t row_bytes, const void* d_tables, void* d_out, uint64_t row_cap,
                                   uint32_t* d_row_sizes, void* stream) {
    if (!d_in || !d_tables || !d_out || !d_row_sizes || row_bytes == 0 || (row_cap & 15) || (reinterpret_cast<uintptr_t>(d_out) & 15)) return ACEAPEX_E_ARG;
    if (row_bytes > ACEAPEX_RANS_STATIC_MAX_ROW_BYTES) return ACEAPEX_E_TOO_LARGE;
    if (row_cap < 256 + 2 * row_bytes) return ACEAPEX_E_ARG;
    if (n_rows == 0) return ACEAPEX_OK;
    uint8_t* sc = nullptr; int sms = 0;
    const int32_t rc = static_scratch_of(&sc, &sms);
    if (rc) return rc;
    // as many warps as the fixed staging area holds (a lane stages at most one word per symbol, in groups of eight)
    const uint64_t per = ((row_bytes + 31) / 32 + 7) & ~7ull, warp_bytes = 32 * per * 2;
    const uint64_t warps = std::min<uint64_t>(std::min<uint64_t>((uint64_t)sms * 32, n_rows), ACEAPEX_RANS_STATIC_SCRATCH_BYTES / warp_bytes);
    const uint64_t wps = warps >= (uint64_t)sms ? std::min<uint64_t>(32, warps / sms) : 1;     // warps per CTA
    const unsigned g = (unsigned)std::min<uint64_t>(sms, warps / wps);                          // g * wps <= warps
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    unsigned long long* ticket = reinterpret_cast<unsigned long long*>(sc);
    if (cudaMemsetAsync(ticket, 0, 8, st) != cudaSuccess) return ACEAPEX_E_CUDA;                // the one part of the array that must start at zero
    k_rans_encode<<<g, (unsigned)(32 * wps), 0, st>>>(static_cast<const uint8_t*>(d_in), n_rows, (uint32_t)row_bytes, static_cast<const EncSym*>(d_tables),
                                                      static_cast<uint8_t*>(d_out), row_cap, d_row_sizes, reinterpret_cast<uint16_t*>(sc + 256), ticket);
    return cudaGetLastError() == cudaSuccess ? ACEAPEX_OK : ACEAPEX_E_CUDA;
}

int32_t aceapex_rans_status(const void* d_scratch, void* stream, uint32_t* status) {
    if (!d_scratch || !status) return ACEAPEX_E_ARG;
    cudaStream_t st = static_cast<cudaStream_t>(stream);
    if (cudaMemcpyAsync(status, static_cast<const uint8_t*>(d_scratch) + 8, 4, cudaMemcpyDeviceToHost, st) != cudaSuccess) return ACEAPEX_E_CUDA;
    return cudaStreamSynchronize(st) == cudaSuccess ? ACEAPEX_OK : ACEAPEX_E_CUDA;
}

} // extern "C"
