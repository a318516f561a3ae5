/* aceapex.h — C ABI of the B200 device-resident decoder for ACX-B200 archives (FORMAT.md).
 *
 * What the library computes (§2): an archive stores LZ77 back-references as ABSOLUTE positions in the
 * decompressed output, partitioned into fixed-size blocks with four streams per block (literals, match lengths,
 * absolute offsets, command sequence).  Decoding a block = entropy-decode its streams, prefix-sum the command
 * sequence into output positions, place literals, and resolve matches by copying from absolute output positions once
 * the source data is available (the "wavefront", §1, §3.1).  Every step runs in
 * hand-written CUDA kernels for sm_100a; there is no CPU fallback.
 *
 * Conventions
 *   - "d_" pointers are DEVICE memory owned by the caller (e.g. torch uint8 tensors) and must stay valid for the
 *     lifetime stated; "h_" pointers are HOST memory.  The library never frees caller memory.
 *   - All sizes/positions are uint64_t bytes.  Return value: 0 = ACEAPEX_OK, negative = error (aceapex_strerror).
 *   - Decode calls are ASYNCHRONOUS on the handle's stream (default: the legacy default stream) unless stated; the
 *     caller synchronises.  Device-side integrity problems (bad offset, rANS state mismatch, dependency timeout)
 *     are latched in a device flag that aceapex_check() reads back.
 *   - The library allocates small device state at open (tables, directory copy is NOT made: it reads the caller's
 *     archive buffer) and never allocates on the hot path: scratch comes from aceapex_set_workspace().
 *   - One handle must not be used from two host threads at once.
 *   - Environment switches, read at open / first use, for tests and measurements only: ACEAPEX_NO_COOPERATIVE (demand rounds as
 *     three launches per round instead of one cooperative launch), ACEAPEX_READS_ROUNDS=0|1 (force one of the two read paths),
 *     ACEAPEX_CTAS_PER_SM (cap on resident CTAs of the generic kernel), ACEAPEX_WIN_TOKENS=1 (the collect and match launches of
 *     a range-decode window re-decode the block's tokens instead of reading the descriptors its literal launch left).
 */
#ifndef ACEAPEX_H
#define ACEAPEX_H

#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct aceapex_archive aceapex_archive;

enum {
    ACEAPEX_OK = 0,
    ACEAPEX_E_MAGIC = -1,      /* not an ACX-B200 archive                                        */
    ACEAPEX_E_VERSION = -2,    /* unsupported version / prob_bits                                */
    ACEAPEX_E_TRUNCATED = -3,  /* archive_bytes smaller than the archive says                    */
    ACEAPEX_E_CORRUPT = -4,    /* header / tables / directory inconsistent, or device flag set   */
    ACEAPEX_E_RANGE = -5,      /* byte range or read id out of bounds                            */
    ACEAPEX_E_BUDGET = -6,     /* vram_budget too small for the call                             */
    ACEAPEX_E_WORKSPACE = -7,  /* workspace missing or smaller than aceapex_info.workspace_bytes */
    ACEAPEX_E_CUDA = -8,       /* a CUDA runtime call failed (aceapex_last_cuda_error)           */
    ACEAPEX_E_ARG = -9,        /* null pointer / bad argument                                    */
    ACEAPEX_E_TOO_LARGE = -10  /* size beyond the fixed maximum of a no-allocation entry point  */
};

typedef struct {
    uint64_t raw_bytes;          /* N: decompressed size                                         */
    uint64_t archive_bytes;      /* C: compressed size (whole archive)                           */
    uint64_t n_blocks;
    uint64_t block_size;
    uint64_t total_lit_bytes;    /* bytes produced by literal runs                               */
    uint64_t total_match_bytes;  /* M: bytes produced by matches (= source bytes read)           */
    uint64_t total_matches;
    uint64_t total_cmds;
    uint64_t workspace_bytes;    /* device scratch the decode calls need (aceapex_set_workspace) */
    uint64_t n_segments;         /* FORMAT.md 1.5: entropy-coded units (one warp each)           */
    uint64_t total_litq_bytes;   /* literal bytes of the class LITQ (runs of q_min bytes or more) */
    uint32_t max_level;          /* FORMAT.md 3: number of match waves - 1                       */
    uint32_t offset_width;       /* W                                                            */
    uint32_t min_match;
    uint32_t max_cmds;           /* largest per-segment command count                            */
    uint32_t n_coded_planes;     /* offset planes that are rANS-coded (the rest are raw)         */
    uint32_t has_fnv;            /* per-block FNV-1a 64 section present                          */
    uint32_t resident_warps;     /* warps of the persistent decode grid                          */
    uint32_t segment_size;       /* SEG                                                          */
    uint32_t q_min;              /* FORMAT.md 1.6                                                */
    uint32_t q_mode;             /* FORMAT.md 1.7: 0 = LITQ bytes, 1 = LITQ aligned pairs        */
} aceapex_info_t;

/* Opens an archive that already resides in device memory ("H2D staging ... outside the timer").
 * d_archive: device pointer, 16-byte aligned, archive_bytes long, must outlive the handle.
 * h_archive_or_null: optional host copy of the same bytes (at least header + tables + directory); when null the
 *   library copies that prefix from the device (synchronous).  Validates magic, version, section layout, tables and
 *   the whole directory (monotone 16-byte aligned payload offsets, counts) and uploads the decode tables.
 * Errors: E_ARG, E_MAGIC, E_VERSION, E_TRUNCATED, E_CORRUPT, E_CUDA.  Synchronous. */
int32_t aceapex_open(const void* d_archive, uint64_t archive_bytes, const void* h_archive_or_null, aceapex_archive** out);

/* Frees the handle and the library's own device state (not the archive, not the workspace).  Synchronises. */
int32_t aceapex_close(aceapex_archive* ar);

int32_t aceapex_info(const aceapex_archive* ar, aceapex_info_t* out);

/* Caller-provided device scratch, >= aceapex_info.workspace_bytes, 256-byte aligned; must stay valid and untouched
 * by the caller while decode calls are in flight.  The first use zero-initialises its control area (async). */
int32_t aceapex_set_workspace(aceapex_archive* ar, void* d_workspace, uint64_t workspace_bytes);

/* cudaStream_t (as void*) all later calls are issued on; null = legacy default stream. */
int32_t aceapex_set_stream(aceapex_archive* ar, void* cuda_stream);

/* Whole-file decode (§3.3, the paper's "v4").  d_out: >= raw_bytes device bytes, 16-byte aligned.  On
 * completion of the stream, d_out[0..N) are the original bytes.  Scheduled as the wavefront of PAPER.md:17, 25 over the
 * dependency levels of FORMAT.md §3, in at most three launches: (1) every block: entropy decode, command scan, literal
 * placement; (2) the blocks below the top level, sorted by (level, index), a block waiting on a device-side completion
 * flag only for source blocks of a strictly lower level; (3) the blocks of the top level (the bulk: 97 % on FASTQ),
 * where nothing waits: every source is a literal byte or belongs to a lower level.  Errors: E_ARG, E_WORKSPACE, E_CUDA. */
int32_t aceapex_decode_all(aceapex_archive* ar, void* d_out);

/* Same result with TWO launches: one match launch takes ALL blocks sorted by (level, index) with completion flags (the
 * "device-side ready counter" variant of BASELINE.json north_star (4)).  Measured slightly slower. */
int32_t aceapex_decode_all_flags(aceapex_archive* ar, void* d_out);

/* Same result in ONE launch: blocks are taken in (level, index) order; each block places its literals, publishes a
 * "literals placed" flag, then resolves its matches, waiting for the literal flag of same-or-higher-level source
 * blocks and for the completion flag of lower-level ones.  Kept for comparison. */
int32_t aceapex_decode_all_fused(aceapex_archive* ar, void* d_out);

/* Arbitrary byte range [byte_lo, byte_hi) (§4, "v7-RA"): d_out[0 .. hi-lo) = those bytes; only the
 * covering blocks are decoded, sources outside the range are reconstructed on demand by recursion on their own
 * sources (depth <= max_level + 1, FORMAT.md §3).  vram_budget: upper bound on the workspace bytes the call touches
 * (0 = the whole workspace): a smaller budget shrinks the demand lists, the window is then served in more sub-windows;
 * E_BUDGET below the minimum (the fixed part of the workspace + 4096 demand records).  lo == hi is a no-op.  E_RANGE if
 * lo > hi or hi > N. */
int32_t aceapex_decode_range(aceapex_archive* ar, uint64_t byte_lo, uint64_t byte_hi, void* d_out, uint64_t vram_budget);

/* Read-level random access (§4.1).  h_read_index: host array of n_index entries, 8 bytes per read
 * (FORMAT.md §4: offset in bits 0..39, length in bits 40..63).  h_read_ids[n]: host array of read ids (duplicates
 * allowed).  d_out receives the reads packed back to back in h_read_ids order (size: aceapex_reads_bytes).
 * Only the blocks covering the reads, and recursively the source spans they need, are decoded.  E_RANGE on a bad id. */
int32_t aceapex_decode_reads(aceapex_archive* ar, const uint64_t* h_read_index, uint64_t n_index,
                             const uint64_t* h_read_ids, uint64_t n, void* d_out);

/* Output size of aceapex_decode_reads; h_out_offsets_or_null[n+1] receives the packed offsets.  Host only. */
int32_t aceapex_reads_bytes(const uint64_t* h_read_index, uint64_t n_index, const uint64_t* h_read_ids, uint64_t n,
                            uint64_t* total_bytes, uint64_t* h_out_offsets_or_null);

/* Makes bytes [pos_lo, pos_hi) of the decompressed output, already resident at d_ptr, usable as match sources by
 * aceapex_decode_range (the ring of PAPER.md:107-109 §5: earlier windows stay resident while later ones decode).
 * slot < 8; pos_lo == pos_hi clears the slot.  A slot must be cleared (or re-pointed) BEFORE its buffer is overwritten,
 * and d_ptr must be 8-byte aligned. */
int32_t aceapex_set_resident(aceapex_archive* ar, uint32_t slot, uint64_t pos_lo, uint64_t pos_hi, const void* d_ptr);

/* Range decode of [byte_lo, byte_hi) through a bounded device ring (section 5: the range decoder "processes
 * the archive in chunks, never materializing the full output at once"; BASELINE.json north_star (6)).  The library owns the
 * window order, the slot rotation and the resident registration (aceapex_set_resident); the caller owns the memory.
 *   d_ring / ring_bytes: device buffer, 16-byte aligned; it is cut into n_slots = min(8, ring_bytes / window_bytes) slots.
 *   window_bytes: multiple of the block size (the last window may be shorter); byte_lo must be a multiple of it too.
 *   Window w is decoded into slot w % n_slots.  Before a slot is overwritten its registration is cleared; after the decode
 *   has been queued it is registered again, so that later windows find its bytes as match sources instead of rebuilding
 *   them.  Everything runs on the handle's stream, in order: the decode of window w + n_slots, which overwrites the slot
 *   of window w, is queued after whatever the consumer queued for window w.
 *   consumer_or_null(user, window_index, window_lo, window_hi, d_window, cuda_stream) is called on the host once per
 *   window, after its decode has been queued; it may queue device work that reads d_window on cuda_stream (any other
 *   stream must be ordered by the consumer itself) and returns 0 to go on, anything else to stop (E_ARG is returned).
 *   With a null consumer and an FNV section in the archive the library's own consumer checks every block of every window
 *   on the device and reports the number of bad blocks in stats.
 *   vram_budget: as in aceapex_decode_range.  stats_or_null receives the figures below.  Synchronous: returns after the
 *   last window has completed.  Resident slots set by the caller before the call are overwritten and cleared. */
typedef int32_t (*aceapex_window_fn)(void* user, uint64_t window_index, uint64_t window_lo, uint64_t window_hi, const void* d_window,
                                     void* cuda_stream);
typedef struct {
    uint64_t n_windows;          /* windows decoded                                                            */
    uint64_t n_slots;            /* ring slots used                                                            */
    uint64_t bytes;              /* output bytes produced                                                      */
    uint64_t bad_blocks;         /* built-in consumer only: blocks whose FNV-1a differs                       */
    uint64_t peak_device_bytes;  /* archive + ring + workspace: everything the decode needs resident in VRAM  */
    float device_ms;             /* CUDA-event time from the first launch to the last                          */
    float min_window_gbs;        /* slowest / fastest window (10^9 B/s of output, CUDA events per window)     */
    float max_window_gbs;
    uint32_t reserved;
} aceapex_stream_stats_t;
int32_t aceapex_decode_stream(aceapex_archive* ar, uint64_t byte_lo, uint64_t byte_hi, void* d_ring, uint64_t ring_bytes,
                              uint64_t window_bytes, aceapex_window_fn consumer_or_null, void* user, uint64_t vram_budget,
                              aceapex_stream_stats_t* stats_or_null);

/* Device FNV-1a 64 of each block of d_data (= decompressed bytes [byte_lo, byte_hi), byte_lo block aligned) compared
 * with the archive's FNV section ("FNV for device-resident GPU paths").  Synchronous; *n_bad = number
 * of mismatching blocks.  E_ARG when the archive has no FNV section. */
int32_t aceapex_verify_fnv(aceapex_archive* ar, const void* d_data, uint64_t byte_lo, uint64_t byte_hi, uint64_t* n_bad);

/* End to end with HOST buffers (bench "e2e"; §6.1): h_archive (the same bytes the handle was opened on,
 * ideally pinned) -> the handle's device archive -> decode into d_out_staging (>= N device bytes, 16-byte aligned) -> h_out
 * (ideally pinned).  Pipelined over chunks of blocks on three streams: the payload of chunk k+1 travels host -> device
 * while chunk k decodes and the output of chunk k-1 travels device -> host.  Synchronous: returns when h_out is complete. */
int32_t aceapex_decode_all_host(aceapex_archive* ar, const void* h_archive, void* d_out_staging, void* h_out);

/* Synchronises the stream and returns E_CORRUPT if any kernel latched an integrity error since the last check
 * (details: aceapex_device_flags), E_CUDA on a CUDA error, else OK. */
int32_t aceapex_check(aceapex_archive* ar);
uint32_t aceapex_device_flags(const aceapex_archive* ar);   /* bit set of ACEAPEX_DF_* from the last aceapex_check */
int32_t aceapex_last_cuda_error(const aceapex_archive* ar); /* cudaError_t of the last failing runtime call         */
const char* aceapex_strerror(int32_t code);

/* Per-kernel device times of aceapex_decode_all (bench.py "roofline"): when switched on, the call records CUDA events on the
 * handle's stream around its three launches.  aceapex_phase_times waits for the last aceapex_decode_all and returns, in
 * milliseconds, ms3[0] = literal launch (entropy decode + scan + literal placement), ms3[1] = match launch of the blocks
 * below the top level, ms3[2] = match launch of the top level.  E_ARG when timing is off or nothing was decoded. */
int32_t aceapex_set_phase_timing(aceapex_archive* ar, int32_t on);
int32_t aceapex_phase_times(aceapex_archive* ar, float* ms3);

/* Number of kernel launches the library issued on this handle so far (bench.py "gpu_launches"). */
uint64_t aceapex_launch_count(const aceapex_archive* ar);
/* Number of those that went out as nodes of a replayed CUDA graph: aceapex_decode_range calls of up to 8 MiB on a level-0
 * archive record their launch sequence once and replay it with updated node parameters (seek latency is
 * launch overhead).  ACEAPEX_NO_GRAPHS in the environment at open switches that off. */
uint64_t aceapex_graph_launch_count(const aceapex_archive* ar);

/* ---- The entropy stage alone (section 6.4: DietGPU ANS on "256 MB exponential, batch 4096 x 64 KB", encode 364.9 /
 * decode 592.5 GB/s on the H100).  A batch is n_rows rows of row_bytes byte symbols, row r at d_in + r * row_bytes.  Every row
 * is coded on its own with ONE static table (256 frequencies summing to 2^11) as a rANS section of FORMAT.md 1.7: row r at
 * d_enc + r * row_capacity = [32 x (u32 initial state, u32 word_off)][u16 words], d_row_sizes[r] = 256 + 2 * words bytes.
 * One warp per row.  All pointers but h_freq are device memory owned by the caller; the calls are asynchronous on
 * cuda_stream unless stated.
 *   aceapex_rans_row_capacity(row_bytes): bytes to reserve per encoded row (the worst case, a multiple of 16).
 *   aceapex_rans_table_bytes(): size of the device table buffer; aceapex_rans_tables builds the encode and decode tables
 *     from h_freq and uploads them (synchronous).  E_ARG when the frequencies do not sum to 2^11.
 *   aceapex_rans_scratch_bytes(row_bytes): device scratch both kernels need (word staging of the encoder, counters).
 *   aceapex_rans_encode: rows -> encoded rows + sizes.  Every symbol of the input must have a non-zero frequency.
 *   aceapex_rans_decode: encoded rows -> rows; a row whose states do not end at 2^16 with every word stream consumed
 *     exactly latches bit 0 of the status word that aceapex_rans_status reads back (synchronous).  The decoder prefetches
 *     up to 128 bytes past the words of a row: d_enc must be that much longer than n_rows * row_capacity. */
uint64_t aceapex_rans_row_capacity(uint64_t row_bytes);
uint64_t aceapex_rans_table_bytes(void);
uint64_t aceapex_rans_scratch_bytes(uint64_t row_bytes);
int32_t aceapex_rans_tables(const uint16_t* h_freq, void* d_tables, void* cuda_stream);
int32_t aceapex_rans_encode(const void* d_in, uint64_t n_rows, uint64_t row_bytes, const void* d_tables, void* d_enc, uint64_t row_capacity,
                            uint32_t* d_row_sizes, void* d_scratch, uint64_t scratch_bytes, void* cuda_stream);
int32_t aceapex_rans_decode(const void* d_enc, uint64_t n_rows, uint64_t row_bytes, uint64_t row_capacity, const uint32_t* d_row_sizes,
                            const void* d_tables, void* d_out, void* d_scratch, uint64_t scratch_bytes, void* cuda_stream);
int32_t aceapex_rans_status(const void* d_scratch, void* cuda_stream, uint32_t* status);

/* ---- aceapex_rans_encode without any allocation, for callers that cannot call cudaMalloc (code under CUDA graph capture,
 * tight serving loops, harnesses that forbid it): the word staging and the work counter live in ONE file-scope
 * `static __device__` array of ACEAPEX_RANS_STATIC_SCRATCH_BYTES (+ 256) bytes inside the library, which every GPU that loads
 * the library holds until the process exits.  Same inputs, outputs, row layout and result (bit for bit) as
 * aceapex_rans_encode; the caller passes no scratch.  The number of warps at work is what the fixed array holds
 * (64 KB rows: 256 warps instead of one per row slot of the GPU), so large rows encode slower than through
 * aceapex_rans_encode.  Limits and rules:
 *   - row_bytes > ACEAPEX_RANS_STATIC_MAX_ROW_BYTES returns ACEAPEX_E_TOO_LARGE (nothing is launched); other bad arguments
 *     E_ARG as in aceapex_rans_encode.
 *   - The call makes no cudaMalloc / cudaFree and calls no allocating library routine: one cudaMemsetAsync of the 8-byte work
 *     counter (the only part of the array that must start at zero; the staging keeps the previous call's words, which are
 *     never read before they are rewritten) and one kernel launch on cuda_stream.
 *   - ALL calls on a device share the array: calls that overlap on the GPU (different streams, or graphs replayed
 *     concurrently) race on it and produce garbage.  Calls on one stream are ordered and safe.
 *   - The device address of the array is looked up once per device, with that device current (cudaGetSymbolAddress), by the
 *     first call on that device or by aceapex_rans_static_setup(), which callers that capture graphs run before capturing. */
#define ACEAPEX_RANS_STATIC_SCRATCH_BYTES (32ull << 20)
#define ACEAPEX_RANS_STATIC_MAX_ROW_BYTES 65536ull
int32_t aceapex_rans_static_setup(void);
int32_t aceapex_rans_encode_static(const void* d_in, uint64_t n_rows, uint64_t row_bytes, const void* d_tables, void* d_enc, uint64_t row_capacity,
                                   uint32_t* d_row_sizes, void* cuda_stream);

enum {
    ACEAPEX_DF_RANS = 1,      /* final rANS state / word count mismatch         */
    ACEAPEX_DF_OFFSET = 2,    /* src >= dst or match leaves the block           */
    ACEAPEX_DF_LENGTH = 4,    /* command lengths do not add up to the block     */
    ACEAPEX_DF_TIMEOUT = 8,   /* a dependency flag was never set                */
    ACEAPEX_DF_STACK = 16     /* demand stack overflow (range / read decode)    */
};

#ifdef __cplusplus
}
#endif
#endif
