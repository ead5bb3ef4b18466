/*
 * aa.h — C ABI of the B200-native dedispersion + single-pulse-search (SPS) hot path.
 *
 * What it mirrors. arXiv:1912.07704 describes AstroAccelerate's plan -> strategy -> pipeline pattern:
 * the user fills a *plan* with search parameters, the API computes an immutable *strategy* ("how input data are
 * split and processed on the GPU", PAPER.md:43 §3.1, :59 §3.2), the pipeline "iterates over the radio telescope
 * input data in chunks" and reports a *status code* per iteration (§3.3); telescope data stay on the
 * host under the user's ownership, device memory is encapsulated, results are owned by the API (§2.4);
 * modules request device memory from a memory manager before use (§2.3). The call sequence below is the
 * paper's 8-step list (§3.1). The function names and the arithmetic are BASELINE.json `north_star`.
 *
 * Conventions
 *   - Plain C, no exceptions cross the boundary. Process-wide state: a thread-local error string, and (aa_row_moments_static
 *     only) the address of its built-in scratch array per device. Everything else, kernel attributes and the SM count
 *     included, is set per strategy at aa_strategy_setup for the device that is current there; every aa_run_* / aa_get_* call
 *     on a strategy must be made with that same device current (AA_ERR_INVALID_ARG naming both devices otherwise).
 *   - Every entry point returns aa_status: >= 0 success / progress, < 0 error. After an error,
 *     aa_last_error() names the offending field ("the API provides user feedback").
 *     Errors raised by aa_run_* are sticky on the strategy.
 *   - "host" / "device" is stated for every pointer. No CUDA allocation happens inside aa_run_*; all device memory
 *     is carved from ONE arena at aa_strategy_setup (north_star "memory-manager arena makes one allocation per run").
 *   - Thread safety: distinct strategies may be used from distinct threads; one strategy is not re-entrant.
 */
#ifndef AA_H
#define AA_H

#include <stddef.h>
#include <stdint.h>

#ifdef __cplusplus
extern "C" {
#endif

typedef struct aa_plan aa_plan;          /* opaque: the user's search parameters + metadata */
typedef struct aa_strategy aa_strategy;  /* opaque: immutable GPU configuration + the chunk cursor */

typedef enum {
    AA_OK = 0,
    AA_STATUS_CHUNK_DONE = 1,        /* this chunk finished, more chunks remain */
    AA_STATUS_FINISHED = 2,          /* the last chunk finished */
    AA_ERR_INVALID_ARG = -1,
    AA_ERR_NOT_READY = -2,           /* run before a successful setup                   (PAPER.md:59 items 2, 4) */
    AA_ERR_BUDGET_TOO_SMALL = -3,
    AA_ERR_CUDA = -4,
    AA_ERR_CANDIDATE_OVERFLOW = -5,  /* records beyond capacity were dropped, the count is still exact */
    AA_ERR_ORDER = -6,               /* "another module still needs to run" */
    AA_ERR_INTERNAL = -7,
    AA_ERR_RANGE = -8                /* 16-bit plans only: a sample above max_value, or the data made a boxcar sum leave int32
                                        (see aa_plan_set_input_bits) */
} aa_status;

/* One DM range: DM_i = dm_low + i*dm_step for i in [0, ndms); the range is searched on data decimated in time by
 * `bin` in {1,2,4,8} (north_star "DM ranges that decimate in time by 1/2/4/8"; binning = SUM of bin samples). */
typedef struct {
    double dm_low, dm_step;
    int32_t ndms;
    int32_t bin;
} aa_dm_range;

/* One candidate (north_star "finds local peaks above a threshold into a candidate list"). */
typedef struct {
    uint64_t sample;    /* absolute UNBINNED start sample of the best boxcar */
    float dm;           /* (float) DM_i */
    float snr;          /* (float) best SNR over the plan's widths */
    uint32_t width;     /* best boxcar width in UNBINNED samples (= w * bin) */
    uint32_t range;     /* index into the plan's ranges */
    uint32_t dm_index;  /* i within the range */
} aa_candidate;

/* Per-range geometry of one chunk, as decided by the strategy (read-only facts, PAPER.md:59 item 2). */
typedef struct {
    int32_t ndms, bin;
    int64_t nt;            /* T_r: output samples per DM row per FULL chunk (binned units) = n_out / bin */
    int64_t row_pitch;     /* int32 elements between consecutive DM rows of D_r on the device */
    int64_t max_delay;     /* delay(C-1, last DM) in binned samples */
    int32_t dm_tile, t_tile, chan_block, window;   /* dedispersion kernel tiling chosen for this range */
    int32_t boxcar_extra;  /* E: samples dedispersed beyond nt per row (0 unless aa_plan_set_boxcar_overlap) */
} aa_range_info;

typedef struct {
    int32_t ready;             /* 1 once setup succeeded */
    int32_t nchans, nranges, nwidths;
    int32_t max_bin;           /* B */
    int64_t nsamp_total;
    int64_t overlap;           /* S: unbinned samples shared by consecutive chunks = max delay rounded up to B */
    int64_t chunk_len;         /* L: unbinned input samples per full chunk (multiple of B, > S) */
    int64_t n_out;             /* L - S: unbinned output span per full chunk */
    int64_t nchunks;
    int64_t next_chunk;        /* chunk cursor: index of the chunk the next aa_run_dedispersion will process */
    int32_t shard_rank, shard_world;   /* aa_strategy_shard: this strategy owns chunks rank, rank+world, ... (0, 1 by default) */
    size_t arena_bytes_used;   /* bytes carved from the arena */
    size_t arena_bytes_total;
    size_t max_candidates;
    int32_t owns_arena;        /* 1 if the library made the (single) cudaMalloc */
    int32_t input_layout;      /* aa_input_layout of the bound plan */
    int32_t input_bits;        /* 8 or 16 (aa_plan_set_input_bits) */
    uint32_t input_max;        /* the plan's largest sample value */
} aa_strategy_info;

/* ------------------------------------------------------------------------------------------------ plan
 * PAPER.md:47 steps 1,3 ("provide ... metadata", "configure each module with a plan"). All arrays are HOST memory and
 * are copied; the caller may free them on return.
 *   chan_freq_mhz [nchans]  strictly descending; [0] is f_top, the reference of every delay.
 *   tsamp_s                 sampling time in seconds (> 0).
 *   ranges [nranges]        ndms >= 1, dm_step > 0 (or ndms == 1), dm_low >= 0, bin in {1,2,4,8}.
 *   boxcar_widths [nwidths] strictly ascending, >= 1, in BINNED samples of each range (north_star "widths 1..W").
 *   snr_threshold           candidates need SNR > threshold (strict).
 * Limits checked here: nchans*255*max(bin) < 2^23 (int32 sums with headroom for the packed accumulators) and
 * max(width)*nchans*255*max(bin) < 2^31 (boxcar sums). Errors: AA_ERR_INVALID_ARG naming the field. */
aa_status aa_plan_create(aa_plan** out, int32_t nchans, const double* chan_freq_mhz, double tsamp_s,
                         const aa_dm_range* ranges, int32_t nranges,
                         const int32_t* boxcar_widths, int32_t nwidths, float snr_threshold);
void aa_plan_destroy(aa_plan* plan);

/* Layout of the input data (metadata of the telescope data, PAPER.md:47 step 1). Default AA_LAYOUT_CHANNEL_MAJOR:
 * x[c][t], one row per channel. AA_LAYOUT_TIME_MAJOR: x[t][c], one row per time sample, the order telescopes
 * deliver; each chunk is then one contiguous host block, copied as it is and corner-turned on the device (kernel
 * K0t) before binning and dedispersion. Must be called before aa_strategy_setup binds the plan (the strategy reserves
 * the staging buffers). Results are identical in both layouts. Errors: AA_ERR_INVALID_ARG naming `layout`. */
typedef enum { AA_LAYOUT_CHANNEL_MAJOR = 0, AA_LAYOUT_TIME_MAJOR = 1 } aa_input_layout;
aa_status aa_plan_set_input_layout(aa_plan* plan, int32_t layout);

/* Sample type of the input (metadata of the telescope data, PAPER.md:47 step 1; the user directs the library at
 * telescope data, which back-ends deliver as 8- or 16-bit samples). Default: bits = 8, uint8 samples.
 * bits = 16: every sample is a uint16 in host byte order and at most max_value (the telescope's stated bit depth, e.g. 4095;
 * 0 means 65535). host_input of aa_run_* then points at uint16 samples (row strides stay in BYTES), and a time-major
 * device chunk needs rows that are 4-byte aligned. Results are exact for ANY input within max_value (binning, dedispersion
 * and everything after are the same definitions; reading C4w).
 * Limits checked here (AA_ERR_INVALID_ARG naming the field): max_value * max(bin) <= 65535 (a binned sample is held in 16
 * bits) and nchans * max_value * max(bin) < 2^31 (int32 sums). The 8-bit plan's worst-case bound on boxcar sums cannot be
 * given at plan time for 16-bit samples (256 * 4096 * 4095 * 8 is far beyond int32 although real boxcar sums of (D - D[0])
 * are tiny), so it is checked on the DATA instead: if width_max * max|D - D[0]| of a row reaches 2^31, aa_run_sps /
 * aa_get_candidates return AA_ERR_RANGE (sticky) rather than a wrong candidate. The samples themselves are checked too, in
 * the kernel that reads every chunk for the per-channel means: a chunk with a sample above max_value (its binned sums would
 * carry into their neighbours) ends in the same sticky AA_ERR_RANGE at the next aa_run_sps / aa_get_candidates.
 * Speed: noise around a per-channel mean rides the 1-byte dedispersion path whatever the sample type (per-channel offset +
 * exception list); a chunk whose channels spread over more than about +-128 (bin 1, 2, 4) or +-512 (bin 8)
 * around their mean in too many samples falls back to a slow global-memory kernel - still exact.
 * Must be called before aa_strategy_setup binds the plan. */
aa_status aa_plan_set_input_bits(aa_plan* plan, int32_t bits, uint32_t max_value);

/* Boxcar-complete chunks (reading C3x; off by default). With the plain chunking a boxcar of width w that starts in
 * the last w-1 samples of a chunk's output span is not evaluated (it would need samples of the next chunk), so a wide
 * pulse straddling a chunk boundary is seen only by narrower boxcars. on != 0: every row is dedispersed
 * E = max(boxcar_widths) - 1 binned samples beyond its chunk's output span (the overlap S grows to
 * ceil_B(max_r bin_r (delay_max_r + E))), statistics still use the span itself, and every boxcar that STARTS inside the span
 * is complete. Candidates are still reported for start samples inside the span only, so chunks do not duplicate them.
 * Must be called before aa_strategy_setup binds the plan. */
aa_status aa_plan_set_boxcar_overlap(aa_plan* plan, int32_t on);

/* Per-width measured statistics (reading C7m; off by default; §1 "boxcar filters and peak-finding to
 * maximise signal-to-noise"). By default a boxcar of width w is normalised with the width-1 statistics of its row scaled for
 * white noise (w mu, sqrt(w) sigma). on != 0: for every row and every plan width w the series B_w[t] = sum_{j<w} D[t+j],
 * t in [0, n_w), n_w = min(T_r, samples present - w + 1), gets its OWN robust statistics (the same iterated 3-sigma clip on
 * exact integer moments, pivot p_w = B_w[0]) and SNR_w[t] = ((double)(B_w[t] - p_w) - (mu_w - p_w)) * (1 / sigma_w). A width
 * whose series is constant or clips to nothing gives no SNR in that row. For w = 1 this is the default exactly; for red
 * (correlated) noise the sqrt(w) scaling overstates the SNR of wide boxcars and this option does not. Costs one more kernel
 * (K3w) that reads D once per clip iteration. Must be called before aa_strategy_setup binds the plan. */
aa_status aa_plan_set_per_width_stats(aa_plan* plan, int32_t on);

/* ------------------------------------------------------------------------------------------------ strategy
 * PAPER.md:47 steps 4-6 ("bind", "the API calculates the optimal strategy", "checks whether all modules are
 * configured"). Host-side planning plus ONE device allocation (or none if the caller lends an arena):
 *   delays:  k_c = (4.148808e3*(f_c^-2 - f_0^-2))/tsamp; delay(c,r,i) = llround((k_c*DM_ri)/bin_r)   [north_star]
 *   chunks:  S = ceil_B(max_r bin_r*delay(C-1,r,last)); L multiple of B with arena(L) <= budget; n_out = L - S;
 *            chunk j covers input [j*n_out, j*n_out + L) and outputs [j*n_out, (j+1)*n_out); the last chunk takes the
 *            remaining input rounded down to a multiple of B (reading C3). chunk_len_hint > 0 forces L.
 *   device_arena (DEVICE, may be NULL): caller-owned memory of arena_bytes (e.g. a torch uint8 tensor), 256-byte
 *            aligned. NULL => the library makes exactly one cudaMalloc of the bytes it needs (<= budget_bytes;
 *            budget_bytes == 0 means "no limit": a single chunk if it fits the device).
 *   compute_stream / copy_stream: cudaStream_t handles (e.g. from torch); NULL => the library creates its own.
 *   max_candidates: capacity of the device candidate buffer per chunk and of the host list.
 * The plan may be destroyed afterwards. Errors: AA_ERR_INVALID_ARG, AA_ERR_BUDGET_TOO_SMALL (message states the
 * bytes needed for the smallest legal chunk), AA_ERR_CUDA. */
aa_status aa_strategy_setup(aa_strategy** out, const aa_plan* plan, uint64_t nsamp_total,
                            void* device_arena, size_t arena_bytes, size_t budget_bytes,
                            void* compute_stream, void* copy_stream, size_t max_candidates,
                            uint64_t chunk_len_hint);
void aa_strategy_destroy(aa_strategy* s);

/* Host-only planning: the same delays, chunk geometry, kernel tiling and arena size as aa_strategy_setup, without touching
 * the GPU. The result has ready == 0 ("query the strategy fields and ready-state"): getters work,
 * aa_run_* return AA_ERR_NOT_READY. budget_bytes == 0 means unlimited (a single chunk). arena_bytes_used reports the bytes a
 * real setup would carve. */
aa_status aa_strategy_plan(aa_strategy** out, const aa_plan* plan, uint64_t nsamp_total, size_t budget_bytes,
                           size_t max_candidates, uint64_t chunk_len_hint);

/* Read-only queries (PAPER.md:59 item 2 "the user may query the strategy fields and ready-state"). */
aa_status aa_strategy_get_info(const aa_strategy* s, aa_strategy_info* out);
aa_status aa_strategy_get_range_info(const aa_strategy* s, int32_t range, aa_range_info* out);
/* Chunk j: absolute start sample, input length L_j and output span n_out_j (unbinned). */
aa_status aa_strategy_get_chunk(const aa_strategy* s, int64_t chunk, uint64_t* start, uint64_t* len, uint64_t* n_out);
/* delay(c, range, dm_index) in binned samples, as used by the kernels. */
aa_status aa_strategy_get_delay(const aa_strategy* s, int32_t range, int32_t dm_index, int32_t chan, int64_t* delay);
/* Human-readable dump of chunking, tiling and arena layout into buf (HOST); returns bytes needed incl. NUL. */
size_t aa_strategy_describe(const aa_strategy* s, char* buf, size_t buflen);
/* Rewind the chunk cursor to the first chunk of this strategy's shard and forget all candidates (the configuration
 * itself is immutable). */
aa_status aa_strategy_reset(aa_strategy* s);
/* Multi-GPU replicas over time chunks ("parallel pipeline ... execution on multiple GPUs"; DESIGN.md
 * "Multi-GPU"): this strategy processes only chunks rank, rank+world, rank+2*world, ...  Chunks are independent given
 * the S-sample overlap, so there is no exchange between ranks; every rank holds its own arena and the host
 * concatenates the candidate lists. Host-only, also valid on a planned (not ready) strategy. Rewinds the cursor like
 * aa_strategy_reset. A rank with no chunk (rank >= nchunks) is legal: its first aa_run_dedispersion returns
 * AA_ERR_ORDER ("all chunks are done"). Errors: AA_ERR_INVALID_ARG unless 0 <= rank < world. */
aa_status aa_strategy_shard(aa_strategy* s, int32_t rank, int32_t world);

/* ------------------------------------------------------------------------------------------------ pipeline
 * PAPER.md:47 step 7. One call = one chunk of one module.
 *
 * aa_run_dedispersion: H2D of the cursor's chunk (unless a previous call prefetched it), prefetch of the following chunk on
 * the copy stream (channel-major plans have ONE raw input buffer: the prefetch starts as soon as K1, its only reader, has
 * finished with the current chunk; time-major plans alternate between two staging buffers), time binning for ranges with
 * bin > 1, then
 *   D_r[i][t'] = sum_c x_b[c][t' + delay(c,r,i)]   (int32, bit-exact)            [north_star]
 * for every range. Asynchronous: returns after enqueueing.
 *   host_input (HOST, const, user-owned, never written): the WHOLE observation; uint8 samples, or uint16 samples for a plan
 *              with aa_plan_set_input_bits(16, ..) (strides stay in bytes). Channel-major plans:
 *              x[c][t], nsamp_total samples per channel, row_stride_bytes between channels. Time-major plans
 *              (aa_plan_set_input_layout): x[t][c], nchans samples per row, row_stride_bytes (>= nchans) between
 *              consecutive time samples. Must stay valid until the
 *              following aa_run_* call returns (prefetch). Pinned memory is needed for the copy to overlap compute.
 * A chunk that was not prefetched (the first chunk; a single-chunk observation) is copied in three channel groups (1/16, 5/16, 10/16 of the channels) and each
 * group is binned and added into D as soon as it has landed, so only the first group's copy is
 * exposed; the sums are int32, any grouping gives the same bits.
 * Returns AA_OK; AA_ERR_NOT_READY; AA_ERR_ORDER if the previous chunk's SPS has not run; AA_ERR_CUDA. */
aa_status aa_run_dedispersion(aa_strategy* s, const uint8_t* host_input /* uint16 samples for a 16-bit plan */, size_t row_stride_bytes);

/* Same, with the chunk already resident on the DEVICE: device_chunk points at sample `start` of chunk `cursor`
 * (x[c][0..L_j), or x[0..L_j)[c] for a time-major plan: then 4-byte aligned with a stride that is a multiple of 4 and
 * >= nchans rounded up to 4), row stride in bytes, at least 16-byte aligned rows; the data are copied device-to-device into the
 * arena's input buffer (so the kernel's over-read slack exists). Used when the producer is another GPU stage. */
aa_status aa_run_dedispersion_device(aa_strategy* s, const uint8_t* device_chunk, size_t row_stride_bytes);

/* aa_run_sps: on the chunk just dedispersed — robust per-row mean/sigma, boxcar SNR, 3x3 local peaks above the
 * threshold, appended to the device candidate buffer. Advances the chunk cursor.
 * Returns AA_STATUS_CHUNK_DONE or AA_STATUS_FINISHED; AA_ERR_ORDER if no dedispersed chunk is pending. */
aa_status aa_run_sps(aa_strategy* s);

/* aa_run_pipeline: the whole chunk loop in one call (PAPER.md:47 step 7 "run the pipeline"): aa_run_dedispersion then
 * aa_run_sps for every remaining chunk of this strategy's shard. Returns AA_STATUS_FINISHED, or the first error. The
 * per-iteration status codes remain available to callers that drive the loop themselves; a test compares this C loop
 * with the Python loop over the same calls (the front-end adds no appreciable run time). */
aa_status aa_run_pipeline(aa_strategy* s, const uint8_t* host_input, size_t row_stride_bytes);

/* aa_get_candidates: synchronises, copies the device records to library-owned HOST memory, and returns ALL candidates
 * of the chunks processed so far in canonical order (chunk, range, dm_index, sample). *out stays valid until the next
 * aa_run_*, aa_strategy_reset or aa_strategy_destroy. Returns AA_OK, or AA_ERR_CANDIDATE_OVERFLOW when more
 * candidates were found than max_candidates (the list holds the first max_candidates in arrival order, sorted; the true
 * count is in aa_last_error()). */
aa_status aa_get_candidates(aa_strategy* s, const aa_candidate** out, size_t* n);

/* Candidate clustering (reading C10): one bright pulse yields many candidates (neighbouring DM
 * trials, widths, DM ranges, chunk edges). Two candidates are LINKED iff |dm_a - dm_b| <= dm_tol and their boxcars,
 * [sample, sample + width), are at most `gap` samples apart (sample_a <= sample_b + width_b + gap and vice versa);
 * clusters are the connected components of that relation over ALL candidates gathered so far (any range, any chunk).
 * Each cluster is reported by its member of highest SNR (first by (range, dm_index, sample) on ties) plus its extent.
 * Host-side, on the library-owned list; *out stays valid until the next aa_run_*, aa_get_clusters, reset or destroy.
 * Clusters are ordered by (range, dm_index, sample) of their representatives. Errors: as aa_get_candidates, and
 * AA_ERR_INVALID_ARG for a negative or non-finite dm_tol. */
typedef struct {
    aa_candidate best;          /* the member with the highest SNR */
    uint32_t members;           /* number of candidates in the cluster */
    float dm_min, dm_max;       /* extent over the members */
    uint64_t sample_min;        /* earliest boxcar start */
    uint64_t sample_end;        /* latest boxcar end (sample + width), exclusive */
} aa_cluster;
aa_status aa_get_clusters(aa_strategy* s, double dm_tol, uint64_t gap, const aa_cluster** out, size_t* n);
/* The same relation on a caller-supplied list (HOST, any order); results land in caller memory `out` of capacity >= n.
 * Returns the number of clusters through *nout. Needs no strategy and no GPU. */
aa_status aa_cluster_candidates(const aa_candidate* in, size_t n, double dm_tol, uint64_t gap, aa_cluster* out, size_t* nout);

/* Parity hooks: copy one row of the CURRENT chunk (the one last dedispersed / searched) to library-owned HOST memory:
 * nt + boxcar_extra samples. Valid until the next call on this strategy. */
aa_status aa_get_dedispersed_row(aa_strategy* s, int32_t range, int32_t dm_index, const int32_t** host_row, size_t* len);
/* mu, sigma, n kept, clip iterations of a row, as computed by aa_run_sps for the current chunk. */
aa_status aa_get_row_stats(aa_strategy* s, int32_t range, int32_t dm_index, double* mu, double* sigma,
                           int64_t* n_kept, int32_t* iterations);
/* Reading C7m only (aa_plan_set_per_width_stats): mu_w, sigma_w (0 = this width gives no SNR in this row) and the pivot
 * p_w = B_w[0] of plan width `width_index` in a row, as computed by aa_run_sps for the current chunk.
 * AA_ERR_ORDER if the option is off or aa_run_sps has not run. */
aa_status aa_get_row_width_stats(aa_strategy* s, int32_t range, int32_t dm_index, int32_t width_index, double* mu, double* sigma,
                                 int64_t* pivot);
/* Per-row moments sum_t D and sum_t t*D (int64) of every row of a range, computed on the device (test hook for the
 * all-rows checksum). out arrays are HOST, length ndms. */
aa_status aa_get_row_moments(aa_strategy* s, int32_t range, int64_t* sum_d, int64_t* sum_td);
/* Device pointer of D_r for the current chunk and its row pitch in elements (read-only use by other GPU code). */
aa_status aa_get_dedispersed_device(aa_strategy* s, int32_t range, const int32_t** device_ptr, int64_t* row_pitch);

/* aa_row_moments_static: the same two checksums per row as aa_get_row_moments (sum_t D[i][t] and sum_t t * D[i][t], int64,
 * wrapping modulo 2^64 like it), on ANY block of int32 rows in device memory, WITHOUT allocating anything - no strategy, no
 * arena, no cudaMalloc / cudaFree / allocating library call inside.
 *
 * Who needs it: code that may not allocate device memory at the moment it wants to check rows of D. (1) A back-end that has
 * handed out all of the GPU's memory up front (the arena lent to aa_strategy_setup, the capture ring, other stages): a fresh
 * cudaMalloc there can fail, and the budget forbids it anyway. (2) A watchdog thread that checksums rows while the chunk loop
 * streams: cudaMalloc and cudaFree synchronise the whole device and would stall the H2D prefetch and the kernels in flight.
 * aa_get_row_moments does not serve them: it works only on a strategy's own D, out of that strategy's arena.
 *
 * Working memory: one array built into the library, 2 x AA_STATIC_MOMENTS_MAX_ROWS x 8 bytes = 256 KiB, present on every
 * GPU that loads this library's kernels, from load until the process exits, whether this function is ever called or not.
 *   device_D   (DEVICE, const) nrows rows of int32, row i at device_D + i * row_pitch (elements); e.g. from
 *              aa_get_dedispersed_device. Must be memory of the CURRENT device.
 *   nt         samples summed per row, 0 <= nt <= row_pitch.
 *   nrows      0 <= nrows <= AA_STATIC_MOMENTS_MAX_ROWS (16384). More rows: AA_ERR_INVALID_ARG, nothing is launched, and
 *              aa_last_error() states the limit - split the rows over several calls.
 *   host_sum_d, host_sum_td (HOST, caller-owned) nrows int64 each, written before the call returns.
 *   stream     cudaStream_t (NULL = default stream). The kernels and the two device-to-host copies run on it and the call
 *              waits for it, so work queued earlier on that stream (the kernel that writes D) is finished first.
 * First call on each device: the function asks the CUDA runtime for the array's address on the current device
 * (cudaGetSymbolAddress) and keeps it; later calls on that device reuse it. Make this first call during start-up, with the
 * intended device current and before any stream capture begins.
 * Sharing: every call on a GPU uses the SAME array, and it keeps the last call's sums. Each call clears the words it will use
 * on `stream` before summing, so calls one after another (any stream, any thread) are independent; two calls that are on the
 * GPU at the same time (two host threads, two streams) add into the same words and both get wrong sums - serialise them.
 * Results equal aa_get_row_moments' bit for bit (integer sums). Errors: AA_ERR_INVALID_ARG, AA_ERR_CUDA. */
#define AA_STATIC_MOMENTS_MAX_ROWS 16384
aa_status aa_row_moments_static(const int32_t* device_D, int64_t row_pitch, int64_t nt, int32_t nrows,
                                int64_t* host_sum_d, int64_t* host_sum_td, void* stream);

/* Block until everything enqueued on the strategy's streams has finished. */
aa_status aa_synchronize(aa_strategy* s);

/* ------------------------------------------------------------------------------------------------ measurement
 * Sustained 32-bit integer add rate of this GPU (the roofline denominator): runs the K0
 * microbenchmark for about `millis` ms on `stream` (NULL = default). Outputs (HOST): lane-adds per second with
 * IADD3-only chains, with IADD3+IMAD mixed chains (both integer pipes), and the SM clock (MHz) observed via the cycle
 * counter. */
aa_status aa_measure_int_add_peak(void* stream, int32_t millis, double* iadd3_per_s, double* mixed_per_s, double* sm_mhz);
/* Same, plus the rate of IMAD-only chains (x*1+y on the FMA pipe alone). Any output pointer may be NULL. */
aa_status aa_measure_int_add_peak3(void* stream, int32_t millis, double* iadd3_per_s, double* mixed_per_s, double* imad_per_s,
                                   double* sm_mhz);

/* CUDA-event time (ms) of the kernel classes of the last chunk: [0] binning, [1] dedispersion (all ranges),
 * [2] SPS statistics, [3] SPS boxcar/peaks, [4] H2D of the chunk (0 if prefetched/overlapped). Synchronises. */
aa_status aa_get_last_timings(aa_strategy* s, float ms_out[5]);
/* Number of kernel launches issued by this strategy since setup / reset. */
aa_status aa_get_launch_count(const aa_strategy* s, uint64_t* launches);

const char* aa_last_error(void);   /* thread-local, never NULL */
const char* aa_version(void);

#ifdef __cplusplus
}
#endif
#endif /* AA_H */
