/*
 * aa_kernels.h — C-style launch wrappers of the CUDA kernels (one per kernel class), called by the host runtime.
 * Follows the separate-compilation practice of PAPER.md:25 (§2.1): CUDA code in its own translation units behind
 * C wrapper functions; host code compiled by the host compiler.
 *
 * All pointers are DEVICE pointers unless named h_*. No wrapper allocates memory. Every wrapper returns the
 * cudaError_t of the launch (cudaGetLastError), as an int.
 */
#ifndef AA_KERNELS_H
#define AA_KERNELS_H

#include <stddef.h>
#include <stdint.h>
#include <vector_types.h>

#ifdef __cplusplus
extern "C" {
#endif

/* ---- K1: time binning, x_b[c][t'] = sum_{j<b} x[c][b*t'+j]  (uint8 -> uint16) --------------------------------- */
/* only_if_cnt (may be NULL): the kernel returns at once unless *only_if_cnt > only_if_above (the uint16 route of a
 * range that also has the offset-uint8 route runs only for chunks with too many exceptions). Same for aak_shift_copy. */
int aak_bin_time(const uint8_t* x, size_t x_pitch, uint16_t* xb, size_t xb_pitch_elems, int32_t nchans,
                 int64_t nbinned, int32_t bin, const unsigned* only_if_cnt, unsigned only_if_above, void* stream);
/* ---- K1b: shifted copy, out[c][j] = in[c][j + shift_bytes] (1..3) for j in [0, row_bytes), rows `pitch` bytes apart.
 * row_bytes and pitch are multiples of 16; only [0, row_bytes) of a source row is read, and the last shift_bytes of an output row
 * (which would come from past the source row) are zero, so out may start right behind the source row (out = in + row_bytes). */
int aak_shift_copy(const uint8_t* in, uint8_t* out, size_t pitch, size_t row_bytes, int32_t nrows, int32_t shift_bytes,
                   const unsigned* only_if_cnt, unsigned only_if_above, void* stream);

/* ---- K1c: offset forms of a binned input, see k_misc.cu: x_b = lo + off_c + r with lo a byte and r an exception list (bin 2, 4),
 * x_8 = 2 y + bit + off_c + r (bin 8, half-byte form). aak_chan_offsets: off_b[c] = clamp(round(b * mean_t x[c][t]) - centre, 0, ..)
 * for rows [0, nrows), centre 128 (bin 2, 4) or 256 (bin 8), and *bias_b += sum of them (any pair may be NULL). aak_prep_fused
 * (below) writes the forms and appends the exceptions (64-bit records: channel 16 bits, residual r 20 bits two's complement,
 * binned sample 28 bits; k_common.cuh) at exc[counter++] while the counter is below cap (one atomic per warp; nothing more is
 * counted once it has passed cap). aak_scatter_exceptions: D[i][t' - delay(c, i)] += r for every exception and every trial of
 * one range; returns at once if *exc_cnt > cap. k = the plan's delay constants (device doubles). */
int aak_chan_offsets(const uint8_t* x, size_t pitch, int64_t len, int32_t nrows, int32_t* off2, int32_t* off4, int32_t* off8, int32_t* bias2,
                     int32_t* bias4, int32_t* bias8, void* stream);
int aak_scatter_exceptions(const uint2* exc, const unsigned* exc_cnt, unsigned cap, const double* k, double dm_low, double dm_step,
                           int32_t ndms, int32_t bin, int64_t nt, int32_t* D, int64_t pitch,
                           int32_t nsm /* SMs of the strategy's device: the grid is 4 CTAs per SM */, void* stream);

/* ---- K1 fused: one read of raw rows [0, nrows) (pointers already offset to the first row; chan0 = its channel index)
 * writes the 4 uint8 copies (x4, may be NULL; rows x4_pitch bytes apart, copy k at + k x4_stride), the offset-uint8 forms lo2 / lo4 with their 4 copies and exceptions (may be
 * NULL; off2/off4 offset to the first row; nb = valid binned samples) and, for bin 8, EITHER the half-byte form (hb8, bits8) OR
 * the 2 copies of the uint16 input (xb8; xb8_pitch in elements, xb8_stride in bytes). ngroups = 16-byte groups per row, a
 * multiple of 16. */
typedef struct {
    const uint8_t* raw; size_t pitch; int64_t ngroups; int32_t chan0; unsigned cap;
    uint8_t* x4; size_t x4_pitch, x4_stride;
    uint8_t* lo2; size_t lo2_pitch, lo2_stride; const int32_t* off2; uint2* exc2; unsigned* cnt2; int64_t nb2;
    uint8_t* lo4; size_t lo4_pitch, lo4_stride; const int32_t* off4; uint2* exc4; unsigned* cnt4; int64_t nb4;
    uint16_t* xb8; size_t xb8_pitch, xb8_stride;
    /* half-byte form of bin 8 (NULL: not used): x_8 = 2 y + bit + off8[c] + r with y a byte (4 shifted copies in hb8), bit the
     * dropped low bit (bits8: one bit per sample, rows of bits8_pitch 32-bit words) and r an exception list; off8[c] =
     * clamp(round(8 mean) - 256, 0, ..) from aak_chan_offsets. K2 sums y with its byte path and doubles the sums,
     * aak_dedisperse_bits adds the dedispersed bit plane, aak_scatter_exceptions the r. */
    uint8_t* hb8; size_t hb8_pitch, hb8_stride; const int32_t* off8; uint2* exc8; unsigned* cnt8; int64_t nb8;
    uint32_t* bits8; size_t bits8_pitch;
} aak_prep_args;
int aak_prep_fused(const aak_prep_args* a, int32_t nrows, void* stream);

/* ---- K1 for 16-bit input samples (k_input16.cu): the offset forms x_b = lo + off_b[c] + r of a uint16 chunk.
 * aak_chan_offsets16: off[k][c] = clamp(round(b mean_t x[c][t]) - centre[k], 0, ..) and *bias[k] += off[k][c], k = 0..3 <-> b = 1, 2, 4, 8
 * (NULL entries are skipped; pointers already offset to the first row). The same read checks every sample against the plan's
 * max_value (the packed sums of K1 and the int32 bound on D rely on it).
 * aak_prep16: one read of raw rows writes the byte forms of bin 1, 2, 4 (lo[k], 4 copies, window [0, 255]) and the uint16 form
 * of bin 8 (lo8, 2 copies, window [0, hi8]) with their exception lists; ngroups = 32-byte groups (16 samples) per row.
 * aak_bin_time16: plain x_b as uint16, one copy (the input of the global-memory route); bin in {1, 2, 4, 8}; conditional like
 * aak_bin_time. aak_corner_turn16: x[c][t] = x_tm[t][c] for uint16 samples. */
int aak_chan_offsets16(const uint16_t* x, size_t pitch_bytes, int64_t len, int32_t nrows, int32_t* const off[4], int32_t* const bias[4],
                       const int32_t centre[4], uint32_t input_max,
                       unsigned* range_flag /* may be NULL; else bit 0 is set if any sample of the rows exceeds input_max */, void* stream);
typedef struct {
    const uint16_t* raw; size_t pitch_bytes; int64_t ngroups; int32_t chan0; unsigned cap;
    uint8_t* lo[3]; size_t pitch[3], stride[3]; const int32_t* off[3]; uint2* exc[3]; unsigned* cnt[3]; int64_t nb[3];
    uint16_t* lo8; size_t pitch8, stride8; const int32_t* off8; uint2* exc8; unsigned* cnt8; int64_t nb8; int32_t hi8;
} aak_prep16_args;
int aak_prep16(const aak_prep16_args* a, int32_t nrows, void* stream);
int aak_bin_time16(const uint16_t* x, size_t x_pitch_bytes, uint16_t* xb, size_t xb_pitch_bytes, int32_t nchans, int64_t nbinned,
                   int32_t bin, const unsigned* only_if_cnt, unsigned only_if_above, void* stream);
int aak_corner_turn16(const uint16_t* in, size_t in_stride_bytes, uint16_t* out, size_t out_pitch_bytes, int32_t nchans, int64_t nsamp,
                      void* stream);

/* ---- K2: dedispersion --------------------------------------------------------------------------------------------
 * Tiled kernel: a CTA owns `dm_tile` (30 or 32) DM trials x T_TILE(=1024) output samples; channels stream through shared
 * memory in blocks of `chan_block` via TMA (tensor map `tmap`, 128 opaque bytes, see aa_strategy.cpp), `ring_stages`-deep
 * mbarrier ring.
 * The input exists as NCOPY = 4 (uint8) or 2 (uint16) sample-shifted copies in ONE global buffer, copy k = x[c][t+k]
 * at byte offset k*copy_stride; tmap points at the 128-byte 4-D CUtensorMap over it (HOST memory).
 * A stage in shared memory is [chan_block][NCOPY][class_wb[wcls[stage]]], and at byte chan_block*NCOPY*window_bytes the stage's
 * slice of etab.
 * etab  [ndm_tiles][nstages][chan_block][32] int32 : shared-memory byte offset of (channel, DM) inside a stage (rows of 32
 *                                                  entries, the first dm_tile are used; ndm_tiles = ceil(ndms / dm_tile))
 * x0tab [ndm_tiles][nstages*chan_block]    int32 : 16-byte aligned BYTE offset of the channel window relative to the
 *                                                  tile's first output sample */
typedef struct {
    const void* tmap;          /* HOST pointer to nclass consecutive 128-byte CUtensorMaps (copied into kernel params): map k loads
                                  windows of class_wb[k] bytes */
    int32_t nclass;            /* 1..8 window classes */
    int32_t class_wb[8];       /* window bytes of each class (multiples of 256, <= window_bytes) */
    const int32_t* wcls;       /* [nstages] class of each stage (channel block) */
    const int32_t* etab;
    const int32_t* x0tab;
    int32_t* D;                /* [ndms][pitch] */
    int64_t pitch;
    int64_t nt;                /* T_r valid outputs per row */
    int32_t ndms;
    int32_t nchans;
    int32_t chan_block;        /* 8, 4 or 2 */
    int32_t window_bytes;      /* WB: the WIDEST (copy, channel) window in shared memory, multiple of 256; sizes the ring slots */
    int32_t spill_stages;      /* carry the 16-bit lanes every this many stages: 256/chan_block (bytes), (256/bin)/chan_block (uint16) */
    int32_t in16;              /* 0: byte input (bin 1, or the offset-uint8 form of a binned input), 1: uint16 binned input */
    int32_t variant;           /* uint8 only: odd-byte lane adds as 0 = IADD3, 1 = IMAD (FMA pipe), 2 = alternating */
    int32_t ring_stages;       /* depth of the shared-memory stage ring (2..8) */
    int32_t skew_q16;          /* CTA order: time tiles skewed by skew_q16 / 65536 per DM tile (0 = plain order) */
    int32_t dm_tile;           /* DM trials per CTA: 32, or 30 (uint8, 2 trials per warp: 15 compute warps with 128 registers) */
    int32_t chan_begin, chan_end; /* sum channels [chan_begin, chan_end) only (multiples of chan_block; chan_end 0 = nchans) */
    int32_t accumulate;        /* 1: D += the partial sums (a later channel group of the same chunk), 0: D = */
    const unsigned* mode_cnt;  /* may be NULL. Else the launch returns at once unless (*mode_cnt > mode_cap) == mode_dense */
    unsigned mode_cap;
    int32_t mode_dense;
    const int32_t* bias;       /* may be NULL. Else *bias is added to every output (sum of the channel offsets) */
    int32_t dms_per_warp;      /* 2 or 4 adjacent DM trials per warp (words of equal-delay trials are reused from registers) */
} aak_dedisp_args;
int aak_dedisperse(const aak_dedisp_args* a, void* stream);
size_t aak_dedisperse_smem_bytes(int32_t chan_block, int32_t window_bytes, int32_t in16, int32_t ring_stages);
int aak_dedisperse_init(void);   /* sets the dynamic shared-memory attribute of every instantiation */

/* ---- K2b: dedispersion of a BIT plane (the low bits the half-byte form of bin 8 drops):
 *   D[i][t] += sum_{c in [chan_begin, chan_end)} bit[c][t + delay(c, i)]
 * bits [nchans][pitch_words] uint32 (bit k of word w = sample 32 w + k; readable up to (nt + max delay) / 32 + window_words + 2
 * words per row), delays [ndms][nchans] int32 (binned samples), window_words = 34 + ceil(largest delay spread inside a tile of
 * 32 trials / 32) <= 256. A CTA owns 32 trials x 1024 samples; channel blocks go through shared memory, every thread extracts its 32
 * samples of a channel with one funnel shift and adds them to bit-sliced (vertical) counters with carry-save adders: about
 * 0.3 instructions per add. Runs only if *mode_cnt <= mode_cap (NULL: always). */
int aak_dedisperse_bits(const uint32_t* bits, size_t pitch_words, const int32_t* delays, int32_t nchans, int32_t chan_begin, int32_t chan_end,
                        int32_t ndms, int64_t nt, int32_t window_words, int32_t* D, int64_t pitch, const unsigned* mode_cnt, unsigned mode_cap,
                        void* stream);
int aak_bits_init(void);         /* sets the dynamic shared-memory attribute (per device: call with the strategy's device current) */

/* One thread per output, global loads (copy 0 of the input, pitch in elements): the route for ranges whose channel window
 * does not fit shared memory, and a cross-check. delays [ndms][nchans] int32; sums channels [chan_begin, chan_end),
 * accumulate as in aak_dedisperse. */
int aak_dedisperse_naive(const void* x, size_t pitch_elems, int32_t in16, const int32_t* delays, int32_t nchans, int32_t chan_begin,
                         int32_t chan_end, int32_t ndms, int64_t nt, int32_t* D, int64_t pitch, int32_t accumulate,
                         const unsigned* mode_cnt /* may be NULL; else runs only if *mode_cnt > mode_cap */, unsigned mode_cap, void* stream);

/* ---- K0t: corner turn of a time-major chunk x_tm[t][c] into channel-major rows x[c][t] (uint8) */
int aak_corner_turn(const uint8_t* in, size_t in_stride, uint8_t* out, size_t out_pitch, int32_t nchans, int64_t nsamp, void* stream);

/* ---- K3: robust row statistics ---------------------------------------------------------------------------------
 * rows: one entry per DM row of all ranges of the chunk. stats out: per row {mu, sigma} doubles and {n, iters} */
typedef struct {
    const int32_t* D;     /* row base */
    int64_t nt;
} aak_row_desc;
int aak_row_stats(const aak_row_desc* rows, int32_t nrows, double* mu_sigma /* [nrows][2] */,
                  int64_t* n_iters /* [nrows][2] */, void* stream);

/* ---- K3w: per-width measured statistics (reading C7m): for every row of one range and every plan width w, the series
 * B_w[t] = sum_{j<w} D[t+j], t in [0, n_w), n_w = min(nt, nt_data - w + 1), is given reading C6 about the pivot p_w = B_w[0]
 * (exact integer moments, iterated 3-sigma clip, at most 8 clips). Outputs per (row, width): wstats = {mu_w, sigma_w} with
 * sigma_w = 0 when the width yields no SNR in this row (n_w < 1, constant series, degenerate clip); wpivot = p_w;
 * wlive[row] = 1 if any width of the row has sigma_w > 0. */
typedef struct {
    const int32_t* D; int64_t pitch; int64_t nt; int64_t nt_data; int32_t ndms;
    int32_t widths[16]; int32_t nwidths;
    double* wstats;       /* [ndms][nwidths][2] */
    int64_t* wpivot;      /* [ndms][nwidths] */
    int32_t* wlive;       /* [ndms] */
} aak_wstats_args;
int aak_row_width_stats(const aak_wstats_args* a, void* stream);

/* ---- K4: boxcar SNR + 3x3 peaks + candidate append ---------------------------------------------------------------- */
typedef struct {
    uint64_t sample; float dm; float snr; uint32_t width; uint32_t range; uint32_t dm_index;
} aak_candidate;
typedef struct {
    const int32_t* D; int64_t pitch; int64_t nt; int32_t ndms; int32_t bin; int32_t range_index;
    int64_t nt_data;           /* samples present per row (>= nt): boxcars may extend to here, candidates start below nt */
    double dm_low, dm_step;
    const double* mu_sigma;    /* [ndms][2] for this range */
    uint64_t chunk_start;
    int32_t widths[16]; int32_t nwidths;
    double threshold;
    aak_candidate* cands; unsigned long long* counter; unsigned long long capacity;
    unsigned* range_flag;      /* may be NULL. Else bit 0 is set if wmax * max|D - D[0]| of a row reaches 2^31: the int32 boxcar sums are
                                  then not trustworthy (plans whose sample maximum is too large for a plan-time guarantee) */
    /* reading C7m (per-width measured statistics), all NULL for reading C7: the outputs of aak_row_width_stats for this range */
    const double* wstats; const int64_t* wpivot; const int32_t* wlive;
} aak_sps_args;
int aak_sps_peaks(const aak_sps_args* a, void* stream);
int aak_sps_init(void);

/* ---- K5 (test hook): per-row moments sum_t D, sum_t t*D ------------------------------------------------------------ */
int aak_row_moments(const int32_t* D, int64_t pitch, int64_t nt, int32_t ndms, long long* sum_d, long long* sum_td,
                    void* stream);

/* ---- K0: integer-add peak microbenchmark ----------------------------------------------------------------------------
 * mode 0: IADD3-only chains, mode 1: IADD3 + IMAD mixed chains. cycles_out [gridDim] receives per-CTA cycle counts. */
int aak_peak_iadd(int32_t mode, int32_t iters, int32_t grid, int32_t threads, uint32_t* sink, unsigned long long* cycles_out,
                  void* stream);
#define AAK_PEAK_ADDS_PER_THREAD_ITER 16

#ifdef __cplusplus
}
#endif
#endif
