/*
 * aa_internal.h — host-side objects behind the opaque handles of include/aa.h.
 * plan = the user's parameters; strategy = immutable GPU configuration + chunk cursor;
 * Arena = the memory manager from which every device buffer is carved once (§2.3).
 */
#ifndef AA_INTERNAL_H
#define AA_INTERNAL_H

#include <cuda.h>
#include <cuda_runtime.h>

#include <cstdint>
#include <string>
#include <vector>

#include "../../include/aa.h"
#include "aa_kernels.h"

namespace aa {

void set_error(const char* fmt, ...);
aa_status cuda_fail(cudaError_t e, const char* what);

constexpr int kDmTile = 32;       /* row length of K2's offset table = the largest DM tile (must match k_dedisp.cu) */
constexpr int kTTile = 1024;
constexpr int kMaxGroups = 4;
constexpr unsigned kExcCap = 1u << 20;   /* exception records per (bin, channel group) */      /* channel groups of a pipelined (not prefetched) chunk copy */
constexpr size_t kSlack = 64 * 1024;   /* readable bytes after every input buffer (TMA windows over-read) */

inline size_t round_up(size_t v, size_t m) { return (v + m - 1) / m * m; }

struct Plan {
    int32_t nchans = 0;
    std::vector<double> freq;
    double tsamp = 0.0;
    std::vector<aa_dm_range> ranges;
    std::vector<int32_t> widths;
    float threshold = 0.f;
    int32_t layout = 0;           /* aa_input_layout */
    bool boxcar_overlap = false;  /* reading C3x */
    bool per_width = false;       /* reading C7m */
    int32_t input_bits = 8;       /* 8: uint8 samples, 16: uint16 samples <= input_max */
    uint32_t input_max = 255;
};

/* Single-allocation bump allocator over caller- or library-owned device memory. */
struct Arena {
    uint8_t* base = nullptr;
    size_t size = 0, used = 0;
    bool dry = false;             /* dry run: only measure */
    void* take(size_t bytes) {
        const size_t off = round_up(used, 256);
        used = off + bytes;
        if (dry || used > size) return nullptr;
        return base + off;
    }
};

/* Tiling of K2 for one range in one input format (uint8 samples, or uint16 binned samples). */
struct K2Plan {
    int32_t in16 = 0, esz = 1, spw = 4, ncopy = 4;
    int32_t chan_block = 8, window_bytes = 0, spill_stages = 0, nstages = 0;
    int32_t skew_q16 = 0;                                     /* CTA rasterisation skew (time tiles per DM tile, 16.16) */
    int32_t dm_tile = 32, ndm_tiles = 0;                      /* DM trials per CTA (32 or 30) and the number of DM tiles */
    int32_t dms_per_warp = 2, variant = 1, ring_stages = 3;   /* K2 tuning chosen by the strategy */
    int32_t* d_etab = nullptr;
    int32_t* d_x0tab = nullptr;
    /* Window classes: a channel block (stage) loads a window only as wide as ITS channels' delay spread inside a DM tile needs
     * (the spread grows down the band), rounded up to 256 bytes; window_bytes is the widest (it sizes the shared-memory ring).
     * One tensor map per distinct width (at most kMaxWinClasses; widths in between are rounded up to the next class). */
    int32_t nclass = 1;
    int32_t class_wb[8] = {0};
    std::vector<int32_t> wcls;    /* [nstages] class of each stage (host copy) */
    int32_t* d_wcls = nullptr;
    CUtensorMap maps[8];          /* 4-D window maps over the NCOPY-copy input buffer of this format, one per class */
};
constexpr int kMaxWinClasses = 8;

struct Range : K2Plan {           /* the base is the range's main plan: uint8 for bin 1, uint16 for binned ranges */
    aa_dm_range r;
    int32_t index = 0;
    int64_t max_delay = 0;        /* binned samples */
    int64_t nt_full = 0;          /* T_r of a full chunk */
    int32_t extra = 0;            /* E: samples dedispersed beyond T_r (reading C3x), 0 by default */
    int64_t pitch = 0;            /* D row pitch, elements */
    std::vector<int32_t> delays;  /* [ndms][nchans], binned samples (host) */
    int32_t* d_D = nullptr;
    size_t first_row = 0;         /* index of this range's first row in the row tables */
    bool naive = false;           /* the tile window does not fit shared memory: one-thread-per-output kernel on a delay table */
    int32_t* d_delays = nullptr;  /* [ndms][nchans] (naive route only) */
    bool has_lo = false;          /* the offset-uint8 route (k_misc.cu "Offset-uint8 form") with its own tiling: bin 2 / 4 of an 8-bit
                                     plan, bin 1 / 2 / 4 of a 16-bit plan */
    K2Plan lo;
    bool half = false;            /* 8-bit plan, bin 8: the offset-uint8 plan reads the HALF-BYTE form (k_bits.cu): sums are doubled and
                                     the dropped low bits are dedispersed as a bit plane */
    int32_t bits_ww = 0;          /* window words of the bit-plane kernel */
    bool main_exc = false;        /* 16-bit plan, bin 8: the main (uint16) plan reads the offset-uint16 form (offsets + exceptions) */
    bool dense_naive = false;     /* 16-bit plan: exception-heavy chunks take the global-memory kernel on the plain binned samples */
};

struct Chunk { uint64_t start, len, n_out; };

struct Strategy {
    bool ready = false;           /* false for a host-only strategy made by aa_strategy_plan */
    Plan plan;
    std::vector<double> k;        /* delay constants, samples per unit DM (unbinned) */
    uint64_t nsamp_total = 0;
    int32_t B = 1;
    int64_t S = 0, L = 0, n_out = 0;
    std::vector<Chunk> chunks;
    std::vector<Range> ranges;
    size_t nrows = 0;

    /* device memory */
    Arena arena;
    bool owns_arena = false;
    int32_t esz_in = 1;                      /* bytes per input sample */
    int32_t lo16_max = 1023;                 /* window of the offset-uint16 form */
    size_t in_pitch = 0;                     /* bytes per channel row of the raw chunk */
    uint8_t* d_raw[2] = {nullptr, nullptr};  /* [0]: the H2D target of a channel-major plan / the corner-turn target; [1] is unused: K2 never
                                                reads the raw chunk (K1 does), so the next chunk's copy may start as soon as K1 is done */
    uint8_t* d_stage[2] = {nullptr, nullptr};   /* time-major plans: H2D targets [L][stage_stride]; d_raw[0] is the corner-turn target */
    size_t stage_stride = 0;
    /* Input forms of K2. Every form of a time-binning factor lives in ONE buffer of nchans rows of 4P bytes (P = samples per
     * row rounded up to 256): a byte form is 4 sample-shifted copies of P bytes (copy k at + k P), a uint16 form 2 copies of
     * 2P bytes (copy k at + 2 k P). The offset-uint8 form of bin 2 / 4 and their uint16 form (the route of exception-heavy
     * chunks) share the rows: a channel group takes one route or the other, never both. */
    uint8_t* d_x4 = nullptr;                 /* bin 1: the 4 sample-shifted copies of the uint8 chunk */
    size_t x4_pitch = 0, x4_stride = 0;      /* bytes between channel rows (4P) and between copies (P) */
    bool need_u8_copies = false;
    size_t xb_pitch[9] = {0};                /* uint16 ELEMENTS between channel rows (2P), indexed by bin */
    uint16_t* d_xb[9] = {nullptr};           /* binned input indexed by bin: copy 0, then copy 1 at +xb_stride bytes (2P) */
    size_t xb_stride[9] = {0};
    /* offset-uint8 form of the binned inputs (bin 2, 4): 4 shifted byte copies, per-channel offsets, exceptions */
    uint8_t* d_lo[9] = {nullptr};            /* copy k at + k*lo_stride bytes (P); the same memory as d_xb of the bin */
    size_t lo_pitch[9] = {0}, lo_stride[9] = {0};   /* bytes between channel rows (4P) and between copies (P) */
    int32_t* d_off[9] = {nullptr};           /* [nchans] */
    uint2* d_exc[9] = {nullptr};             /* [kMaxGroups][exc_cap] */
    unsigned* d_exc_cnt[9] = {nullptr};      /* [kMaxGroups] exception counters, then [kMaxGroups] int32 biases (one memset clears both) */
    unsigned exc_limit[9] = {0};             /* a group with more exceptions than this takes the uint16 route */
    uint32_t* d_bits[9] = {nullptr};         /* bit plane of the half-byte form (bin 8): [nchans][bits_pitch] words */
    size_t bits_pitch[9] = {0};
    double* d_k = nullptr;                   /* delay constants on the device (exception scatter) */
    bool d_k_needed = false;
    aak_row_desc* d_rows[2] = {nullptr, nullptr};   /* [0] full chunk geometry, [1] last (short) chunk */
    double* d_mu_sigma = nullptr;            /* [nrows][2] */
    int64_t* d_n_iters = nullptr;            /* [nrows][2] */
    double* d_wstats = nullptr;              /* reading C7m: [nrows][nwidths][2] = mu_w, sigma_w */
    int64_t* d_wpivot = nullptr;             /* [nrows][nwidths] p_w */
    int32_t* d_wlive = nullptr;              /* [nrows] */
    aak_candidate* d_cands = nullptr;
    unsigned long long* d_counter = nullptr;
    long long* d_moments = nullptr;          /* [2][max ndms] */
    size_t max_candidates = 0;

    /* the device this strategy was set up on (arena, streams, events and kernel attributes all belong to it) */
    int device = -1;
    int nsm = 0;                                      /* its SM count */

    /* streams / events */
    cudaStream_t compute = nullptr, copy = nullptr;
    cudaStream_t aux = nullptr;                       /* library-owned: every other DM range's K2 runs here, so that the tail
                                                         wave of one range overlaps the first wave of the next */
    cudaStream_t d2h = nullptr;                       /* library-owned: candidate records leave the device here */
    cudaEvent_t ev_fork = nullptr, ev_join = nullptr;
    bool owns_compute = false, owns_copy = false;
    cudaEvent_t ev_copied[2] = {nullptr, nullptr};    /* chunk landed in d_raw[b] (copy stream) */
    cudaEvent_t ev_raw_free[2] = {nullptr, nullptr};  /* last reader of d_raw[b] finished (compute stream) */
    cudaEvent_t ev_group[kMaxGroups] = {nullptr};     /* channel group g of the current chunk landed (copy stream) */
    cudaEvent_t ev_count = nullptr;                   /* candidate counter copied to the host */
    cudaEvent_t ev_t[6] = {nullptr};                  /* timing marks on the compute stream */
    cudaEvent_t ev_h2d[2] = {nullptr, nullptr};       /* timing marks on the copy stream */
    bool h2d_timed = false;

    /* cursor / state */
    int64_t next_chunk = 0;
    int32_t shard_rank = 0, shard_world = 1;   /* aa_strategy_shard */
    int64_t current_chunk = -1;        /* chunk whose D is on the device */
    bool pending_sps = false;
    int64_t raw_holds[2] = {-1, -1};   /* which chunk each raw buffer holds (or is receiving) */
    bool raw_free_recorded[2] = {false, false};
    bool harvest_pending = false;
    int64_t harvest_chunk = -1;
    aa_status sticky = AA_OK;
    uint64_t launches = 0;
    bool timed = false, stats_timed = false;

    /* host results */
    unsigned long long* h_counter = nullptr;    /* pinned */
    std::vector<aa_candidate> cands;
    std::vector<aa_cluster> clusters;
    uint64_t true_count = 0;
    bool overflow = false;
    std::vector<int32_t> host_row;
};

/* aa_strategy.cpp */
int64_t delay_of(const Strategy& s, const Range& rg, int32_t chan, int32_t dm_index);

}  // namespace aa

struct aa_plan { aa::Plan p; };
struct aa_strategy { aa::Strategy s; };

#endif
