/*
 * aa_strategy.cpp — strategy object: "how input data are split and processed on the GPU" (§3.1).
 * Host-only planning (delays, chunk geometry, kernel tiling, offset tables, tensor maps) plus the memory manager
 * (§2.3): every device buffer is carved from ONE arena here; aa_run_* never allocates.
 *
 * Arithmetic of the delays is BASELINE.json north_star, evaluated in IEEE double in the order of DESIGN.md reading C2
 * (this file is compiled with -ffp-contract=off):
 *     k_c = (4.148808e3 * (1/f_c^2 - 1/f_0^2)) / tsamp;  DM_i = dm_low + i*dm_step;  delay = llround((k_c*DM_i)/bin)
 */
#include <algorithm>
#include <cmath>
#include <cstdio>
#include <cstdlib>
#include <cstring>
#include <new>

#include "aa_internal.h"

namespace aa {

typedef CUresult (*EncodeTiledFn)(CUtensorMap*, CUtensorMapDataType, cuuint32_t, void*, const cuuint64_t*, const cuuint64_t*,
                                  const cuuint32_t*, const cuuint32_t*, CUtensorMapInterleave, CUtensorMapSwizzle,
                                  CUtensorMapL2promotion, CUtensorMapFloatOOBfill);

static EncodeTiledFn encode_fn() {
    static EncodeTiledFn fn = nullptr;
    if (!fn) {
        void* p = nullptr;
        cudaDriverEntryPointQueryResult q;
        if (cudaGetDriverEntryPoint("cuTensorMapEncodeTiled", &p, cudaEnableDefault, &q) == cudaSuccess && q == cudaDriverEntryPointSuccess)
            fn = (EncodeTiledFn)p;
    }
    return fn;
}

static double dm_of(const aa_dm_range& r, int32_t i) { return r.dm_low + (double)i * r.dm_step; }

static int64_t delay_calc(double k_c, double dm, int32_t bin) { return (int64_t)llround((k_c * dm) / (double)bin); }

int64_t delay_of(const Strategy& s, const Range& rg, int32_t chan, int32_t dm_index) {
    return delay_calc(s.k[(size_t)chan], dm_of(rg.r, dm_index), rg.r.bin);
}

/* Channel rows of the NCOPY shifted copies seen as overlapping 256-byte segments: a {256, nseg, NCOPY, 1} box lands as
 * NCOPY linear windows of window_bytes each (k_dedisp.cu). Rows are pitch_bytes apart, the copies of a row copy_stride. */
static bool make_window_map1(CUtensorMap* map, void* base, size_t row_bytes, size_t pitch_bytes, size_t copy_stride, int32_t ncopy,
                             int32_t nchans, int32_t window_bytes) {
    EncodeTiledFn enc = encode_fn();
    if (!enc) { set_error("aa_strategy_setup: cuTensorMapEncodeTiled is not available from this driver"); return false; }
    const cuuint32_t nseg = (cuuint32_t)(window_bytes / 256);
    cuuint64_t dims[4] = {(cuuint64_t)row_bytes, nseg, (cuuint64_t)ncopy, (cuuint64_t)nchans};   /* row_bytes: one copy of one channel */
    cuuint64_t strides[3] = {256, (cuuint64_t)copy_stride, (cuuint64_t)pitch_bytes};
    cuuint32_t box[4] = {256, nseg, (cuuint32_t)ncopy, 1};
    cuuint32_t es[4] = {1, 1, 1, 1};
    const CUresult r = enc(map, CU_TENSOR_MAP_DATA_TYPE_UINT8, 4, base, dims, strides, box, es, CU_TENSOR_MAP_INTERLEAVE_NONE,
                           CU_TENSOR_MAP_SWIZZLE_NONE, CU_TENSOR_MAP_L2_PROMOTION_L2_256B, CU_TENSOR_MAP_FLOAT_OOB_FILL_NONE);
    if (r != CUDA_SUCCESS) { set_error("aa_strategy_setup: cuTensorMapEncodeTiled failed with CUresult %d", (int)r); return false; }
    return true;
}

/* The maps of all window classes of one K2 plan. */
static bool make_window_maps(K2Plan& p, void* base, size_t row_bytes, size_t pitch_bytes, size_t copy_stride, int32_t ncopy, int32_t nchans) {
    for (int k = 0; k < p.nclass; ++k)
        if (!make_window_map1(&p.maps[k], base, row_bytes, pitch_bytes, copy_stride, ncopy, nchans, p.class_wb[k])) return false;
    return true;
}

/* Everything that depends on the chunk length L. Carves (or, on a dry arena, only measures) the device buffers. */
static void carve(Strategy& s, int64_t L, bool two_stage) {
    Arena& a = s.arena;
    a.used = 0;
    const size_t esz = (size_t)s.esz_in;
    s.in_pitch = round_up((size_t)L * esz, 256);
    const size_t raw_bytes = (size_t)s.plan.nchans * s.in_pitch + kSlack;
    /* ONE raw buffer also when chunks are double-buffered: only K1 reads it (3 ms of a 200 ms step), so the copy of the next
     * chunk starts when K1 of this one is done and still overlaps the whole of K2 */
    s.d_raw[0] = (uint8_t*)a.take(raw_bytes);
    s.d_raw[1] = nullptr;
    s.d_stage[0] = s.d_stage[1] = nullptr;
    if (s.plan.layout == AA_LAYOUT_TIME_MAJOR) {
        /* the chunk lands time-major in a staging buffer (two when chunks are double-buffered); one channel-major buffer */
        s.stage_stride = round_up((size_t)s.plan.nchans * esz, 16);
        const size_t stage_bytes = (size_t)L * s.stage_stride + kSlack;
        s.d_stage[0] = (uint8_t*)a.take(stage_bytes);
        s.d_stage[1] = two_stage ? (uint8_t*)a.take(stage_bytes) : nullptr;
    }
    /* input forms: nchans rows of 4P bytes per binning factor (aa_internal.h), kSlack readable bytes after the last row */
    s.d_x4 = nullptr; s.x4_stride = s.x4_pitch = 0;
    for (int b = 1; b <= 8; b *= 2) {
        bool used = false, lo = false, sparse = false;
        int64_t nd = 0;
        for (const Range& rg : s.ranges) {
            if (rg.r.bin != b) continue;
            used = true;
            lo = lo || rg.has_lo;
            if (rg.has_lo || rg.main_exc) { sparse = true; nd += rg.r.ndms; }
        }
        const size_t P = used ? round_up((size_t)(L / b), 256) : 0;
        uint8_t* base = used ? (uint8_t*)a.take((size_t)s.plan.nchans * 4 * P + kSlack) : nullptr;
        if (b == 1 && s.plan.input_bits == 8) {       /* plain bytes: the 4 sample-shifted copies of the chunk itself */
            s.d_x4 = base; s.x4_pitch = 4 * P; s.x4_stride = P;
            s.d_xb[b] = nullptr; s.d_lo[b] = nullptr;
            continue;
        }
        s.d_xb[b] = (uint16_t*)base;
        s.xb_pitch[b] = 2 * P;                     /* elements: a row is 2 copies of 2P bytes */
        s.xb_stride[b] = 2 * P;                    /* bytes */
        s.d_lo[b] = lo ? base : nullptr;           /* the same rows as 4 copies of P bytes */
        s.lo_pitch[b] = lo ? 4 * P : 0;
        s.lo_stride[b] = lo ? P : 0;
        s.d_off[b] = sparse ? (int32_t*)a.take((size_t)s.plan.nchans * 4) : nullptr;
        s.d_exc[b] = sparse ? (uint2*)a.take((size_t)kMaxGroups * kExcCap * sizeof(uint2)) : nullptr;
        s.d_exc_cnt[b] = sparse ? (unsigned*)a.take(2 * kMaxGroups * 4) : nullptr;
        /* Route test = an exception RATE. The scatter costs one atomic per (exception, trial) at a measured 2.7e10 atomics/s; the
         * dense route costs the range about 2.9e-14 s more per add (16 against 30 Tadd/s measured). Both grow with the number of
         * trials, so the break-even is a fraction of the bin's samples, 2.9e-14 x 2.7e10 = 8e-4; half of it is allowed (Gaussian
         * noise: 2e-8 at bin 2, 6e-5 at bin 4, 5e-3 at bin 8). The earlier absolute budget of 1e8 atomics sent the bin-4 range of
         * the low-frequency configuration (1.3e5 exceptions x 2500 trials) down the uint16 route: 257 ms instead of ~150. */
        (void)nd;
        s.exc_limit[b] = sparse ? (unsigned)std::min<double>((double)kMaxGroups * kExcCap, std::max(1.0, 4.0e-4 * (double)s.plan.nchans * (double)(L / b))) : 0;
        if (sparse && !s.d_k_needed) s.d_k_needed = true;
        bool half = false;
        for (const Range& rg : s.ranges) half = half || (rg.r.bin == b && rg.half);
        s.bits_pitch[b] = half ? round_up(P / 32 + 1024 + 64, 64) : 0;        /* + the widest window the bit-plane kernel may read */
        s.d_bits[b] = half ? (uint32_t*)a.take((size_t)s.plan.nchans * s.bits_pitch[b] * 4) : nullptr;
    }
    s.d_k = s.d_k_needed ? (double*)a.take((size_t)s.plan.nchans * 8) : nullptr;
    const int64_t n_out = L - s.S;
    for (Range& rg : s.ranges) {
        rg.nt_full = n_out / rg.r.bin;
        rg.pitch = (int64_t)round_up((size_t)(rg.nt_full + rg.extra), 128);
        rg.d_D = (int32_t*)a.take((size_t)rg.r.ndms * (size_t)rg.pitch * 4);
        rg.d_delays = (rg.naive || rg.dense_naive || rg.half) ? (int32_t*)a.take((size_t)rg.r.ndms * s.plan.nchans * 4) : nullptr;
        rg.d_etab = (int32_t*)a.take((size_t)rg.ndm_tiles * rg.nstages * rg.chan_block * kDmTile * 4);   /* rg. = the main plan */
        rg.d_x0tab = (int32_t*)a.take((size_t)rg.ndm_tiles * rg.nstages * rg.chan_block * 4);
        rg.d_wcls = (int32_t*)a.take((size_t)rg.nstages * 4);
        if (rg.has_lo) {
            rg.lo.d_etab = (int32_t*)a.take((size_t)rg.lo.ndm_tiles * rg.lo.nstages * rg.lo.chan_block * kDmTile * 4);
            rg.lo.d_x0tab = (int32_t*)a.take((size_t)rg.lo.ndm_tiles * rg.lo.nstages * rg.lo.chan_block * 4);
            rg.lo.d_wcls = (int32_t*)a.take((size_t)rg.lo.nstages * 4);
        }
    }
    s.d_rows[0] = (aak_row_desc*)a.take(s.nrows * sizeof(aak_row_desc));
    s.d_rows[1] = (aak_row_desc*)a.take(s.nrows * sizeof(aak_row_desc));
    s.d_mu_sigma = (double*)a.take(s.nrows * 2 * sizeof(double));
    s.d_n_iters = (int64_t*)a.take(s.nrows * 2 * sizeof(int64_t));
    const size_t nwd = s.plan.widths.size();
    s.d_wstats = s.plan.per_width ? (double*)a.take(s.nrows * nwd * 2 * sizeof(double)) : nullptr;
    s.d_wpivot = s.plan.per_width ? (int64_t*)a.take(s.nrows * nwd * sizeof(int64_t)) : nullptr;
    s.d_wlive = s.plan.per_width ? (int32_t*)a.take(s.nrows * sizeof(int32_t)) : nullptr;
    s.d_cands = (aak_candidate*)a.take(s.max_candidates * sizeof(aak_candidate));
    s.d_counter = (unsigned long long*)a.take(256);
    int32_t maxnd = 0;
    for (const Range& rg : s.ranges) maxnd = std::max(maxnd, rg.r.ndms);
    s.d_moments = (long long*)a.take((size_t)2 * maxnd * sizeof(long long));
    a.used = round_up(a.used, 256);
}

static std::vector<Chunk> make_chunks(uint64_t nsamp, int64_t B, int64_t S, int64_t L) {
    std::vector<Chunk> v;
    const int64_t n_out = L - S;
    const int64_t usable = (int64_t)(nsamp / (uint64_t)B) * B;
    int64_t start = 0;
    while (start < usable) {
        const int64_t len = std::min<int64_t>(L, usable - start);
        if (len <= S) break;
        v.push_back(Chunk{(uint64_t)start, (uint64_t)len, (uint64_t)(len - S)});
        if (len < L) break;
        start += n_out;
    }
    return v;
}

/* Tiling and offset tables of K2 for one range in one input format (in16: uint16 binned samples, else bytes). */
static bool plan_format(const Strategy& s, const Range& rg, K2Plan& p, int in16, int carry_channels, std::vector<int32_t>& etab,
                        std::vector<int32_t>& x0tab) {
    const int32_t C = s.plan.nchans, nd = rg.r.ndms;
    p.in16 = in16; p.esz = in16 ? 2 : 1; p.spw = 4 / p.esz; p.ncopy = p.spw;
    /* uint8 samples: 15 compute warps x 2 trials (+ the producer = 16 warps, 128 registers per thread, 30 trials per CTA):
     * measured 216.6 -> 204.9 ms on SKA-like against 16 + 1 warps at 96 registers (11 or 7 warps are slower again, and
     * 14 + 1 warps change nothing for the uint16 kernel, which is bound by shared-memory bytes, not by loads in flight);
     * binned uint16 samples: 16 warps x (4 adjacent trials, half the tile), 32 trials per CTA */
    p.dm_tile = in16 ? kDmTile : 30;
    p.ndm_tiles = (nd + p.dm_tile - 1) / p.dm_tile;
    /* in-tile delay spread of every channel (largest over the DM tiles); the widest window: T_TILE + spread + alignment
     * residue (< 16 bytes) */
    std::vector<int64_t> spread((size_t)C, 0);
    int64_t omax = 0;
    for (int32_t t = 0; t < p.ndm_tiles; ++t) {
        const int32_t i0 = t * p.dm_tile, i1 = std::min(nd - 1, i0 + p.dm_tile - 1);
        const int32_t* a = rg.delays.data() + (size_t)i0 * C;
        const int32_t* b = rg.delays.data() + (size_t)i1 * C;
        for (int32_t c = 0; c < C; ++c) spread[(size_t)c] = std::max<int64_t>(spread[(size_t)c], (int64_t)b[c] - a[c]);
    }
    for (int32_t c = 0; c < C; ++c) omax = std::max(omax, spread[(size_t)c]);
    auto window_of = [&](int64_t o) { return (int32_t)round_up((size_t)((kTTile + o + 16 / p.esz) * p.esz), 256); };
    const int64_t wsamp = kTTile + omax + 16 / p.esz;
    p.window_bytes = (int32_t)round_up((size_t)(wsamp * p.esz), 256);
    if (p.window_bytes > 65536) return false;
    /* the largest channel block that still leaves a 2-deep ring, then the deepest ring (<= 5) that fits: measured on the
     * low-frequency config (wide windows), 8 channels x 2 stages beats 4 x 4 by 6 %; ring depth alone moves < 1 % */
    p.chan_block = 0;
    p.ring_stages = 2;
    for (int cb = 8; cb >= 2; cb /= 2)
        if (aak_dedisperse_smem_bytes(cb, p.window_bytes, p.in16, 2) <= 227 * 1024) { p.chan_block = cb; break; }
    if (!p.chan_block) return false;
    for (int n = 3; n <= 5; ++n)
        if (aak_dedisperse_smem_bytes(p.chan_block, p.window_bytes, p.in16, n) <= 227 * 1024) p.ring_stages = n;
    /* measured on B200 (profiles/): binned ranges are shared-memory bound and gain 13 % from 4 trials per warp with
     * register reuse; the uint8 ranges are issue bound and lose 7 % to the extra branches, so they keep 2 trials per warp
     * with the odd-byte adds on the FMA pipe */
    p.dms_per_warp = p.in16 ? 4 : 2;
    p.variant = 1;
    /* rasterisation skew = the channel-averaged delay growth per DM tile, in time tiles (only worth it above ~1/4 tile) */
    {
        double sum = 0.0;
        const int32_t* last = rg.delays.data() + (size_t)(nd - 1) * C;
        for (int32_t c = 0; c < C; ++c) sum += (double)last[c];
        const double per_tile = (sum / C) / std::max(1, p.ndm_tiles - 1) / (double)kTTile;
        p.skew_q16 = per_tile >= 0.25 ? (int32_t)std::min(per_tile * 65536.0, 2.0e9) : 0;
    }
    p.nstages = (C + p.chan_block - 1) / p.chan_block;
    /* 16-bit lanes are carried every 65536 / (largest sample value + 1) channels: bytes 256, uint16 sums of b bytes 256/b,
     * the offset-uint16 form 65536 / (lo16_max + 1) */
    p.spill_stages = carry_channels / p.chan_block;
    if (p.spill_stages < 1) return false;
    const int32_t CB = p.chan_block, Cpad = p.nstages * CB;
    /* window classes: the width each channel block needs, at most kMaxWinClasses distinct values (rounded up to the next kept one) */
    std::vector<int32_t> need((size_t)p.nstages, 256);
    for (int32_t st = 0; st < p.nstages; ++st) {
        int64_t o = 0;
        for (int32_t c = st * CB; c < std::min(C, (st + 1) * CB); ++c) o = std::max(o, spread[(size_t)c]);
        need[(size_t)st] = window_of(o);
    }
    {
        std::vector<int32_t> vals(need);
        std::sort(vals.begin(), vals.end());
        vals.erase(std::unique(vals.begin(), vals.end()), vals.end());
        while ((int)vals.size() > kMaxWinClasses) {                 /* drop the value whose removal rounds the fewest bytes up */
            size_t best = 0; int64_t cost = -1;
            for (size_t k = 0; k + 1 < vals.size(); ++k) {
                int64_t n = 0;
                for (int32_t v : need) if (v == vals[k]) ++n;
                const int64_t cst = n * (int64_t)(vals[k + 1] - vals[k]);
                if (cost < 0 || cst < cost) { cost = cst; best = k; }
            }
            for (int32_t& v : need) if (v == vals[best]) v = vals[best + 1];
            vals.erase(vals.begin() + (ptrdiff_t)best);
        }
        p.nclass = (int32_t)vals.size();
        for (int k = 0; k < 8; ++k) p.class_wb[k] = k < p.nclass ? vals[(size_t)k] : 0;
        p.wcls.assign((size_t)p.nstages, 0);
        for (int32_t st = 0; st < p.nstages; ++st)
            p.wcls[(size_t)st] = (int32_t)(std::lower_bound(vals.begin(), vals.end(), need[(size_t)st]) - vals.begin());
    }
    etab.assign((size_t)p.ndm_tiles * Cpad * kDmTile, 0);
    x0tab.assign((size_t)p.ndm_tiles * Cpad, 0);
    for (int32_t t = 0; t < p.ndm_tiles; ++t) {
        const int32_t i0 = t * p.dm_tile;
        for (int32_t c = 0; c < Cpad; ++c) {
            int32_t* e = etab.data() + ((size_t)t * Cpad + c) * kDmTile;     /* [tile][stage][c_local][m] */
            const int32_t cl = c % CB;
            const int32_t WB = need[(size_t)(c / CB)];                         /* this channel block's window */
            if (c >= C) {                                                   /* padding channel: TMA zero-fills it */
                for (int m = 0; m < kDmTile; ++m) e[m] = cl * p.ncopy * WB;
                continue;
            }
            const int64_t d0 = rg.delays[(size_t)i0 * C + c];
            const int64_t xs = d0 * p.esz, xa = xs & ~(int64_t)15;
            const int64_t res = (xs - xa) / p.esz;                          /* samples folded into the offsets */
            x0tab[(size_t)t * Cpad + c] = (int32_t)xa;
            for (int m = 0; m < kDmTile; ++m) {
                const int32_t i = std::min(nd - 1, i0 + m);
                const int64_t o = (int64_t)rg.delays[(size_t)i * C + c] - d0 + res;
                const int64_t copy = o & (p.spw - 1);
                e[m] = (int32_t)((cl * p.ncopy + copy) * WB + (o - copy) * p.esz);
            }
        }
    }
    return true;
}

/* Delays and the K2 plan(s) of one range (host side). Returns false with the error set. */
static bool plan_range(Strategy& s, Range& rg, std::vector<int32_t>& etab, std::vector<int32_t>& x0tab,
                       std::vector<int32_t>& etab_lo, std::vector<int32_t>& x0tab_lo) {
    const int32_t C = s.plan.nchans, nd = rg.r.ndms;
    rg.delays.resize((size_t)nd * C);
    for (int32_t i = 0; i < nd; ++i) {
        const double dm = dm_of(rg.r, i);
        int32_t* row = rg.delays.data() + (size_t)i * C;
        for (int32_t c = 0; c < C; ++c) {
            const int64_t d = delay_calc(s.k[(size_t)c], dm, rg.r.bin);
            if (d < 0 || d > 0x3fffffff) { set_error("aa_strategy_setup: delay(%d, range %d, %d) = %lld out of range", c, rg.index, i, (long long)d); return false; }
            row[c] = (int32_t)d;
        }
    }
    rg.max_delay = rg.delays[(size_t)(nd - 1) * C + (C - 1)];
    auto no_main = [&]() {                 /* no tiled plan on the main input form */
        rg.in16 = (rg.r.bin > 1 || s.plan.input_bits == 16); rg.esz = rg.in16 ? 2 : 1; rg.spw = 4 / rg.esz; rg.ncopy = rg.spw;
        rg.dm_tile = kDmTile; rg.ndm_tiles = 0; rg.nstages = 0; rg.chan_block = 8; rg.window_bytes = 0;
        etab.clear(); x0tab.clear();
    };
    rg.naive = false; rg.has_lo = false; rg.main_exc = false; rg.dense_naive = false; rg.half = false;
    if (s.plan.input_bits == 16) {
        /* 16-bit samples (k_input16.cu): bin 1 / 2 / 4 ride the byte path on the offset-uint8 form, bin 8 the uint16 path on the
         * offset-uint16 form; a chunk with too many exceptions, or a range whose window does not fit, takes the global-memory
         * kernel on the plain binned samples */
        rg.dense_naive = true;
        if (rg.r.bin <= 4) {
            no_main();
            rg.has_lo = plan_format(s, rg, rg.lo, 0, 256, etab_lo, x0tab_lo);
            if (!rg.has_lo) { rg.naive = true; rg.dense_naive = false; }
        } else {
            if (plan_format(s, rg, rg, 1, 65536 / (s.lo16_max + 1), etab, x0tab)) rg.main_exc = true;
            else { no_main(); rg.naive = true; rg.dense_naive = false; }
        }
        return true;
    }
    if (!plan_format(s, rg, rg, rg.r.bin > 1, rg.r.bin > 1 ? 256 / rg.r.bin : 256, etab, x0tab)) {
        /* a window that does not fit shared memory is not an error of the plan: such a range (DM step very coarse for the
         * band) takes the one-thread-per-output kernel on a device delay table; everything else about it stays the same */
        no_main();
        rg.naive = true;
        return true;
    }
    /* bin 2 and 4 also get the offset-uint8 route (half the shared-memory bytes per add); the uint16 plan above stays as
     * the route for chunks with too many exceptions. */
    rg.has_lo = (rg.r.bin == 2 || rg.r.bin == 4 || rg.r.bin == 8);
    if (rg.has_lo && !plan_format(s, rg, rg.lo, 0, 256, etab_lo, x0tab_lo)) rg.has_lo = false;
    if (rg.has_lo && rg.r.bin == 8) {
        /* bin 8: the byte plan reads the half-byte form, its low bits go through the bit-plane kernel (k_bits.cu): tiles of 32
         * trials, window = 34 words + the largest delay spread inside such a tile */
        int64_t sp = 0;
        for (int32_t i0 = 0; i0 < nd; i0 += 32) {
            const int32_t i1 = std::min(nd - 1, i0 + 31);
            for (int32_t c = 0; c < C; ++c) sp = std::max<int64_t>(sp, (int64_t)rg.delays[(size_t)i1 * C + c] - rg.delays[(size_t)i0 * C + c]);
        }
        rg.bits_ww = (int32_t)(34 + (sp + 31) / 32);
        if (rg.bits_ww > 256) rg.has_lo = false;
        else { rg.half = true; rg.lo.variant = 3; }
    }
    return true;
}

/* Host-only part of the setup: delays, overlap, tiling, tables, chunk length under `limit` bytes (0 = unlimited). */
static aa_status plan_host(aa_strategy* h, const aa_plan* plan, uint64_t nsamp_total, size_t limit, size_t max_candidates,
                           uint64_t chunk_len_hint, std::vector<std::vector<int32_t>>& etabs, std::vector<std::vector<int32_t>>& x0tabs,
                           size_t* bytes_needed) {
    Strategy& s = h->s;
    s.plan = plan->p;
    s.nsamp_total = nsamp_total;
    s.max_candidates = max_candidates;
    const int32_t C = s.plan.nchans;

    /* delays and overlap (reading C2, C3) */
    s.k.resize((size_t)C);
    const double f0 = s.plan.freq[0];
    for (int32_t c = 0; c < C; ++c) {
        const double f = s.plan.freq[(size_t)c];
        s.k[(size_t)c] = (4.148808e3 * (1.0 / (f * f) - 1.0 / (f0 * f0))) / s.plan.tsamp;
    }
    s.B = 1;
    for (const aa_dm_range& r : s.plan.ranges) s.B = std::max(s.B, r.bin);
    s.esz_in = s.plan.input_bits == 16 ? 2 : 1;
    s.lo16_max = C <= 16384 ? 1023 : 255;      /* nchans * lo16_max < 2^24: the packed accumulators of the uint16 kernel */
    s.ranges.resize(s.plan.ranges.size());
    etabs.resize(2 * s.ranges.size()); x0tabs.resize(2 * s.ranges.size());      /* [r]: main plan, [nranges + r]: offset-uint8 plan */
    int64_t smax = 0;
    s.nrows = 0;
    for (size_t r = 0; r < s.ranges.size(); ++r) {
        Range& rg = s.ranges[r];
        rg.r = s.plan.ranges[r];
        rg.index = (int32_t)r;
        if (!plan_range(s, rg, etabs[r], x0tabs[r], etabs[s.ranges.size() + r], x0tabs[s.ranges.size() + r])) return AA_ERR_INVALID_ARG;
        rg.extra = s.plan.boxcar_overlap ? s.plan.widths.back() - 1 : 0;       /* reading C3x */
        smax = std::max<int64_t>(smax, (rg.max_delay + rg.extra) * rg.r.bin);
        rg.first_row = s.nrows;
        s.nrows += (size_t)rg.r.ndms;
        if (rg.r.bin == 1 && s.plan.input_bits == 8) s.need_u8_copies = true;
    }
    /* a naive range reads the uint16 form of its bin on every chunk, so that bin keeps no offset-uint8 route */
    for (const Range& nv : s.ranges)
        if (nv.naive) for (Range& rg : s.ranges) if (rg.r.bin == nv.r.bin) rg.has_lo = false;
    /* the uint16 input of a bin is written per BIN (only for exception-heavy chunks once the bin has an offset-uint8 buffer),
     * while its ranges pick their route per RANGE: a range without the offset-uint8 plan (its byte window did not fit) would
     * then read a uint16 buffer that a sparse chunk never filled. So a bin keeps the route only if all its ranges have it. */
    for (const Range& nl : s.ranges)
        if (!nl.has_lo) for (Range& rg : s.ranges) if (rg.r.bin == nl.r.bin) rg.has_lo = false;
    for (Range& rg : s.ranges) if (!rg.has_lo) rg.half = false;
    /* 16-bit plans: a bin's rows hold EITHER its offset form (with the plain samples written only for exception-heavy chunks) OR,
     * if one of its ranges has only the global-memory route, the plain samples always: then every range of the bin takes it */
    if (s.plan.input_bits == 16)
        for (const Range& nv : s.ranges)
            if (nv.naive)
                for (Range& rg : s.ranges)
                    if (rg.r.bin == nv.r.bin && !rg.naive) {
                        rg.naive = true; rg.dense_naive = false; rg.has_lo = false; rg.main_exc = false;
                        rg.ndm_tiles = 0; rg.nstages = 0; etabs[(size_t)rg.index].clear(); x0tabs[(size_t)rg.index].clear();
                    }
    s.S = (int64_t)round_up((size_t)smax, (size_t)s.B);
    const int64_t usable = (int64_t)(nsamp_total / (uint64_t)s.B) * s.B;
    if (usable <= s.S) {
        set_error("aa_strategy_setup: nsamp_total = %llu is not longer than the maximum delay %lld samples", (unsigned long long)nsamp_total, (long long)s.S);
        return AA_ERR_INVALID_ARG;
    }

    /* chunk length under the budget (reading C3): whole observation if it fits, else the largest power of two */
    s.arena.dry = true; s.arena.base = nullptr; s.arena.size = 0;
    auto need = [&](int64_t L) { const bool two = (L < usable); carve(s, L, two); return s.arena.used; };   /* two: double-buffered staging */
    /* a chunk row stays below 2^28 samples: the sample field of an exception record (k_common.cuh) has 28 bits */
    const int64_t Lmax = (((int64_t)1 << 28) - 1) / s.B * s.B;
    auto fits = [&](int64_t L) { return L <= Lmax && (!limit || need(L) <= limit); };
    int64_t L = 0;
    if (chunk_len_hint) {
        L = (int64_t)chunk_len_hint;
        if (L % s.B || L <= s.S) { set_error("aa_strategy_setup: chunk_len_hint = %lld must be a multiple of %d and > overlap %lld", (long long)L, s.B, (long long)s.S); return AA_ERR_INVALID_ARG; }
        if (L > usable) L = usable;
        if (L > Lmax) { set_error("aa_strategy_setup: chunk_len_hint = %lld exceeds the largest chunk of %lld samples", (long long)L, (long long)Lmax); return AA_ERR_INVALID_ARG; }
        if (limit && need(L) > limit) { set_error("aa_strategy_setup: chunk_len_hint = %lld needs %zu bytes, budget is %zu", (long long)L, need(L), limit); return AA_ERR_BUDGET_TOO_SMALL; }
    } else if (fits(usable)) {
        L = usable;
    } else {
        int64_t p2 = 1;
        while (p2 <= s.S) p2 <<= 1;
        if (p2 % s.B) p2 = (int64_t)round_up((size_t)p2, (size_t)s.B);
        if (p2 >= usable || !fits(p2)) {
            if (p2 > Lmax) { set_error("aa_strategy_setup: the maximum delay (%lld samples) exceeds the largest chunk of %lld samples", (long long)s.S, (long long)Lmax); return AA_ERR_INVALID_ARG; }
            set_error("aa_strategy_setup: budget of %zu bytes is too small: the smallest chunk (%lld samples, overlap %lld) needs %zu bytes",
                      limit, (long long)p2, (long long)s.S, need(std::min(p2, usable)));
            return AA_ERR_BUDGET_TOO_SMALL;
        }
        while (p2 * 2 < usable && fits(p2 * 2)) p2 *= 2;
        L = p2;
        /* then grow in eighths of that power of two while the arena still fits: every chunk recomputes S samples of
         * overlap, so longer chunks waste less (600 s stream under 40 GB: L = 2^19 -> 3 * 2^18, 19 -> 13 chunks) */
        const int64_t step = (int64_t)round_up((size_t)std::max<int64_t>(p2 / 8, s.B), (size_t)s.B);
        while (L + step < usable && fits(L + step)) L += step;
    }
    s.L = L;
    s.n_out = L - s.S;
    s.chunks = make_chunks(nsamp_total, s.B, s.S, L);
    carve(s, L, s.chunks.size() > 1);
    *bytes_needed = s.arena.used;
    return AA_OK;
}

}  // namespace aa

using namespace aa;

extern "C" aa_status aa_strategy_plan(aa_strategy** out, const aa_plan* plan, uint64_t nsamp_total, size_t budget_bytes,
                                      size_t max_candidates, uint64_t chunk_len_hint) {
    if (!out) { set_error("aa_strategy_plan: out is NULL"); return AA_ERR_INVALID_ARG; }
    *out = nullptr;
    if (!plan) { set_error("aa_strategy_plan: plan is NULL (configure a plan first)"); return AA_ERR_NOT_READY; }
    if (max_candidates < 1) { set_error("aa_strategy_plan: max_candidates must be >= 1"); return AA_ERR_INVALID_ARG; }
    aa_strategy* h = new (std::nothrow) aa_strategy();
    if (!h) { set_error("aa_strategy_plan: out of host memory"); return AA_ERR_INTERNAL; }
    std::vector<std::vector<int32_t>> etabs, x0tabs;
    size_t bytes = 0;
    const aa_status st = plan_host(h, plan, nsamp_total, budget_bytes, max_candidates, chunk_len_hint, etabs, x0tabs, &bytes);
    if (st != AA_OK) { delete h; return st; }
    h->s.arena.size = 0;
    h->s.ready = false;
    *out = h;
    return AA_OK;
}

extern "C" aa_status aa_strategy_setup(aa_strategy** out, const aa_plan* plan, uint64_t nsamp_total, void* device_arena,
                                       size_t arena_bytes, size_t budget_bytes, void* compute_stream, void* copy_stream,
                                       size_t max_candidates, uint64_t chunk_len_hint) {
    if (!out) { set_error("aa_strategy_setup: out is NULL"); return AA_ERR_INVALID_ARG; }
    *out = nullptr;
    if (!plan) { set_error("aa_strategy_setup: plan is NULL (configure and bind a plan first)"); return AA_ERR_NOT_READY; }
    if (max_candidates < 1) { set_error("aa_strategy_setup: max_candidates must be >= 1"); return AA_ERR_INVALID_ARG; }
    if (device_arena && ((uintptr_t)device_arena & 255)) { set_error("aa_strategy_setup: device_arena must be 256-byte aligned"); return AA_ERR_INVALID_ARG; }
    aa_strategy* h = new (std::nothrow) aa_strategy();
    if (!h) { set_error("aa_strategy_setup: out of host memory"); return AA_ERR_INTERNAL; }
    Strategy& s = h->s;
    auto fail = [&](aa_status st) { aa_strategy_destroy(h); return st; };
    size_t limit = budget_bytes;
    if (device_arena) limit = limit ? std::min(limit, arena_bytes) : arena_bytes;
    if (!device_arena && limit == 0) {
        size_t fr = 0, tot = 0;
        cudaError_t e0 = cudaMemGetInfo(&fr, &tot);
        if (e0 != cudaSuccess) return fail(cuda_fail(e0, "cudaMemGetInfo"));
        limit = fr - std::min<size_t>(fr / 16, (size_t)1 << 30);
    }
    std::vector<std::vector<int32_t>> etabs, x0tabs;
    size_t bytes_needed = 0;
    {
        const aa_status st = plan_host(h, plan, nsamp_total, limit, max_candidates, chunk_len_hint, etabs, x0tabs, &bytes_needed);
        if (st != AA_OK) return fail(st);
    }
    const int32_t C = s.plan.nchans;
    const int64_t L = s.L;
    const bool two_stage = s.chunks.size() > 1;

    /* the single allocation (north_star "one allocation per run") */
    if (device_arena) {
        if (bytes_needed > arena_bytes) { set_error("aa_strategy_setup: arena of %zu bytes is too small, %zu needed", arena_bytes, bytes_needed); return fail(AA_ERR_BUDGET_TOO_SMALL); }
        s.arena.base = (uint8_t*)device_arena; s.arena.size = arena_bytes; s.owns_arena = false;
    } else {
        void* p = nullptr;
        cudaError_t e = cudaMalloc(&p, bytes_needed);
        if (e != cudaSuccess) { cudaGetLastError(); set_error("aa_strategy_setup: cudaMalloc of %zu bytes failed: %s", bytes_needed, cudaGetErrorString(e)); return fail(AA_ERR_BUDGET_TOO_SMALL); }
        s.arena.base = (uint8_t*)p; s.arena.size = bytes_needed; s.owns_arena = true;
    }
    s.arena.dry = false;
    carve(s, L, two_stage);

    /* streams, events, pinned counter */
    cudaError_t e;
    if ((e = cudaGetDevice(&s.device)) != cudaSuccess) return fail(cuda_fail(e, "cudaGetDevice"));
    if ((e = cudaDeviceGetAttribute(&s.nsm, cudaDevAttrMultiProcessorCount, s.device)) != cudaSuccess || s.nsm < 1) return fail(cuda_fail(e, "cudaDeviceGetAttribute (SM count)"));
    if (compute_stream) s.compute = (cudaStream_t)compute_stream;
    else { if ((e = cudaStreamCreateWithFlags(&s.compute, cudaStreamNonBlocking)) != cudaSuccess) return fail(cuda_fail(e, "cudaStreamCreate")); s.owns_compute = true; }
    if (copy_stream) s.copy = (cudaStream_t)copy_stream;
    else { if ((e = cudaStreamCreateWithFlags(&s.copy, cudaStreamNonBlocking)) != cudaSuccess) return fail(cuda_fail(e, "cudaStreamCreate")); s.owns_copy = true; }
    for (int b = 0; b < 2; ++b) {
        if ((e = cudaEventCreateWithFlags(&s.ev_copied[b], cudaEventDisableTiming)) != cudaSuccess) return fail(cuda_fail(e, "cudaEventCreate"));
        if ((e = cudaEventCreateWithFlags(&s.ev_raw_free[b], cudaEventDisableTiming)) != cudaSuccess) return fail(cuda_fail(e, "cudaEventCreate"));
        if ((e = cudaEventCreate(&s.ev_h2d[b])) != cudaSuccess) return fail(cuda_fail(e, "cudaEventCreate"));
    }
    if ((e = cudaEventCreateWithFlags(&s.ev_count, cudaEventDisableTiming)) != cudaSuccess) return fail(cuda_fail(e, "cudaEventCreate"));
    if ((e = cudaStreamCreateWithFlags(&s.aux, cudaStreamNonBlocking)) != cudaSuccess) return fail(cuda_fail(e, "cudaStreamCreate"));
    if ((e = cudaStreamCreateWithFlags(&s.d2h, cudaStreamNonBlocking)) != cudaSuccess) return fail(cuda_fail(e, "cudaStreamCreate"));
    if ((e = cudaEventCreateWithFlags(&s.ev_fork, cudaEventDisableTiming)) != cudaSuccess) return fail(cuda_fail(e, "cudaEventCreate"));
    if ((e = cudaEventCreateWithFlags(&s.ev_join, cudaEventDisableTiming)) != cudaSuccess) return fail(cuda_fail(e, "cudaEventCreate"));
    for (int g = 0; g < kMaxGroups; ++g)
        if ((e = cudaEventCreateWithFlags(&s.ev_group[g], cudaEventDisableTiming)) != cudaSuccess) return fail(cuda_fail(e, "cudaEventCreate"));
    for (int i = 0; i < 6; ++i)
        if ((e = cudaEventCreate(&s.ev_t[i])) != cudaSuccess) return fail(cuda_fail(e, "cudaEventCreate"));
    if ((e = cudaHostAlloc((void**)&s.h_counter, 64, cudaHostAllocDefault)) != cudaSuccess) return fail(cuda_fail(e, "cudaHostAlloc"));
    *s.h_counter = 0;
    if ((e = (cudaError_t)aak_dedisperse_init()) != cudaSuccess) return fail(cuda_fail(e, "kernel attribute setup (dedispersion)"));
    if ((e = (cudaError_t)aak_sps_init()) != cudaSuccess) return fail(cuda_fail(e, "kernel attribute setup (sps)"));
    if ((e = (cudaError_t)aak_bits_init()) != cudaSuccess) return fail(cuda_fail(e, "kernel attribute setup (bit plane)"));

    /* upload tables, build tensor maps and row descriptors */
    std::vector<aak_row_desc> rows_full(s.nrows), rows_last(s.nrows);
    const Chunk& last = s.chunks.back();
    for (size_t r = 0; r < s.ranges.size(); ++r) {
        Range& rg = s.ranges[r];
        if ((rg.naive || rg.dense_naive || rg.half) && (e = cudaMemcpyAsync(rg.d_delays, rg.delays.data(), rg.delays.size() * 4, cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "delay table upload"));
        if (rg.naive) { for (int32_t i = 0; i < rg.r.ndms; ++i) { const int32_t* base = rg.d_D + (size_t)i * (size_t)rg.pitch; rows_full[rg.first_row + i] = aak_row_desc{base, rg.nt_full}; rows_last[rg.first_row + i] = aak_row_desc{base, (int64_t)(last.n_out / (uint64_t)rg.r.bin)}; } continue; }
        const bool has_main = rg.ndm_tiles > 0;
        if (has_main && (e = cudaMemcpyAsync(rg.d_etab, etabs[r].data(), etabs[r].size() * 4, cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "table upload"));
        if (has_main && (e = cudaMemcpyAsync(rg.d_x0tab, x0tabs[r].data(), x0tabs[r].size() * 4, cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "table upload"));
        if (has_main && (e = cudaMemcpyAsync(rg.d_wcls, rg.wcls.data(), rg.wcls.size() * 4, cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "table upload"));
        if (rg.has_lo) {
            const size_t n = s.ranges.size();
            if ((e = cudaMemcpyAsync(rg.lo.d_etab, etabs[n + r].data(), etabs[n + r].size() * 4, cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "table upload"));
            if ((e = cudaMemcpyAsync(rg.lo.d_x0tab, x0tabs[n + r].data(), x0tabs[n + r].size() * 4, cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "table upload"));
            if ((e = cudaMemcpyAsync(rg.lo.d_wcls, rg.lo.wcls.data(), rg.lo.wcls.size() * 4, cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "table upload"));
            if (!make_window_maps(rg.lo, s.d_lo[rg.r.bin], s.lo_stride[rg.r.bin], s.lo_pitch[rg.r.bin], s.lo_stride[rg.r.bin], 4, C)) return fail(AA_ERR_CUDA);
        }
        if (!has_main) {
        } else if (rg.in16) {
            if (!make_window_maps(rg, s.d_xb[rg.r.bin], s.xb_stride[rg.r.bin], s.xb_pitch[rg.r.bin] * 2, s.xb_stride[rg.r.bin], 2, C)) return fail(AA_ERR_CUDA);
        } else {
            if (!make_window_maps(rg, s.d_x4, s.x4_stride, s.x4_pitch, s.x4_stride, 4, C)) return fail(AA_ERR_CUDA);
        }
        for (int32_t i = 0; i < rg.r.ndms; ++i) {
            const int32_t* base = rg.d_D + (size_t)i * (size_t)rg.pitch;
            rows_full[rg.first_row + i] = aak_row_desc{base, rg.nt_full};
            rows_last[rg.first_row + i] = aak_row_desc{base, (int64_t)(last.n_out / (uint64_t)rg.r.bin)};
        }
    }
    if ((e = cudaMemcpyAsync(s.d_rows[0], rows_full.data(), s.nrows * sizeof(aak_row_desc), cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "row table upload"));
    if ((e = cudaMemcpyAsync(s.d_rows[1], rows_last.data(), s.nrows * sizeof(aak_row_desc), cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "row table upload"));
    if ((e = cudaMemsetAsync(s.d_counter, 0, 256, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "cudaMemsetAsync"));
    if (s.d_k && (e = cudaMemcpyAsync(s.d_k, s.k.data(), (size_t)C * 8, cudaMemcpyHostToDevice, s.compute)) != cudaSuccess) return fail(cuda_fail(e, "delay constants upload"));
    if ((e = cudaStreamSynchronize(s.compute)) != cudaSuccess) return fail(cuda_fail(e, "strategy upload"));   /* host tables go out of scope */
    s.ready = true;
    *out = h;
    return AA_OK;
}

extern "C" void aa_strategy_destroy(aa_strategy* h) {
    if (!h) return;
    Strategy& s = h->s;
    if (s.compute) cudaStreamSynchronize(s.compute);
    if (s.copy) cudaStreamSynchronize(s.copy);
    for (int b = 0; b < 2; ++b) {
        if (s.ev_copied[b]) cudaEventDestroy(s.ev_copied[b]);
        if (s.ev_raw_free[b]) cudaEventDestroy(s.ev_raw_free[b]);
        if (s.ev_h2d[b]) cudaEventDestroy(s.ev_h2d[b]);
    }
    if (s.aux) { cudaStreamSynchronize(s.aux); cudaStreamDestroy(s.aux); }
    if (s.d2h) { cudaStreamSynchronize(s.d2h); cudaStreamDestroy(s.d2h); }
    if (s.ev_fork) cudaEventDestroy(s.ev_fork);
    if (s.ev_join) cudaEventDestroy(s.ev_join);
    if (s.ev_count) cudaEventDestroy(s.ev_count);
    for (int g = 0; g < kMaxGroups; ++g) if (s.ev_group[g]) cudaEventDestroy(s.ev_group[g]);
    for (int i = 0; i < 6; ++i) if (s.ev_t[i]) cudaEventDestroy(s.ev_t[i]);
    if (s.owns_compute && s.compute) cudaStreamDestroy(s.compute);
    if (s.owns_copy && s.copy) cudaStreamDestroy(s.copy);
    if (s.h_counter) cudaFreeHost(s.h_counter);
    if (s.owns_arena && s.arena.base) cudaFree(s.arena.base);
    delete h;
}

extern "C" aa_status aa_strategy_get_info(const aa_strategy* h, aa_strategy_info* out) {
    if (!h || !out) { set_error("aa_strategy_get_info: NULL argument"); return h ? AA_ERR_INVALID_ARG : AA_ERR_NOT_READY; }
    const Strategy& s = h->s;
    out->ready = s.ready ? 1 : 0;
    out->nchans = s.plan.nchans; out->nranges = (int32_t)s.ranges.size(); out->nwidths = (int32_t)s.plan.widths.size();
    out->max_bin = s.B; out->nsamp_total = (int64_t)s.nsamp_total; out->overlap = s.S; out->chunk_len = s.L; out->n_out = s.n_out;
    out->nchunks = (int64_t)s.chunks.size(); out->next_chunk = s.next_chunk;
    out->shard_rank = s.shard_rank; out->shard_world = s.shard_world;
    out->arena_bytes_used = s.arena.used; out->arena_bytes_total = s.arena.size; out->max_candidates = s.max_candidates;
    out->owns_arena = s.owns_arena ? 1 : 0;
    out->input_layout = s.plan.layout;
    out->input_bits = s.plan.input_bits; out->input_max = s.plan.input_max;
    return AA_OK;
}

extern "C" aa_status aa_strategy_get_range_info(const aa_strategy* h, int32_t range, aa_range_info* out) {
    if (!h) { set_error("aa_strategy_get_range_info: strategy is NULL"); return AA_ERR_NOT_READY; }
    if (!out || range < 0 || range >= (int32_t)h->s.ranges.size()) { set_error("aa_strategy_get_range_info: range %d out of bounds", range); return AA_ERR_INVALID_ARG; }
    const Range& rg = h->s.ranges[(size_t)range];
    out->ndms = rg.r.ndms; out->bin = rg.r.bin; out->nt = rg.nt_full; out->row_pitch = rg.pitch; out->max_delay = rg.max_delay;
    const K2Plan& kp = (rg.ndm_tiles > 0 || !rg.has_lo) ? static_cast<const K2Plan&>(rg) : rg.lo;     /* the tiled plan that exists */
    out->dm_tile = kp.dm_tile; out->t_tile = kTTile; out->chan_block = kp.chan_block; out->window = kp.window_bytes;
    out->boxcar_extra = rg.extra;
    return AA_OK;
}

extern "C" aa_status aa_strategy_get_chunk(const aa_strategy* h, int64_t chunk, uint64_t* start, uint64_t* len, uint64_t* n_out) {
    if (!h) { set_error("aa_strategy_get_chunk: strategy is NULL"); return AA_ERR_NOT_READY; }
    if (chunk < 0 || chunk >= (int64_t)h->s.chunks.size()) { set_error("aa_strategy_get_chunk: chunk %lld out of bounds (nchunks = %zu)", (long long)chunk, h->s.chunks.size()); return AA_ERR_INVALID_ARG; }
    const Chunk& c = h->s.chunks[(size_t)chunk];
    if (start) *start = c.start;
    if (len) *len = c.len;
    if (n_out) *n_out = c.n_out;
    return AA_OK;
}

extern "C" aa_status aa_strategy_get_delay(const aa_strategy* h, int32_t range, int32_t dm_index, int32_t chan, int64_t* delay) {
    if (!h) { set_error("aa_strategy_get_delay: strategy is NULL"); return AA_ERR_NOT_READY; }
    const Strategy& s = h->s;
    if (!delay || range < 0 || range >= (int32_t)s.ranges.size() || chan < 0 || chan >= s.plan.nchans || dm_index < 0 ||
        dm_index >= s.ranges[(size_t)range].r.ndms) { set_error("aa_strategy_get_delay: index out of bounds"); return AA_ERR_INVALID_ARG; }
    *delay = s.ranges[(size_t)range].delays[(size_t)dm_index * s.plan.nchans + chan];
    return AA_OK;
}

extern "C" size_t aa_strategy_describe(const aa_strategy* h, char* buf, size_t buflen) {
    if (!h) return 0;
    const Strategy& s = h->s;
    std::string o;
    char line[512];
    snprintf(line, sizeof line, "strategy: nchans=%d nsamp=%llu B=%d overlap S=%lld chunk L=%lld n_out=%lld nchunks=%zu\n", s.plan.nchans,
             (unsigned long long)s.nsamp_total, s.B, (long long)s.S, (long long)s.L, (long long)s.n_out, s.chunks.size());
    o += line;
    snprintf(line, sizeof line, "arena: %zu bytes used of %zu (%s), input pitch %zu, H2D buffers %d, uint8 shifted copies %s\n", s.arena.used,
             s.arena.size, s.owns_arena ? "library-owned, one cudaMalloc" : "caller-owned", s.in_pitch, s.d_stage[0] ? (s.d_stage[1] ? 2 : 1) : 1,
             s.need_u8_copies ? "4" : "none");
    o += line;
    for (const Range& rg : s.ranges) {
        snprintf(line, sizeof line,
                 "range %d: dm_low=%g step=%g ndms=%d bin=%d max_delay=%lld T=%lld pitch=%lld | tile %dx%d chan_block=%d window=%dB stages=%d "
                 "dm_tiles=%d spill/%d smem=%zuB\n",
                 rg.index, rg.r.dm_low, rg.r.dm_step, rg.r.ndms, rg.r.bin, (long long)rg.max_delay, (long long)rg.nt_full, (long long)rg.pitch,
                 rg.dm_tile, kTTile, rg.chan_block, rg.window_bytes, rg.nstages, rg.ndm_tiles, rg.spill_stages,
                 aak_dedisperse_smem_bytes(rg.chan_block, rg.window_bytes, rg.in16, rg.ring_stages));
        o += line;
        {
            const K2Plan& kp = (rg.ndm_tiles > 0 || !rg.has_lo) ? static_cast<const K2Plan&>(rg) : rg.lo;
            if (kp.nclass > 1 && !kp.wcls.empty()) {
                double sum = 0.0;
                for (int32_t c : kp.wcls) sum += kp.class_wb[c];
                snprintf(line, sizeof line, "         %d window classes, %d..%d bytes, %.0f on average over the channel blocks\n", kp.nclass, kp.class_wb[0],
                         kp.class_wb[kp.nclass - 1], sum / (double)kp.wcls.size());
                o += line;
            }
        }
        if (rg.naive) o += "         tile window does not fit shared memory: one-thread-per-output kernel on a device delay table\n";
        if (rg.half) o += "         the offset-uint8 route reads the half-byte form; the dropped low bits are dedispersed as a bit plane\n";
        if (rg.main_exc) o += "         the uint16 plan reads the offset-uint16 form (per-channel offsets + exceptions)\n";
        if (rg.dense_naive) o += "         exception-heavy chunks take the one-thread-per-output kernel on the plain binned samples\n";
        if (rg.has_lo) {
            snprintf(line, sizeof line, "         offset-uint8 route: chan_block=%d window=%dB stages=%d ring=%d exception limit %u per chunk\n",
                     rg.lo.chan_block, rg.lo.window_bytes, rg.lo.nstages, rg.lo.ring_stages, s.exc_limit[rg.r.bin]);
            o += line;
        }
    }
    for (size_t j = 0; j < s.chunks.size() && j < 4; ++j) {
        snprintf(line, sizeof line, "chunk %zu: start=%llu len=%llu n_out=%llu\n", j, (unsigned long long)s.chunks[j].start,
                 (unsigned long long)s.chunks[j].len, (unsigned long long)s.chunks[j].n_out);
        o += line;
    }
    if (s.chunks.size() > 4) {
        const Chunk& c = s.chunks.back();
        snprintf(line, sizeof line, "... chunk %zu: start=%llu len=%llu n_out=%llu\n", s.chunks.size() - 1, (unsigned long long)c.start,
                 (unsigned long long)c.len, (unsigned long long)c.n_out);
        o += line;
    }
    if (buf && buflen) { const size_t n = std::min(buflen - 1, o.size()); memcpy(buf, o.data(), n); buf[n] = 0; }
    return o.size() + 1;
}
