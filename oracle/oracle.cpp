/*
 * oracle/oracle.cpp — the ORACLE: a plain, slow, single-threaded CPU statement of what the hot path
 * computes (incoherent dedispersion + single-pulse search). TEST INFRASTRUCTURE ONLY.
 *
 *   * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs may
 *     build, load or call anything in oracle/. The product (paper_1912_07704_b200/, include/) never does.
 *   * It shares no code, header, table or constant generator with the CUDA path; neither includes
 *     nor imports the other. Inputs come from datagen/ (which holds none of this arithmetic).
 *   * The method is exact (brute force), so each function is the plain definition written out, in
 *     int64 / __int128 / IEEE double, compiled with -O2 -ffp-contract=off (no fused multiply-add).
 *
 * Authority. /root/reference/PAPER.md gives no formula (it is an API paper): it fixes only that data are
 * "dedispersed and analysed entirely on the GPU" and that SPS "uses boxcar filters and peak-finding to
 * maximise signal-to-noise" (§1). The formulas are BASELINE.json `north_star`:
 *   D[dm][t] = sum_c x[c][t + delay(c,dm)],
 *   delay = round(4.148808e3 * DM * (f_c^-2 - f_top^-2) / tsamp),  DM ranges decimating by 1/2/4/8,
 *   SPS: boxcars of widths 1..W, robust per-DM mean and sigma -> SNR, local peaks above a threshold.
 * Wherever both are silent this file follows the readings C1..C9 of SURVEY.md §8(c), restated with the
 * changes listed in DESIGN.md "Readings".
 *
 * Pin status (tests/test_oracle_pins.py, -m "not gpu"):
 *   delays            pinned: 60-digit decimal evaluation of the north_star formula + SURVEY §8(c) values
 *   binning           pinned: constant input, sum conservation (8- and 16-bit input; the 16-bit entry also against numpy
 *                             reshape-sums and, through dedispersion, the pure-Python brute force and DM 0 = channel sum)
 *   dedispersion      pinned: DM=0 = channel sum, pure-Python brute force, constant input, impulse response,
 *                             all-rows moment identity, injected-pulse recovery
 *   row statistics    pinned for the definition of (n, S1, S2) -> (mu, sigma) (exact rational checks, Gaussian
 *                             closed form 0.98485*sigma, outlier rejection, shuffle invariance);
 *                     the CONSTANTS 3.0 (clip) and 8 (iteration cap) are conventions: "parity unpinned"
 *   boxcar / SNR      pinned: direct summation, hand-worked rational example, injected-pulse SNR closed form
 *   peaks             pinned on hand-built maps; the plateau tie rule and strict '>' at the threshold are
 *                             conventions: "parity unpinned" beyond self-consistency
 *   delay table       pinned: entry by entry against orc_delay and the golden delays (test_delay_table_*)
 *   candidate record  pinned: pulses injected at known unbinned samples in a bin-4 range and in later chunks
 *   per-width stats   pinned: w = 1 equals C7 bit for bit, hand-worked rational example, white-noise closed form
 *                             sigma_w = 0.98485 sigma sqrt(w), AR(1) closed form where sqrt(w) scaling is wrong by 2x,
 *                             invariance under a constant shift of D
 */
#include <cmath>
#include <cstdint>
#include <cstddef>
#include <cstring>
#include <vector>

typedef __int128 i128;

extern "C" {

/* ---- C2: delay -------------------------------------------------------------------------------------
 * north_star: delay = round(4.148808e3 * DM * (f_c^-2 - f_top^-2) / tsamp), f in MHz, tsamp in s.
 * Reading C2: evaluated in IEEE double in exactly this order; channel 0 is f_top;
 * a range with time bin b uses the delay in BINNED samples, llround( (k_c*DM) / b ). */
void orc_delay_constants(int32_t nchans, const double* freq_mhz, double tsamp_s, double* k_out) {
    const double f0 = freq_mhz[0];
    for (int32_t c = 0; c < nchans; ++c) {
        const double f = freq_mhz[c];
        k_out[c] = (4.148808e3 * (1.0 / (f * f) - 1.0 / (f0 * f0))) / tsamp_s;
    }
}

double orc_dm(double dm_low, double dm_step, int32_t i) {   /* DM_i = dm_low + i*dm_step, never accumulated */
    return dm_low + (double)i * dm_step;
}

int64_t orc_delay(double k_c, double dm, int32_t bin) {
    return (int64_t)llround((k_c * dm) / (double)bin);   /* round half away from zero */
}

/* Table form of orc_delay for one range: out[i][c] = orc_delay(k[c], orc_dm(dm_low, dm_step, i), bin), i in [i0, i1).
 * A plain loop over the function above (no arithmetic of its own); lets tests build whole delay tables quickly. */
void orc_delay_table(const double* k, int32_t nchans, double dm_low, double dm_step, int32_t bin, int32_t i0, int32_t i1,
                     int64_t* out) {
    for (int32_t i = i0; i < i1; ++i) {
        const double dm = orc_dm(dm_low, dm_step, i);
        for (int32_t c = 0; c < nchans; ++c) out[(size_t)(i - i0) * (size_t)nchans + (size_t)c] = orc_delay(k[c], dm, bin);
    }
}

/* ---- C4: time binning (reading: SUM of b consecutive samples, no division, held in uint16) -----------
 * out[c][t'] = sum_{j<b} x[c][start + b*t' + j],  t' in [0, nbinned) */
void orc_bin(const uint8_t* x, size_t row_stride, int32_t nchans, int64_t start, int64_t nbinned, int32_t b,
             uint16_t* out) {
    for (int32_t c = 0; c < nchans; ++c) {
        const uint8_t* row = x + (size_t)c * row_stride + start;
        uint16_t* o = out + (size_t)c * (size_t)nbinned;
        for (int64_t t = 0; t < nbinned; ++t) {
            uint32_t s = 0;
            for (int32_t j = 0; j < b; ++j) s += row[(int64_t)b * t + j];
            o[t] = (uint16_t)s;
        }
    }
}

/* The same sum for 16-bit input samples (PAPER.md:47 step 1 "telescope data, metadata": back-ends deliver 8- or
 * 16-bit samples). row_stride in BYTES. The caller guarantees b * max(x) <= 65535 so that a sum fits the uint16 it is held in
 * (reading C4w: the plan states the largest sample value; the Python wrapper checks the data). */
void orc_bin16(const uint16_t* x, size_t row_stride_bytes, int32_t nchans, int64_t start, int64_t nbinned, int32_t b,
               uint16_t* out) {
    for (int32_t c = 0; c < nchans; ++c) {
        const uint16_t* row = (const uint16_t*)((const uint8_t*)x + (size_t)c * row_stride_bytes) + start;
        uint16_t* o = out + (size_t)c * (size_t)nbinned;
        for (int64_t t = 0; t < nbinned; ++t) {
            uint32_t s = 0;
            for (int32_t j = 0; j < b; ++j) s += row[(int64_t)b * t + j];
            o[t] = (uint16_t)s;
        }
    }
}

/* ---- C5: dedispersion (north_star: D[dm][t] = sum over channels c of x[c][t + delay(c,dm)]) ----------
 * xb is the binned chunk [nchans][nbinned]; rows i in [i0, i1) of the range (dm_low, dm_step, bin);
 * D is [(i1-i0)][T] int64. The caller guarantees T + delay(C-1, i1-1) <= nbinned (C3). */
void orc_dedisperse(const uint16_t* xb, int64_t nbinned, int32_t nchans, const double* k,
                    double dm_low, double dm_step, int32_t bin, int32_t i0, int32_t i1, int64_t T, int64_t* D) {
    for (int32_t i = i0; i < i1; ++i) {
        int64_t* row = D + (size_t)(i - i0) * (size_t)T;
        for (int64_t t = 0; t < T; ++t) row[t] = 0;
        const double dm = orc_dm(dm_low, dm_step, i);
        for (int32_t c = 0; c < nchans; ++c) {
            const int64_t d = orc_delay(k[c], dm, bin);
            const uint16_t* src = xb + (size_t)c * (size_t)nbinned + d;
            for (int64_t t = 0; t < T; ++t) row[t] += src[t];
        }
    }
}

/* ---- C6: robust per-row statistics (north_star: "robust per-DM mean and sigma") ----------------------
 * Reading C6: iterated 3-sigma clipping on exact integer sums about the pivot p = D[0]:
 *   keep = all; repeat (at most 8 clips): n,S1,S2 over keep; mu = p + S1/n; var = (n*S2 - S1^2)/n^2 (population);
 *   sigma = sqrt(var); lo = ceil(mu - 3 sigma), hi = floor(mu + 3 sigma); keep' = {t: lo <= D[t] <= hi};
 *   stop when (n,S1,S2) do not change. mu, sigma are those of the final keep set. No truncation correction.
 * out_int = {n, iterations, lo, hi}; returns 0, or 1 if the final keep set is degenerate (n == 0). */
static void orc_moments(const int64_t* D, int64_t T, int64_t p, int64_t lo, int64_t hi, int clip,
                        int64_t* n, i128* s1, i128* s2) {
    int64_t cnt = 0; i128 a = 0, b = 0;
    for (int64_t t = 0; t < T; ++t) {
        if (clip && (D[t] < lo || D[t] > hi)) continue;
        const i128 d = (i128)(D[t] - p);
        ++cnt; a += d; b += d * d;
    }
    *n = cnt; *s1 = a; *s2 = b;
}

static void orc_mu_sigma(int64_t p, int64_t n, i128 s1, i128 s2, double* mu, double* sigma) {
    const i128 num = (i128)n * s2 - s1 * s1;                  /* n^2 * variance, exact, >= 0 */
    *mu = (double)p + (double)s1 / (double)n;
    const double var = (double)num / ((double)n * (double)n);
    *sigma = sqrt(var);
}

int32_t orc_row_stats(const int64_t* D, int64_t T, double* mu_out, double* sigma_out, int64_t* out_int) {
    const int64_t p = D[0];
    int64_t n, lo = 0, hi = 0; i128 s1, s2; double mu, sigma; int32_t it = 0;
    orc_moments(D, T, p, 0, 0, 0, &n, &s1, &s2);
    orc_mu_sigma(p, n, s1, s2, &mu, &sigma);
    for (it = 0; it < 8; ++it) {
        lo = (int64_t)ceil(mu - 3.0 * sigma);
        hi = (int64_t)floor(mu + 3.0 * sigma);
        int64_t n2; i128 a2, b2;
        orc_moments(D, T, p, lo, hi, 1, &n2, &a2, &b2);
        if (n2 == 0) { out_int[0] = 0; out_int[1] = it + 1; out_int[2] = lo; out_int[3] = hi; *mu_out = mu; *sigma_out = 0.0; return 1; }
        const bool same = (n2 == n && a2 == s1 && b2 == s2);
        n = n2; s1 = a2; s2 = b2;
        orc_mu_sigma(p, n, s1, s2, &mu, &sigma);
        if (same) { ++it; break; }
    }
    out_int[0] = n; out_int[1] = it; out_int[2] = lo; out_int[3] = hi;
    *mu_out = mu; *sigma_out = sigma;
    return 0;
}

/* ---- C7: boxcars and SNR ("boxcar filters ... to maximise signal-to-noise") ----------------
 *   B_w[t] = sum_{j<w} D[t+j],  t in [0, T-w]           (t = START of the boxcar)
 *   SNR_w[t] = ( (double)(B_w[t] - w*p) - (double)w*(mu - p) ) * inv_w,   inv_w = 1/(sqrt((double)w)*sigma)
 *   S[t] = max_w SNR_w[t] over the widths valid at t (t + w <= T); wbest = smallest w attaining it;
 *   no valid width (or sigma == 0): S = -inf, wbest = 0.
 * p = D[0] is the same pivot as in C6 (keeps the subtraction exact). The white-noise scaling w*mu, sqrt(w)*sigma
 * of the width-1 statistics is reading C7. DESIGN.md "Readings": the division is done once per (row, w) as inv_w
 * and applied as a multiplication, so that the GPU can follow the same double operations. */
void orc_boxcar_snr(const int64_t* D, int64_t T, const int32_t* widths, int32_t nwidths, double mu, double sigma,
                    double* S, int32_t* wbest) {
    const int64_t p = D[0];
    const double ninf = -INFINITY;
    for (int64_t t = 0; t < T; ++t) { S[t] = ninf; wbest[t] = 0; }
    if (!(sigma > 0.0)) return;
    const double mrel = mu - (double)p;
    for (int32_t iw = 0; iw < nwidths; ++iw) {            /* ascending widths: strict '>' keeps the smallest */
        const int64_t w = widths[iw];
        const double a_w = (double)w * mrel;
        const double inv_w = 1.0 / (sqrt((double)w) * sigma);
        for (int64_t t = 0; t + w <= T; ++t) {
            int64_t B = 0;
            for (int64_t j = 0; j < w; ++j) B += D[t + j];
            const double snr = ((double)(B - w * p) - a_w) * inv_w;
            if (snr > S[t]) { S[t] = snr; wbest[t] = (int32_t)w; }
        }
    }
}

/* Same B_w through a running prefix sum: an O(T) route to the same exact integers, used only so the
 * oracle finishes on full-length rows; tests check it against orc_boxcar_snr's direct summation. */
void orc_boxcar_snr_prefix(const int64_t* D, int64_t T, const int32_t* widths, int32_t nwidths, double mu, double sigma,
                           double* S, int32_t* wbest) {
    const int64_t p = D[0];
    const double ninf = -INFINITY;
    for (int64_t t = 0; t < T; ++t) { S[t] = ninf; wbest[t] = 0; }
    if (!(sigma > 0.0)) return;
    std::vector<int64_t> P((size_t)T + 1);
    P[0] = 0;
    for (int64_t t = 0; t < T; ++t) P[(size_t)t + 1] = P[(size_t)t] + D[t];
    const double mrel = mu - (double)p;
    for (int32_t iw = 0; iw < nwidths; ++iw) {
        const int64_t w = widths[iw];
        const double a_w = (double)w * mrel;
        const double inv_w = 1.0 / (sqrt((double)w) * sigma);
        for (int64_t t = 0; t + w <= T; ++t) {
            const int64_t B = P[(size_t)(t + w)] - P[(size_t)t];
            const double snr = ((double)(B - w * p) - a_w) * inv_w;
            if (snr > S[t]) { S[t] = snr; wbest[t] = (int32_t)w; }
        }
    }
}

/* ---- C7m: per-width MEASURED statistics (reading C7m; SURVEY §8(f3) "per-width measured sigma instead of
 * sqrt(w) scaling"; "boxcar filters ... to maximise signal-to-noise"). Optional, off by default.
 * For each plan width w the series of boxcar sums of the row
 *     B_w[t] = sum_{j<w} D[t+j],   t in [0, n_w),   n_w = min(T, Tx - w + 1)      (T: the chunk's output span, Tx = T + E
 *                                                                                   samples present; E = 0 unless C3x)
 * is itself given reading C6 (orc_row_stats on the integer series B_w: pivot p_w = B_w[0], exact integer moments,
 * iterated 3-sigma clip, at most 8 clips) -> mu_w, sigma_w, and
 *     SNR_w[t] = ( (double)(B_w[t] - p_w) - (mu_w - (double)p_w) ) * (1.0 / sigma_w)
 * replaces the white-noise scaling w*mu, sqrt(w)*sigma of C7. A width with n_w < 1, or sigma_w == 0 (or a degenerate
 * clip) gives no SNR in this row. S = max over the remaining widths, smallest width on ties; S = -inf if none.
 * For w = 1 this is C7 exactly (B_1 = D). wstats_out (may be NULL): [nwidths][3] = mu_w, sigma_w, (double)p_w. */
void orc_boxcar_snr_perwidth(const int64_t* D, int64_t T, int64_t Tx, const int32_t* widths, int32_t nwidths,
                             double* S, int32_t* wbest, double* wstats_out) {
    const double ninf = -INFINITY;
    for (int64_t t = 0; t < T; ++t) { S[t] = ninf; wbest[t] = 0; }
    std::vector<int64_t> B;
    for (int32_t iw = 0; iw < nwidths; ++iw) {
        const int64_t w = widths[iw];
        if (wstats_out) { wstats_out[3 * iw] = 0.0; wstats_out[3 * iw + 1] = 0.0; wstats_out[3 * iw + 2] = 0.0; }
        int64_t nw = Tx - w + 1;
        if (nw > T) nw = T;
        if (nw < 1) continue;
        B.assign((size_t)nw, 0);
        for (int64_t t = 0; t < nw; ++t) {
            int64_t b = 0;
            for (int64_t j = 0; j < w; ++j) b += D[t + j];
            B[(size_t)t] = b;
        }
        double mu, sigma; int64_t info[4];
        const int32_t degenerate = orc_row_stats(B.data(), nw, &mu, &sigma, info);
        const int64_t pw = B[0];
        if (wstats_out) { wstats_out[3 * iw] = mu; wstats_out[3 * iw + 1] = degenerate ? 0.0 : sigma; wstats_out[3 * iw + 2] = (double)pw; }
        if (degenerate || !(sigma > 0.0)) continue;
        const double mrel = mu - (double)pw;
        const double inv = 1.0 / sigma;
        for (int64_t t = 0; t < nw; ++t) {
            const double snr = ((double)(B[(size_t)t] - pw) - mrel) * inv;
            if (snr > S[t]) { S[t] = snr; wbest[t] = (int32_t)w; }
        }
    }
}

/* ---- C8: peak finding ("peak-finding"; north_star "finds local peaks above a threshold") ---
 * On the map S[row][t] of ONE range in ONE chunk: (row, t) is a candidate iff S > threshold (strict) and, for
 * each of the 8 neighbours that exist (rows inside [0,nrows), t inside [0,T)):  S > neighbour when the neighbour
 * precedes (row,t) lexicographically, S >= neighbour otherwise (a plateau yields exactly one candidate, its
 * first point). -inf neighbours never block. Only rows [r0, r1) are reported (the others are halo).
 * out_row/out_t receive up to cap entries in (row, t) order; returns the TRUE count. */
int64_t orc_find_peaks(const double* S, int32_t nrows, int64_t T, double threshold, int32_t r0, int32_t r1,
                       int32_t* out_row, int64_t* out_t, int64_t cap) {
    int64_t cnt = 0;
    for (int32_t r = r0; r < r1; ++r) {
        for (int64_t t = 0; t < T; ++t) {
            const double s = S[(size_t)r * (size_t)T + (size_t)t];
            if (!(s > threshold)) continue;
            bool peak = true;
            for (int32_t dr = -1; dr <= 1 && peak; ++dr) {
                for (int64_t dt = -1; dt <= 1; ++dt) {
                    if (dr == 0 && dt == 0) continue;
                    const int32_t rr = r + dr; const int64_t tt = t + dt;
                    if (rr < 0 || rr >= nrows || tt < 0 || tt >= T) continue;
                    const double v = S[(size_t)rr * (size_t)T + (size_t)tt];
                    const bool before = (dr < 0) || (dr == 0 && dt < 0);
                    if (before ? !(s > v) : !(s >= v)) { peak = false; break; }
                }
            }
            if (peak) {
                if (cnt < cap) { out_row[cnt] = r; out_t[cnt] = t; }
                ++cnt;
            }
        }
    }
    return cnt;
}

/* ---- C9 + driver: search rows [i0, i1) of one range on one chunk ---------------------------------------
 * Follows steps a4..a7 of SURVEY §8(a) in order on a chunk already binned by orc_bin (a2): dedisperse (with one halo row each side) -> row statistics
 * -> boxcar/SNR -> peaks -> candidate records. sample = chunk_start + bin*t, width = bin*wbest (unbinned units). */
typedef struct {
    uint64_t sample; float dm; float snr; uint32_t width; uint32_t range; uint32_t dm_index;
} orc_candidate;

/* `extra` = E (reading C3x, optional "boxcar-complete chunks"): each row is dedispersed for T + E samples, the
 * statistics use the first T (the chunk's own output span), a boxcar starting at t < T may extend into the E extra samples
 * (valid while t + w <= T + E), and S / peaks are defined on t in [0, T). extra = 0 is readings C3/C7 as they were. */
int64_t orc_search_rows(const uint16_t* xb /* binned chunk [nchans][nbinned], from orc_bin */, int64_t nbinned, int32_t nchans,
                        const double* k, double dm_low, double dm_step, int32_t ndms, int32_t bin, int32_t range_index,
                        int64_t T, int64_t extra, const int32_t* widths, int32_t nwidths, double threshold, uint64_t chunk_start,
                        int32_t i0, int32_t i1, int32_t per_width /* 0: reading C7; 1: reading C7m */,
                        int64_t* D_out /* [(i1-i0)][T+extra] or NULL */, double* stats_out /* [(i1-i0)][2] or NULL */,
                        double* S_out /* [(i1-i0)][T] or NULL */, int32_t* w_out /* [(i1-i0)][T] or NULL */,
                        orc_candidate* cands, int64_t cap) {
    const int32_t h0 = i0 > 0 ? i0 - 1 : i0, h1 = i1 < ndms ? i1 + 1 : i1;   /* halo rows for the 3x3 test */
    const int32_t nr = h1 - h0;
    const int64_t Tx = T + extra;
    std::vector<int64_t> D((size_t)nr * (size_t)Tx);
    orc_dedisperse(xb, nbinned, nchans, k, dm_low, dm_step, bin, h0, h1, Tx, D.data());
    std::vector<double> S((size_t)nr * (size_t)T), Sx((size_t)Tx);
    std::vector<int32_t> W((size_t)nr * (size_t)T), Wx((size_t)Tx);
    for (int32_t r = 0; r < nr; ++r) {
        double mu, sigma; int64_t info[4];
        orc_row_stats(D.data() + (size_t)r * Tx, T, &mu, &sigma, info);
        if (per_width) orc_boxcar_snr_perwidth(D.data() + (size_t)r * Tx, T, Tx, widths, nwidths, Sx.data(), Wx.data(), nullptr);
        else orc_boxcar_snr_prefix(D.data() + (size_t)r * Tx, Tx, widths, nwidths, mu, sigma, Sx.data(), Wx.data());
        memcpy(S.data() + (size_t)r * T, Sx.data(), sizeof(double) * (size_t)T);
        memcpy(W.data() + (size_t)r * T, Wx.data(), sizeof(int32_t) * (size_t)T);
        const int32_t i = h0 + r;
        if (i >= i0 && i < i1) {
            if (stats_out) { stats_out[2 * (i - i0)] = mu; stats_out[2 * (i - i0) + 1] = sigma; }
            if (D_out) memcpy(D_out + (size_t)(i - i0) * Tx, D.data() + (size_t)r * Tx, sizeof(int64_t) * (size_t)Tx);
            if (S_out) memcpy(S_out + (size_t)(i - i0) * T, S.data() + (size_t)r * T, sizeof(double) * (size_t)T);
            if (w_out) memcpy(w_out + (size_t)(i - i0) * T, W.data() + (size_t)r * T, sizeof(int32_t) * (size_t)T);
        }
    }
    std::vector<int32_t> pr((size_t)(cap > 0 ? cap : 1)); std::vector<int64_t> pt((size_t)(cap > 0 ? cap : 1));
    /* rows outside [h0,h1) are not neighbours of [i0,i1), so treating the band as the whole map is exact,
     * EXCEPT that a halo row that is a real row must exist: nrows below is the band height. */
    const int64_t cnt = orc_find_peaks(S.data(), nr, T, threshold, i0 - h0, i1 - h0, pr.data(), pt.data(), cap);
    const int64_t m = cnt < cap ? cnt : cap;
    for (int64_t q = 0; q < m; ++q) {
        const int32_t i = h0 + pr[(size_t)q];
        orc_candidate c;
        c.sample = chunk_start + (uint64_t)bin * (uint64_t)pt[(size_t)q];
        c.dm = (float)orc_dm(dm_low, dm_step, i);
        c.snr = (float)S[(size_t)pr[(size_t)q] * (size_t)T + (size_t)pt[(size_t)q]];
        c.width = (uint32_t)bin * (uint32_t)W[(size_t)pr[(size_t)q] * (size_t)T + (size_t)pt[(size_t)q]];
        c.range = (uint32_t)range_index; c.dm_index = (uint32_t)i;
        cands[q] = c;
    }
    return cnt;
}

/* C3 helper: maximum delay of a range in UNBINNED samples, S_r = b * delay(C-1, last DM). */
int64_t orc_range_max_delay_unbinned(const double* k, int32_t nchans, double dm_low, double dm_step, int32_t ndms, int32_t bin) {
    return (int64_t)bin * orc_delay(k[nchans - 1], orc_dm(dm_low, dm_step, ndms - 1), bin);
}

}  /* extern "C" */
