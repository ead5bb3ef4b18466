/*
 * aa_plan.cpp — plan object: the user's search parameters, validated once ("If there are configuration
 * errors the API provides user feedback"; PAPER.md:59 item 3 "plan and strategy error checking are encapsulated").
 */
#include <cmath>
#include <cstdarg>
#include <cstdio>
#include <new>

#include "aa_internal.h"

namespace aa {

static thread_local char g_err[1024] = "";

void set_error(const char* fmt, ...) {
    va_list ap;
    va_start(ap, fmt);
    vsnprintf(g_err, sizeof(g_err), fmt, ap);
    va_end(ap);
}

aa_status cuda_fail(cudaError_t e, const char* what) {
    set_error("CUDA error in %s: %s (%s)", what, cudaGetErrorName(e), cudaGetErrorString(e));
    return AA_ERR_CUDA;
}

}  // namespace aa

extern "C" const char* aa_last_error(void) { return aa::g_err; }
extern "C" const char* aa_version(void) { return "paper_1912_07704_b200 0.1 (sm_100a)"; }

extern "C" aa_status aa_plan_create(aa_plan** out, int32_t nchans, const double* chan_freq_mhz, double tsamp_s,
                                    const aa_dm_range* ranges, int32_t nranges, const int32_t* boxcar_widths,
                                    int32_t nwidths, float snr_threshold) {
    using aa::set_error;
    if (!out) { set_error("aa_plan_create: out is NULL"); return AA_ERR_INVALID_ARG; }
    *out = nullptr;
    if (nchans < 1 || nchans > 65535) { set_error("aa_plan_create: nchans = %d must be in 1..65535", nchans); return AA_ERR_INVALID_ARG; }
    if (!chan_freq_mhz) { set_error("aa_plan_create: chan_freq_mhz is NULL"); return AA_ERR_INVALID_ARG; }
    for (int32_t c = 0; c < nchans; ++c) {
        if (!(chan_freq_mhz[c] > 0.0) || !std::isfinite(chan_freq_mhz[c])) {
            set_error("aa_plan_create: chan_freq_mhz[%d] = %g must be a positive frequency", c, chan_freq_mhz[c]);
            return AA_ERR_INVALID_ARG;
        }
        if (c > 0 && !(chan_freq_mhz[c] < chan_freq_mhz[c - 1])) {
            set_error("aa_plan_create: chan_freq_mhz must be strictly descending (channel 0 is f_top); [%d] = %g >= [%d] = %g",
                      c, chan_freq_mhz[c], c - 1, chan_freq_mhz[c - 1]);
            return AA_ERR_INVALID_ARG;
        }
    }
    if (!(tsamp_s > 0.0) || !std::isfinite(tsamp_s)) { set_error("aa_plan_create: tsamp_s = %g must be > 0", tsamp_s); return AA_ERR_INVALID_ARG; }
    if (nranges < 1 || nranges > 64 || !ranges) { set_error("aa_plan_create: nranges = %d must be in 1..64 with ranges non-NULL", nranges); return AA_ERR_INVALID_ARG; }
    int32_t max_bin = 1;
    for (int32_t r = 0; r < nranges; ++r) {
        const aa_dm_range& g = ranges[r];
        if (g.ndms < 1 || g.ndms > 65535) { set_error("aa_plan_create: ranges[%d].ndms = %d must be in 1..65535 (empty range)", r, g.ndms); return AA_ERR_INVALID_ARG; }
        if (!(g.dm_low >= 0.0) || !std::isfinite(g.dm_low)) { set_error("aa_plan_create: ranges[%d].dm_low = %g must be >= 0", r, g.dm_low); return AA_ERR_INVALID_ARG; }
        if (!std::isfinite(g.dm_step) || (g.ndms > 1 && !(g.dm_step > 0.0)) || g.dm_step < 0.0) {
            set_error("aa_plan_create: ranges[%d].dm_step = %g must be > 0", r, g.dm_step); return AA_ERR_INVALID_ARG;
        }
        if (g.bin != 1 && g.bin != 2 && g.bin != 4 && g.bin != 8) { set_error("aa_plan_create: ranges[%d].bin = %d must be 1, 2, 4 or 8", r, g.bin); return AA_ERR_INVALID_ARG; }
        if (g.bin > max_bin) max_bin = g.bin;
    }
    if (nwidths < 1 || nwidths > 16 || !boxcar_widths) { set_error("aa_plan_create: nwidths = %d must be in 1..16 with boxcar_widths non-NULL", nwidths); return AA_ERR_INVALID_ARG; }
    for (int32_t i = 0; i < nwidths; ++i) {
        if (boxcar_widths[i] < 1 || boxcar_widths[i] > 2048) { set_error("aa_plan_create: boxcar_widths[%d] = %d must be in 1..2048", i, boxcar_widths[i]); return AA_ERR_INVALID_ARG; }
        if (i > 0 && boxcar_widths[i] <= boxcar_widths[i - 1]) { set_error("aa_plan_create: boxcar_widths must be strictly ascending; [%d] = %d", i, boxcar_widths[i]); return AA_ERR_INVALID_ARG; }
    }
    if (!std::isfinite(snr_threshold)) { set_error("aa_plan_create: snr_threshold must be finite"); return AA_ERR_INVALID_ARG; }
    /* arithmetic limits of the packed int32 accumulators and of the int32 boxcar sums */
    if ((int64_t)nchans * max_bin > 65536) {
        set_error("aa_plan_create: nchans * max bin = %lld exceeds 65536 (16-bit carry lanes of the dedispersion kernel)", (long long)nchans * max_bin);
        return AA_ERR_INVALID_ARG;
    }
    if ((int64_t)boxcar_widths[nwidths - 1] * nchans * 255 * max_bin >= (int64_t)1 << 31) {
        set_error("aa_plan_create: max width * nchans * 255 * max bin = %lld does not fit int32 boxcar sums",
                  (long long)boxcar_widths[nwidths - 1] * nchans * 255 * max_bin);
        return AA_ERR_INVALID_ARG;
    }
    aa_plan* p = new (std::nothrow) aa_plan();
    if (!p) { set_error("aa_plan_create: out of host memory"); return AA_ERR_INTERNAL; }
    p->p.nchans = nchans;
    p->p.freq.assign(chan_freq_mhz, chan_freq_mhz + nchans);
    p->p.tsamp = tsamp_s;
    p->p.ranges.assign(ranges, ranges + nranges);
    p->p.widths.assign(boxcar_widths, boxcar_widths + nwidths);
    p->p.threshold = snr_threshold;
    *out = p;
    return AA_OK;
}

extern "C" void aa_plan_destroy(aa_plan* plan) { delete plan; }

extern "C" aa_status aa_plan_set_boxcar_overlap(aa_plan* plan, int32_t on) {
    if (!plan) { aa::set_error("aa_plan_set_boxcar_overlap: plan is NULL"); return AA_ERR_NOT_READY; }
    plan->p.boxcar_overlap = on != 0;
    return AA_OK;
}

extern "C" aa_status aa_plan_set_input_bits(aa_plan* plan, int32_t bits, uint32_t max_value) {
    using aa::set_error;
    if (!plan) { set_error("aa_plan_set_input_bits: plan is NULL"); return AA_ERR_NOT_READY; }
    if (bits != 8 && bits != 16) { set_error("aa_plan_set_input_bits: bits = %d must be 8 or 16", bits); return AA_ERR_INVALID_ARG; }
    if (bits == 8) { plan->p.input_bits = 8; plan->p.input_max = 255; return AA_OK; }
    if (max_value == 0) max_value = 65535;
    if (max_value > 65535) { set_error("aa_plan_set_input_bits: max_value = %u does not fit 16 bits", max_value); return AA_ERR_INVALID_ARG; }
    int64_t max_bin = 1;
    for (const aa_dm_range& g : plan->p.ranges) max_bin = g.bin > max_bin ? g.bin : max_bin;
    if ((int64_t)max_value * max_bin > 65535) {
        set_error("aa_plan_set_input_bits: max_value * max bin = %lld exceeds 65535 (a binned sample is held in 16 bits)", (long long)max_value * max_bin);
        return AA_ERR_INVALID_ARG;
    }
    if ((int64_t)plan->p.nchans * max_value * max_bin >= (int64_t)1 << 31) {
        set_error("aa_plan_set_input_bits: nchans * max_value * max bin = %lld does not fit the int32 dedispersed sums",
                  (long long)plan->p.nchans * max_value * max_bin);
        return AA_ERR_INVALID_ARG;
    }
    plan->p.input_bits = 16; plan->p.input_max = max_value;
    return AA_OK;
}

extern "C" aa_status aa_plan_set_per_width_stats(aa_plan* plan, int32_t on) {
    if (!plan) { aa::set_error("aa_plan_set_per_width_stats: plan is NULL"); return AA_ERR_NOT_READY; }
    plan->p.per_width = on != 0;
    return AA_OK;
}

extern "C" aa_status aa_plan_set_input_layout(aa_plan* plan, int32_t layout) {
    if (!plan) { aa::set_error("aa_plan_set_input_layout: plan is NULL"); return AA_ERR_NOT_READY; }
    if (layout != AA_LAYOUT_CHANNEL_MAJOR && layout != AA_LAYOUT_TIME_MAJOR) {
        aa::set_error("aa_plan_set_input_layout: layout = %d must be AA_LAYOUT_CHANNEL_MAJOR (0) or AA_LAYOUT_TIME_MAJOR (1)", layout);
        return AA_ERR_INVALID_ARG;
    }
    plan->p.layout = layout;
    return AA_OK;
}
