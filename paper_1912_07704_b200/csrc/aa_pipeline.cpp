/*
 * aa_pipeline.cpp — the pipeline: "iterates over the radio telescope input data in chunks. On each iteration, the user may
 * query the pipeline via a status code" (§3.3). One aa_run_* call = one module on one chunk; nothing here
 * allocates device memory and the dedispersed data never leave the GPU between the modules.
 * Host input is const and user-owned; results are copied into library-owned host memory.
 */
#include <algorithm>
#include <cstring>

#include "aa_internal.h"

using namespace aa;

namespace {

#define AA_CUDA(call, what)                                              \
    do {                                                                 \
        cudaError_t e_ = (call);                                         \
        if (e_ != cudaSuccess) { s.sticky = cuda_fail(e_, what); return s.sticky; } \
    } while (0)
#define AA_LAUNCH(call, what)                                            \
    do {                                                                 \
        int e_ = (call);                                                 \
        ++s.launches;                                                    \
        if (e_ != 0) { s.sticky = cuda_fail((cudaError_t)e_, what); return s.sticky; } \
    } while (0)

aa_status check_ready(aa_strategy* h, const char* fn) {
    if (!h) { set_error("%s: strategy is NULL — configure a plan and call aa_strategy_setup first", fn); return AA_ERR_NOT_READY; }
    if (!h->s.ready) { set_error("%s: this strategy was only planned (aa_strategy_plan); call aa_strategy_setup to make it ready", fn); return AA_ERR_NOT_READY; }
    if (h->s.sticky < 0) { return h->s.sticky; }
    /* arena, streams, events, tensor maps and kernel attributes belong to the device the strategy was set up on: running it with
     * another device current would launch on the wrong GPU (one arena per device; one strategy per device) */
    int dev = -1;
    const cudaError_t e = cudaGetDevice(&dev);
    if (e != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if (dev != h->s.device) {
        set_error("%s: this strategy was set up on CUDA device %d but device %d is current; cudaSetDevice(%d) first (one strategy per device)",
                  fn, h->s.device, dev, h->s.device);
        return AA_ERR_INVALID_ARG;
    }
    return AA_OK;
}

/* Enqueue the H2D copy of chunk j into raw buffer b on the copy stream. */
aa_status enqueue_h2d(Strategy& s, int64_t j, int b, const uint8_t* host_input, size_t row_stride, bool timed) {
    const Chunk& c = s.chunks[(size_t)j];
    if (s.raw_free_recorded[b]) AA_CUDA(cudaStreamWaitEvent(s.copy, s.ev_raw_free[b], 0), "cudaStreamWaitEvent");
    if (timed) AA_CUDA(cudaEventRecord(s.ev_h2d[0], s.copy), "cudaEventRecord");
    const size_t esz = (size_t)s.esz_in;
    if (s.plan.layout == AA_LAYOUT_TIME_MAJOR)      /* one contiguous block of c.len time rows */
        AA_CUDA(cudaMemcpy2DAsync(s.d_stage[b], s.stage_stride, host_input + (size_t)c.start * row_stride, row_stride, (size_t)s.plan.nchans * esz,
                                  (size_t)c.len, cudaMemcpyHostToDevice, s.copy), "cudaMemcpy2DAsync (H2D chunk, time-major)");
    else
        AA_CUDA(cudaMemcpy2DAsync(s.d_raw[b], s.in_pitch, host_input + c.start * esz, row_stride, (size_t)c.len * esz, (size_t)s.plan.nchans,
                                  cudaMemcpyHostToDevice, s.copy), "cudaMemcpy2DAsync (H2D chunk)");
    if (timed) AA_CUDA(cudaEventRecord(s.ev_h2d[1], s.copy), "cudaEventRecord");
    AA_CUDA(cudaEventRecord(s.ev_copied[b], s.copy), "cudaEventRecord");
    s.raw_holds[b] = j;
    return AA_OK;
}

/* Channel groups of a chunk whose H2D copy is pipelined with its own dedispersion (boundaries are multiples of 8, the
 * largest channel block of K2). */
struct ChannelGroups { int n; int32_t c[kMaxGroups + 1]; };

/* Exception budget of a channel group: the chunk's budget in proportion to the group's channels. */
static unsigned group_limit(const Strategy& s, int bin, int32_t c0, int32_t c1) {
    const uint64_t v = (uint64_t)s.exc_limit[bin] * (uint64_t)(c1 - c0) / (uint64_t)s.plan.nchans;
    return (unsigned)std::max<uint64_t>(1, std::min<uint64_t>(v, kExcCap));
}

/* K1 for channel rows [c0, c1) (= channel group g) of the chunk in raw buffer b: sample-shifted uint8 copies, the
 * offset-uint8 form of the bin 2 / 4 inputs (per-channel offsets, byte copies, exception list), and the uint16 binned
 * inputs with their shifted copies (for bin 2 / 4 only when the group has too many exceptions). */
/* K1 of a 16-bit plan (k_input16.cu): per-channel offsets, the offset forms of every bin with their exception lists, and the
 * plain binned samples for the groups / bins that take the global-memory route. */
aa_status enqueue_prep16(Strategy& s, const Chunk& c, int b, int32_t c0, int32_t c1, int g) {
    const int32_t n = c1 - c0;
    const uint16_t* raw = (const uint16_t*)(s.d_raw[b] + (size_t)c0 * s.in_pitch);
    int32_t* off[4]; int32_t* bias[4]; int32_t centre[4];
    bool any = false;
    for (int k = 0; k < 4; ++k) {
        const int bin = 1 << k;
        const bool sparse = s.d_exc_cnt[bin] != nullptr;
        off[k] = sparse ? s.d_off[bin] + c0 : nullptr;
        bias[k] = sparse ? (int32_t*)(s.d_exc_cnt[bin] + kMaxGroups + g) : nullptr;
        centre[k] = bin == 8 ? (s.lo16_max + 1) / 2 : 128;
        any = any || sparse;
    }
    /* runs for every 16-bit chunk, also when no bin has an offset form: the same read checks the samples against max_value */
    AA_LAUNCH(aak_chan_offsets16(raw, s.in_pitch, (int64_t)c.len, n, off, bias, centre, s.plan.input_max, (unsigned*)(s.d_counter + 2), s.compute),
              "channel offsets (16-bit)");
    if (any) {
        aak_prep16_args a;
        memset(&a, 0, sizeof a);
        a.raw = raw; a.pitch_bytes = s.in_pitch; a.ngroups = (int64_t)(s.in_pitch / 32); a.chan0 = c0; a.cap = kExcCap;
        for (int k = 0; k < 3; ++k) {
            const int bin = 1 << k;
            if (!s.d_lo[bin] || !s.d_exc_cnt[bin]) continue;
            a.lo[k] = s.d_lo[bin] + (size_t)c0 * s.lo_pitch[bin]; a.pitch[k] = s.lo_pitch[bin]; a.stride[k] = s.lo_stride[bin]; a.off[k] = s.d_off[bin] + c0;
            a.exc[k] = s.d_exc[bin] + (size_t)g * kExcCap; a.cnt[k] = s.d_exc_cnt[bin] + g; a.nb[k] = (int64_t)(c.len / (uint64_t)bin);
        }
        if (s.d_xb[8] && s.d_exc_cnt[8]) {
            a.lo8 = s.d_xb[8] + (size_t)c0 * s.xb_pitch[8]; a.pitch8 = s.xb_pitch[8] * 2; a.stride8 = s.xb_stride[8]; a.off8 = s.d_off[8] + c0;
            a.exc8 = s.d_exc[8] + (size_t)g * kExcCap; a.cnt8 = s.d_exc_cnt[8] + g; a.nb8 = (int64_t)(c.len / 8); a.hi8 = s.lo16_max;
        }
        AA_LAUNCH(aak_prep16(&a, n, s.compute), "input forms (16-bit)");
    }
    for (int bin = 1; bin <= 8; bin *= 2) {
        if (!s.d_xb[bin]) continue;
        const unsigned* cnt = s.d_exc_cnt[bin] ? s.d_exc_cnt[bin] + g : nullptr;     /* NULL: the bin has only the global-memory route */
        const unsigned lim = cnt ? group_limit(s, bin, c0, c1) : 0u;
        AA_LAUNCH(aak_bin_time16(raw, s.in_pitch, s.d_xb[bin] + (size_t)c0 * s.xb_pitch[bin], s.xb_pitch[bin] * 2, n, (int64_t)(c.len / (uint64_t)bin), bin, cnt,
                                 lim, s.compute), "time binning (16-bit)");
    }
    return AA_OK;
}

aa_status enqueue_prep(Strategy& s, const Chunk& c, int b, int32_t c0, int32_t c1, int g) {
    if (s.plan.input_bits == 16) return enqueue_prep16(s, c, b, c0, c1, g);
    const int32_t n = c1 - c0;
    const uint8_t* raw = s.d_raw[b] + (size_t)c0 * s.in_pitch;
    if (s.d_lo[2] || s.d_lo[4] || s.d_lo[8])
        AA_LAUNCH(aak_chan_offsets(raw, s.in_pitch, (int64_t)c.len, n, s.d_lo[2] ? s.d_off[2] + c0 : nullptr, s.d_lo[4] ? s.d_off[4] + c0 : nullptr,
                                   s.d_lo[8] ? s.d_off[8] + c0 : nullptr,
                                   s.d_lo[2] ? (int32_t*)(s.d_exc_cnt[2] + kMaxGroups + g) : nullptr,
                                   s.d_lo[4] ? (int32_t*)(s.d_exc_cnt[4] + kMaxGroups + g) : nullptr,
                                   s.d_lo[8] ? (int32_t*)(s.d_exc_cnt[8] + kMaxGroups + g) : nullptr, s.compute), "channel offsets");
    /* one read of the raw rows writes every input form K2 may read, except the uint16 forms of bin 2 / 4 */
    aak_prep_args a;
    memset(&a, 0, sizeof a);
    a.raw = raw; a.pitch = s.in_pitch; a.ngroups = (int64_t)(s.in_pitch / 16); a.chan0 = c0; a.cap = kExcCap;
    if (s.need_u8_copies) { a.x4 = s.d_x4 + (size_t)c0 * s.x4_pitch; a.x4_pitch = s.x4_pitch; a.x4_stride = s.x4_stride; }
    if (s.d_lo[2]) {
        a.lo2 = s.d_lo[2] + (size_t)c0 * s.lo_pitch[2]; a.lo2_pitch = s.lo_pitch[2]; a.lo2_stride = s.lo_stride[2]; a.off2 = s.d_off[2] + c0;
        a.exc2 = s.d_exc[2] + (size_t)g * kExcCap; a.cnt2 = s.d_exc_cnt[2] + g; a.nb2 = (int64_t)(c.len / 2);
    }
    if (s.d_lo[4]) {
        a.lo4 = s.d_lo[4] + (size_t)c0 * s.lo_pitch[4]; a.lo4_pitch = s.lo_pitch[4]; a.lo4_stride = s.lo_stride[4]; a.off4 = s.d_off[4] + c0;
        a.exc4 = s.d_exc[4] + (size_t)g * kExcCap; a.cnt4 = s.d_exc_cnt[4] + g; a.nb4 = (int64_t)(c.len / 4);
    }
    if (s.d_lo[8]) {                                 /* the half-byte form and its bit plane; the uint16 form only for exception-heavy chunks */
        a.hb8 = s.d_lo[8] + (size_t)c0 * s.lo_pitch[8]; a.hb8_pitch = s.lo_pitch[8]; a.hb8_stride = s.lo_stride[8]; a.off8 = s.d_off[8] + c0;
        a.exc8 = s.d_exc[8] + (size_t)g * kExcCap; a.cnt8 = s.d_exc_cnt[8] + g; a.nb8 = (int64_t)(c.len / 8);
        a.bits8 = s.d_bits[8] + (size_t)c0 * s.bits_pitch[8]; a.bits8_pitch = s.bits_pitch[8];
    } else if (s.d_xb[8]) { a.xb8 = s.d_xb[8] + (size_t)c0 * s.xb_pitch[8]; a.xb8_pitch = s.xb_pitch[8]; a.xb8_stride = s.xb_stride[8]; }
    AA_LAUNCH(aak_prep_fused(&a, n, s.compute), "input forms (fused)");
    for (int bin = 2; bin <= 8; bin *= 2) {
        if (bin == 8 && !s.d_lo[8]) continue;         /* bin 8 without the half-byte route: the fused kernel wrote its uint16 form */
        if (!s.d_xb[bin]) continue;
        const unsigned* cnt = s.d_lo[bin] ? s.d_exc_cnt[bin] + g : nullptr;      /* NULL: the range has no offset-uint8 route */
        const unsigned lim = cnt ? group_limit(s, bin, c0, c1) : 0u;
        const size_t pitch_bytes = s.xb_pitch[bin] * 2;           /* a row = 2 copies of xb_stride bytes */
        uint16_t* xb = s.d_xb[bin] + (size_t)c0 * s.xb_pitch[bin];
        AA_LAUNCH(aak_bin_time(raw, s.in_pitch, xb, s.xb_pitch[bin], n, (int64_t)(c.len / (uint64_t)bin), bin, cnt, lim, s.compute), "time binning");
        AA_LAUNCH(aak_shift_copy((const uint8_t*)xb, (uint8_t*)xb + s.xb_stride[bin], pitch_bytes, s.xb_stride[bin], n, 2, cnt, lim, s.compute), "shift copy (uint16)");
    }
    return AA_OK;
}

/* K2 of every range over channels [c0, c1) (channel group g); accumulate = add to the D already there. A bin 2 / 4 range
 * launches both of its routes; each tests the group's exception counter and only one of them runs. */
aa_status enqueue_k2(Strategy& s, const Chunk& c, int32_t c0, int32_t c1, bool accumulate, int g) {
    /* ranges are independent: odd ranges go to the auxiliary stream so the last, partly filled wave of one range's K2
     * overlaps the first wave of the next one (fork after the prep kernels, join before anything reads D) */
    const bool two = s.ranges.size() > 1 && s.aux;
    if (two) {
        AA_CUDA(cudaEventRecord(s.ev_fork, s.compute), "cudaEventRecord");
        AA_CUDA(cudaStreamWaitEvent(s.aux, s.ev_fork, 0), "cudaStreamWaitEvent");
    }
    for (Range& rg : s.ranges) {
        cudaStream_t st = (two && (rg.index & 1)) ? s.aux : s.compute;
        const int bin = rg.r.bin;
        aak_dedisp_args a;
        a.D = rg.d_D; a.pitch = rg.pitch;
        a.nt = (int64_t)(c.n_out / (uint64_t)bin) + rg.extra;      /* reading C3x: E samples beyond the output span */
        a.ndms = rg.r.ndms; a.nchans = s.plan.nchans;
        a.chan_begin = c0; a.chan_end = c1; a.accumulate = accumulate ? 1 : 0;
        const bool plain_u8 = bin == 1 && s.plan.input_bits == 8;
        const void* x0 = plain_u8 ? (const void*)s.d_x4 : (const void*)s.d_xb[bin];            /* copy 0 of the range's plain input form */
        const size_t pitch_elems = plain_u8 ? s.x4_pitch : s.xb_pitch[bin];
        if (rg.naive) {
            AA_LAUNCH(aak_dedisperse_naive(x0, pitch_elems, !plain_u8, rg.d_delays, s.plan.nchans, c0, c1, rg.r.ndms, a.nt, rg.d_D, rg.pitch,
                                           accumulate ? 1 : 0, nullptr, 0u, st), "dedispersion (global-memory route)");
            continue;
        }
        /* routes: [offset-uint8 plan] [main plan: plain input, or the offset-uint16 form] [global-memory kernel]. Where a range
         * has a sparse route (offsets + exceptions) and a dense one, both are launched; each tests the group's exception
         * counter and only one of them runs. */
        const bool sparse = rg.has_lo || rg.main_exc;
        const bool has_main = rg.ndm_tiles > 0;
        const unsigned* cnt = sparse ? s.d_exc_cnt[bin] + g : nullptr;
        const unsigned lim = sparse ? group_limit(s, bin, c0, c1) : 0u;
        for (int route = 0; route < 2; ++route) {
            if (route == 0 && !rg.has_lo) continue;
            if (route == 1 && !has_main) continue;
            const K2Plan& p = route == 0 ? rg.lo : static_cast<const K2Plan&>(rg);
            const bool route_sparse = route == 0 || rg.main_exc;
            a.tmap = p.maps; a.etab = p.d_etab; a.x0tab = p.d_x0tab;
            a.nclass = p.nclass; a.wcls = p.d_wcls;
            for (int k = 0; k < 8; ++k) a.class_wb[k] = p.class_wb[k];
            a.chan_block = p.chan_block; a.window_bytes = p.window_bytes; a.spill_stages = p.spill_stages; a.in16 = p.in16;
            a.variant = p.variant; a.dms_per_warp = p.dms_per_warp; a.ring_stages = p.ring_stages; a.dm_tile = p.dm_tile; a.skew_q16 = p.skew_q16;
            a.mode_cnt = cnt; a.mode_cap = lim; a.mode_dense = route_sparse ? 0 : 1;
            a.bias = route_sparse ? (const int32_t*)(s.d_exc_cnt[bin] + kMaxGroups + g) : nullptr;
            AA_LAUNCH(aak_dedisperse(&a, st), "dedispersion");
        }
        if (rg.half)                                  /* the low bits the half-byte form dropped */
            AA_LAUNCH(aak_dedisperse_bits(s.d_bits[bin], s.bits_pitch[bin], rg.d_delays, s.plan.nchans, c0, c1, rg.r.ndms, a.nt, rg.bits_ww, rg.d_D,
                                          rg.pitch, cnt, lim, st), "bit-plane dedispersion");
        if (sparse)
            AA_LAUNCH(aak_scatter_exceptions(s.d_exc[bin] + (size_t)g * kExcCap, s.d_exc_cnt[bin] + g, lim, s.d_k, rg.r.dm_low, rg.r.dm_step,
                                             rg.r.ndms, bin, a.nt, rg.d_D, rg.pitch, s.nsm, st), "exception scatter");
        if (rg.dense_naive)
            AA_LAUNCH(aak_dedisperse_naive(x0, pitch_elems, 1, rg.d_delays, s.plan.nchans, c0, c1, rg.r.ndms, a.nt, rg.d_D, rg.pitch,
                                           accumulate ? 1 : 0, cnt, lim, st), "dedispersion (global-memory route of an exception-heavy chunk)");
    }
    if (two) {
        AA_CUDA(cudaEventRecord(s.ev_join, s.aux), "cudaEventRecord");
        AA_CUDA(cudaStreamWaitEvent(s.compute, s.ev_join, 0), "cudaStreamWaitEvent");
    }
    return AA_OK;
}

/* H2D of chunk j into raw buffer b as `groups.n` row blocks, one event per block (channel-major plans). */
aa_status enqueue_h2d_groups(Strategy& s, int64_t j, int b, const uint8_t* host_input, size_t row_stride, const ChannelGroups& groups) {
    const Chunk& c = s.chunks[(size_t)j];
    if (s.raw_free_recorded[b]) AA_CUDA(cudaStreamWaitEvent(s.copy, s.ev_raw_free[b], 0), "cudaStreamWaitEvent");
    AA_CUDA(cudaEventRecord(s.ev_h2d[0], s.copy), "cudaEventRecord");
    for (int g = 0; g < groups.n; ++g) {
        const int32_t c0 = groups.c[g], c1 = groups.c[g + 1];
        AA_CUDA(cudaMemcpy2DAsync(s.d_raw[b] + (size_t)c0 * s.in_pitch, s.in_pitch, host_input + (size_t)c0 * row_stride + c.start * (size_t)s.esz_in, row_stride,
                                  (size_t)c.len * (size_t)s.esz_in, (size_t)(c1 - c0), cudaMemcpyHostToDevice, s.copy), "cudaMemcpy2DAsync (H2D channel group)");
        AA_CUDA(cudaEventRecord(s.ev_group[g], s.copy), "cudaEventRecord");
    }
    AA_CUDA(cudaEventRecord(s.ev_h2d[1], s.copy), "cudaEventRecord");
    AA_CUDA(cudaEventRecord(s.ev_copied[b], s.copy), "cudaEventRecord");
    s.raw_holds[b] = j;
    return AA_OK;
}

/* Corner turn (time-major plans), shifted copies, binning and the dedispersion launches for the chunk resident in input
 * buffer b. tm_src/tm_stride: the time-major source of the corner turn (the staging buffer, or the caller's device chunk). */
aa_status enqueue_dedispersion(Strategy& s, int64_t j, int b, const uint8_t* tm_src = nullptr, size_t tm_stride = 0,
                               const ChannelGroups* groups = nullptr) {
    const Chunk& c = s.chunks[(size_t)j];
    const int32_t C = s.plan.nchans;
    const int slot = b;                               /* the buffer whose reuse the raw_free event guards */
    AA_CUDA(cudaEventRecord(s.ev_t[0], s.compute), "cudaEventRecord");
    if (s.plan.layout == AA_LAYOUT_TIME_MAJOR) {
        if (!tm_src) { tm_src = s.d_stage[b]; tm_stride = s.stage_stride; }
        if (s.plan.input_bits == 16)
            AA_LAUNCH(aak_corner_turn16((const uint16_t*)tm_src, tm_stride, (uint16_t*)s.d_raw[0], s.in_pitch, C, (int64_t)c.len, s.compute), "corner turn (16-bit)");
        else
            AA_LAUNCH(aak_corner_turn(tm_src, tm_stride, s.d_raw[0], s.in_pitch, C, (int64_t)c.len, s.compute), "corner turn");
        b = 0;                                        /* the channel-major copy lives in d_raw[0] */
    }
    if (s.plan.input_bits == 16)                   /* [2]: "a sample exceeds max_value" flag of this chunk (k_chan_offsets16) */
        AA_CUDA(cudaMemsetAsync(s.d_counter + 2, 0, sizeof(unsigned long long), s.compute), "cudaMemsetAsync");
    for (int bn = 1; bn <= 8; bn *= 2)             /* exception counters and biases of this chunk's channel groups */
        if (s.d_exc_cnt[bn]) AA_CUDA(cudaMemsetAsync(s.d_exc_cnt[bn], 0, 2 * kMaxGroups * 4, s.compute), "cudaMemsetAsync");
    if (groups) {
        /* the chunk is still arriving: channel group g is prepared and added to D as soon as its rows have landed, so only
         * the first group's copy is exposed (D is accumulated over the groups: int32 sums, any grouping gives the same bits) */
        for (int g = 0; g < groups->n; ++g) {
            AA_CUDA(cudaStreamWaitEvent(s.compute, s.ev_group[g], 0), "cudaStreamWaitEvent");
            aa_status st = enqueue_prep(s, c, b, groups->c[g], groups->c[g + 1], g);
            if (st != AA_OK) return st;
            if (g == 0) AA_CUDA(cudaEventRecord(s.ev_t[1], s.compute), "cudaEventRecord");
            if (g == groups->n - 1) { AA_CUDA(cudaEventRecord(s.ev_raw_free[slot], s.compute), "cudaEventRecord"); s.raw_free_recorded[slot] = true; }
            if ((st = enqueue_k2(s, c, groups->c[g], groups->c[g + 1], g > 0, g)) != AA_OK) return st;
        }
    } else {
        aa_status st = enqueue_prep(s, c, b, 0, C, 0);
        if (st != AA_OK) return st;
        AA_CUDA(cudaEventRecord(s.ev_t[1], s.compute), "cudaEventRecord");
        /* K1 was the last reader of the H2D buffer (K2 reads the input forms K1 wrote): the next chunk's copy may start now */
        AA_CUDA(cudaEventRecord(s.ev_raw_free[slot], s.compute), "cudaEventRecord");
        s.raw_free_recorded[slot] = true;
        if ((st = enqueue_k2(s, c, 0, C, false, 0)) != AA_OK) return st;
    }
    AA_CUDA(cudaEventRecord(s.ev_t[2], s.compute), "cudaEventRecord");
    s.timed = true; s.stats_timed = false;
    s.current_chunk = j;
    s.pending_sps = true;
    return AA_OK;
}

bool cand_less(const aa_candidate& a, const aa_candidate& b) {
    if (a.range != b.range) return a.range < b.range;
    if (a.dm_index != b.dm_index) return a.dm_index < b.dm_index;
    return a.sample < b.sample;
}

/* Bring the candidates of the last searched chunk to the host (PAPER.md:47 step 8). Synchronises on the counter copy. */
aa_status harvest(Strategy& s) {
    if (!s.harvest_pending) return AA_OK;
    AA_CUDA(cudaEventSynchronize(s.ev_count), "cudaEventSynchronize");
    const unsigned long long found = s.h_counter[0];
    if (s.plan.input_bits == 16 && (s.h_counter[2] & 1ull)) {
        s.harvest_pending = false;
        set_error("aa_run_sps: chunk %lld holds a sample above the plan's max_value = %u (aa_plan_set_input_bits): the binned sums and D of "
                  "this chunk cannot be trusted", (long long)s.harvest_chunk, s.plan.input_max);
        s.sticky = AA_ERR_RANGE;
        return s.sticky;
    }
    if (s.h_counter[1] & 1ull) {
        s.harvest_pending = false;
        set_error("aa_run_sps: in chunk %lld the widest boxcar times the largest |D - D[0]| of a row reaches 2^31: the int32 boxcar sums cannot be "
                  "trusted for this data (16-bit plan; narrow the widths or the sample maximum)", (long long)s.harvest_chunk);
        s.sticky = AA_ERR_RANGE;
        return s.sticky;
    }
    s.true_count += found;
    unsigned long long take = std::min<unsigned long long>(found, s.max_candidates);
    const size_t room = s.max_candidates - std::min(s.max_candidates, s.cands.size());
    if (take > room) take = room;
    if (take < found) s.overflow = true;
    if (take) {
        const size_t old = s.cands.size();
        s.cands.resize(old + (size_t)take);
        static_assert(sizeof(aa_candidate) == sizeof(aak_candidate), "candidate layouts must match");
        /* on the library's own stream: the compute stream may already hold the next chunk's K2 (200 ms), and ev_count says the
         * records are complete; the next K4 is enqueued only after this returns */
        AA_CUDA(cudaMemcpyAsync(s.cands.data() + old, s.d_cands, (size_t)take * sizeof(aa_candidate), cudaMemcpyDeviceToHost, s.d2h), "candidate D2H");
        AA_CUDA(cudaStreamSynchronize(s.d2h), "cudaStreamSynchronize");
        std::sort(s.cands.begin() + (ptrdiff_t)old, s.cands.end(), cand_less);   /* chunks arrive in order: canonical */
    }
    s.harvest_pending = false;
    return AA_OK;
}

}  // namespace

extern "C" aa_status aa_run_dedispersion(aa_strategy* h, const uint8_t* host_input, size_t row_stride_bytes) {
    aa_status st = check_ready(h, "aa_run_dedispersion");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (!host_input) { set_error("aa_run_dedispersion: host_input is NULL"); return AA_ERR_INVALID_ARG; }
    const bool tmajor = s.plan.layout == AA_LAYOUT_TIME_MAJOR;
    const size_t esz = (size_t)s.esz_in;
    if (!tmajor && row_stride_bytes < s.nsamp_total * esz) { set_error("aa_run_dedispersion: row_stride_bytes = %zu is shorter than nsamp_total = %llu samples of %zu byte(s)", row_stride_bytes, (unsigned long long)s.nsamp_total, esz); return AA_ERR_INVALID_ARG; }
    if (tmajor && row_stride_bytes < (size_t)s.plan.nchans * esz) { set_error("aa_run_dedispersion: row_stride_bytes = %zu is shorter than nchans = %d samples of %zu byte(s) (time-major plan)", row_stride_bytes, s.plan.nchans, esz); return AA_ERR_INVALID_ARG; }
    if (esz == 2 && (((uintptr_t)host_input | row_stride_bytes) & 1)) { set_error("aa_run_dedispersion: a 16-bit plan needs host_input and row_stride_bytes = %zu aligned to 2 bytes", row_stride_bytes); return AA_ERR_INVALID_ARG; }
    const bool two_buffers = s.d_stage[1] != nullptr;      /* time-major staging; a channel-major plan has ONE H2D buffer */
    const bool prefetch = s.chunks.size() > 1;
    if (s.pending_sps) { set_error("aa_run_dedispersion: chunk %lld is dedispersed but aa_run_sps has not run on it yet", (long long)s.current_chunk); return AA_ERR_ORDER; }
    if (s.next_chunk >= (int64_t)s.chunks.size()) { set_error("aa_run_dedispersion: all %zu chunks are done (aa_strategy_reset rewinds)", s.chunks.size()); return AA_ERR_ORDER; }
    const int64_t j = s.next_chunk;
    const int b = two_buffers ? (int)((j / s.shard_world) & 1) : 0;
    s.h2d_timed = false;
    ChannelGroups groups; groups.n = 0;
    if (s.raw_holds[b] != j) {
        /* not prefetched (first chunk, or a single-chunk observation): pipeline the copy with the compute by channel groups */
        const int32_t C = s.plan.nchans;
        if (!tmajor && C >= 64 * kMaxGroups) {
            /* the copy is several times faster than the compute (PCIe ~55 GB/s against ~10 GB/s of input consumed), so only
             * the FIRST group's copy is exposed: 1/16 of the channels, then 5/16 (lands while group 0 computes), then the rest.
             * Every extra group costs one more read-modify-write pass over D, so three groups, not more. */
            groups.n = 3;
            groups.c[0] = 0;
            groups.c[1] = std::max<int32_t>(8, (C / 16) & ~7);
            groups.c[2] = std::max<int32_t>(groups.c[1] + 8, (int32_t)(((int64_t)C * 6 / 16) & ~7));
            groups.c[3] = C;
            if ((st = enqueue_h2d_groups(s, j, b, host_input, row_stride_bytes, groups)) != AA_OK) return st;
        } else {
            if ((st = enqueue_h2d(s, j, b, host_input, row_stride_bytes, true)) != AA_OK) return st;
        }
        s.h2d_timed = true;
    }
    if (!groups.n) AA_CUDA(cudaStreamWaitEvent(s.compute, s.ev_copied[b], 0), "cudaStreamWaitEvent");
    if ((st = enqueue_dedispersion(s, j, b, nullptr, 0, groups.n ? &groups : nullptr)) != AA_OK) return st;
    /* double buffering: start moving chunk j+1 while chunk j computes (north_star "Streaming") */
    const int64_t jn = j + s.shard_world;           /* the next chunk of this strategy's shard */
    const int bn = two_buffers ? (b ^ 1) : 0;       /* the single buffer is free again once K1 of chunk j has run (ev_raw_free) */
    if (prefetch && jn < (int64_t)s.chunks.size() && s.raw_holds[bn] != jn)
        if ((st = enqueue_h2d(s, jn, bn, host_input, row_stride_bytes, false)) != AA_OK) return st;
    return AA_OK;
}

extern "C" aa_status aa_run_dedispersion_device(aa_strategy* h, const uint8_t* device_chunk, size_t row_stride_bytes) {
    aa_status st = check_ready(h, "aa_run_dedispersion_device");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (!device_chunk) { set_error("aa_run_dedispersion_device: device_chunk is NULL"); return AA_ERR_INVALID_ARG; }
    if (s.pending_sps) { set_error("aa_run_dedispersion_device: chunk %lld is dedispersed but aa_run_sps has not run on it yet", (long long)s.current_chunk); return AA_ERR_ORDER; }
    if (s.next_chunk >= (int64_t)s.chunks.size()) { set_error("aa_run_dedispersion_device: all %zu chunks are done", s.chunks.size()); return AA_ERR_ORDER; }
    const int64_t j = s.next_chunk;
    const Chunk& c = s.chunks[(size_t)j];
    s.h2d_timed = false;
    if (s.plan.layout == AA_LAYOUT_TIME_MAJOR) {
        if (((uintptr_t)device_chunk & 3) || (row_stride_bytes & 3) || row_stride_bytes < (size_t)((s.plan.nchans * s.esz_in + 3) & ~3)) {
            set_error("aa_run_dedispersion_device: a time-major device chunk must be 4-byte aligned with row_stride_bytes a multiple of 4 and >= nchans rounded up to 4 (got %zu)", row_stride_bytes);
            return AA_ERR_INVALID_ARG;
        }
        /* the corner turn writes d_raw[0]; nothing else is in flight into it (host prefetches of a time-major plan go to d_stage) */
        return enqueue_dedispersion(s, j, 0, device_chunk, row_stride_bytes);
    }
    if (row_stride_bytes < c.len * (size_t)s.esz_in) { set_error("aa_run_dedispersion_device: row_stride_bytes = %zu is shorter than the chunk (%llu samples)", row_stride_bytes, (unsigned long long)c.len); return AA_ERR_INVALID_ARG; }
    const int b = 0;
    /* a host prefetch of an earlier aa_run_dedispersion(host) may still be writing this buffer on the copy stream */
    if (s.raw_holds[b] >= 0) AA_CUDA(cudaStreamWaitEvent(s.compute, s.ev_copied[b], 0), "cudaStreamWaitEvent");
    AA_CUDA(cudaMemcpy2DAsync(s.d_raw[b], s.in_pitch, device_chunk, row_stride_bytes, (size_t)c.len * (size_t)s.esz_in, (size_t)s.plan.nchans,
                              cudaMemcpyDeviceToDevice, s.compute), "cudaMemcpy2DAsync (D2D chunk)");
    s.raw_holds[b] = j;
    return enqueue_dedispersion(s, j, b);
}

extern "C" aa_status aa_run_sps(aa_strategy* h) {
    aa_status st = check_ready(h, "aa_run_sps");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (!s.pending_sps) { set_error("aa_run_sps: no dedispersed chunk is pending — aa_run_dedispersion must run first"); return AA_ERR_ORDER; }
    if ((st = harvest(s)) != AA_OK) return st;      /* previous chunk's records leave the device buffer first */
    const int64_t j = s.current_chunk;
    const Chunk& c = s.chunks[(size_t)j];
    const bool is_short = c.len != (uint64_t)s.L;
    AA_CUDA(cudaMemsetAsync(s.d_counter, 0, 2 * sizeof(unsigned long long), s.compute), "cudaMemsetAsync");   /* [0] candidates, [1] range flag */
    AA_CUDA(cudaEventRecord(s.ev_t[3], s.compute), "cudaEventRecord");
    AA_LAUNCH(aak_row_stats(s.d_rows[is_short ? 1 : 0], (int32_t)s.nrows, s.d_mu_sigma, s.d_n_iters, s.compute), "row statistics");
    const size_t nwd = s.plan.widths.size();
    if (s.plan.per_width) {                        /* reading C7m: every width's own statistics, range by range (K3w) */
        for (Range& rg : s.ranges) {
            aak_wstats_args a;
            a.D = rg.d_D; a.pitch = rg.pitch; a.nt = (int64_t)(c.n_out / (uint64_t)rg.r.bin); a.nt_data = a.nt + rg.extra; a.ndms = rg.r.ndms;
            a.nwidths = (int32_t)nwd;
            for (int k = 0; k < 16; ++k) a.widths[k] = k < a.nwidths ? s.plan.widths[(size_t)k] : 0;
            a.wstats = s.d_wstats + 2 * nwd * rg.first_row; a.wpivot = s.d_wpivot + nwd * rg.first_row; a.wlive = s.d_wlive + rg.first_row;
            AA_LAUNCH(aak_row_width_stats(&a, s.compute), "per-width row statistics");
        }
    }
    AA_CUDA(cudaEventRecord(s.ev_t[4], s.compute), "cudaEventRecord");
    /* the ranges' K4 launches are independent (one atomic counter): odd ranges go to the auxiliary stream, as for K2, so that the
     * short launches of the binned ranges run beside the others instead of each ending in its own partly filled wave */
    const bool two = s.ranges.size() > 1 && s.aux;
    if (two) {
        AA_CUDA(cudaEventRecord(s.ev_fork, s.compute), "cudaEventRecord");
        AA_CUDA(cudaStreamWaitEvent(s.aux, s.ev_fork, 0), "cudaStreamWaitEvent");
    }
    for (Range& rg : s.ranges) {
        aak_sps_args a;
        a.D = rg.d_D; a.pitch = rg.pitch; a.nt = (int64_t)(c.n_out / (uint64_t)rg.r.bin); a.nt_data = a.nt + rg.extra; a.ndms = rg.r.ndms; a.bin = rg.r.bin;
        a.range_index = rg.index; a.dm_low = rg.r.dm_low; a.dm_step = rg.r.dm_step;
        a.mu_sigma = s.d_mu_sigma + 2 * rg.first_row; a.chunk_start = c.start;
        a.nwidths = (int32_t)s.plan.widths.size();
        for (int k = 0; k < 16; ++k) a.widths[k] = k < a.nwidths ? s.plan.widths[(size_t)k] : 0;
        a.threshold = (double)s.plan.threshold;
        a.cands = s.d_cands; a.counter = s.d_counter; a.capacity = s.max_candidates;
        a.range_flag = s.plan.input_bits == 16 ? (unsigned*)(s.d_counter + 1) : nullptr;      /* no plan-time bound on boxcar sums */
        a.wstats = s.plan.per_width ? s.d_wstats + 2 * nwd * rg.first_row : nullptr;
        a.wpivot = s.plan.per_width ? s.d_wpivot + nwd * rg.first_row : nullptr;
        a.wlive = s.plan.per_width ? s.d_wlive + rg.first_row : nullptr;
        AA_LAUNCH(aak_sps_peaks(&a, (two && (rg.index & 1)) ? s.aux : s.compute), "sps peaks");
    }
    if (two) {
        AA_CUDA(cudaEventRecord(s.ev_join, s.aux), "cudaEventRecord");
        AA_CUDA(cudaStreamWaitEvent(s.compute, s.ev_join, 0), "cudaStreamWaitEvent");
    }
    AA_CUDA(cudaEventRecord(s.ev_t[5], s.compute), "cudaEventRecord");
    AA_CUDA(cudaMemcpyAsync(s.h_counter, s.d_counter, 3 * sizeof(unsigned long long), cudaMemcpyDeviceToHost, s.compute), "counter D2H");
    AA_CUDA(cudaEventRecord(s.ev_count, s.compute), "cudaEventRecord");
    s.harvest_pending = true; s.harvest_chunk = j; s.stats_timed = true;
    s.pending_sps = false;
    s.next_chunk = j + s.shard_world;
    return s.next_chunk >= (int64_t)s.chunks.size() ? AA_STATUS_FINISHED : AA_STATUS_CHUNK_DONE;
}

extern "C" aa_status aa_run_pipeline(aa_strategy* h, const uint8_t* host_input, size_t row_stride_bytes) {
    aa_status st = check_ready(h, "aa_run_pipeline");
    if (st != AA_OK) return st;
    if (h->s.pending_sps && (st = aa_run_sps(h)) < 0) return st;
    while (h->s.next_chunk < (int64_t)h->s.chunks.size()) {
        if ((st = aa_run_dedispersion(h, host_input, row_stride_bytes)) < 0) return st;
        if ((st = aa_run_sps(h)) < 0) return st;
    }
    return AA_STATUS_FINISHED;
}

extern "C" aa_status aa_get_candidates(aa_strategy* h, const aa_candidate** out, size_t* n) {
    aa_status st = check_ready(h, "aa_get_candidates");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (!out || !n) { set_error("aa_get_candidates: NULL output argument"); return AA_ERR_INVALID_ARG; }
    if ((st = harvest(s)) != AA_OK) return st;
    *out = s.cands.data();
    *n = s.cands.size();
    if (s.overflow) {
        set_error("aa_get_candidates: %llu candidates were found but max_candidates = %zu; %zu are returned", (unsigned long long)s.true_count, s.max_candidates, s.cands.size());
        return AA_ERR_CANDIDATE_OVERFLOW;
    }
    return AA_OK;
}

extern "C" aa_status aa_strategy_reset(aa_strategy* h) {
    if (!h) { set_error("aa_strategy_reset: strategy is NULL"); return AA_ERR_NOT_READY; }
    Strategy& s = h->s;
    if (s.compute) cudaStreamSynchronize(s.compute);
    if (s.copy) cudaStreamSynchronize(s.copy);
    s.next_chunk = s.shard_rank; s.current_chunk = -1; s.pending_sps = false; s.harvest_pending = false;
    s.raw_holds[0] = s.raw_holds[1] = -1;
    s.cands.clear(); s.true_count = 0; s.overflow = false; s.launches = 0; s.timed = false; s.stats_timed = false;
    if (s.sticky != AA_ERR_CUDA) s.sticky = AA_OK;
    return AA_OK;
}

extern "C" aa_status aa_strategy_shard(aa_strategy* h, int32_t rank, int32_t world) {
    if (!h) { set_error("aa_strategy_shard: strategy is NULL"); return AA_ERR_NOT_READY; }
    if (world < 1 || rank < 0 || rank >= world) { set_error("aa_strategy_shard: need 0 <= rank < world, got rank = %d, world = %d", rank, world); return AA_ERR_INVALID_ARG; }
    h->s.shard_rank = rank; h->s.shard_world = world;
    return aa_strategy_reset(h);
}

extern "C" aa_status aa_synchronize(aa_strategy* h) {
    aa_status st = check_ready(h, "aa_synchronize");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    AA_CUDA(cudaStreamSynchronize(s.compute), "cudaStreamSynchronize");
    AA_CUDA(cudaStreamSynchronize(s.copy), "cudaStreamSynchronize");
    return AA_OK;
}

extern "C" aa_status aa_get_dedispersed_row(aa_strategy* h, int32_t range, int32_t dm_index, const int32_t** host_row, size_t* len) {
    aa_status st = check_ready(h, "aa_get_dedispersed_row");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (s.current_chunk < 0) { set_error("aa_get_dedispersed_row: no chunk has been dedispersed yet"); return AA_ERR_ORDER; }
    if (!host_row || !len || range < 0 || range >= (int32_t)s.ranges.size() || dm_index < 0 || dm_index >= s.ranges[(size_t)range].r.ndms) {
        set_error("aa_get_dedispersed_row: range %d / dm_index %d out of bounds", range, dm_index); return AA_ERR_INVALID_ARG;
    }
    const Range& rg = s.ranges[(size_t)range];
    const size_t nt = (size_t)(s.chunks[(size_t)s.current_chunk].n_out / (uint64_t)rg.r.bin) + (size_t)rg.extra;
    s.host_row.resize(nt);
    AA_CUDA(cudaMemcpyAsync(s.host_row.data(), rg.d_D + (size_t)dm_index * (size_t)rg.pitch, nt * 4, cudaMemcpyDeviceToHost, s.compute), "row D2H");
    AA_CUDA(cudaStreamSynchronize(s.compute), "cudaStreamSynchronize");
    *host_row = s.host_row.data();
    *len = nt;
    return AA_OK;
}

extern "C" aa_status aa_get_dedispersed_device(aa_strategy* h, int32_t range, const int32_t** device_ptr, int64_t* row_pitch) {
    aa_status st = check_ready(h, "aa_get_dedispersed_device");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (!device_ptr || !row_pitch || range < 0 || range >= (int32_t)s.ranges.size()) { set_error("aa_get_dedispersed_device: bad argument"); return AA_ERR_INVALID_ARG; }
    *device_ptr = s.ranges[(size_t)range].d_D;
    *row_pitch = s.ranges[(size_t)range].pitch;
    return AA_OK;
}

extern "C" aa_status aa_get_row_stats(aa_strategy* h, int32_t range, int32_t dm_index, double* mu, double* sigma, int64_t* n_kept,
                                      int32_t* iterations) {
    aa_status st = check_ready(h, "aa_get_row_stats");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (!s.stats_timed) { set_error("aa_get_row_stats: aa_run_sps has not run on the current chunk"); return AA_ERR_ORDER; }
    if (range < 0 || range >= (int32_t)s.ranges.size() || dm_index < 0 || dm_index >= s.ranges[(size_t)range].r.ndms) {
        set_error("aa_get_row_stats: range %d / dm_index %d out of bounds", range, dm_index); return AA_ERR_INVALID_ARG;
    }
    const size_t row = s.ranges[(size_t)range].first_row + (size_t)dm_index;
    double ms[2]; int64_t ni[2];
    AA_CUDA(cudaMemcpyAsync(ms, s.d_mu_sigma + 2 * row, sizeof ms, cudaMemcpyDeviceToHost, s.compute), "stats D2H");
    AA_CUDA(cudaMemcpyAsync(ni, s.d_n_iters + 2 * row, sizeof ni, cudaMemcpyDeviceToHost, s.compute), "stats D2H");
    AA_CUDA(cudaStreamSynchronize(s.compute), "cudaStreamSynchronize");
    if (mu) *mu = ms[0];
    if (sigma) *sigma = ms[1];
    if (n_kept) *n_kept = ni[0];
    if (iterations) *iterations = (int32_t)ni[1];
    return AA_OK;
}

extern "C" aa_status aa_get_row_width_stats(aa_strategy* h, int32_t range, int32_t dm_index, int32_t width_index, double* mu, double* sigma,
                                            int64_t* pivot) {
    aa_status st = check_ready(h, "aa_get_row_width_stats");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (!s.plan.per_width) { set_error("aa_get_row_width_stats: the plan does not ask for per-width statistics (aa_plan_set_per_width_stats)"); return AA_ERR_ORDER; }
    if (!s.stats_timed) { set_error("aa_get_row_width_stats: aa_run_sps has not run on the current chunk"); return AA_ERR_ORDER; }
    const size_t nwd = s.plan.widths.size();
    if (range < 0 || range >= (int32_t)s.ranges.size() || dm_index < 0 || dm_index >= s.ranges[(size_t)range].r.ndms || width_index < 0 ||
        width_index >= (int32_t)nwd) {
        set_error("aa_get_row_width_stats: range %d / dm_index %d / width_index %d out of bounds", range, dm_index, width_index); return AA_ERR_INVALID_ARG;
    }
    const size_t o = (s.ranges[(size_t)range].first_row + (size_t)dm_index) * nwd + (size_t)width_index;
    double ms[2]; int64_t pv;
    AA_CUDA(cudaMemcpyAsync(ms, s.d_wstats + 2 * o, sizeof ms, cudaMemcpyDeviceToHost, s.compute), "width stats D2H");
    AA_CUDA(cudaMemcpyAsync(&pv, s.d_wpivot + o, sizeof pv, cudaMemcpyDeviceToHost, s.compute), "width stats D2H");
    AA_CUDA(cudaStreamSynchronize(s.compute), "cudaStreamSynchronize");
    if (mu) *mu = ms[0];
    if (sigma) *sigma = ms[1];
    if (pivot) *pivot = pv;
    return AA_OK;
}

extern "C" aa_status aa_get_row_moments(aa_strategy* h, int32_t range, int64_t* sum_d, int64_t* sum_td) {
    aa_status st = check_ready(h, "aa_get_row_moments");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (s.current_chunk < 0) { set_error("aa_get_row_moments: no chunk has been dedispersed yet"); return AA_ERR_ORDER; }
    if (!sum_d || !sum_td || range < 0 || range >= (int32_t)s.ranges.size()) { set_error("aa_get_row_moments: bad argument"); return AA_ERR_INVALID_ARG; }
    const Range& rg = s.ranges[(size_t)range];
    const int64_t nt = (int64_t)(s.chunks[(size_t)s.current_chunk].n_out / (uint64_t)rg.r.bin) + rg.extra;
    long long* a = s.d_moments;
    long long* b = s.d_moments + rg.r.ndms;
    AA_LAUNCH(aak_row_moments(rg.d_D, rg.pitch, nt, rg.r.ndms, a, b, s.compute), "row moments");
    AA_CUDA(cudaMemcpyAsync(sum_d, a, (size_t)rg.r.ndms * 8, cudaMemcpyDeviceToHost, s.compute), "moments D2H");
    AA_CUDA(cudaMemcpyAsync(sum_td, b, (size_t)rg.r.ndms * 8, cudaMemcpyDeviceToHost, s.compute), "moments D2H");
    AA_CUDA(cudaStreamSynchronize(s.compute), "cudaStreamSynchronize");
    return AA_OK;
}

extern "C" aa_status aa_get_last_timings(aa_strategy* h, float ms_out[5]) {
    aa_status st = check_ready(h, "aa_get_last_timings");
    if (st != AA_OK) return st;
    Strategy& s = h->s;
    if (!ms_out) { set_error("aa_get_last_timings: ms_out is NULL"); return AA_ERR_INVALID_ARG; }
    for (int i = 0; i < 5; ++i) ms_out[i] = 0.f;
    if (!s.timed) return AA_OK;
    AA_CUDA(cudaStreamSynchronize(s.compute), "cudaStreamSynchronize");
    AA_CUDA(cudaEventElapsedTime(&ms_out[0], s.ev_t[0], s.ev_t[1]), "cudaEventElapsedTime");
    AA_CUDA(cudaEventElapsedTime(&ms_out[1], s.ev_t[1], s.ev_t[2]), "cudaEventElapsedTime");
    if (s.stats_timed) {
        AA_CUDA(cudaEventElapsedTime(&ms_out[2], s.ev_t[3], s.ev_t[4]), "cudaEventElapsedTime");
        AA_CUDA(cudaEventElapsedTime(&ms_out[3], s.ev_t[4], s.ev_t[5]), "cudaEventElapsedTime");
    }
    if (s.h2d_timed) {
        AA_CUDA(cudaStreamSynchronize(s.copy), "cudaStreamSynchronize");
        AA_CUDA(cudaEventElapsedTime(&ms_out[4], s.ev_h2d[0], s.ev_h2d[1]), "cudaEventElapsedTime");
    }
    return AA_OK;
}

extern "C" aa_status aa_get_launch_count(const aa_strategy* h, uint64_t* launches) {
    if (!h || !launches) { set_error("aa_get_launch_count: NULL argument"); return h ? AA_ERR_INVALID_ARG : AA_ERR_NOT_READY; }
    *launches = h->s.launches;
    return AA_OK;
}

extern "C" aa_status aa_measure_int_add_peak(void* stream, int32_t millis, double* iadd3_per_s, double* mixed_per_s, double* sm_mhz) {
    return aa_measure_int_add_peak3(stream, millis, iadd3_per_s, mixed_per_s, nullptr, sm_mhz);
}

extern "C" aa_status aa_measure_int_add_peak3(void* stream, int32_t millis, double* iadd3_per_s, double* mixed_per_s, double* imad_per_s, double* sm_mhz) {
    cudaStream_t st = (cudaStream_t)stream;
    int dev = 0, nsm = 0;
    cudaError_t e;
    if ((e = cudaGetDevice(&dev)) != cudaSuccess) return cuda_fail(e, "cudaGetDevice");
    if ((e = cudaDeviceGetAttribute(&nsm, cudaDevAttrMultiProcessorCount, dev)) != cudaSuccess) return cuda_fail(e, "cudaDeviceGetAttribute");
    const int threads = 1024, grid = nsm;
    uint32_t* sink = nullptr; unsigned long long* cyc = nullptr;
    if ((e = cudaMalloc(&sink, (size_t)grid * threads * 4)) != cudaSuccess) return cuda_fail(e, "cudaMalloc (peak scratch)");
    if ((e = cudaMalloc(&cyc, (size_t)grid * 8)) != cudaSuccess) { cudaFree(sink); return cuda_fail(e, "cudaMalloc (peak scratch)"); }
    cudaEvent_t e0, e1;
    cudaEventCreate(&e0); cudaEventCreate(&e1);
    std::vector<unsigned long long> hc((size_t)grid);
    double rate[3] = {0, 0, 0}, mhz = 0;
    aa_status ret = AA_OK;
    if (millis < 1) millis = 1;
    for (int mode = 0; mode < 3 && ret == AA_OK; ++mode) {
        int iters = 4096;
        for (int pass = 0; pass < 2; ++pass) {       /* pass 0 calibrates the iteration count */
            cudaEventRecord(e0, st);
            int le = aak_peak_iadd(mode, iters, grid, threads, sink, cyc, st);
            cudaEventRecord(e1, st);
            if (le != 0 || (e = cudaEventSynchronize(e1)) != cudaSuccess) { ret = cuda_fail(le ? (cudaError_t)le : e, "peak microbenchmark"); break; }
            float ms = 0.f;
            cudaEventElapsedTime(&ms, e0, e1);
            if (pass == 0) {
                double want = (double)iters * (double)millis / std::max(1e-3, (double)ms);
                iters = (int)std::min(2.0e9, std::max(4096.0, want));
            } else {
                cudaMemcpy(hc.data(), cyc, (size_t)grid * 8, cudaMemcpyDeviceToHost);
                double sum = 0;
                for (unsigned long long v : hc) sum += (double)v;
                rate[mode] = (double)AAK_PEAK_ADDS_PER_THREAD_ITER * iters * (double)threads * grid / ((double)ms * 1e-3);
                mhz = (sum / grid) / ((double)ms * 1e-3) * 1e-6;
            }
        }
    }
    cudaEventDestroy(e0); cudaEventDestroy(e1);
    cudaFree(sink); cudaFree(cyc);
    if (ret != AA_OK) return ret;
    if (iadd3_per_s) *iadd3_per_s = rate[0];
    if (mixed_per_s) *mixed_per_s = rate[1];
    if (imad_per_s) *imad_per_s = rate[2];
    if (sm_mhz) *sm_mhz = mhz;
    return AA_OK;
}
