/*
 * k_input16.cu — K1 for 16-bit input samples (§3.1 step 1 "Provide telescope data, metadata":
 * back-ends deliver 8- or 16-bit samples).
 *
 * K2 adds bytes fastest (one shared-memory byte per add), and radio data are noise around a per-channel mean whatever the
 * sample type, so a 16-bit chunk is turned into the same OFFSET forms the binned 8-bit inputs use (k_misc.cu "Offset-uint8
 * form"):   x_b[c][t] = lo[c][t] + off_b[c] + r[c][t],   lo = clamp(x_b - off_b, 0, hi_b),   r = 0 except for rare outliers,
 * with hi_b = 255 (a byte, 4 sample-shifted copies) for bin 1, 2, 4 and hi_8 = 1023 (a uint16, 2 copies) for bin 8, whose noise
 * (sigma sqrt 8) does not fit a byte. K2 sums lo, adds sum_c off_b[c] to every output, and k_scatter_exceptions adds every r
 * exactly; a channel group with too many exceptions takes the global-memory kernel on the plain binned uint16 samples
 * (k_bin_time16) instead. D is therefore bit-exact for ANY input within the plan's stated sample maximum.
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include "aa_kernels.h"
#include "k_common.cuh"

namespace {

/* off_b[c] = clamp(round(b * mean_t x[c][t]) - centre_b, 0, 65535 * 8): centres the channel's noise in the window of its form;
 * any value is CORRECT. bias_b += off_b[c]. Entries k = 0..3 are b = 1, 2, 4, 8; a NULL off[k] is skipped. */
struct Off16 { int32_t* off[4]; int32_t* bias[4]; int32_t centre[4]; };

__global__ void __launch_bounds__(256)
k_chan_offsets16(const uint16_t* __restrict__ x, size_t pitch_bytes, long long len, const Off16 o, unsigned input_max,
                 unsigned* __restrict__ range_flag) {
    __shared__ unsigned long long red[8];
    const uint16_t* row = reinterpret_cast<const uint16_t*>(reinterpret_cast<const uint8_t*>(x) + (size_t)blockIdx.x * pitch_bytes);
    unsigned long long s = 0;
    unsigned mx2 = 0;                        /* largest sample seen, per 16-bit half */
    const long long nvec = len >> 3;
    for (long long q = threadIdx.x; q < nvec; q += 256) {
        const uint4 v = *reinterpret_cast<const uint4*>(row + q * 8);
        s += (v.x & 0xFFFFu) + (v.x >> 16) + (v.y & 0xFFFFu) + (v.y >> 16) + (v.z & 0xFFFFu) + (v.z >> 16) + (v.w & 0xFFFFu) + (v.w >> 16);
        mx2 = __vmaxu2(__vmaxu2(mx2, v.x), __vmaxu2(__vmaxu2(v.y, v.z), v.w));
    }
    for (long long t = (nvec << 3) + threadIdx.x; t < len; t += 256) { const unsigned v = row[t]; s += v; mx2 = __vmaxu2(mx2, v); }
    /* a sample above the plan's max_value breaks the packed 16-bit sums of K1 and the int32 bound on D: flag the chunk */
    if (range_flag && max(mx2 & 0xFFFFu, mx2 >> 16) > input_max) atomicOr(range_flag, 1u);
#pragma unroll
    for (int d = 16; d > 0; d >>= 1) s += __shfl_down_sync(0xffffffffu, s, d);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long tot = 0;
        for (int w = 0; w < 8; ++w) tot += red[w];
        const long long n = len > 0 ? len : 1;
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            if (!o.off[k]) continue;
            long long v = (long long)((((unsigned long long)(1 << k)) * tot + (unsigned long long)(n / 2)) / (unsigned long long)n) - o.centre[k];
            v = v < 0 ? 0 : (v > 65535ll * 8 ? 65535ll * 8 : v);
            o.off[k][blockIdx.x] = (int32_t)v;
            atomicAdd(o.bias[k], (int32_t)v);
        }
    }
}

/* One read of raw uint16 rows writes every offset form. A thread owns 16 raw samples and looks 16 ahead (the shifted copies
 * of the coarsest byte form need 3 more bin-4 samples = 12 raw samples). */
struct Prep16 {
    const uint16_t* raw; size_t pitch_bytes; long long ngroups; int chan0; unsigned cap;
    /* byte forms of bin 1, 2, 4 (k = 0, 1, 2): 4 copies, copy j at + j*stride, rows pitch bytes apart */
    uint8_t* lo[3]; size_t pitch[3], stride[3]; const int32_t* off[3]; uint2* exc[3]; unsigned* cnt[3]; long long nb[3];
    /* uint16 form of bin 8: 2 copies */
    uint16_t* lo8; size_t pitch8, stride8; const int32_t* off8; uint2* exc8; unsigned* cnt8; long long nb8; int hi8;
};

__global__ void __launch_bounds__(256)
k_prep16(const Prep16 p) {
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= p.ngroups) return;
    const int c = blockIdx.y;
    const uint8_t* src = reinterpret_cast<const uint8_t*>(p.raw) + (size_t)c * p.pitch_bytes + (size_t)g * 32;
    int v[32];
#pragma unroll
    for (int q = 0; q < 4; ++q) {                                       /* rows are padded: readable past the chunk */
        const uint4 w = *reinterpret_cast<const uint4*>(src + 16 * q);
        v[8 * q + 0] = (int)(w.x & 0xFFFFu); v[8 * q + 1] = (int)(w.x >> 16);
        v[8 * q + 2] = (int)(w.y & 0xFFFFu); v[8 * q + 3] = (int)(w.y >> 16);
        v[8 * q + 4] = (int)(w.z & 0xFFFFu); v[8 * q + 5] = (int)(w.z >> 16);
        v[8 * q + 6] = (int)(w.w & 0xFFFFu); v[8 * q + 7] = (int)(w.w >> 16);
    }
    const int chan = p.chan0 + c;
    if (p.lo[0]) {                                                      /* bin 1: 16 own samples + 3 ahead */
        const int oc = p.off[0][c];
        uint32_t l[19];
#pragma unroll
        for (int k = 0; k < 19; ++k) {
            const int y = v[k] - oc;
            const int q = y < 0 ? 0 : (y > 255 ? 255 : y);
            l[k] = (uint32_t)q;
            const long long t = g * 16 + k;
            if (k < 16 && y != q && t < p.nb[0]) append_exception(p.exc[0], p.cnt[0], p.cap, make_exception(chan, t, y - q));
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            uint4 o;
            o.x = l[j] | (l[j + 1] << 8) | (l[j + 2] << 16) | (l[j + 3] << 24);
            o.y = l[j + 4] | (l[j + 5] << 8) | (l[j + 6] << 16) | (l[j + 7] << 24);
            o.z = l[j + 8] | (l[j + 9] << 8) | (l[j + 10] << 16) | (l[j + 11] << 24);
            o.w = l[j + 12] | (l[j + 13] << 8) | (l[j + 14] << 16) | (l[j + 15] << 24);
            *reinterpret_cast<uint4*>(p.lo[0] + (size_t)j * p.stride[0] + (size_t)c * p.pitch[0] + (size_t)g * 16) = o;
        }
    }
    if (p.lo[1]) {                                                      /* bin 2: 8 own + 3 ahead */
        const int oc = p.off[1][c];
        uint32_t l[11];
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            const int y = v[2 * k] + v[2 * k + 1] - oc;
            const int q = y < 0 ? 0 : (y > 255 ? 255 : y);
            l[k] = (uint32_t)q;
            const long long t = g * 8 + k;
            if (k < 8 && y != q && t < p.nb[1]) append_exception(p.exc[1], p.cnt[1], p.cap, make_exception(chan, t, y - q));
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t a = l[j] | (l[j + 1] << 8) | (l[j + 2] << 16) | (l[j + 3] << 24);
            const uint32_t b = l[j + 4] | (l[j + 5] << 8) | (l[j + 6] << 16) | (l[j + 7] << 24);
            *reinterpret_cast<uint2*>(p.lo[1] + (size_t)j * p.stride[1] + (size_t)c * p.pitch[1] + (size_t)g * 8) = make_uint2(a, b);
        }
    }
    if (p.lo[2]) {                                                      /* bin 4: 4 own + 3 ahead */
        const int oc = p.off[2][c];
        uint32_t l[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) {
            const int y = v[4 * k] + v[4 * k + 1] + v[4 * k + 2] + v[4 * k + 3] - oc;
            const int q = y < 0 ? 0 : (y > 255 ? 255 : y);
            l[k] = (uint32_t)q;
            const long long t = g * 4 + k;
            if (k < 4 && y != q && t < p.nb[2]) append_exception(p.exc[2], p.cnt[2], p.cap, make_exception(chan, t, y - q));
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
            *reinterpret_cast<uint32_t*>(p.lo[2] + (size_t)j * p.stride[2] + (size_t)c * p.pitch[2] + (size_t)g * 4) =
                l[j] | (l[j + 1] << 8) | (l[j + 2] << 16) | (l[j + 3] << 24);
    }
    if (p.lo8) {                                                        /* bin 8: 2 own + 1 ahead, uint16 window [0, hi8] */
        const int oc = p.off8[c];
        uint32_t l[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            int y = -oc;
#pragma unroll
            for (int j = 0; j < 8; ++j) y += v[8 * k + j];
            const int q = y < 0 ? 0 : (y > p.hi8 ? p.hi8 : y);
            l[k] = (uint32_t)q;
            const long long t = g * 2 + k;
            if (k < 2 && y != q && t < p.nb8) append_exception(p.exc8, p.cnt8, p.cap, make_exception(chan, t, y - q));
        }
        uint8_t* d0 = reinterpret_cast<uint8_t*>(p.lo8) + (size_t)c * p.pitch8 + (size_t)g * 4;
        *reinterpret_cast<uint32_t*>(d0) = l[0] | (l[1] << 16);
        *reinterpret_cast<uint32_t*>(d0 + p.stride8) = l[1] | (l[2] << 16);
    }
}

/* Plain binned uint16 samples x_b (no offset), one copy: the input of the global-memory route of exception-heavy chunks.
 * Runs only if *only_if_cnt > only_if_above (NULL: always). One thread turns 8 raw samples into 8/B outputs. */
template <int B>
__global__ void __launch_bounds__(256)
k_bin_time16(const uint16_t* __restrict__ x, size_t x_pitch_bytes, uint16_t* __restrict__ xb, size_t xb_pitch_bytes, long long ngroups,
             const unsigned* __restrict__ only_if_cnt, unsigned only_if_above) {
    if (only_if_cnt && *only_if_cnt <= only_if_above) return;
    const int c = blockIdx.y;
#pragma unroll 1
    for (int it = 0; it < 8; ++it) {
        const long long g = ((long long)blockIdx.x * 8 + it) * blockDim.x + threadIdx.x;
        if (g >= ngroups) return;
        const uint4 w = *reinterpret_cast<const uint4*>(reinterpret_cast<const uint8_t*>(x) + (size_t)c * x_pitch_bytes + (size_t)g * 16);
        const uint32_t v[8] = {w.x & 0xFFFFu, w.x >> 16, w.y & 0xFFFFu, w.y >> 16, w.z & 0xFFFFu, w.z >> 16, w.w & 0xFFFFu, w.w >> 16};
        uint8_t* dst = reinterpret_cast<uint8_t*>(xb) + (size_t)c * xb_pitch_bytes + (size_t)g * (16 / B);
        if (B == 1) *reinterpret_cast<uint4*>(dst) = w;
        else if (B == 2) *reinterpret_cast<uint2*>(dst) = make_uint2((v[0] + v[1]) | ((v[2] + v[3]) << 16), (v[4] + v[5]) | ((v[6] + v[7]) << 16));
        else if (B == 4) *reinterpret_cast<uint32_t*>(dst) = (v[0] + v[1] + v[2] + v[3]) | ((v[4] + v[5] + v[6] + v[7]) << 16);
        else *reinterpret_cast<uint16_t*>(dst) = (uint16_t)(v[0] + v[1] + v[2] + v[3] + v[4] + v[5] + v[6] + v[7]);
    }
}

/* Corner turn of a time-major 16-bit chunk x_tm[t][c] into channel-major rows x[c][t]: 64 x 64 tiles through shared memory
 * (one padding word per row keeps both phases free of bank conflicts). */
__global__ void __launch_bounds__(256)
k_corner_turn16(const uint16_t* __restrict__ in, size_t in_stride_bytes, uint16_t* __restrict__ out, size_t out_pitch_bytes, int nchans,
                long long nsamp) {
    __shared__ uint32_t T[64][33];                                   /* T[t][c/2] = channels (c, c+1) of sample t */
    const int x = threadIdx.x & 31, y = threadIdx.x >> 5;
    const long long t_tile = (long long)blockIdx.x * 64;
    const int c_tile = blockIdx.y * 64;
    for (int r = y; r < 64; r += 8) {
        const long long t = t_tile + r;
        const int c = c_tile + 2 * x;
        uint32_t w = 0;
        if (t < nsamp && c < nchans) w = *reinterpret_cast<const uint32_t*>(reinterpret_cast<const uint8_t*>(in) + (size_t)t * in_stride_bytes + (size_t)c * 2);
        T[r][x] = w;
    }
    __syncthreads();
    for (int r = y; r < 64; r += 8) {                                 /* r = channel inside the tile; lane x = samples 2x, 2x+1 */
        const int c = c_tile + r;
        if (c >= nchans) break;
        const uint32_t a = T[2 * x][r >> 1], b = T[2 * x + 1][r >> 1];
        const uint32_t v = (r & 1) ? ((a >> 16) | (b & 0xFFFF0000u)) : ((a & 0xFFFFu) | (b << 16));
        const long long t = t_tile + 2 * x;
        if (t < nsamp) *reinterpret_cast<uint32_t*>(reinterpret_cast<uint8_t*>(out) + (size_t)c * out_pitch_bytes + (size_t)t * 2) = v;   /* rows are padded to 256 bytes */
    }
}

}  // namespace

extern "C" int aak_chan_offsets16(const uint16_t* x, size_t pitch_bytes, int64_t len, int32_t nrows, int32_t* const off[4], int32_t* const bias[4],
                                  const int32_t centre[4], uint32_t input_max, unsigned* range_flag, void* stream) {
    if (nrows <= 0) return 0;
    Off16 o;
    for (int k = 0; k < 4; ++k) { o.off[k] = off[k]; o.bias[k] = bias[k]; o.centre[k] = centre[k]; }
    k_chan_offsets16<<<(unsigned)nrows, 256, 0, (cudaStream_t)stream>>>(x, pitch_bytes, len, o, input_max, range_flag);
    return (int)cudaGetLastError();
}

extern "C" int aak_prep16(const aak_prep16_args* a, int32_t nrows, void* stream) {
    if (nrows <= 0 || a->ngroups <= 0) return 0;
    Prep16 p;
    p.raw = a->raw; p.pitch_bytes = a->pitch_bytes; p.ngroups = a->ngroups; p.chan0 = a->chan0; p.cap = a->cap;
    for (int k = 0; k < 3; ++k) {
        p.lo[k] = a->lo[k]; p.pitch[k] = a->pitch[k]; p.stride[k] = a->stride[k]; p.off[k] = a->off[k]; p.exc[k] = a->exc[k]; p.cnt[k] = a->cnt[k];
        p.nb[k] = a->nb[k];
    }
    p.lo8 = a->lo8; p.pitch8 = a->pitch8; p.stride8 = a->stride8; p.off8 = a->off8; p.exc8 = a->exc8; p.cnt8 = a->cnt8; p.nb8 = a->nb8; p.hi8 = a->hi8;
    dim3 grid((unsigned)((a->ngroups + 255) / 256), (unsigned)nrows);
    k_prep16<<<grid, 256, 0, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}

extern "C" int aak_bin_time16(const uint16_t* x, size_t x_pitch_bytes, uint16_t* xb, size_t xb_pitch_bytes, int32_t nchans, int64_t nbinned,
                              int32_t bin, const unsigned* only_if_cnt, unsigned only_if_above, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const long long ngroups = (nbinned * bin + 7) / 8;
    if (ngroups <= 0 || nchans <= 0) return 0;
    dim3 grid((unsigned)((ngroups + 256 * 8 - 1) / (256 * 8)), (unsigned)nchans);
    switch (bin) {
        case 1: k_bin_time16<1><<<grid, 256, 0, st>>>(x, x_pitch_bytes, xb, xb_pitch_bytes, ngroups, only_if_cnt, only_if_above); break;
        case 2: k_bin_time16<2><<<grid, 256, 0, st>>>(x, x_pitch_bytes, xb, xb_pitch_bytes, ngroups, only_if_cnt, only_if_above); break;
        case 4: k_bin_time16<4><<<grid, 256, 0, st>>>(x, x_pitch_bytes, xb, xb_pitch_bytes, ngroups, only_if_cnt, only_if_above); break;
        case 8: k_bin_time16<8><<<grid, 256, 0, st>>>(x, x_pitch_bytes, xb, xb_pitch_bytes, ngroups, only_if_cnt, only_if_above); break;
        default: return (int)cudaErrorInvalidValue;
    }
    return (int)cudaGetLastError();
}

extern "C" int aak_corner_turn16(const uint16_t* in, size_t in_stride_bytes, uint16_t* out, size_t out_pitch_bytes, int32_t nchans, int64_t nsamp,
                                 void* stream) {
    if (((uintptr_t)in & 3) || (in_stride_bytes & 3) || (out_pitch_bytes & 3) || in_stride_bytes < (size_t)(((nchans + 1) & ~1) * 2)) return (int)cudaErrorInvalidValue;
    if (nsamp <= 0 || nchans <= 0) return 0;
    dim3 grid((unsigned)((nsamp + 63) / 64), (unsigned)((nchans + 63) / 64));
    k_corner_turn16<<<grid, 256, 0, (cudaStream_t)stream>>>(in, in_stride_bytes, out, out_pitch_bytes, nchans, nsamp);
    return (int)cudaGetLastError();
}
