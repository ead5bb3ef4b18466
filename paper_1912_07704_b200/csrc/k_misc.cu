/*
 * k_misc.cu — K1 (time binning), K5 (row-moment test hook) and K0 (integer-add peak microbenchmark) for sm_100a.
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include "aa_kernels.h"
#include "k_common.cuh"

namespace {

constexpr int K1_GROUPS_PER_THREAD = 8;   /* 16-byte groups per thread of the binning / shifted-copy kernels */

/* ---- K1: x_b[c][t'] = sum_{j<b} x[c][b*t'+j] (north_star "DM ranges that decimate in time by 1/2/4/8";
 * DESIGN.md reading C4: binning is a SUM held in uint16). One thread turns 16 input bytes into 16/b outputs. */
template <int B>
__global__ void __launch_bounds__(256)
k_bin_time(const uint8_t* __restrict__ x, size_t x_pitch, uint16_t* __restrict__ xb, size_t xb_pitch, long long ngroups,
           const unsigned* __restrict__ only_if_cnt, unsigned only_if_above) {
    if (only_if_cnt && *only_if_cnt <= only_if_above) return;      /* the offset-uint8 route handles this chunk */
    const int c = blockIdx.y;
#pragma unroll 1
    for (int it = 0; it < K1_GROUPS_PER_THREAD; ++it) {            /* few, fat CTAs: a skipped launch costs microseconds */
    const long long g = ((long long)blockIdx.x * K1_GROUPS_PER_THREAD + it) * blockDim.x + threadIdx.x;
    if (g >= ngroups) return;
    const uint4 v = *reinterpret_cast<const uint4*>(x + (size_t)c * x_pitch + (size_t)g * 16);
    const uint32_t w[4] = {v.x, v.y, v.z, v.w};
    uint16_t o[16 / B];
#pragma unroll
    for (int k = 0; k < 16 / B; ++k) {
        uint32_t s = 0;
#pragma unroll
        for (int j = 0; j < B; ++j) {
            const int byte = k * B + j;
            s += (w[byte >> 2] >> (8 * (byte & 3))) & 0xFFu;
        }
        o[k] = (uint16_t)s;
    }
    uint16_t* dst = xb + (size_t)c * xb_pitch + (size_t)g * (16 / B);
    if (B == 2) {
        uint4 r;
        r.x = o[0] | ((uint32_t)o[1] << 16); r.y = o[2] | ((uint32_t)o[3] << 16);
        r.z = o[4] | ((uint32_t)o[5] << 16); r.w = o[6] | ((uint32_t)o[7] << 16);
        *reinterpret_cast<uint4*>(dst) = r;
    } else if (B == 4) {
        uint2 r;
        r.x = o[0] | ((uint32_t)o[1] << 16); r.y = o[2] | ((uint32_t)o[3] << 16);
        *reinterpret_cast<uint2*>(dst) = r;
    } else {
        *reinterpret_cast<uint32_t*>(dst) = o[0] | ((uint32_t)o[1] << 16);
    }
    }
}

/* ---- K1b: out[c][j] = in[c][j + shift] (shift = 1, 2 or 3 bytes): the sample-shifted copies K2's TMA loads need
 * (TMA wants 16-byte aligned global coordinates, so a window at an odd sample offset is read from a shifted copy). */
__global__ void __launch_bounds__(256)
k_shift_copy(const uint8_t* __restrict__ in, uint8_t* __restrict__ out, size_t pitch, long long ngroups, int shift,
             const unsigned* __restrict__ only_if_cnt, unsigned only_if_above) {
    if (only_if_cnt && *only_if_cnt <= only_if_above) return;
#pragma unroll 1
    for (int it = 0; it < K1_GROUPS_PER_THREAD; ++it) {
    const long long g = ((long long)blockIdx.x * K1_GROUPS_PER_THREAD + it) * blockDim.x + threadIdx.x;
    if (g >= ngroups) return;
    const uint8_t* src = in + (size_t)blockIdx.y * pitch + (size_t)g * 16;
    const uint4 a = *reinterpret_cast<const uint4*>(src);
    /* The last group of a row has no look-ahead word: its last `shift` output bytes would be in[row_bytes ..], which lie past the
     * row (padding no reader uses) and are written as zero. Reading src + 16 there would also be a data race when the copies are
     * interleaved in one buffer (out = in + row_bytes, the uint16 forms): that word is the first word of THIS launch's output. */
    const uint32_t nx = g + 1 < ngroups ? *reinterpret_cast<const uint32_t*>(src + 16) : 0u;
    const int bs = shift * 8;
    uint4 o;
    o.x = __funnelshift_r(a.x, a.y, bs);
    o.y = __funnelshift_r(a.y, a.z, bs);
    o.z = __funnelshift_r(a.z, a.w, bs);
    o.w = __funnelshift_r(a.w, nx, bs);
    *reinterpret_cast<uint4*>(out + (size_t)blockIdx.y * pitch + (size_t)g * 16) = o;
    }
}

/* ---- K0t: corner turn. Telescopes deliver TIME-major samples x_tm[t][c] (PAPER.md:47 step 1 "telescope data");
 * the dedispersion kernels read CHANNEL-major rows x[c][t]. A CTA transposes a 128-channel x 128-sample tile:
 * each thread loads 4 words = 4 samples x 4 channels, transposes the 4x4 bytes in registers (8 PRMT), and stores four
 * words (one channel x 4 samples each) into an XOR-swizzled shared-memory tile, so that both the stores and the
 * row reads that follow are bank-conflict free; a warp then writes one 128-byte channel row segment per instruction. */
constexpr int CT_TILE = 128;
__global__ void __launch_bounds__(256)
k_corner_turn(const uint8_t* __restrict__ in, size_t in_stride, uint8_t* __restrict__ out, size_t out_pitch, int nchans, long long nsamp) {
    __shared__ uint32_t T[CT_TILE][32];                          /* T[c][(t/4) ^ (c/4)] = 4 consecutive samples of channel c */
    const int x = threadIdx.x & 31, y = threadIdx.x >> 5;
    const long long t_tile = (long long)blockIdx.x * CT_TILE;
    const int c_tile = blockIdx.y * CT_TILE;
    const int c0 = c_tile + 4 * x;
#pragma unroll
    for (int q = 0; q < 4; ++q) {
        const int tq = y + 8 * q;                                /* sample quad inside the tile */
        uint32_t w[4];
#pragma unroll
        for (int k = 0; k < 4; ++k) {
            const long long t = t_tile + 4 * tq + k;
            w[k] = (t < nsamp && c0 < nchans) ? *reinterpret_cast<const uint32_t*>(in + (size_t)t * in_stride + c0) : 0u;
        }
        /* 4x4 byte transpose: o[j] = (w0.bj, w1.bj, w2.bj, w3.bj) */
        const uint32_t a0 = __byte_perm(w[0], w[1], 0x5140), a1 = __byte_perm(w[0], w[1], 0x7362);
        const uint32_t b0 = __byte_perm(w[2], w[3], 0x5140), b1 = __byte_perm(w[2], w[3], 0x7362);
        const uint32_t o0 = __byte_perm(a0, b0, 0x5410), o1 = __byte_perm(a0, b0, 0x7632);
        const uint32_t o2 = __byte_perm(a1, b1, 0x5410), o3 = __byte_perm(a1, b1, 0x7632);
        T[4 * x + 0][tq ^ x] = o0;
        T[4 * x + 1][tq ^ x] = o1;
        T[4 * x + 2][tq ^ x] = o2;
        T[4 * x + 3][tq ^ x] = o3;
    }
    __syncthreads();
    for (int r = y; r < CT_TILE; r += 8) {
        const int c = c_tile + r;
        if (c >= nchans) break;
        const uint32_t v = T[r][x ^ (r >> 2)];
        const long long t = t_tile + 4 * x;
        if (t < nsamp) *reinterpret_cast<uint32_t*>(out + (size_t)c * out_pitch + (size_t)t) = v;   /* rows are padded to 256 bytes */
    }
}

/* ---- Offset-uint8 form of a binned input (ranges with bin 2 and 4). A binned sample x_b <= 255*b needs 9-10 bits, and as
 * uint16 it costs K2 two shared-memory bytes per add - the crossbar is what limits K2. Radio data are noise around a
 * per-channel mean, so x_b - off_c (off_c = the channel's mean binned value - 128) fits a byte almost always:
 *     x_b[c][t] = lo[c][t] + off_c + r[c][t],   lo = clamp(x_b - off_c, 0, 255),   r = 0 except for rare outliers.
 * K2 then runs its 1-byte path on lo (half the shared-memory traffic), adds sum_c off_c to every output, and the few
 * (c, t, r != 0) EXCEPTIONS are scattered into D exactly by k_scatter_exceptions. Nothing is approximated: if a chunk has
 * too many exceptions (counter above `cap`), the uint16 kernels run instead (every kernel of both routes tests the same
 * counter and returns at once when it is not its turn). */
__global__ void __launch_bounds__(256)
k_chan_offsets(const uint8_t* __restrict__ x, size_t pitch, long long len, int32_t* __restrict__ off2, int32_t* __restrict__ off4,
               int32_t* __restrict__ off8, int32_t* __restrict__ bias2, int32_t* __restrict__ bias4, int32_t* __restrict__ bias8) {
    __shared__ unsigned long long red[8];
    const uint8_t* row = x + (size_t)blockIdx.x * pitch;
    unsigned long long s = 0;
    const long long nvec = len >> 4;
    for (long long q = threadIdx.x; q < nvec; q += 256) {
        const uint4 v = *reinterpret_cast<const uint4*>(row + q * 16);
        s += __dp4a(v.x, 0x01010101u, 0u) + __dp4a(v.y, 0x01010101u, 0u) + __dp4a(v.z, 0x01010101u, 0u) + __dp4a(v.w, 0x01010101u, 0u);
    }
    for (long long t = (nvec << 4) + threadIdx.x; t < len; t += 256) s += row[t];
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) s += __shfl_down_sync(0xffffffffu, s, o);
    if ((threadIdx.x & 31) == 0) red[threadIdx.x >> 5] = s;
    __syncthreads();
    if (threadIdx.x == 0) {
        unsigned long long tot = 0;
        for (int w = 0; w < 8; ++w) tot += red[w];
        const long long n = len > 0 ? len : 1;
        /* any offset is CORRECT; this one centres the channel's noise on 128 */
        if (off2) { long long o = (long long)((2 * tot + n / 2) / n) - 128; o = o < 0 ? 0 : (o > 255 ? 255 : o); off2[blockIdx.x] = (int32_t)o; atomicAdd(bias2, (int32_t)o); }
        if (off4) { long long o = (long long)((4 * tot + n / 2) / n) - 128; o = o < 0 ? 0 : (o > 765 ? 765 : o); off4[blockIdx.x] = (int32_t)o; atomicAdd(bias4, (int32_t)o); }
        /* bin 8, half-byte form: (x_8 - off) >> 1 is centred on 128 */
        if (off8) { long long o = (long long)((8 * tot + n / 2) / n) - 256; o = o < 0 ? 0 : (o > 1785 ? 1785 : o); off8[blockIdx.x] = (int32_t)o; atomicAdd(bias8, (int32_t)o); }
    }
}

/* D[i][t - delay(c, i)] += r for every exception (c, t, r) and every DM trial i of one range. The delay is reading C2
 * evaluated in IEEE double with explicit round-to-nearest operations, the same operation order as the host tables. */
__global__ void __launch_bounds__(256)
k_scatter_exceptions(const uint2* __restrict__ exc, const unsigned* __restrict__ exc_cnt, unsigned cap, const double* __restrict__ k,
                     double dm_low, double dm_step, int ndms, int bin, long long nt, int32_t* __restrict__ D, long long pitch) {
    const unsigned n = *exc_cnt;
    if (n > cap) return;                                               /* dense chunk: the uint16 route produced D */
    const unsigned long long total = (unsigned long long)n * (unsigned)ndms;
    for (unsigned long long q = (unsigned long long)blockIdx.x * blockDim.x + threadIdx.x; q < total; q += (unsigned long long)gridDim.x * blockDim.x) {
        const unsigned e = (unsigned)(q / (unsigned)ndms);
        const int i = (int)(q - (unsigned long long)e * (unsigned)ndms);
        const uint2 rec = exc[e];
        const int c = (int)(rec.x & 0xFFFFu);
        const int r = ((int)(((rec.x >> 16) | ((rec.y >> 28) << 16)) << 12)) >> 12;          /* sign-extend 20 bits */
        const double dm = __dadd_rn(dm_low, __dmul_rn((double)i, dm_step));
        const long long delay = llround(__ddiv_rn(__dmul_rn(k[c], dm), (double)bin));
        const long long t = (long long)(rec.y & 0x0FFFFFFFu) - delay;
        if (t >= 0 && t < nt) atomicAdd(D + (size_t)i * (size_t)pitch + (size_t)t, r);
    }
}

/* ---- K1 fused: ONE read of the raw chunk produces everything K2's TMA windows need: the 4 sample-shifted uint8 copies,
 * the offset-uint8 forms of the bin-2 and bin-4 inputs (4 shifted byte copies each, exceptions appended), and the two
 * copies of the uint16 bin-8 input. A thread owns 16 raw samples and looks 16 samples ahead for the shifted copies.
 * (The uint16 forms of bin 2 / 4 are written by k_bin_time / k_shift_copy, only for exception-heavy chunks.) */
struct PrepFused {
    const uint8_t* raw; size_t pitch; long long ngroups; int chan0; unsigned cap;
    uint8_t* x4; size_t x4_pitch, x4_stride;
    uint8_t* lo2; size_t lo2_pitch, lo2_stride; const int32_t* off2; uint2* exc2; unsigned* cnt2; long long nb2;
    uint8_t* lo4; size_t lo4_pitch, lo4_stride; const int32_t* off4; uint2* exc4; unsigned* cnt4; long long nb4;
    uint16_t* xb8; size_t xb8_pitch, xb8_stride;
    /* half-byte form of bin 8: hb8 = 4 byte copies of y = clamp((x_8 - off8) >> 1, 0, 255), bits8 = the dropped low bits, one
     * bit per sample (bit k of word w of a row = sample 32 w + k), exceptions r = x_8 - off8 - 2 y - bit */
    uint8_t* hb8; size_t hb8_pitch, hb8_stride; const int32_t* off8; uint2* exc8; unsigned* cnt8; long long nb8;
    uint32_t* bits8; size_t bits8_pitch;
};

__device__ __forceinline__ uint32_t spread16(uint32_t x) {             /* bit k of the low half -> bit 2k */
    x = (x | (x << 8)) & 0x00FF00FFu; x = (x | (x << 4)) & 0x0F0F0F0Fu; x = (x | (x << 2)) & 0x33333333u; x = (x | (x << 1)) & 0x55555555u;
    return x;
}

__device__ __forceinline__ uint32_t byte_of(const uint32_t (&w)[8], int i) { return (w[i >> 2] >> (8 * (i & 3))) & 0xFFu; }


__global__ void __launch_bounds__(256)
k_prep_fused(const PrepFused p) {
    const long long g = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    if (g >= p.ngroups) return;                                         /* ngroups is a multiple of 16: whole half-warps leave */
    const int c = blockIdx.y;
    const uint8_t* src = p.raw + (size_t)c * p.pitch + (size_t)g * 16;
    const uint4 a = *reinterpret_cast<const uint4*>(src);
    const uint4 n = *reinterpret_cast<const uint4*>(src + 16);          /* rows are padded: readable past the chunk */
    const uint32_t w[8] = {a.x, a.y, a.z, a.w, n.x, n.y, n.z, n.w};
    if (p.x4) {
        const size_t off = (size_t)c * p.x4_pitch + (size_t)g * 16;
        *reinterpret_cast<uint4*>(p.x4 + off) = a;
#pragma unroll
        for (int k = 1; k < 4; ++k) {
            uint4 o;
            o.x = __funnelshift_r(a.x, a.y, 8 * k); o.y = __funnelshift_r(a.y, a.z, 8 * k);
            o.z = __funnelshift_r(a.z, a.w, 8 * k); o.w = __funnelshift_r(a.w, n.x, 8 * k);
            *reinterpret_cast<uint4*>(p.x4 + (size_t)k * p.x4_stride + off) = o;
        }
    }
    if (p.lo2) {
        const int oc = p.off2[c];
        uint32_t l[11];
#pragma unroll
        for (int k = 0; k < 11; ++k) {
            /* x_2 - off in ONE instruction: IDP.2A sums the two bytes of a half word into the accumulator (-off) */
            const int y = (int)((k & 1) ? __dp2a_hi(0x00010001u, w[k >> 1], (unsigned)-oc) : __dp2a_lo(0x00010001u, w[k >> 1], (unsigned)-oc));
            const int v = y < 0 ? 0 : (y > 255 ? 255 : y);
            l[k] = (uint32_t)v;
            const long long t = g * 8 + k;
            if (k < 8 && y != v && t < p.nb2)
                append_exception(p.exc2, p.cnt2, p.cap, make_exception(p.chan0 + c, t, y - v));
        }
#pragma unroll
        for (int j = 0; j < 4; ++j) {
            const uint32_t lo = l[j] | (l[j + 1] << 8) | (l[j + 2] << 16) | (l[j + 3] << 24);
            const uint32_t hi = l[j + 4] | (l[j + 5] << 8) | (l[j + 6] << 16) | (l[j + 7] << 24);
            *reinterpret_cast<uint2*>(p.lo2 + (size_t)j * p.lo2_stride + (size_t)c * p.lo2_pitch + (size_t)g * 8) = make_uint2(lo, hi);
        }
    }
    if (p.lo4) {
        const int oc = p.off4[c];
        uint32_t l[7];
#pragma unroll
        for (int k = 0; k < 7; ++k) {
            const int y = (int)__dp4a(w[k], 0x01010101u, (unsigned)-oc);      /* x_4 - off: IDP.4A */
            const int v = y < 0 ? 0 : (y > 255 ? 255 : y);
            l[k] = (uint32_t)v;
            const long long t = g * 4 + k;
            if (k < 4 && y != v && t < p.nb4)
                append_exception(p.exc4, p.cnt4, p.cap, make_exception(p.chan0 + c, t, y - v));
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
            *reinterpret_cast<uint32_t*>(p.lo4 + (size_t)j * p.lo4_stride + (size_t)c * p.lo4_pitch + (size_t)g * 4) =
                l[j] | (l[j + 1] << 8) | (l[j + 2] << 16) | (l[j + 3] << 24);
    }
    if (p.hb8) {
        /* 2 own samples of bin 8 and 3 ahead (the 4 shifted copies): 40 raw samples */
        const uint2 n2 = *reinterpret_cast<const uint2*>(src + 32);
        const int oc = p.off8[c];
        uint32_t y[5], bit[2] = {0u, 0u};
#pragma unroll
        for (int k = 0; k < 5; ++k) {
            const uint32_t wa = k < 4 ? w[2 * k] : n2.x, wb = k < 4 ? w[2 * k + 1] : n2.y;
            const int z = (int)__dp4a(wa, 0x01010101u, __dp4a(wb, 0x01010101u, (unsigned)-oc));     /* x_8 - off */
            const int h = z >> 1;                                       /* arithmetic: floor(z / 2), z = 2 h + (z & 1) */
            const int v = h < 0 ? 0 : (h > 255 ? 255 : h);
            y[k] = (uint32_t)v;
            const long long t = g * 2 + k;
            if (k < 2) {
                bit[k] = (uint32_t)(z & 1);
                if (h != v && t < p.nb8) append_exception(p.exc8, p.cnt8, p.cap, make_exception(p.chan0 + c, t, z - 2 * v - (z & 1)));
            }
        }
#pragma unroll
        for (int j = 0; j < 4; ++j)
            *reinterpret_cast<uint16_t*>(p.hb8 + (size_t)j * p.hb8_stride + (size_t)c * p.hb8_pitch + (size_t)g * 2) = (uint16_t)(y[j] | (y[j + 1] << 8));
        /* the bit plane: lane L of the warp holds samples 2L, 2L+1 of a 64-sample run */
        const int lane = threadIdx.x & 31;
        const unsigned am = (g - lane + 16 < p.ngroups) ? 0xffffffffu : 0x0000ffffu;   /* the lanes that did not leave at the top */
        const uint32_t m0 = __ballot_sync(am, bit[0]), m1 = __ballot_sync(am, bit[1]);
        if ((lane & 15) == 0) {
            const uint32_t h0 = lane ? (m0 >> 16) : (m0 & 0xFFFFu), h1 = lane ? (m1 >> 16) : (m1 & 0xFFFFu);
            p.bits8[(size_t)c * p.bits8_pitch + (size_t)(g >> 4)] = spread16(h0) | (spread16(h1) << 1);
        }
    }
    if (p.xb8) {
        uint32_t s8[3];
#pragma unroll
        for (int k = 0; k < 3; ++k) {
            uint32_t t = 0;
#pragma unroll
            for (int j = 0; j < 8; ++j) t += byte_of(w, 8 * k + j);
            s8[k] = t;
        }
        uint8_t* d0 = reinterpret_cast<uint8_t*>(p.xb8 + (size_t)c * p.xb8_pitch + (size_t)g * 2);
        *reinterpret_cast<uint32_t*>(d0) = s8[0] | (s8[1] << 16);
        *reinterpret_cast<uint32_t*>(d0 + p.xb8_stride) = s8[1] | (s8[2] << 16);
    }
}

/* ---- K5: sum_t D[i][t] and sum_t t*D[i][t] per row, int64 (all-rows checksum against the prefix-sum identity) */
__global__ void __launch_bounds__(256)
k_row_moments(const int32_t* __restrict__ D, long long pitch, long long nt, long long* __restrict__ sum_d,
              long long* __restrict__ sum_td) {
    __shared__ long long red[16];
    const int32_t* row = D + (size_t)blockIdx.x * (size_t)pitch;
    long long a = 0, b = 0;
    for (long long t = threadIdx.x; t < nt; t += blockDim.x) { const long long v = row[t]; a += v; b += v * t; }
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) { a += __shfl_down_sync(0xffffffffu, a, o); b += __shfl_down_sync(0xffffffffu, b, o); }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    if (lane == 0) { red[warp * 2] = a; red[warp * 2 + 1] = b; }
    __syncthreads();
    if (threadIdx.x == 0) {
        long long sa = 0, sb = 0;
        for (int w = 0; w < 8; ++w) { sa += red[w * 2]; sb += red[w * 2 + 1]; }
        sum_d[blockIdx.x] = sa; sum_td[blockIdx.x] = sb;
    }
}

/* ---- K0: sustained 32-bit integer add rate. 16 independent chains per thread, each step one add instruction.
 * mode 0: every step an IADD3 (ALU pipe). mode 1: chains alternate IADD3 and IMAD (x*m + y with a runtime m = 1),
 * which is how a kernel spreads integer adds over both 64-lane integer-capable pipes of an SM. */
__global__ void __launch_bounds__(1024)
k_peak_iadd(int mode, int iters, uint32_t* __restrict__ sink, unsigned long long* __restrict__ cycles, uint32_t b, uint32_t m) {
    uint32_t a[AAK_PEAK_ADDS_PER_THREAD_ITER];
#pragma unroll
    for (int i = 0; i < AAK_PEAK_ADDS_PER_THREAD_ITER; ++i) a[i] = b * (i + 1) + threadIdx.x;
    __syncthreads();
    const unsigned long long t0 = clock64();
    if (mode == 0) {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < AAK_PEAK_ADDS_PER_THREAD_ITER; ++i)
                asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(a[i]) : "r"(b), "r"(m));   /* one IADD3 */
        }
    } else if (mode == 2) {                                       /* every step an IMAD (FMA pipe only) */
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < AAK_PEAK_ADDS_PER_THREAD_ITER; ++i)
                asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a[i]) : "r"(b), "r"(m));
        }
    } else {
        for (int it = 0; it < iters; ++it) {
#pragma unroll
            for (int i = 0; i < AAK_PEAK_ADDS_PER_THREAD_ITER; i += 2) {
                asm volatile("{.reg .u32 t; add.u32 t, %0, %1; add.u32 %0, t, %2;}" : "+r"(a[i]) : "r"(b), "r"(m));
                asm volatile("mad.lo.u32 %0, %1, %2, %0;" : "+r"(a[i + 1]) : "r"(b), "r"(m));                        /* IMAD */
            }
        }
    }
    const unsigned long long t1 = clock64();
    uint32_t s = 0;
#pragma unroll
    for (int i = 0; i < AAK_PEAK_ADDS_PER_THREAD_ITER; ++i) s += a[i];
    sink[(size_t)blockIdx.x * blockDim.x + threadIdx.x] = s;
    if (threadIdx.x == 0) cycles[blockIdx.x] = t1 - t0;
}

}  // namespace

extern "C" int aak_bin_time(const uint8_t* x, size_t x_pitch, uint16_t* xb, size_t xb_pitch_elems, int32_t nchans,
                            int64_t nbinned, int32_t bin, const unsigned* only_if_cnt, unsigned only_if_above, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const long long ngroups = (nbinned * bin + 15) / 16;
    dim3 grid((unsigned)((ngroups + 256 * K1_GROUPS_PER_THREAD - 1) / (256 * K1_GROUPS_PER_THREAD)), (unsigned)nchans);
    switch (bin) {
        case 2: k_bin_time<2><<<grid, 256, 0, st>>>(x, x_pitch, xb, xb_pitch_elems, ngroups, only_if_cnt, only_if_above); break;
        case 4: k_bin_time<4><<<grid, 256, 0, st>>>(x, x_pitch, xb, xb_pitch_elems, ngroups, only_if_cnt, only_if_above); break;
        case 8: k_bin_time<8><<<grid, 256, 0, st>>>(x, x_pitch, xb, xb_pitch_elems, ngroups, only_if_cnt, only_if_above); break;
        default: return (int)cudaErrorInvalidValue;
    }
    return (int)cudaGetLastError();
}

extern "C" int aak_shift_copy(const uint8_t* in, uint8_t* out, size_t pitch, size_t row_bytes, int32_t nrows, int32_t shift_bytes,
                              const unsigned* only_if_cnt, unsigned only_if_above, void* stream) {
    if (shift_bytes < 1 || shift_bytes > 3 || (row_bytes & 15) || (pitch & 15)) return (int)cudaErrorInvalidValue;
    const long long ngroups = (long long)(row_bytes / 16);
    dim3 grid((unsigned)((ngroups + 256 * K1_GROUPS_PER_THREAD - 1) / (256 * K1_GROUPS_PER_THREAD)), (unsigned)nrows);
    k_shift_copy<<<grid, 256, 0, (cudaStream_t)stream>>>(in, out, pitch, ngroups, shift_bytes, only_if_cnt, only_if_above);
    return (int)cudaGetLastError();
}

extern "C" int aak_row_moments(const int32_t* D, int64_t pitch, int64_t nt, int32_t ndms, long long* sum_d, long long* sum_td,
                               void* stream) {
    k_row_moments<<<(unsigned)ndms, 256, 0, (cudaStream_t)stream>>>(D, pitch, nt, sum_d, sum_td);
    return (int)cudaGetLastError();
}

extern "C" int aak_peak_iadd(int32_t mode, int32_t iters, int32_t grid, int32_t threads, uint32_t* sink,
                             unsigned long long* cycles_out, void* stream) {
    k_peak_iadd<<<(unsigned)grid, (unsigned)threads, 0, (cudaStream_t)stream>>>(mode, iters, sink, cycles_out, 12345u, 1u);
    return (int)cudaGetLastError();
}

/* in: [nsamp][in_stride] time-major (in_stride >= round_up(nchans, 4), in and in_stride 4-byte aligned);
 * out: [nchans][out_pitch] channel-major, out_pitch a multiple of 4 with room for round_up(nsamp, 4) bytes per row. */
extern "C" int aak_corner_turn(const uint8_t* in, size_t in_stride, uint8_t* out, size_t out_pitch, int32_t nchans, int64_t nsamp,
                               void* stream) {
    if (((uintptr_t)in & 3) || (in_stride & 3) || (out_pitch & 3) || in_stride < (size_t)((nchans + 3) & ~3)) return (int)cudaErrorInvalidValue;
    if (nsamp <= 0 || nchans <= 0) return 0;
    dim3 grid((unsigned)((nsamp + CT_TILE - 1) / CT_TILE), (unsigned)((nchans + CT_TILE - 1) / CT_TILE));
    k_corner_turn<<<grid, 256, 0, (cudaStream_t)stream>>>(in, in_stride, out, out_pitch, nchans, nsamp);
    return (int)cudaGetLastError();
}

extern "C" int aak_chan_offsets(const uint8_t* x, size_t pitch, int64_t len, int32_t nrows, int32_t* off2, int32_t* off4, int32_t* off8,
                                int32_t* bias2, int32_t* bias4, int32_t* bias8, void* stream) {
    if (nrows <= 0) return 0;
    k_chan_offsets<<<(unsigned)nrows, 256, 0, (cudaStream_t)stream>>>(x, pitch, len, off2, off4, off8, bias2, bias4, bias8);
    return (int)cudaGetLastError();
}

extern "C" int aak_scatter_exceptions(const uint2* exc, const unsigned* exc_cnt, unsigned cap, const double* k, double dm_low,
                                      double dm_step, int32_t ndms, int32_t bin, int64_t nt, int32_t* D, int64_t pitch, int32_t nsm,
                                      void* stream) {
    if (nsm < 1) return (int)cudaErrorInvalidValue;
    k_scatter_exceptions<<<nsm * 4, 256, 0, (cudaStream_t)stream>>>(exc, exc_cnt, cap, k, dm_low, dm_step, ndms, bin, nt, D, pitch);
    return (int)cudaGetLastError();
}

extern "C" int aak_prep_fused(const aak_prep_args* a, int32_t nrows, void* stream) {
    if (nrows <= 0 || a->ngroups <= 0) return 0;
    PrepFused p;
    p.raw = a->raw; p.pitch = a->pitch; p.ngroups = a->ngroups; p.chan0 = a->chan0; p.cap = a->cap;
    p.x4 = a->x4; p.x4_pitch = a->x4_pitch; p.x4_stride = a->x4_stride;
    p.lo2 = a->lo2; p.lo2_pitch = a->lo2_pitch; p.lo2_stride = a->lo2_stride; p.off2 = a->off2; p.exc2 = a->exc2; p.cnt2 = a->cnt2; p.nb2 = a->nb2;
    p.lo4 = a->lo4; p.lo4_pitch = a->lo4_pitch; p.lo4_stride = a->lo4_stride; p.off4 = a->off4; p.exc4 = a->exc4; p.cnt4 = a->cnt4; p.nb4 = a->nb4;
    p.xb8 = a->xb8; p.xb8_pitch = a->xb8_pitch; p.xb8_stride = a->xb8_stride;
    p.hb8 = a->hb8; p.hb8_pitch = a->hb8_pitch; p.hb8_stride = a->hb8_stride; p.off8 = a->off8; p.exc8 = a->exc8; p.cnt8 = a->cnt8; p.nb8 = a->nb8;
    p.bits8 = a->bits8; p.bits8_pitch = a->bits8_pitch;
    dim3 grid((unsigned)((a->ngroups + 255) / 256), (unsigned)nrows);
    k_prep_fused<<<grid, 256, 0, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}
