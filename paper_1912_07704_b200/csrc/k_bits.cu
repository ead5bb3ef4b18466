/*
 * k_bits.cu — K2b, dedispersion of a bit plane for sm_100a.
 *
 * The bin-8 input x_8 (a sum of 8 bytes, noise sigma 45) does not fit the 1-byte path of K2: as uint16 it costs two
 * shared-memory bytes per add, and that crossbar is what limits K2 (the bin-8 range ran at 0.49 of the add roofline). The
 * HALF-BYTE form splits it exactly:   x_8[c][t] = 2 y[c][t] + bit[c][t] + off8[c] + r[c][t],   y = clamp((x_8 - off8) >> 1, 0, 255)
 * (sigma 23: a byte), bit = the dropped low bit, r = exceptions (1.5e-8 of Gaussian samples). K2 sums y on its byte path and
 * doubles the sums, k_scatter_exceptions adds the r, and this kernel adds
 *        D[i][t] += sum_c bit[c][t + delay(c, i)]                   (BASELINE.json north_star, applied to the bit plane)
 * with bit-sliced arithmetic: a thread owns 32 consecutive output samples of one DM trial as VERTICAL counters (plane p holds
 * bit p of all 32 counts); a channel contributes one 32-bit word of the plane, cut out of two shared-memory words by a funnel
 * shift at the (channel, trial) delay; 32 such words are folded by a carry-save adder tree (2 LOP3 each) before one ripple
 * into the high planes. That is about 0.3 instructions per algorithmic add against 0.9 on the byte path, on 1/8 byte per add.
 */
#include <cuda_runtime.h>
#include <stdint.h>
#include "aa_kernels.h"

namespace {

constexpr int BK_THREADS = 256;               /* 8 warps: warp w owns trials NM w .. NM w + NM - 1 of the tile; lane l owns word l */
constexpr int BK_NM = 4;                      /* adjacent DM trials per thread: their delays in a channel differ by a few samples, so the
                                                 two shared-memory words one trial needs nearly always serve the next one as well */
constexpr int BK_DMS = BK_NM * BK_THREADS / 32;   /* 32 DM trials per CTA */
constexpr int BK_T = 1024;                    /* output samples per CTA = 32 words */
constexpr int BK_CB = 128;                    /* channels per shared-memory block */
constexpr int BK_NP = 16;                     /* counter planes: counts up to 65535 channels */

/* sum = a ^ b ^ c, carry = majority(a, b, c): one LOP3 each */
__device__ __forceinline__ void csa(uint32_t& h, uint32_t& l, uint32_t a, uint32_t b, uint32_t c) {
    uint32_t s, m;
    asm("lop3.b32 %0, %1, %2, %3, 0x96;" : "=r"(s) : "r"(a), "r"(b), "r"(c));
    asm("lop3.b32 %0, %1, %2, %3, 0xE8;" : "=r"(m) : "r"(a), "r"(b), "r"(c));
    l = s; h = m;
}

struct BitsParams {
    const uint32_t* bits; size_t pitchw; const int32_t* delays; int nchans, c0, c1, ndms; long long nt; int ww;
    int32_t* D; long long dpitch; const unsigned* mode_cnt; unsigned mode_cap;
};

/* the words of NM adjacent trials of one channel: trial m reuses the pair loaded for trial m - 1 when it starts in the same word
 * (a warp-uniform test of two table entries; the first version loaded two words per trial and was bound by the shared-memory
 * load path: ncu l1tex 89 %, mio_throttle the top stall) */
__device__ __forceinline__ void bk_words(const uint8_t* Sb, const uint32_t* e, uint32_t (&x)[BK_NM]) {
    uint32_t lo = 0, hi = 0, off = 0xffffffffu;
    static_assert(BK_NM == 4, "one 16-byte load fetches the four entries");
    const uint4 e4 = *reinterpret_cast<const uint4*>(e);
    const uint32_t ev[4] = {e4.x, e4.y, e4.z, e4.w};
#pragma unroll
    for (int m = 0; m < BK_NM; ++m) {
        const uint32_t o = ev[m] & 0x00FFFFFFu;
        if (o != off) {
            off = o;
            lo = *reinterpret_cast<const uint32_t*>(Sb + off);
            hi = *reinterpret_cast<const uint32_t*>(Sb + off + 4);
        }
        x[m] = __funnelshift_r(lo, hi, ev[m] >> 24);
    }
}

__global__ void __launch_bounds__(BK_THREADS, 2)
k_dedisperse_bits(const BitsParams p) {
    if (p.mode_cnt && *p.mode_cnt > p.mode_cap) return;               /* exception-heavy chunk: the uint16 route produced D */
    extern __shared__ __align__(16) uint32_t bk_smem[];
    uint32_t* S = bk_smem;                                           /* [BK_CB][ww] window words of the block's channels */
    uint32_t* ent = S + (size_t)BK_CB * p.ww;                        /* [BK_CB][BK_DMS]: byte offset of the first word | shift << 24 */
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const long long t0 = (long long)blockIdx.x * BK_T;
    const int i0 = blockIdx.y * BK_DMS;
    uint32_t P[BK_NM][BK_NP];
#pragma unroll
    for (int m = 0; m < BK_NM; ++m)
#pragma unroll
        for (int q = 0; q < BK_NP; ++q) P[m][q] = 0u;

    for (int cb = p.c0; cb < p.c1; cb += BK_CB) {
        /* ---- warp w stages channels w, w + 8, ...: the lanes fetch the channel's delay for the tile's 32 trials (trial index
         * clamped to the range; trial i0 has the smallest), then the warp copies the window words and writes the entries. All
         * loads of a block are in flight together (one channel at a time cost two dependent round trips per channel). */
        constexpr int NK = BK_CB / (BK_THREADS / 32);
#pragma unroll 1
        for (int k0 = 0; k0 < NK; k0 += 8) {
            int d[8];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int c = cb + warp + (k0 + k) * (BK_THREADS / 32);
                d[k] = c < p.c1 ? __ldg(p.delays + (size_t)min(i0 + lane, p.ndms - 1) * p.nchans + c) : 0;
            }
            uint32_t wv[8][2];
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int cl = warp + (k0 + k) * (BK_THREADS / 32), c = cb + cl;
                const bool live = c < p.c1;                           /* channels past the group read as zero bits */
                const int d0 = __shfl_sync(0xffffffffu, d[k], 0);
                const long long w0 = (t0 + d0) >> 5;
                const uint32_t* src = p.bits + (size_t)c * p.pitchw + (size_t)w0;
                wv[k][0] = (live && lane < p.ww) ? __ldg(src + lane) : 0u;
                wv[k][1] = (live && lane + 32 < p.ww) ? __ldg(src + lane + 32) : 0u;
                const int o = (int)(t0 + d[k] - (w0 << 5));           /* bit offset inside the window, >= 0 */
                ent[cl * BK_DMS + lane] = (uint32_t)((cl * p.ww + (o >> 5)) * 4) | ((uint32_t)(o & 31) << 24);
            }
#pragma unroll
            for (int k = 0; k < 8; ++k) {
                const int cl = warp + (k0 + k) * (BK_THREADS / 32), c = cb + cl;
                if (lane < p.ww) S[cl * p.ww + lane] = wv[k][0];
                if (lane + 32 < p.ww) S[cl * p.ww + lane + 32] = wv[k][1];
                if (p.ww > 64) {                                      /* wide windows (large delay spreads): the rest, plainly */
                    const int d0 = __shfl_sync(0xffffffffu, d[k], 0);
                    const uint32_t* src = p.bits + (size_t)c * p.pitchw + (size_t)((t0 + d0) >> 5);
                    for (int j = lane + 64; j < p.ww; j += 32) S[cl * p.ww + j] = c < p.c1 ? __ldg(src + j) : 0u;
                }
            }
        }
        __syncthreads();
        /* ---- every thread: its word of every channel for each of its trials; 32 channels per carry-save tree, the four weight-32
         * carries of the block through a second tree, one ripple into the high planes per block */
        const uint8_t* Sb = reinterpret_cast<const uint8_t*>(S) + lane * 4;
        const uint32_t* eb = ent + BK_NM * warp;
        uint32_t c32v[BK_NM][BK_CB / 32];
#pragma unroll
        for (int c32 = 0; c32 < BK_CB; c32 += 32) {
            uint32_t sixteen[BK_NM][2];
#pragma unroll
            for (int h = 0; h < 2; ++h) {
                uint32_t eight[BK_NM][2];
#pragma unroll
                for (int q = 0; q < 2; ++q) {
                    uint32_t four[BK_NM][2];
#pragma unroll
                    for (int r = 0; r < 2; ++r) {
                        uint32_t two[BK_NM][2];
#pragma unroll
                        for (int u = 0; u < 2; ++u) {
                            const int cl = c32 + ((h * 2 + q) * 2 + r) * 4 + u * 2;
                            uint32_t x0[BK_NM], x1[BK_NM];
                            bk_words(Sb, eb + cl * BK_DMS, x0);
                            bk_words(Sb, eb + (cl + 1) * BK_DMS, x1);
#pragma unroll
                            for (int m = 0; m < BK_NM; ++m) csa(two[m][u], P[m][0], P[m][0], x0[m], x1[m]);
                        }
#pragma unroll
                        for (int m = 0; m < BK_NM; ++m) csa(four[m][r], P[m][1], P[m][1], two[m][0], two[m][1]);
                    }
#pragma unroll
                    for (int m = 0; m < BK_NM; ++m) csa(eight[m][q], P[m][2], P[m][2], four[m][0], four[m][1]);
                }
#pragma unroll
                for (int m = 0; m < BK_NM; ++m) csa(sixteen[m][h], P[m][3], P[m][3], eight[m][0], eight[m][1]);
            }
#pragma unroll
            for (int m = 0; m < BK_NM; ++m) csa(c32v[m][c32 / 32], P[m][4], P[m][4], sixteen[m][0], sixteen[m][1]);
        }
        static_assert(BK_CB == 128, "the second-level tree below folds four weight-32 carries");
#pragma unroll
        for (int m = 0; m < BK_NM; ++m) {
            uint32_t a64, b64, carry;
            csa(a64, P[m][5], P[m][5], c32v[m][0], c32v[m][1]);
            csa(b64, P[m][5], P[m][5], c32v[m][2], c32v[m][3]);
            csa(carry, P[m][6], P[m][6], a64, b64);
#pragma unroll
            for (int q = 7; q < BK_NP; ++q) { const uint32_t t = P[m][q] & carry; P[m][q] ^= carry; carry = t; }
        }
        __syncthreads();
    }

    /* ---- unpack the vertical counters and add them to D (32 consecutive samples per thread and trial) */
#pragma unroll
    for (int m = 0; m < BK_NM; ++m) {
        const int i = i0 + BK_NM * warp + m;
        if (i >= p.ndms) continue;
        int32_t* row = p.D + (size_t)i * (size_t)p.dpitch;
        const long long tb = t0 + 32 * lane;
#pragma unroll
        for (int k4 = 0; k4 < 8; ++k4) {
            if (tb + 4 * k4 >= p.nt) break;                          /* rows are padded to 128 samples: whole int4 groups exist */
            int cnt[4] = {0, 0, 0, 0};
#pragma unroll
            for (int q = 0; q < BK_NP; ++q)
#pragma unroll
                for (int k = 0; k < 4; ++k) cnt[k] += (int)((P[m][q] >> (4 * k4 + k)) & 1u) << q;
            int4* dst = reinterpret_cast<int4*>(row + tb + 4 * k4);
            int4 v = *dst;
            v.x += cnt[0]; v.y += cnt[1]; v.z += cnt[2]; v.w += cnt[3];
            *dst = v;
        }
    }
}

}  // namespace

extern "C" int aak_dedisperse_bits(const uint32_t* bits, size_t pitch_words, const int32_t* delays, int32_t nchans, int32_t chan_begin,
                                   int32_t chan_end, int32_t ndms, int64_t nt, int32_t window_words, int32_t* D, int64_t pitch,
                                   const unsigned* mode_cnt, unsigned mode_cap, void* stream) {
    if (ndms <= 0 || nt <= 0 || chan_begin >= chan_end) return 0;
    if (window_words < 34 || window_words > 256) return (int)cudaErrorInvalidValue;      /* 128 channels x 256 words = 128 KB of shared memory */
    BitsParams p;
    p.bits = bits; p.pitchw = pitch_words; p.delays = delays; p.nchans = nchans; p.c0 = chan_begin; p.c1 = chan_end; p.ndms = ndms; p.nt = nt;
    p.ww = window_words; p.D = D; p.dpitch = pitch; p.mode_cnt = mode_cnt; p.mode_cap = mode_cap;
    const size_t smem = ((size_t)BK_CB * window_words + BK_CB * BK_DMS) * 4;
    dim3 grid((unsigned)((nt + BK_T - 1) / BK_T), (unsigned)((ndms + BK_DMS - 1) / BK_DMS));
    if (grid.y > 65535) return (int)cudaErrorInvalidConfiguration;
    k_dedisperse_bits<<<grid, BK_THREADS, smem, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}

/* Function attributes belong to a device: called by aa_strategy_setup with the strategy's device current, like
 * aak_dedisperse_init and aak_sps_init (no process-wide "already done" flag). */
extern "C" int aak_bits_init(void) {
    return (int)cudaFuncSetAttribute(k_dedisperse_bits, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
}
