/*
 * k_dedisp.cu — K2, brute-force incoherent dedispersion for sm_100a.
 *
 *   D[i][t] = sum_{c<C} x_b[c][t + delay(c,i)]          (BASELINE.json north_star; every term is added individually)
 *
 * Design:
 *   * A CTA owns 30 or 32 DM trials x T_TILE = 1024 output samples, held in registers by its compute warps; one more
 *     warp is the TMA producer. uint8 input: 15 compute warps x (2 DMs x 1024 samples) + producer = 16 warps, so a thread
 *     may use 128 registers (measured 5 % faster than 16 + 1 warps at 96 registers: ptxas keeps more shared-memory loads
 *     in flight). Binned uint16 input: 16 compute warps x (4 adjacent DMs x 512 samples) + producer.
 *     Channels stream through shared memory in blocks of CB channels,
 *     NSTAGE-deep ring, full/empty mbarriers (no __syncthreads in the main loop).
 *   * Shared memory holds SPW sample-shifted copies of every channel window (SPW = samples per 32-bit word: 4 for uint8,
 *     2 for uint16), so that ANY sample offset t+delay is a word-aligned, bank-conflict-free LDS.32: copy k holds the
 *     window shifted by k samples. TMA needs 16-byte aligned global coordinates (measured: an unaligned inner
 *     coordinate raises an illegal-instruction fault on sm_100a), so the shifted copies exist in GLOBAL memory
 *     (K1 writes them: x_k[c][t] = x[c][t+k], copy k at byte offset k*copy_stride of one buffer); the window start is
 *     aligned down to 16 bytes and the residue is folded into the host-built offset table.
 *   * The window of a channel block is only as wide as its channels' delay spread inside a DM tile needs (window classes, one
 *     tensor map each): with the low-frequency configuration's spreads (up to 1600 samples per tile at the bottom of the band,
 *     none at the top) a uniform window made the L2 -> shared-memory fill (4 copies x 2816 bytes x 8 channels per 1920 clocks of
 *     adds = 47 B/clk/SM, the chip-wide TMA rate) the limiter of K2; per-block windows cut it by a third.
 *   * ONE TMA per channel moves the windows of all copies: the tensor map views the buffer as OVERLAPPING 256-byte
 *     segments (dims {pitch, nseg, NCOPY, C}, strides {256, copy_stride, pitch}), so a {256, nseg, NCOPY, 1} box lands
 *     as NCOPY linear windows of WB bytes. A stage is therefore CB tensor copies + one bulk copy of the offset table,
 *     issued by one elected thread (ncu on the first version, one TMA per (copy, channel) issued from 32 divergent
 *     lanes, showed the producer warp busy 85 % of the time and the compute warps starved: profiles/r01_*).
 *   * Packed arithmetic (uint8): a loaded word w = (b0,b1,b2,b3) is four consecutive time samples of one channel.
 *         A += w                      (whole word, lanes overlap at 8-bit spacing, wraps mod 2^32)
 *         H += (b1, 0, b3, 0)         (one PRMT; two clean 16-bit lanes)
 *     and L = A - (H << 8) = (b0 sums, b2 sums) is recovered exactly when the lanes are read, so one 32-bit add
 *     instruction performs two (H) or four (A) algorithmic adds and only ONE unpack instruction is spent per four
 *     samples. Two channels are folded per three-input IADD3 (A += w1 + w2); the H adds are issued as IMAD (x*1+y) so
 *     that they run on the FMA pipe while PRMT/IADD3 use the ALU pipe. 16-bit lanes are carried into a second pair of
 *     packed registers every 256/bin channels (255 + 256*255 = 65535 never overflows), so the result is bit-exact
 *     int32 for any uint8 input.
 *     uint16 (binned) input is already a pair of 16-bit lanes: A += w1 + w2, same carry rule.
 *   * The per-(channel, DM) shared-memory offsets come from a host-built table (exact double delays), streamed with
 *     the data by a 1-D bulk copy; inside the loop an address is one integer add.
 */
#include <cuda.h>
#include <cuda_runtime.h>
#include <stdint.h>
#include <string.h>
#include "aa_kernels.h"

namespace {

constexpr int DM_TILE = 32;          /* row length of the offset table: at most this many DM trials per CTA */
constexpr int T_TILE = 1024;         /* output samples per CTA */
#ifndef AA_PRODUCER_SLEEP_NS
#define AA_PRODUCER_SLEEP_NS 400
#endif
#ifndef AA_CONSUMER_SLEEP_NS
#define AA_CONSUMER_SLEEP_NS 0
#endif
constexpr int PRODUCER_SLEEP_NS = AA_PRODUCER_SLEEP_NS, CONSUMER_SLEEP_NS = AA_CONSUMER_SLEEP_NS;
constexpr int MAX_RING = 8;          /* shared-memory ring depth is a launch parameter (2..MAX_RING) */
constexpr int SMEM_HEADER = 1024;    /* mbarriers live here; keeps the stages 1024-byte aligned */


/* one tensor map per window class (boxes of 256 x nseg bytes, nseg = class_wb / 256) */
template <int N> struct WindowMaps { CUtensorMap m[N]; };

/* Kernel parameters. VW (plans with several window classes) adds the class table; plans with one class keep the parameter
 * block of the first version of this kernel byte for byte: ptxas schedules the main loop differently when the block grows,
 * and the schedule it picks for the original block is 0.5 % faster (measured, identical opcode mix). */
#define AA_DEDISP_PARAMS_HEAD \
    const int32_t* etab; \
    const int32_t* x0tab; \
    int32_t* D; \
    long long pitch; \
    long long nt; \
    int ndms; \
    int nstages; \
    int window_bytes; \
    int spill_stages; \
    int nring;                 /* ring depth */ \
    int stage_begin, stage_end; /* channel blocks [stage_begin, stage_end) of the nstages are summed by this launch */ \
    int accumulate;            /* 1: add to the values already in D (a later channel group of the same chunk) */ \
    const unsigned* mode_cnt;  /* NULL, or: run only if (*mode_cnt > mode_cap) == mode_dense */ \
    unsigned mode_cap; \
    int mode_dense; \
    const int* bias;           /* NULL, or a constant added to every output */
#define AA_DEDISP_PARAMS_TAIL \
    int skew_q16;              /* CTA order: time tile = blockIdx / ndm_tiles - (skew_q16 * dm_tile >> 16), see launch() */ \
    int nt_tiles; \
    unsigned one;              /* always 1; a runtime value so that x*one+y stays an IMAD (FMA pipe) */
template <bool VW> struct DedispParamsT { AA_DEDISP_PARAMS_HEAD AA_DEDISP_PARAMS_TAIL };
template <> struct DedispParamsT<true> {
    AA_DEDISP_PARAMS_HEAD
    const int* wcls;           /* [nstages] window class of each stage */
    int class_wb[8];           /* window bytes per class */
    AA_DEDISP_PARAMS_TAIL
};

__device__ __forceinline__ uint32_t smem_u32(const void* p) { return (uint32_t)__cvta_generic_to_shared(p); }

__device__ __forceinline__ void mbar_init(uint32_t bar, uint32_t count) {
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"(bar), "r"(count) : "memory");
}
__device__ __forceinline__ bool mbar_try_wait(uint32_t bar, uint32_t parity) {
    uint32_t ok;
    asm volatile(
        "{\n"
        ".reg .pred p;\n"
        "mbarrier.try_wait.parity.shared::cta.b64 p, [%1], %2, %3;\n"
        "selp.u32 %0, 1, 0, p;\n"
        "}\n"
        : "=r"(ok)
        : "r"(bar), "r"(parity), "r"(0x989680u)      /* suspend-time hint: sleep in hardware until the phase completes */
        : "memory");
    return ok != 0;
}
/* SLEEP_NS > 0: back off between polls. A polling warp takes issue slots from the compute warps of its scheduler
 * (ncu: the producer's empty-barrier polls were 5.8 % of all instructions executed, all on one of the four schedulers). */
template <int SLEEP_NS>
__device__ __forceinline__ void mbar_wait(uint32_t bar, uint32_t parity) {
    while (!mbar_try_wait(bar, parity)) {
        if (SLEEP_NS > 0) __nanosleep(SLEEP_NS);
    }
}
__device__ __forceinline__ void mbar_arrive(uint32_t bar) {
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"(bar) : "memory");
}
__device__ __forceinline__ void mbar_arrive_expect_tx(uint32_t bar, uint32_t bytes) {
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"(bar), "r"(bytes) : "memory");
}
__device__ __forceinline__ void tma_load_4d(uint32_t dst, const CUtensorMap* map, int x, int y, int z, int w, uint32_t bar) {
    asm volatile(
        "cp.async.bulk.tensor.4d.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1, {%2, %3, %4, %5}], [%6];" ::"r"(dst),
        "l"(reinterpret_cast<uint64_t>(map)), "r"(x), "r"(y), "r"(z), "r"(w), "r"(bar)
        : "memory");
}
__device__ __forceinline__ void bulk_load_1d(uint32_t dst, const void* src, uint32_t bytes, uint32_t bar) {
    asm volatile("cp.async.bulk.shared::cluster.global.mbarrier::complete_tx::bytes [%0], [%1], %2, [%3];" ::"r"(dst),
                 "l"(src), "r"(bytes), "r"(bar)
                 : "memory");
}
/* x*1 + y on the FMA pipe: `one` is a runtime 1 so ptxas keeps the IMAD. */
__device__ __forceinline__ uint32_t add_fma_pipe(uint32_t x, uint32_t one, uint32_t y) {
    uint32_t d;
    asm("mad.lo.u32 %0, %1, %2, %3;" : "=r"(d) : "r"(x), "r"(one), "r"(y));
    return d;
}
__device__ __forceinline__ uint32_t odd_bytes(uint32_t w) { /* (b1, 0, b3, 0) */
    uint32_t d;
    asm("prmt.b32 %0, %1, 0, 0x4341;" : "=r"(d) : "r"(w));
    return d;
}

/* M = adjacent DM trials per warp. The 16 compute warps form 32/M DM groups x NTH = 16*M/32 time parts of the tile.
 * Adjacent DM trials often have the SAME delay in a channel (the delay grows by less than one sample per DM step over
 * much of the band): the words loaded for trial m-1 are then exactly the words trial m needs, and are reused from
 * registers instead of being read from shared memory again (a warp-uniform test of two table entries). */
/* NWC = compute warps: 16 (+1 producer = 17 warps, 96 registers per thread) or 15 (+1 = 16 warps, 128 registers per
 * thread, 30 trials per CTA: the extra registers let ptxas keep more shared-memory loads in flight). */
/* VW: the plan has more than one window class (the producer looks the class of every channel block up); plans with ONE class
 * keep the constant map and window of the first version of this kernel (measured: the look-up costs the byte kernel 2 %). */
template <int IN16, int CB, int FMA_H, int M, int NWC, bool VW>
__global__ void __launch_bounds__((NWC + 1) * 32, 1)
k_dedisperse(const __grid_constant__ WindowMaps<VW ? 8 : 1> maps, const DedispParamsT<VW> p) {
    constexpr int ESZ = IN16 ? 2 : 1;
    constexpr int SPW = 4 / ESZ;                 /* samples per word */
    constexpr int NCOPY = SPW;                   /* shifted copies */
    constexpr int NW = NWC;
    constexpr int NTH = (M == 2) ? 1 : 2;        /* time parts of the tile */
    constexpr int NG = NWC / NTH;                /* DM groups */
    constexpr int DMT = NG * M;                  /* DM trials per CTA: 32 or 30 */
    constexpr int T_PART = T_TILE / NTH;
    constexpr int J = T_PART / (32 * SPW);       /* words per thread per DM */
    constexpr int ENT_BYTES = CB * DM_TILE * 4;
    static_assert(NG * NTH == NW && NTH >= 1 && J >= 1 && DMT <= DM_TILE, "warp layout");

    if (p.mode_cnt && ((*p.mode_cnt > p.mode_cap) ? 1 : 0) != p.mode_dense) return;     /* the other input format handles this chunk */
    extern __shared__ __align__(1024) uint8_t smem[];
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const int ndm_tiles = (p.ndms + DMT - 1) / DMT;
    /* DM tile fastest, and the time tile skewed by the average delay of the DM tile: CTAs that run together then read the
     * same stretch of the INPUT (t + delay), so the windows of neighbouring DM tiles are L2 hits also where the delay grows
     * by more than a tile per DM tile (low-frequency bands). skew 0 = plain (DM tile, time tile) order. */
    const int dt = blockIdx.x % ndm_tiles;
    const int tt = blockIdx.x / ndm_tiles - (int)(((long long)p.skew_q16 * dt) >> 16);
    if (tt < 0 || tt >= p.nt_tiles) return;
    const long long t0 = (long long)tt * T_TILE;
    const int WB = p.window_bytes;
    const int data_bytes = NCOPY * CB * WB;
    const int stage_bytes = data_bytes + ENT_BYTES;
    const int NSTAGE = p.nring;
    const uint32_t bar_full = smem_u32(smem);            /* NSTAGE x 8 bytes */
    const uint32_t bar_empty = bar_full + 8 * MAX_RING;
    uint8_t* const stages = smem + SMEM_HEADER;

    if (threadIdx.x == 0) {
        for (int s = 0; s < NSTAGE; ++s) {
            mbar_init(bar_full + 8 * s, 1);
            mbar_init(bar_empty + 8 * s, NW);
        }
        asm volatile("fence.mbarrier_init.release.cluster;" ::: "memory");
        asm volatile("fence.proxy.async.shared::cta;" ::: "memory");
    }
    __syncthreads();

    if (warp == NW) {
        /* ------------------------------------------------------------------ producer: one elected thread */
        if (lane == 0) {
            const int32_t* x0row = p.x0tab + (size_t)dt * (size_t)p.nstages * CB;
            const int32_t* erow = p.etab + (size_t)dt * (size_t)p.nstages * (CB * DM_TILE);
            const long long tb = t0 * ESZ;
            int slot = 0; uint32_t ph = 0;
            for (int s = p.stage_begin; s < p.stage_end; ++s) {
                int x0[CB];
#pragma unroll
                for (int c = 0; c < CB; ++c) x0[c] = __ldg(x0row + s * CB + c);
                if constexpr (VW) {
                    const int cls = __ldg(p.wcls + s);
                    const int WBs = p.class_wb[cls];                         /* this channel block's window (<= WB) */
                    const CUtensorMap* map = &maps.m[cls];
                    mbar_wait<PRODUCER_SLEEP_NS>(bar_empty + 8 * slot, ph ^ 1u);
                    const uint32_t fb = bar_full + 8 * slot;
                    mbar_arrive_expect_tx(fb, (uint32_t)(NCOPY * CB * WBs + ENT_BYTES));
                    const uint32_t sbase = smem_u32(stages + (size_t)slot * stage_bytes);
#pragma unroll
                    for (int c = 0; c < CB; ++c) {
                        const long long xs = tb + x0[c];                     /* 16-byte aligned byte coordinate of the window */
                        const int xi = xs > 0x7fff0000ll ? 0x7fff0000 : (int)xs;   /* far out of bounds is zero-filled anyway */
                        tma_load_4d(sbase + (uint32_t)(c * NCOPY * WBs), map, xi, 0, 0, s * CB + c, fb);
                    }
                    bulk_load_1d(sbase + data_bytes, erow + (size_t)s * (CB * DM_TILE), ENT_BYTES, fb);
                } else {
                    mbar_wait<PRODUCER_SLEEP_NS>(bar_empty + 8 * slot, ph ^ 1u);
                    const uint32_t fb = bar_full + 8 * slot;
                    mbar_arrive_expect_tx(fb, (uint32_t)stage_bytes);
                    const uint32_t sbase = smem_u32(stages + (size_t)slot * stage_bytes);
#pragma unroll
                    for (int c = 0; c < CB; ++c) {
                        const long long xs = tb + x0[c];                     /* 16-byte aligned byte coordinate of the window */
                        const int xi = xs > 0x7fff0000ll ? 0x7fff0000 : (int)xs;   /* far out of bounds is zero-filled anyway */
                        tma_load_4d(sbase + (uint32_t)(c * NCOPY * WB), &maps.m[0], xi, 0, 0, s * CB + c, fb);
                    }
                    bulk_load_1d(sbase + data_bytes, erow + (size_t)s * (CB * DM_TILE), ENT_BYTES, fb);
                }
                if (++slot == NSTAGE) { slot = 0; ph ^= 1u; }
            }
        }
        return;
    }

    /* ---------------------------------------------------------------------- compute warps */
    const uint32_t one = p.one;
    uint32_t A[M][J], C1[M][J];
    uint32_t H[IN16 ? 1 : M][IN16 ? 1 : J], C2[IN16 ? 1 : M][IN16 ? 1 : J];
#pragma unroll
    for (int m = 0; m < M; ++m)
#pragma unroll
        for (int j = 0; j < J; ++j) {
            A[m][j] = 0; C1[m][j] = 0;
            if (!IN16) { H[m][j] = 0; C2[m][j] = 0; }
        }

    const int grp = warp % NG, part = warp / NG;
    const int ent_off = data_bytes + grp * M * 4;
    int until_spill = p.spill_stages;
    int slot = 0; uint32_t ph = 0;
    for (int s = p.stage_begin; s < p.stage_end; ++s) {
        mbar_wait<CONSUMER_SLEEP_NS>(bar_full + 8 * slot, ph);
        const uint8_t* sb = stages + (size_t)slot * stage_bytes;
        const uint8_t* db = sb + lane * 4 + part * (T_PART * ESZ);
        if (M == 2) {
            /* two trials per warp: every word is loaded where it is used (no registers to spare for reuse) */
#pragma unroll
            for (int cp = 0; cp < CB / 2; ++cp) {
                const uint2 e1 = *reinterpret_cast<const uint2*>(sb + ent_off + (2 * cp) * (DM_TILE * 4));
                const uint2 e2 = *reinterpret_cast<const uint2*>(sb + ent_off + (2 * cp + 1) * (DM_TILE * 4));
#pragma unroll
                for (int m = 0; m < 2; ++m) {
                    const uint8_t* a1 = db + (m == 0 ? e1.x : e1.y);
                    const uint8_t* a2 = db + (m == 0 ? e2.x : e2.y);
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        const uint32_t w1 = *reinterpret_cast<const uint32_t*>(a1 + j * 128);
                        const uint32_t w2 = *reinterpret_cast<const uint32_t*>(a2 + j * 128);
                        A[m][j] = A[m][j] + w1 + w2;
                        if (!IN16) {
                            if ((FMA_H & 1) || (FMA_H == 2 && (j & 1))) {
                                H[m][j] = add_fma_pipe(odd_bytes(w1), one, H[m][j]);
                                H[m][j] = add_fma_pipe(odd_bytes(w2), one, H[m][j]);
                            } else {
                                H[m][j] = H[m][j] + odd_bytes(w1) + odd_bytes(w2);
                            }
                        }
                    }
                }
            }
        } else {
            /* four adjacent trials per warp: the words of trial m-1 are reused when trial m has the same delay */
#pragma unroll 1
            for (int cp = 0; cp < CB / 2; ++cp) {
                const uint4 ea = *reinterpret_cast<const uint4*>(sb + ent_off + (2 * cp) * (DM_TILE * 4));
                const uint4 eb = *reinterpret_cast<const uint4*>(sb + ent_off + (2 * cp + 1) * (DM_TILE * 4));
                const uint32_t e1[4] = {ea.x, ea.y, ea.z, ea.w};
                const uint32_t e2[4] = {eb.x, eb.y, eb.z, eb.w};
                uint32_t w1[J], w2[J];
#pragma unroll
                for (int m = 0; m < M; ++m) {
                    if (m == 0 || e1[m] != e1[m - 1]) {             /* warp-uniform: one table entry for all lanes */
                        const uint8_t* a1 = db + e1[m];
#pragma unroll
                        for (int j = 0; j < J; ++j) w1[j] = *reinterpret_cast<const uint32_t*>(a1 + j * 128);
                    }
                    if (m == 0 || e2[m] != e2[m - 1]) {
                        const uint8_t* a2 = db + e2[m];
#pragma unroll
                        for (int j = 0; j < J; ++j) w2[j] = *reinterpret_cast<const uint32_t*>(a2 + j * 128);
                    }
#pragma unroll
                    for (int j = 0; j < J; ++j) {
                        A[m][j] = A[m][j] + w1[j] + w2[j];
                        if (!IN16) {
                            if ((FMA_H & 1) || (FMA_H == 2 && (j & 1))) {
                                H[m][j] = add_fma_pipe(odd_bytes(w1[j]), one, H[m][j]);
                                H[m][j] = add_fma_pipe(odd_bytes(w2[j]), one, H[m][j]);
                            } else {
                                H[m][j] = H[m][j] + odd_bytes(w1[j]) + odd_bytes(w2[j]);
                            }
                        }
                    }
                }
            }
        }
        __syncwarp();
        if (lane == 0) mbar_arrive(bar_empty + 8 * slot);
        if (++slot == NSTAGE) { slot = 0; ph ^= 1u; }
        if (--until_spill == 0) {
            until_spill = p.spill_stages;
#pragma unroll
            for (int m = 0; m < M; ++m)
#pragma unroll
                for (int j = 0; j < J; ++j) {
                    if (!IN16) {
                        uint32_t L = A[m][j] - (H[m][j] << 8);
                        C1[m][j] += (L >> 8) & 0x00FF00FFu;
                        C2[m][j] += (H[m][j] >> 8) & 0x00FF00FFu;
                        L &= 0x00FF00FFu;
                        H[m][j] &= 0x00FF00FFu;
                        A[m][j] = L + (H[m][j] << 8);
                    } else {
                        C1[m][j] += (A[m][j] >> 8) & 0x00FF00FFu;
                        A[m][j] &= 0x00FF00FFu;
                    }
                }
        }
    }

    /* ---------------------------------------------------------------------- unpack and store */
    const int bias = p.bias ? *p.bias : 0;
#pragma unroll
    for (int m = 0; m < M; ++m) {
        const int i = dt * DMT + grp * M + m;
        if (i >= p.ndms) continue;
        int32_t* row = p.D + (size_t)i * (size_t)p.pitch;
#pragma unroll
        for (int j = 0; j < J; ++j) {
            const long long t = t0 + part * T_PART + (long long)(j * 32 + lane) * SPW;
            if (t >= p.nt) continue;
            if (!IN16) {
                const uint32_t L = A[m][j] - (H[m][j] << 8);
                int4 v;
                constexpr int SH = (FMA_H == 3) ? 1 : 0;             /* half-byte form of bin 8: the sums of y count twice */
                v.x = bias + (int)(((L & 0xFFFFu) + ((C1[m][j] & 0xFFFFu) << 8)) << SH);
                v.y = bias + (int)(((H[m][j] & 0xFFFFu) + ((C2[m][j] & 0xFFFFu) << 8)) << SH);
                v.z = bias + (int)(((L >> 16) + ((C1[m][j] >> 16) << 8)) << SH);
                v.w = bias + (int)(((H[m][j] >> 16) + ((C2[m][j] >> 16) << 8)) << SH);
                if (p.accumulate) {
                    const int4 o = *reinterpret_cast<const int4*>(row + t);
                    v.x += o.x; v.y += o.y; v.z += o.z; v.w += o.w;
                }
                *reinterpret_cast<int4*>(row + t) = v;
            } else {
                int2 v;
                v.x = (int)((A[m][j] & 0xFFFFu) + ((C1[m][j] & 0xFFFFu) << 8));
                v.y = (int)((A[m][j] >> 16) + ((C1[m][j] >> 16) << 8));
                if (FMA_H) { v.x += bias; v.y += bias; }         /* uint16 kernels: FMA_H = 1 marks the offset-uint16 form (16-bit plans) */
                if (p.accumulate) {
                    const int2 o = *reinterpret_cast<const int2*>(row + t);
                    v.x += o.x; v.y += o.y;
                }
                *reinterpret_cast<int2*>(row + t) = v;
            }
        }
    }
}

/* One thread per output, global loads: the route for ranges whose per-tile channel window does not fit shared memory (a DM
 * step so coarse for the band that 30 trials spread over more than ~14 000 samples), and a cross-check. */
template <typename T>
__global__ void k_dedisperse_naive(const T* __restrict__ x, size_t pitch, const int32_t* __restrict__ delays, int nchans, int c0, int c1,
                                   int ndms, long long nt, int32_t* __restrict__ D, long long dpitch, int accumulate,
                                   const unsigned* __restrict__ mode_cnt, unsigned mode_cap) {
    if (mode_cnt && *mode_cnt <= mode_cap) return;                   /* the offset form handles this chunk */
    const long long t = (long long)blockIdx.x * blockDim.x + threadIdx.x;
    const int i = blockIdx.y;
    if (t >= nt || i >= ndms) return;
    const int32_t* dl = delays + (size_t)i * nchans;
    int acc = accumulate ? D[(size_t)i * dpitch + t] : 0;
    for (int c = c0; c < c1; ++c) acc += (int)x[(size_t)c * pitch + (size_t)(t + dl[c])];
    D[(size_t)i * dpitch + t] = acc;
}

template <int IN16, int CB, int FMA_H, int M, int NWC, bool VW>
int launch_vw(const aak_dedisp_args* a, cudaStream_t st) {
    constexpr int NCOPY = IN16 ? 2 : 4;
    DedispParamsT<VW> p;
    p.etab = a->etab; p.x0tab = a->x0tab; p.D = a->D; p.pitch = a->pitch; p.nt = a->nt; p.ndms = a->ndms;
    p.nstages = (a->nchans + CB - 1) / CB;
    /* channel group [chan_begin, chan_end): whole channel blocks (chan_end == 0 means all channels) */
    const int cend = a->chan_end > 0 ? a->chan_end : a->nchans;
    if (a->chan_begin % CB || (cend % CB && cend != a->nchans) || a->chan_begin >= cend) return (int)cudaErrorInvalidValue;
    p.stage_begin = a->chan_begin / CB; p.stage_end = (cend + CB - 1) / CB; p.accumulate = a->accumulate;
    p.mode_cnt = a->mode_cnt; p.mode_cap = a->mode_cap; p.mode_dense = a->mode_dense; p.bias = a->bias;
    p.window_bytes = a->window_bytes; p.spill_stages = a->spill_stages; p.one = 1u;
    if (a->nclass < 1 || a->nclass > 8 || !a->wcls) return (int)cudaErrorInvalidValue;
    if constexpr (VW) {
        p.wcls = a->wcls;
        for (int k = 0; k < 8; ++k) p.class_wb[k] = k < a->nclass ? a->class_wb[k] : 0;
    }
    p.nring = a->ring_stages;
    if (p.nring < 2 || p.nring > MAX_RING) return (int)cudaErrorInvalidValue;
    const size_t smem = SMEM_HEADER + (size_t)p.nring * ((size_t)NCOPY * CB * a->window_bytes + CB * DM_TILE * 4);
    constexpr int DMT = 2 * NWC;                 /* M = 2: NWC groups of 2; M = 4: NWC / 2 groups of 4 */
    if (a->dm_tile != DMT) return (int)cudaErrorInvalidValue;
    const long long ndm_tiles = (a->ndms + DMT - 1) / DMT;
    const long long nt_tiles = (a->nt + T_TILE - 1) / T_TILE;
    p.skew_q16 = a->skew_q16 > 0 ? a->skew_q16 : 0; p.nt_tiles = (int)nt_tiles;
    const long long extra_rows = ((long long)p.skew_q16 * (ndm_tiles - 1)) >> 16;     /* diagonals that start before time tile 0 */
    const long long grid = ndm_tiles * (nt_tiles + extra_rows);
    if (grid <= 0 || grid > 0x7fffffffll) return (int)cudaErrorInvalidConfiguration;
    WindowMaps<VW ? 8 : 1> maps;
    memset(&maps, 0, sizeof maps);
    memcpy(maps.m, a->tmap, sizeof(CUtensorMap) * (size_t)(VW ? a->nclass : 1));
    k_dedisperse<IN16, CB, FMA_H, M, NWC, VW><<<(unsigned)grid, (NWC + 1) * 32, smem, st>>>(maps, p);
    return (int)cudaGetLastError();
}

template <int IN16, int CB, int FMA_H, int M, int NWC>
int launch(const aak_dedisp_args* a, cudaStream_t st) {
    return a->nclass > 1 ? launch_vw<IN16, CB, FMA_H, M, NWC, true>(a, st) : launch_vw<IN16, CB, FMA_H, M, NWC, false>(a, st);
}

template <int IN16, int CB, int FMA_H, int M, int NWC>
int set_attr() {
    int e = (int)cudaFuncSetAttribute(k_dedisperse<IN16, CB, FMA_H, M, NWC, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
    if (e) return e;
    return (int)cudaFuncSetAttribute(k_dedisperse<IN16, CB, FMA_H, M, NWC, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, 227 * 1024);
}

}  // namespace

extern "C" size_t aak_dedisperse_smem_bytes(int32_t chan_block, int32_t window_bytes, int32_t in16, int32_t ring_stages) {
    const size_t ncopy = in16 ? 2 : 4;
    return SMEM_HEADER + (size_t)ring_stages * (ncopy * chan_block * (size_t)window_bytes + (size_t)chan_block * DM_TILE * 4);
}

/* The instantiations the strategy can select (aa_strategy.cpp plan_format): bytes (uint8 input and the offset-uint8 form) =
 * 15 compute warps x 2 trials, odd-byte adds on the FMA pipe (third parameter 3: the same with every sum doubled, for the
 * half-byte form of bin 8, k_bits.cu); binned uint16 = 16 compute warps x 4 adjacent trials with
 * equal-delay reuse (third parameter 1: the offset-uint16 form of a 16-bit plan, which adds the sum of the channel offsets -
 * kept apart because the plain uint16 kernel, at 96 registers with spills, loses 8 % to any change of its epilogue);
 * channel block 8, 4 or 2 by window size. The variants measured and rejected are in profiles/r01c_profiles.md
 * and profiles/r02_all_configs.md (IDP.2A accumulators, 16-byte table loads). */
#define AA_FOR_ALL_VARIANTS(X) \
    X(0, 8, 1, 2, 15) X(0, 4, 1, 2, 15) X(0, 2, 1, 2, 15) \
    X(0, 8, 3, 2, 15) X(0, 4, 3, 2, 15) X(0, 2, 3, 2, 15) \
    X(1, 8, 0, 4, 16) X(1, 4, 0, 4, 16) X(1, 2, 0, 4, 16) \
    X(1, 8, 1, 4, 16) X(1, 4, 1, 4, 16) X(1, 2, 1, 4, 16)

extern "C" int aak_dedisperse_init(void) {
    int e = 0;
#define X(I, C, F, MM, W) if ((e = set_attr<I, C, F, MM, W>())) return e;
    AA_FOR_ALL_VARIANTS(X)
#undef X
    return 0;
}

/* variant (uint8 only): 0 = odd-byte adds as IADD3, 1 = as IMAD (FMA pipe), 2 = alternating; dms_per_warp in {2, 4} */
extern "C" int aak_dedisperse(const aak_dedisp_args* a, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    const int fma = a->in16 ? (a->bias ? 1 : 0) : (a->dms_per_warp == 4 ? (a->variant & 1) : a->variant);
    const int mm = a->dms_per_warp == 4 ? 4 : 2;
    const int nwc = a->dm_tile / 2;
#define X(I, C, F, MM, W) if (a->in16 == I && a->chan_block == C && fma == F && mm == MM && nwc == W) return launch<I, C, F, MM, W>(a, st);
    AA_FOR_ALL_VARIANTS(X)
#undef X
    return (int)cudaErrorInvalidValue;
}

extern "C" int aak_dedisperse_naive(const void* x, size_t pitch_elems, int32_t in16, const int32_t* delays, int32_t nchans,
                                    int32_t chan_begin, int32_t chan_end, int32_t ndms, int64_t nt, int32_t* D, int64_t pitch,
                                    int32_t accumulate, const unsigned* mode_cnt, unsigned mode_cap, void* stream) {
    cudaStream_t st = (cudaStream_t)stream;
    if (ndms <= 0 || nt <= 0) return 0;
    if (ndms > 65535) return (int)cudaErrorInvalidConfiguration;
    dim3 grid((unsigned)((nt + 255) / 256), (unsigned)ndms);
    if (in16)
        k_dedisperse_naive<uint16_t><<<grid, 256, 0, st>>>((const uint16_t*)x, pitch_elems, delays, nchans, chan_begin, chan_end, ndms, nt, D, pitch, accumulate, mode_cnt, mode_cap);
    else
        k_dedisperse_naive<uint8_t><<<grid, 256, 0, st>>>((const uint8_t*)x, pitch_elems, delays, nchans, chan_begin, chan_end, ndms, nt, D, pitch, accumulate, mode_cnt, mode_cap);
    return (int)cudaGetLastError();
}
