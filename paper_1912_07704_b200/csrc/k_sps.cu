/*
 * k_sps.cu — K3 (robust row statistics) and K4 (boxcar SNR + 3x3 peak finding + candidate compaction) for sm_100a.
 *
 * PAPER.md:19 (§1): SPS "uses boxcar filters and peak-finding to maximise signal-to-noise"; data stay on the GPU
 * between dedispersion and SPS. BASELINE.json north_star: "boxcar prefix sums, warp-shuffle reductions for the robust
 * statistics, and peak-finding; candidates are compacted with a warp-aggregated atomic append".
 *
 * Arithmetic (DESIGN.md "Readings" C6-C9). Every floating-point step is an explicit round-to-nearest double operation
 * (__dadd_rn, __dmul_rn, ... are never contracted into FMAs), in the order the definition states, so the values that
 * DECIDE integers (clip bounds, best width, peak comparisons, threshold) are taken in plain IEEE double:
 *   statistics  pivot p = D[0]; exact integer n, S1 = sum(D-p), S2 = sum((D-p)^2) over the kept samples;
 *               mu = p + S1/n; sigma = sqrt((n*S2 - S1^2) / (n*n)); keep = [ceil(mu-3 sigma), floor(mu+3 sigma)];
 *               repeat until (n,S1,S2) repeat, at most 8 clips.
 *   SNR         B_w[t] = sum_{j<w} D[t+j]; snr = ((double)(B_w - w p) - w (mu-p)) * (1/(sqrt(w) sigma));
 *               S[t] = max over valid widths (t+w <= T), smallest width on ties.
 *   peak        S > threshold and S > earlier neighbours, S >= later neighbours in the 3x3 (row, t) neighbourhood.
 */
#include <cuda_runtime.h>
#include <math_constants.h>
#include <stdint.h>
#include "aa_kernels.h"

namespace {

typedef unsigned long long u64;
typedef long long i64;
typedef unsigned __int128 u128;

/* ------------------------------------------------------------------------------------------------ K3 */
constexpr int STAT_THREADS = 512;

__device__ __forceinline__ double u128_to_double_rn(u128 v) {
    const u64 hi = (u64)(v >> 64);
    if (hi == 0) return __ull2double_rn((u64)v);
    const int lz = __clzll((i64)hi);
    const u128 n = v << lz;
    u64 top = (u64)(n >> 64);
    if ((u64)n != 0) top |= 1ull;                 /* sticky bit, far below the rounding position */
    return ldexp(__ull2double_rn(top), 64 - lz);  /* exact scaling */
}

struct Moments { u64 n; i64 s1; u64 s2lo, s2hi; };   /* s2 = s2hi*2^32 + s2lo (sums of the 32-bit halves) */

__device__ __forceinline__ void acc_sample(int v, int p, int lo, int hi, bool clip, unsigned& n, i64& s1, u64& s2) {
    if (clip && (v < lo || v > hi)) return;
    const i64 d = (i64)v - (i64)p;
    ++n; s1 += d; s2 += (u64)(d * d);
}

__device__ Moments block_moments(const int32_t* __restrict__ D, i64 T, int p, int lo, int hi, bool clip, u64* red) {
    unsigned n = 0; i64 s1 = 0; u64 s2 = 0;
    const i64 nvec = T >> 2;
    const int4* Dv = reinterpret_cast<const int4*>(D);
    for (i64 q = threadIdx.x; q < nvec; q += STAT_THREADS) {
        const int4 v = Dv[q];
        acc_sample(v.x, p, lo, hi, clip, n, s1, s2);
        acc_sample(v.y, p, lo, hi, clip, n, s1, s2);
        acc_sample(v.z, p, lo, hi, clip, n, s1, s2);
        acc_sample(v.w, p, lo, hi, clip, n, s1, s2);
    }
    for (i64 t = (nvec << 2) + threadIdx.x; t < T; t += STAT_THREADS) acc_sample(D[t], p, lo, hi, clip, n, s1, s2);
    u64 a = n, b = (u64)s1, c = s2 & 0xFFFFFFFFull, d = s2 >> 32;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
        c += __shfl_down_sync(0xffffffffu, c, o);
        d += __shfl_down_sync(0xffffffffu, d, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();                       /* red[] may still be read from the previous pass */
    if (lane == 0) { red[warp * 4 + 0] = a; red[warp * 4 + 1] = b; red[warp * 4 + 2] = c; red[warp * 4 + 3] = d; }
    __syncthreads();
    Moments m; m.n = 0; m.s1 = 0; m.s2lo = 0; m.s2hi = 0;
    for (int w = 0; w < STAT_THREADS / 32; ++w) {
        m.n += red[w * 4 + 0]; m.s1 += (i64)red[w * 4 + 1]; m.s2lo += red[w * 4 + 2]; m.s2hi += red[w * 4 + 3];
    }
    return m;                              /* every thread holds the same totals */
}

__device__ __forceinline__ void mu_sigma_of(int p, const Moments& m, double& mu, double& sigma) {
    const u128 s2 = ((u128)m.s2hi << 32) + (u128)m.s2lo;
    const u128 s1sq = (u128)((unsigned __int128)((__int128)m.s1 * (__int128)m.s1));
    const u128 num = (u128)m.n * s2 - s1sq;                         /* n^2 * variance, exact, >= 0 */
    const double nd = __ull2double_rn(m.n);
    mu = __dadd_rn((double)p, __ddiv_rn(__ll2double_rn(m.s1), nd));
    const double var = __ddiv_rn(u128_to_double_rn(num), __dmul_rn(nd, nd));
    sigma = __dsqrt_rn(var);
}

__device__ __forceinline__ int clamp_i32(double x) {
    if (x <= -2147483648.0) return INT32_MIN;
    if (x >= 2147483647.0) return INT32_MAX;
    return (int)x;                          /* x is integral here */
}

__global__ void __launch_bounds__(STAT_THREADS)
k_row_stats(const aak_row_desc* __restrict__ rows, double* __restrict__ mu_sigma, i64* __restrict__ n_iters) {
    __shared__ u64 red[(STAT_THREADS / 32) * 4];
    const aak_row_desc rd = rows[blockIdx.x];
    const int32_t* D = rd.D;
    const i64 T = rd.nt;
    const int p = D[0];
    Moments m = block_moments(D, T, p, 0, 0, false, red);
    double mu, sigma;
    mu_sigma_of(p, m, mu, sigma);
    int it = 0;
    bool degenerate = false;
    for (it = 0; it < 8; ++it) {
        const double t3 = __dmul_rn(3.0, sigma);
        const int lo = clamp_i32(ceil(__dsub_rn(mu, t3)));
        const int hi = clamp_i32(floor(__dadd_rn(mu, t3)));
        const Moments m2 = block_moments(D, T, p, lo, hi, true, red);
        if (m2.n == 0) { degenerate = true; ++it; break; }
        const bool same = (m2.n == m.n && m2.s1 == m.s1 && m2.s2lo == m.s2lo && m2.s2hi == m.s2hi);
        m = m2;
        mu_sigma_of(p, m, mu, sigma);
        if (same) { ++it; break; }
    }
    if (threadIdx.x == 0) {
        mu_sigma[2 * (size_t)blockIdx.x] = mu;
        mu_sigma[2 * (size_t)blockIdx.x + 1] = degenerate ? 0.0 : sigma;
        n_iters[2 * (size_t)blockIdx.x] = degenerate ? 0 : (i64)m.n;
        n_iters[2 * (size_t)blockIdx.x + 1] = it;
    }
}

/* ------------------------------------------------------------------------------------------------ K4 */
constexpr int SPS_ROWS = 8;                    /* centre rows per CTA */
constexpr int SPS_TT = 512;                    /* centre samples per CTA */
constexpr int SPS_WARPS = SPS_ROWS + 2;        /* one warp per row incl. the two halo rows */
constexpr int SPS_THREADS = SPS_WARPS * 32;
constexpr int SPS_Q = SPS_TT + 2;              /* positions per row incl. the two halo columns */
constexpr int SPS_MAXW = 16;

struct SpsParams {
    const int32_t* D; i64 pitch; i64 nt; int ndms; int bin; int range_index;
    double dm_low, dm_step;
    const double* mu_sigma;
    u64 chunk_start;
    int widths[SPS_MAXW]; int nwidths; int wmax;
    double threshold;
    aak_candidate* cands; u64* counter; u64 capacity;
};

__global__ void __launch_bounds__(SPS_THREADS)
k_sps_peaks(const SpsParams p) {
    extern __shared__ __align__(16) uint8_t sm[];
    const int NE = SPS_Q + p.wmax;                                   /* samples loaded per row */
    double* S = reinterpret_cast<double*>(sm);                       /* [SPS_WARPS][SPS_Q] */
    double* cst = S + SPS_WARPS * SPS_Q;                             /* [SPS_WARPS][2*SPS_MAXW]: a_w, inv_w */
    int* P = reinterpret_cast<int*>(cst + SPS_WARPS * 2 * SPS_MAXW); /* [SPS_WARPS][NE+1] */
    unsigned short* Wb = reinterpret_cast<unsigned short*>(P + SPS_WARPS * (NE + 1));   /* [SPS_WARPS][SPS_Q] */

    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    const i64 t0 = (i64)blockIdx.x * SPS_TT;
    const int i_base = blockIdx.y * SPS_ROWS;
    const int rr = i_base - 1 + warp;                                /* this warp's DM row */
    double* Srow = S + warp * SPS_Q;
    unsigned short* Wrow = Wb + warp * SPS_Q;
    const double ninf = -CUDART_INF;

    bool live = (rr >= 0 && rr < p.ndms);
    double sigma = 0.0, mu = 0.0;
    if (live) { mu = p.mu_sigma[2 * (size_t)rr]; sigma = p.mu_sigma[2 * (size_t)rr + 1]; live = sigma > 0.0; }
    if (!live) {
        for (int q = lane; q < SPS_Q; q += 32) { Srow[q] = ninf; Wrow[q] = 0; }
    } else {
        const int32_t* Drow = p.D + (size_t)rr * (size_t)p.pitch;
        const int pv = Drow[0];
        int* Prow = P + warp * (NE + 1);
        double* crow = cst + warp * 2 * SPS_MAXW;
        if (lane < p.nwidths) {
            const double w = (double)p.widths[lane];
            crow[lane] = __dmul_rn(w, __dsub_rn(mu, (double)pv));
            crow[SPS_MAXW + lane] = __ddiv_rn(1.0, __dmul_rn(__dsqrt_rn(w), sigma));
        }
        /* prefix sums of d = D - p over [t0-1, t0-1+NE): wrapping int32, differences are exact (plan limit) */
        int carry = 0;
        if (lane == 0) Prow[0] = 0;
        for (int e0 = 0; e0 < NE; e0 += 32) {
            const int e = e0 + lane;
            const i64 t = t0 - 1 + e;
            int d = 0;
            if (e < NE && t >= 0 && t < p.nt) d = Drow[t] - pv;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const int u = __shfl_up_sync(0xffffffffu, d, o);
                if (lane >= o) d += u;
            }
            d += carry;
            if (e < NE) Prow[e + 1] = d;
            carry = __shfl_sync(0xffffffffu, d, 31);
        }
        __syncwarp();
        for (int q = lane; q < SPS_Q; q += 32) {
            const i64 t = t0 - 1 + q;
            double best = ninf; int bw = 0;
            if (t >= 0 && t < p.nt) {
                const int base = Prow[q];
                for (int iw = 0; iw < p.nwidths; ++iw) {
                    const int w = p.widths[iw];
                    if (t + w > p.nt) break;                       /* ascending widths */
                    const int B = Prow[q + w] - base;
                    const double snr = __dmul_rn(__dsub_rn(__int2double_rn(B), crow[iw]), crow[SPS_MAXW + iw]);
                    if (snr > best) { best = snr; bw = w; }
                }
            }
            Srow[q] = best; Wrow[q] = (unsigned short)bw;
        }
    }
    __syncthreads();

    /* 3x3 local maxima on the centre rows/columns; warp-aggregated append */
    constexpr int NPOS = SPS_ROWS * SPS_TT;
    for (int k = 0; k < (NPOS + SPS_THREADS - 1) / SPS_THREADS; ++k) {      /* uniform trip count: ballots need every lane */
        const int idx = k * SPS_THREADS + threadIdx.x;
        bool is = false; int r = 0, q = 0; double s = 0.0;
        if (idx < NPOS) {
            r = idx / SPS_TT + 1; q = idx % SPS_TT + 1;
            const int i = i_base + r - 1; const i64 t = t0 + q - 1;
            if (i < p.ndms && t < p.nt) {
                s = S[r * SPS_Q + q];
                if (s > p.threshold) {
                    is = true;
#pragma unroll
                    for (int dr = -1; dr <= 1; ++dr)
#pragma unroll
                        for (int dq = -1; dq <= 1; ++dq) {
                            if (dr == 0 && dq == 0) continue;
                            const double v = S[(r + dr) * SPS_Q + (q + dq)];
                            const bool before = (dr < 0) || (dr == 0 && dq < 0);
                            if (before ? !(s > v) : !(s >= v)) is = false;
                        }
                }
            }
        }
        const unsigned mask = __ballot_sync(0xffffffffu, is);
        if (mask) {
            const int leader = __ffs(mask) - 1;
            u64 base = 0;
            if (lane == leader) base = atomicAdd(p.counter, (u64)__popc(mask));
            base = __shfl_sync(0xffffffffu, base, leader);
            if (is) {
                const u64 slot = base + (u64)__popc(mask & ((1u << lane) - 1u));
                if (slot < p.capacity) {
                    const int i = i_base + r - 1;
                    aak_candidate c;
                    c.sample = p.chunk_start + (u64)p.bin * (u64)(t0 + q - 1);
                    c.dm = (float)__dadd_rn(p.dm_low, __dmul_rn((double)i, p.dm_step));
                    c.snr = (float)s;
                    c.width = (uint32_t)p.bin * (uint32_t)Wb[r * SPS_Q + q];
                    c.range = (uint32_t)p.range_index;
                    c.dm_index = (uint32_t)i;
                    p.cands[slot] = c;
                }
            }
        }
    }
}

size_t sps_smem_bytes(int wmax) {
    const int NE = SPS_Q + wmax;
    return (size_t)SPS_WARPS * SPS_Q * 8 + (size_t)SPS_WARPS * 2 * SPS_MAXW * 8 + (size_t)SPS_WARPS * (NE + 1) * 4 +
           (size_t)SPS_WARPS * SPS_Q * 2 + 16;
}

}  // namespace

extern "C" int aak_row_stats(const aak_row_desc* rows, int32_t nrows, double* mu_sigma, int64_t* n_iters, void* stream) {
    if (nrows <= 0) return 0;
    k_row_stats<<<(unsigned)nrows, STAT_THREADS, 0, (cudaStream_t)stream>>>(rows, mu_sigma, (i64*)n_iters);
    return (int)cudaGetLastError();
}

extern "C" int aak_sps_init(void) {
    return (int)cudaFuncSetAttribute(k_sps_peaks, cudaFuncAttributeMaxDynamicSharedMemorySize, 200 * 1024);
}

extern "C" int aak_sps_peaks(const aak_sps_args* a, void* stream) {
    if (a->nwidths < 1 || a->nwidths > SPS_MAXW) return (int)cudaErrorInvalidValue;
    SpsParams p;
    p.D = a->D; p.pitch = a->pitch; p.nt = a->nt; p.ndms = a->ndms; p.bin = a->bin; p.range_index = a->range_index;
    p.dm_low = a->dm_low; p.dm_step = a->dm_step; p.mu_sigma = a->mu_sigma; p.chunk_start = a->chunk_start;
    p.nwidths = a->nwidths; p.wmax = 0;
    for (int k = 0; k < SPS_MAXW; ++k) { p.widths[k] = k < a->nwidths ? a->widths[k] : 0; if (p.widths[k] > p.wmax) p.wmax = p.widths[k]; }
    p.threshold = a->threshold; p.cands = a->cands; p.counter = (u64*)a->counter; p.capacity = a->capacity;
    const size_t smem = sps_smem_bytes(p.wmax);
    if (smem > 200 * 1024) return (int)cudaErrorInvalidValue;
    dim3 grid((unsigned)((a->nt + SPS_TT - 1) / SPS_TT), (unsigned)((a->ndms + SPS_ROWS - 1) / SPS_ROWS));
    k_sps_peaks<<<grid, SPS_THREADS, smem, (cudaStream_t)stream>>>(p);
    return (int)cudaGetLastError();
}
