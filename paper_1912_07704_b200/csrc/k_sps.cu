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
constexpr int STAT_THREADS = 256;
constexpr int SPS_MAXW = 16;                 /* aa_plan_create: at most 16 boxcar widths */

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

/* Single-pass form. The clip iterations only ever move samples in the TAILS of the row's distribution in or out, so the
 * row is read once: samples inside a provisional CORE interval [clo, chi] (about +-2.75 sigma, estimated from the head
 * of the row) are reduced to their exact moments straight away, every other sample is kept in a list in shared memory
 * (0.6 % of a Gaussian row). Each iteration of reading C6 then needs core + (list entries inside its bounds), the same
 * exact integers the full passes give (integer sums do not depend on the order or grouping). If a bound ever cuts into
 * the core, or the list overflows, the row falls back to the plain multi-pass loop below - same result, more reads. */
constexpr int STAT_LIST_CAP = 12288;                 /* int32 entries of shared memory per row (48 KB: 4 CTAs per SM) */
constexpr double STAT_CORE_Z = 2.75;                 /* core half-width in head sigmas: 0.6 % of a Gaussian row goes to the list */
constexpr int STAT_HEAD = 8192;                      /* samples used for the provisional core */

struct StatSmem {
    u64 red[(STAT_THREADS / 32) * 4];
    int cnt;
    int overflow;
    int list[STAT_LIST_CAP];
};

__device__ Moments list_moments(const int* list, int n_list, int p, int lo, int hi, u64* red) {
    unsigned n = 0; i64 s1 = 0; u64 s2 = 0;
    for (int q = threadIdx.x; q < n_list; q += STAT_THREADS) acc_sample(list[q], p, lo, hi, true, n, s1, s2);
    u64 a = n, b = (u64)s1, c = s2 & 0xFFFFFFFFull, d = s2 >> 32;
#pragma unroll
    for (int o = 16; o > 0; o >>= 1) {
        a += __shfl_down_sync(0xffffffffu, a, o);
        b += __shfl_down_sync(0xffffffffu, b, o);
        c += __shfl_down_sync(0xffffffffu, c, o);
        d += __shfl_down_sync(0xffffffffu, d, o);
    }
    const int warp = threadIdx.x >> 5, lane = threadIdx.x & 31;
    __syncthreads();
    if (lane == 0) { red[warp * 4 + 0] = a; red[warp * 4 + 1] = b; red[warp * 4 + 2] = c; red[warp * 4 + 3] = d; }
    __syncthreads();
    Moments m; m.n = 0; m.s1 = 0; m.s2lo = 0; m.s2hi = 0;
    for (int w = 0; w < STAT_THREADS / 32; ++w) {
        m.n += red[w * 4 + 0]; m.s1 += (i64)red[w * 4 + 1]; m.s2lo += red[w * 4 + 2]; m.s2hi += red[w * 4 + 3];
    }
    return m;
}

__device__ __forceinline__ Moments add_moments(const Moments& a, const Moments& b) {
    Moments m; m.n = a.n + b.n; m.s1 = a.s1 + b.s1; m.s2lo = a.s2lo + b.s2lo; m.s2hi = a.s2hi + b.s2hi; return m;
}
__device__ __forceinline__ bool same_moments(const Moments& a, const Moments& b) {
    /* s2 is carried as two partial sums whose split depends on the grouping: compare the value s2hi*2^32 + s2lo */
    const u128 x = ((u128)a.s2hi << 32) + (u128)a.s2lo, y = ((u128)b.s2hi << 32) + (u128)b.s2lo;
    return a.n == b.n && a.s1 == b.s1 && x == y;
}

/* one core-vs-list decision per sample; a list append is one shared-memory atomic (0.6 % of the samples of a Gaussian row) */
__device__ __forceinline__ void split_sample(bool valid, int v, int p, int clo, int chi, unsigned& n, i64& s1, u64& s2,
                                             StatSmem& sm, int lane) {
    if (!valid) return;
    if (v >= clo && v <= chi) {
        const i64 d = (i64)v - (i64)p;
        ++n; s1 += d; s2 += (u64)(d * d);
    } else {
        const int slot = atomicAdd(&sm.cnt, 1);
        if (slot < STAT_LIST_CAP) sm.list[slot] = v; else sm.overflow = 1;
    }
}

__global__ void __launch_bounds__(STAT_THREADS, 4)
k_row_stats(const aak_row_desc* __restrict__ rows, double* __restrict__ mu_sigma, i64* __restrict__ n_iters) {
    extern __shared__ __align__(16) uint8_t stat_raw[];
    StatSmem& sm = *reinterpret_cast<StatSmem*>(stat_raw);
    u64* red = sm.red;
    const aak_row_desc rd = rows[blockIdx.x];
    const int32_t* D = rd.D;
    const i64 T = rd.nt;
    const int p = D[0];
    const int lane = threadIdx.x & 31;
    double mu, sigma;
    Moments m;
    bool fast = false;
    Moments core; core.n = 0; core.s1 = 0; core.s2lo = 0; core.s2hi = 0;
    int clo = 0, chi = -1, n_list = 0;

    /* ---- provisional core from the head of the row (any interval would be CORRECT; this one makes the list short) */
    {
        const i64 Th = T < STAT_HEAD ? T : STAT_HEAD;
        const Moments h = block_moments(D, Th, p, 0, 0, false, red);
        double hm, hs;
        mu_sigma_of(p, h, hm, hs);
        if (hs > 0.0 && hs < 1.0e8) {
            clo = clamp_i32(ceil(hm - STAT_CORE_Z * hs));
            chi = clamp_i32(floor(hm + STAT_CORE_Z * hs));
        }
        if (threadIdx.x == 0) { sm.cnt = 0; sm.overflow = 0; }
        __syncthreads();
    }
    if (chi >= clo) {
        /* ---- the single pass over the row */
        unsigned n = 0; i64 s1 = 0; u64 s2 = 0;
        const i64 nvec = T >> 2;
        const int4* Dv = reinterpret_cast<const int4*>(D);
        const i64 nvec_pad = (nvec + STAT_THREADS - 1) / STAT_THREADS * STAT_THREADS;     /* uniform trip count for the ballots */
        constexpr int U = 8;                                                            /* 128 bytes in flight per thread */
        for (i64 q0 = 0; q0 < nvec_pad; q0 += U * STAT_THREADS) {
            int4 v[U]; bool ok[U];
#pragma unroll
            for (int u = 0; u < U; ++u) {
                const i64 q = q0 + u * STAT_THREADS + threadIdx.x;
                ok[u] = q < nvec;
                v[u] = ok[u] ? __ldg(Dv + q) : make_int4(0, 0, 0, 0);
            }
#pragma unroll
            for (int u = 0; u < U; ++u) {
                split_sample(ok[u], v[u].x, p, clo, chi, n, s1, s2, sm, lane);
                split_sample(ok[u], v[u].y, p, clo, chi, n, s1, s2, sm, lane);
                split_sample(ok[u], v[u].z, p, clo, chi, n, s1, s2, sm, lane);
                split_sample(ok[u], v[u].w, p, clo, chi, n, s1, s2, sm, lane);
            }
        }
        {
            const i64 t = (nvec << 2) + threadIdx.x;                                    /* at most 3 tail samples */
            const bool ok = t < T;
            split_sample(ok, ok ? D[t] : 0, p, clo, chi, n, s1, s2, sm, lane);
        }
        u64 a = n, b = (u64)s1, c = s2 & 0xFFFFFFFFull, d = s2 >> 32;
#pragma unroll
        for (int o = 16; o > 0; o >>= 1) {
            a += __shfl_down_sync(0xffffffffu, a, o);
            b += __shfl_down_sync(0xffffffffu, b, o);
            c += __shfl_down_sync(0xffffffffu, c, o);
            d += __shfl_down_sync(0xffffffffu, d, o);
        }
        const int warp = threadIdx.x >> 5;
        __syncthreads();
        if (lane == 0) { red[warp * 4 + 0] = a; red[warp * 4 + 1] = b; red[warp * 4 + 2] = c; red[warp * 4 + 3] = d; }
        __syncthreads();
        for (int w = 0; w < STAT_THREADS / 32; ++w) {
            core.n += red[w * 4 + 0]; core.s1 += (i64)red[w * 4 + 1]; core.s2lo += red[w * 4 + 2]; core.s2hi += red[w * 4 + 3];
        }
        n_list = sm.cnt;
        fast = (sm.overflow == 0) && n_list <= STAT_LIST_CAP;
    }

    int it = 0;
    bool degenerate = false;
    if (fast) {
        m = add_moments(core, list_moments(sm.list, n_list, p, INT32_MIN, INT32_MAX, red));      /* unclipped row */
        mu_sigma_of(p, m, mu, sigma);
        for (it = 0; it < 8; ++it) {
            const double t3 = __dmul_rn(3.0, sigma);
            const int lo = clamp_i32(ceil(__dsub_rn(mu, t3)));
            const int hi = clamp_i32(floor(__dadd_rn(mu, t3)));
            if (lo > clo || hi < chi) { fast = false; break; }       /* a bound cuts into the core: take the plain route */
            const Moments m2 = add_moments(core, list_moments(sm.list, n_list, p, lo, hi, red));
            if (m2.n == 0) { degenerate = true; ++it; break; }
            const bool same = same_moments(m2, m);
            m = m2;
            mu_sigma_of(p, m, mu, sigma);
            if (same) { ++it; break; }
        }
    }
    if (!fast) {
        /* ---- plain route: one pass over the row per iteration (reading C6 written out) */
        degenerate = false;
        m = block_moments(D, T, p, 0, 0, false, red);
        mu_sigma_of(p, m, mu, sigma);
        for (it = 0; it < 8; ++it) {
            const double t3 = __dmul_rn(3.0, sigma);
            const int lo = clamp_i32(ceil(__dsub_rn(mu, t3)));
            const int hi = clamp_i32(floor(__dadd_rn(mu, t3)));
            const Moments m2 = block_moments(D, T, p, lo, hi, true, red);
            if (m2.n == 0) { degenerate = true; ++it; break; }
            const bool same = same_moments(m2, m);
            m = m2;
            mu_sigma_of(p, m, mu, sigma);
            if (same) { ++it; break; }
        }
    }
    if (threadIdx.x == 0) {
        mu_sigma[2 * (size_t)blockIdx.x] = mu;
        mu_sigma[2 * (size_t)blockIdx.x + 1] = degenerate ? 0.0 : sigma;
        n_iters[2 * (size_t)blockIdx.x] = degenerate ? 0 : (i64)m.n;
        n_iters[2 * (size_t)blockIdx.x + 1] = it;
    }
}


/* ------------------------------------------------------------------------------------------------ K3w
 * Per-width measured statistics (reading C7m; SURVEY §8(f3) "per-width measured sigma instead of sqrt(w)
 * scaling"). One CTA per DM row. The row is walked in tiles: exclusive prefix sums of d = D - D[0] in shared memory (thread
 * scan + warp shuffle scan + cross-warp carry), then e = B_w[t] - w D[0] = I[t+w] - I[t] for every width that is still
 * iterating, and the exact integer moments (n, sum e, sum e^2) of the kept samples. One pass over the row per clip iteration
 * (pass 0 unclipped, then at most 8 clips), all widths in the same pass. The moments are taken about w D[0] (e fits int32 by
 * the plan's boxcar limit; sum e^2 is carried to 96 bits) and moved to the definition's pivot p_w = B_w[0] exactly in
 * 128-bit integers before the double arithmetic, which follows reading C6 operation by operation. */
constexpr int PW_THREADS = 512;
constexpr int PW_TILE = 4096;                 /* series samples per tile */
constexpr int PW_MAXW = 2048;                 /* aa_plan_create: boxcar widths <= 2048 */
constexpr int PW_EPT = (PW_TILE + PW_MAXW) / PW_THREADS;     /* 12 contiguous elements per thread */
static_assert(PW_EPT * PW_THREADS == PW_TILE + PW_MAXW && PW_EPT % 4 == 0, "prefix tile layout");

struct PwParams {
    const int32_t* D; i64 pitch; i64 nt; i64 ntd; int widths[SPS_MAXW]; int nwidths; int wmax;
    double* wstats; i64* wpivot; int* wlive;
};

struct PwSmem {
    unsigned I[PW_TILE + PW_MAXW + 8];        /* I[e] = sum_{j<e} d[t0+j] (mod 2^32) */
    unsigned wtot[PW_THREADS / 32];
    u64 red[SPS_MAXW][PW_THREADS / 32][6];    /* per width and warp: n, sum e, and sum e^2 as four 32-bit limbs */
    i64 nw[SPS_MAXW];                         /* series length n_w */
    int q[SPS_MAXW];                          /* B_w[0] - w p */
    int lo[SPS_MAXW], hi[SPS_MAXW];           /* clip bounds on e, clamped to int32 (lo > hi: nothing is kept) */
    int active[SPS_MAXW];                     /* still iterating */
    u64 pn[SPS_MAXW]; i64 ps1[SPS_MAXW]; u64 ps2lo[SPS_MAXW], ps2hi[SPS_MAXW];      /* previous keep set */
    double mu[SPS_MAXW], sigma[SPS_MAXW];
    int nactive;
};

__device__ __forceinline__ i64 clamp_i64(double x) {
    if (!(x > -9.0e18)) return (i64)(-9000000000000000000ll);
    if (!(x < 9.0e18)) return (i64)(9000000000000000000ll);
    return (i64)x;                            /* x is integral here */
}

template <int NWT>
__global__ void __launch_bounds__(PW_THREADS, 1)
k_row_width_stats(const PwParams p) {
    __shared__ PwSmem sm;
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const int32_t* D = p.D + (size_t)blockIdx.x * (size_t)p.pitch;
    const int pv = D[0];
    const i64 T = p.nt, Tx = p.ntd;
    if (tid < SPS_MAXW) {
        i64 n = 0;
        if (tid < p.nwidths) { n = Tx - p.widths[tid] + 1; if (n > T) n = T; if (n < 0) n = 0; }
        sm.nw[tid] = n; sm.active[tid] = n >= 1 ? 1 : 0; sm.q[tid] = 0; sm.lo[tid] = INT32_MIN; sm.hi[tid] = INT32_MAX;
        sm.mu[tid] = 0.0; sm.sigma[tid] = 0.0;
    }
    if (tid == 0) sm.nactive = 1;
    __syncthreads();

    for (int pass = 0; pass <= 8 && sm.nactive > 0; ++pass) {
        unsigned an[NWT], ahi[NWT]; i64 as1[NWT]; u64 alo[NWT];
#pragma unroll
        for (int iw = 0; iw < NWT; ++iw) { an[iw] = 0; ahi[iw] = 0; as1[iw] = 0; alo[iw] = 0; }
        for (i64 t0 = 0; t0 < T; t0 += PW_TILE) {
            /* ---- exclusive prefix sums of the segment [t0, t0 + PW_TILE + wmax) that exists */
            const i64 avail = Tx - t0;
            const int ne = (int)(avail < (i64)(PW_TILE + p.wmax) ? avail : (i64)(PW_TILE + p.wmax));
            const int e0 = tid * PW_EPT;
            unsigned loc[PW_EPT];
            unsigned run = 0;
#pragma unroll
            for (int v = 0; v < PW_EPT / 4; ++v) {
                const int e = e0 + 4 * v;
                int4 x = make_int4(pv, pv, pv, pv);
                if (e < ne) x = __ldg(reinterpret_cast<const int4*>(D + t0 + e));      /* rows are padded to 128 elements */
                loc[4 * v + 0] = run; run += (unsigned)(x.x - pv);
                loc[4 * v + 1] = run; run += (unsigned)(x.y - pv);
                loc[4 * v + 2] = run; run += (unsigned)(x.z - pv);
                loc[4 * v + 3] = run; run += (unsigned)(x.w - pv);
            }
            unsigned incl = run;
#pragma unroll
            for (int o = 1; o < 32; o <<= 1) {
                const unsigned u = __shfl_up_sync(0xffffffffu, incl, o);
                if (lane >= o) incl += u;
            }
            if (lane == 31) sm.wtot[warp] = incl;
            __syncthreads();
            unsigned carry = incl - run;
#pragma unroll
            for (int w = 0; w < PW_THREADS / 32; ++w) carry += (w < warp) ? sm.wtot[w] : 0u;
#pragma unroll
            for (int v = 0; v < PW_EPT / 4; ++v)
                *reinterpret_cast<uint4*>(&sm.I[e0 + 4 * v]) = make_uint4(loc[4 * v] + carry, loc[4 * v + 1] + carry, loc[4 * v + 2] + carry, loc[4 * v + 3] + carry);
            if (tid == PW_THREADS - 1) sm.I[PW_TILE + PW_MAXW] = run + carry;
            __syncthreads();
            if (pass == 0 && t0 == 0 && tid < p.nwidths && sm.nw[tid] >= 1) sm.q[tid] = (int)sm.I[p.widths[tid]];   /* B_w[0] - w p */

            /* ---- moments of the kept samples of every width that is still iterating */
            int klim[NWT], lo[NWT], hi[NWT];                          /* samples of this tile that belong to the width's series */
            int kmax = 0;
#pragma unroll
            for (int iw = 0; iw < NWT; ++iw) {
                const i64 left = sm.nw[iw] - t0;
                klim[iw] = sm.active[iw] ? (int)(left < 0 ? 0 : (left > (i64)PW_TILE ? (i64)PW_TILE : left)) : 0;
                lo[iw] = sm.lo[iw]; hi[iw] = sm.hi[iw];
                kmax = klim[iw] > kmax ? klim[iw] : kmax;
            }
#pragma unroll 2
            for (int k = tid; k < kmax; k += PW_THREADS) {
                const unsigned base = sm.I[k];
#pragma unroll
                for (int iw = 0; iw < NWT; ++iw) {
                    if (k >= klim[iw]) continue;
                    const int e = (int)(sm.I[k + p.widths[iw]] - base);
                    if (e < lo[iw] || e > hi[iw]) continue;
                    const u64 e2 = (u64)((i64)e * (i64)e);
                    ++an[iw]; as1[iw] += e;
                    alo[iw] += e2; ahi[iw] += (alo[iw] < e2) ? 1u : 0u;
                }
            }
            __syncthreads();
        }
        /* ---- block totals per width */
#pragma unroll
        for (int iw = 0; iw < NWT; ++iw) {
            if (!sm.active[iw]) continue;                             /* block-uniform */
            u64 v[6] = {(u64)an[iw], (u64)as1[iw], alo[iw] & 0xFFFFFFFFull, alo[iw] >> 32, (u64)ahi[iw], 0ull};
#pragma unroll
            for (int o = 16; o > 0; o >>= 1) {
#pragma unroll
                for (int j = 0; j < 5; ++j) v[j] += __shfl_down_sync(0xffffffffu, v[j], o);
            }
            if (lane == 0) {
#pragma unroll
                for (int j = 0; j < 5; ++j) sm.red[iw][warp][j] = v[j];
            }
        }
        __syncthreads();
        if (tid < p.nwidths && sm.active[tid]) {
            const int iw = tid;
            u64 n2 = 0; i64 s1e = 0; u128 s2e = 0;
            for (int w = 0; w < PW_THREADS / 32; ++w) {
                n2 += sm.red[iw][w][0]; s1e += (i64)sm.red[iw][w][1];
                s2e += (u128)sm.red[iw][w][2] + ((u128)sm.red[iw][w][3] << 32) + ((u128)sm.red[iw][w][4] << 64);
            }
            bool done = false;
            if (pass > 0 && n2 == 0) {                                /* degenerate clip: the width yields no SNR in this row */
                sm.sigma[iw] = 0.0; done = true;
            } else {
                const bool same = pass > 0 && n2 == sm.pn[iw] && s1e == sm.ps1[iw] && (u64)s2e == sm.ps2lo[iw] && (u64)(s2e >> 64) == sm.ps2hi[iw];
                sm.pn[iw] = n2; sm.ps1[iw] = s1e; sm.ps2lo[iw] = (u64)s2e; sm.ps2hi[iw] = (u64)(s2e >> 64);
                /* to the pivot of the definition, p_w = B_w[0] = w p + q: d = e - q */
                const i64 q = sm.q[iw];
                const __int128 S1 = (__int128)s1e - (__int128)n2 * q;
                const __int128 S2 = (__int128)s2e - 2 * (__int128)q * (__int128)s1e + (__int128)n2 * ((__int128)q * q);
                const u128 num = (u128)((__int128)n2 * S2 - S1 * S1);           /* n^2 * variance, exact, >= 0 */
                const i64 pw = (i64)p.widths[iw] * (i64)pv + q;
                const double nd = __ull2double_rn(n2);
                const double mu = __dadd_rn(__ll2double_rn(pw), __ddiv_rn(__ll2double_rn((i64)S1), nd));
                const double sigma = __dsqrt_rn(__ddiv_rn(u128_to_double_rn(num), __dmul_rn(nd, nd)));
                sm.mu[iw] = mu; sm.sigma[iw] = sigma;
                if (same || pass == 8) done = true;
                else {
                    const double t3 = __dmul_rn(3.0, sigma);
                    const i64 shift = (i64)p.widths[iw] * (i64)pv;            /* bounds on B_w -> bounds on e = B_w - w p */
                    const i64 l = clamp_i64(ceil(__dsub_rn(mu, t3))) - shift, h = clamp_i64(floor(__dadd_rn(mu, t3))) - shift;
                    if (l > (i64)INT32_MAX || h < (i64)INT32_MIN || l > h) { sm.lo[iw] = 1; sm.hi[iw] = 0; }
                    else { sm.lo[iw] = l < (i64)INT32_MIN ? INT32_MIN : (int)l; sm.hi[iw] = h > (i64)INT32_MAX ? INT32_MAX : (int)h; }
                }
            }
            if (done) sm.active[iw] = 0;
        }
        __syncthreads();
        if (tid == 0) { int n = 0; for (int iw = 0; iw < p.nwidths; ++iw) n += sm.active[iw]; sm.nactive = n; }
        __syncthreads();
    }
    if (tid < p.nwidths) {
        const size_t o = (size_t)blockIdx.x * (size_t)p.nwidths + (size_t)tid;
        const bool has = sm.nw[tid] >= 1;
        p.wstats[2 * o] = has ? sm.mu[tid] : 0.0;
        p.wstats[2 * o + 1] = has ? sm.sigma[tid] : 0.0;
        p.wpivot[o] = has ? (i64)p.widths[tid] * (i64)pv + (i64)sm.q[tid] : 0;
    }
    if (tid == 0) {
        int live = 0;
        for (int iw = 0; iw < p.nwidths; ++iw) live |= (sm.nw[iw] >= 1 && sm.sigma[iw] > 0.0) ? 1 : 0;
        p.wlive[blockIdx.x] = live;
    }
}

/* ------------------------------------------------------------------------------------------------ K4
 * One CTA walks DOWN a band of K4_RB DM rows (plus one halo row above and below, recomputed, not exchanged) for one
 * strip of TT output samples. Per row step:
 *   1. the row segment (TT + 5 + wmax samples, loaded as int4 one step ahead into registers) is turned into inclusive
 *      prefix sums of d = D - pivot: thread-local serial scan of 4V contiguous samples, warp shuffle scan of the thread
 *      totals, cross-warp carry through shared memory; the prefix row goes into a 3-row ring in shared memory;
 *   2. INTEGER prefilter: position t can only exceed the threshold if for some width B_w - w p >= bmin_w, where
 *      bmin_w = floor(a_w + threshold/inv_w) - 2 is computed once per (row, width) in double (2 below the exact bound:
 *      conservative, the rounding error of the SNR expression is < 2^-20 in these units). That is 3 integer
 *      instructions per (sample, width) and no double arithmetic on the common path. Flagged positions are appended
 *      to a per-row list in shared memory (warp-aggregated);
 *   3. for each flagged position of the PREVIOUS row (whose lower neighbour row is now in the ring) the exact double
 *      SNR map S is evaluated on demand for the position and its 8 neighbours, in the operation order of reading C7,
 *      then S > threshold and the 3x3 rule of reading C8 decide; candidates are appended to the global list with one
 *      atomic per warp (ballot + popc).
 * Two __syncthreads per row step. The result is the same set the plain definition gives: step 2 never drops a
 * position whose S exceeds the threshold, and step 3 is the definition itself.
 */
constexpr int K4_THREADS = 256;
constexpr int K4_WARPS = K4_THREADS / 32;
constexpr int K4_RB = 32;                      /* centre rows per CTA (fewer when the grid would not fill the GPU) */

struct SpsParams {
    const int32_t* D; i64 pitch; i64 nt; i64 ntd; int ndms; int bin; int range_index;   /* ntd: samples present per row >= nt */
    double dm_low, dm_step;
    const double* mu_sigma;
    u64 chunk_start;
    int widths[SPS_MAXW]; int nwidths; int wmax; int pow2;      /* pow2: widths[i] == 1 << i */
    int tt;                                    /* centre samples per strip, multiple of 4 */
    int rb;                                    /* centre rows per CTA */
    double threshold;
    aak_candidate* cands; u64* counter; u64 capacity;
    const double* wstats; const i64* wpivot; const int* wlive;     /* reading C7m (NULL: reading C7) */
    unsigned* range_flag;                                          /* NULL, or: bit 0 set when wmax * max|d| of a row reaches 2^31 */
};

struct K4RowConst {                            /* per ring slot */
    double a[SPS_MAXW];                        /* C7: w * (mu - p);          C7m: mu_w - p_w */
    double inv[SPS_MAXW];                      /* C7: 1 / (sqrt(w) * sigma); C7m: 1 / sigma_w, or 0 = this width gives no SNR in this row */
    int bmin[SPS_MAXW];
    int q[SPS_MAXW];                           /* C7m: p_w - w p = B_w[0] - w p (0 for C7) */
    int live;                                  /* row exists and has a positive sigma */
    int pad[3];
};

template <int V>
struct K4Smem {
    unsigned I[3][1024 * V];                   /* inclusive prefix sums of d, ring of 3 rows */
    K4RowConst rc[4];
    unsigned wtot[K4_WARPS];
    int cnt[2];
    unsigned short list[2][1024 * V];
};

/* exact S (reading C7) of one position from a prefix row: e = element index of the position, t = its sample index */
template <bool PW>
__device__ __forceinline__ double k4_eval(const unsigned* I, const K4RowConst& rc, const SpsParams& p, int e, i64 t, int& bw) {
    double best = -CUDART_INF; bw = 0;
    const unsigned base = I[e - 1];
    constexpr bool pw = PW;
    for (int iw = 0; iw < p.nwidths; ++iw) {
        const int w = p.widths[iw];
        if (t + w > p.ntd) break;                                  /* ascending widths */
        const int B = (int)(I[e + w - 1] - base);
        double snr;
        if (pw) {                                                  /* reading C7m: ((double)(B_w - p_w) - (mu_w - p_w)) * (1 / sigma_w) */
            if (!(rc.inv[iw] > 0.0)) continue;
            snr = __dmul_rn(__dsub_rn(__ll2double_rn((i64)B - (i64)rc.q[iw]), rc.a[iw]), rc.inv[iw]);
        } else {
            snr = __dmul_rn(__dsub_rn(__int2double_rn(B), rc.a[iw]), rc.inv[iw]);
        }
        if (snr > best) { best = snr; bw = w; }
    }
    return best;
}

/* integer prefilter of one row: flags positions that may exceed the threshold, appends them to list (shared memory).
 * qmax = centre positions of this strip that exist (t < nt); qfull = those for which every width fits (t + wmax <= ntd);
 * nloc = ntd - t0 (samples of the row from the strip's first centre sample on), all as 32-bit strip-local numbers. */
template <int NW, bool POW2>
__device__ __forceinline__ void k4_prefilter(const unsigned* __restrict__ I, const K4RowConst& rc, const SpsParams& p, int qmax, int qfull,
                                             int nloc, unsigned short* list, int* cnt, int tid, int lane) {
    /* POW2: the plan's widths are 1, 2, 4, ... (every BASELINE.json config): the prefix offsets are then immediates of the
     * shared-memory loads instead of values re-read from the parameter bank and added per sample */
    int bm[NW], wd[NW];
#pragma unroll
    for (int iw = 0; iw < NW; ++iw) { bm[iw] = rc.bmin[iw]; wd[iw] = POW2 ? (1 << iw) : p.widths[iw]; }
    for (int q0 = 0; q0 < p.tt; q0 += K4_THREADS) {                  /* uniform trip count: ballots need every lane */
        const int q = q0 + tid;
        bool f = false;
        if (q < qmax) {
            const unsigned* Iq = I + q + 3;                          /* B_w(t) = I[e+w-1] - I[e-1], e = q + 4 */
            const unsigned base = Iq[0];
            if (q < qfull) {
#pragma unroll
                for (int iw = 0; iw < NW; ++iw) f |= ((int)(Iq[wd[iw]] - base) >= bm[iw]);
            } else {
#pragma unroll
                for (int iw = 0; iw < NW; ++iw)
                    if (q + wd[iw] <= nloc) f |= ((int)(Iq[wd[iw]] - base) >= bm[iw]);
            }
        }
        const unsigned mask = __ballot_sync(0xffffffffu, f);
        if (mask) {
            const int leader = __ffs(mask) - 1;
            int base = 0;
            if (lane == leader) base = atomicAdd(cnt, __popc(mask));
            base = __shfl_sync(0xffffffffu, base, leader);
            if (f) list[base + __popc(mask & ((1u << lane) - 1u))] = (unsigned short)q;
        }
    }
}

template <int V, bool PW>
__global__ void __launch_bounds__(K4_THREADS)
k_sps_peaks(const SpsParams p) {
    extern __shared__ __align__(16) uint8_t k4_raw[];
    K4Smem<V>& sm = *reinterpret_cast<K4Smem<V>*>(k4_raw);
    const int tid = threadIdx.x, warp = tid >> 5, lane = tid & 31;
    const i64 t0 = (i64)blockIdx.x * p.tt;
    const i64 tb = t0 - 4;                                           /* sample index of element 0 of the segment */
    const int i0 = blockIdx.y * p.rb;
    const int i1 = min(i0 + p.rb, p.ndms);
    const int e0 = tid * 4 * V;                                      /* this thread's 4V contiguous elements */
    const int ne = p.tt + 4 + p.wmax;                                /* elements the strip needs */
    /* 32-bit strip-local bounds (the 64-bit sample indices stay out of the per-sample code) */
    const i64 nd_loc = p.ntd - tb;                                   /* elements of the segment that exist: e < nd_loc */
    const int e_hi = (int)(nd_loc < (i64)ne ? (nd_loc < 0 ? 0 : nd_loc) : (i64)ne);
    const int e_lo = tb < 0 ? (int)(-tb) : 0;                        /* first element with a sample (t >= 0) */
    const i64 c_loc = p.nt - t0;
    const int qmax = (int)(c_loc < (i64)p.tt ? (c_loc < 0 ? 0 : c_loc) : (i64)p.tt);
    const i64 f_loc = p.ntd - t0 - p.wmax + 1;
    const int qfull = (int)(f_loc < (i64)qmax ? (f_loc < 0 ? 0 : f_loc) : (i64)qmax);
    const i64 n_loc64 = p.ntd - t0;
    const int nloc = (int)(n_loc64 > 0x3fffffff ? 0x3fffffff : (n_loc64 < 0 ? 0 : n_loc64));

    int4 cur[V], nxt[V];
    int pv_c = 0, pv_n = 0;
    double mu_c = 0.0, sg_c = 0.0, mu_n = 0.0, sg_n = 0.0;

    auto load_row = [&](int r, int4 (&buf)[V], int& pv, double& mu, double& sg) {
        sg = 0.0; mu = 0.0; pv = 0;
        if (r < 0 || r >= p.ndms) return;
        const int32_t* row = p.D + (size_t)r * (size_t)p.pitch;
        pv = __ldg(row);
        mu = __ldg(p.mu_sigma + 2 * (size_t)r);
        sg = __ldg(p.mu_sigma + 2 * (size_t)r + 1);
        if (PW) sg = __ldg(p.wlive + r) ? 1.0 : 0.0;            /* reading C7m: the row is live if any width has a sigma_w > 0 */
#pragma unroll
        for (int v = 0; v < V; ++v) {
            const int e = e0 + 4 * v;                                /* tb and nt are multiples of 4 or the row is padded to 128 */
            if (e >= e_lo && e < e_hi) buf[v] = __ldg(reinterpret_cast<const int4*>(row + (tb + e)));
            else buf[v] = make_int4(0, 0, 0, 0);
        }
    };

    load_row(i0 - 1, cur, pv_c, mu_c, sg_c);
    if (tid < 2) sm.cnt[tid] = 0;
    __syncthreads();

    int s = 0;
    for (int r = i0 - 1; r <= i1; ++r, ++s) {
        const int s3 = s % 3, s4 = s & 3, sl = s & 1;
        if (r + 1 <= i1) load_row(r + 1, nxt, pv_n, mu_n, sg_n);      /* one row ahead, in registers */
        const bool live = sg_c > 0.0;                                /* exists and sigma > 0 */

        /* ---- phase 1: per-row constants, thread-local + warp scan */
        if (tid < SPS_MAXW) {
            K4RowConst& rc = sm.rc[s4];
            if (tid == 0) rc.live = live ? 1 : 0;
            if (live && tid < p.nwidths) {
                double a, inv, qd = 0.0;
                int q = 0;
                if (PW) {                                            /* reading C7m: this row's own statistics of B_w */
                    const size_t o = (size_t)r * (size_t)p.nwidths + (size_t)tid;
                    const double mu_w = __ldg(p.wstats + 2 * o), sg_w = __ldg(p.wstats + 2 * o + 1);
                    const i64 pw = __ldg(p.wpivot + o);
                    q = (int)(pw - (i64)p.widths[tid] * (i64)pv_c);
                    qd = (double)q;
                    a = __dsub_rn(mu_w, __ll2double_rn(pw));
                    inv = sg_w > 0.0 ? __ddiv_rn(1.0, sg_w) : 0.0;
                } else {
                    const double w = (double)p.widths[tid];
                    a = __dmul_rn(w, __dsub_rn(mu_c, (double)pv_c));
                    inv = __ddiv_rn(1.0, __dmul_rn(__dsqrt_rn(w), sg_c));
                }
                rc.a[tid] = a; rc.inv[tid] = inv; if (PW) rc.q[tid] = q;
                /* x = the computed value of X = q + a + threshold/inv, the real-valued bound on e = B_w - w p. DESIGN.md §2 "K4
                 * prefilter margin" proves SNR_w > threshold => e >= floor(x): the rounding of the SNR expression and of x together
                 * move the bound by < 2^-16 while e is an integer; the kernel keeps 2 whole units of slack on top. */
                const double x = qd + a + p.threshold / inv;
                int bm;
                if (!(inv > 0.0)) bm = INT32_MAX;                    /* no SNR from this width: never flagged */
                else if (x != x) bm = INT32_MIN;
                else if (x >= 2147483000.0) bm = 2147482998;         /* e > x - 2^-16 is still possible up to INT32_MAX: keep the rule */
                else if (x <= -2147483000.0) bm = INT32_MIN;
                else bm = (int)floor(x) - 2;
                rc.bmin[tid] = bm;
            }
        }
        unsigned loc[V][4];
        unsigned run = 0;
        if (live) {
#pragma unroll
            for (int v = 0; v < V; ++v) {
                const int e = e0 + 4 * v;
                const int d[4] = {cur[v].x, cur[v].y, cur[v].z, cur[v].w};
#pragma unroll
                for (int k = 0; k < 4; ++k) {
                    const bool in = (e + k >= e_lo) && (e + k < e_hi);
                    run += in ? (unsigned)(d[k] - pv_c) : 0u;
                    loc[v][k] = run;
                }
            }
            if (p.range_flag) {                                      /* block-uniform; plans without a plan-time bound only */
                long long mx = 0;
#pragma unroll
                for (int v = 0; v < V; ++v) {
                    const int e = e0 + 4 * v;
                    const int d[4] = {cur[v].x, cur[v].y, cur[v].z, cur[v].w};
#pragma unroll
                    for (int k = 0; k < 4; ++k) {
                        const long long a = (long long)d[k] - (long long)pv_c;
                        if ((e + k >= e_lo) && (e + k < e_hi)) mx = max(mx, a < 0 ? -a : a);
                    }
                }
                if (mx * (long long)p.wmax >= (1ll << 31)) atomicOr(p.range_flag, 1u);
            }
        }
        unsigned incl = run;
#pragma unroll
        for (int o = 1; o < 32; o <<= 1) {
            const unsigned u = __shfl_up_sync(0xffffffffu, incl, o);
            if (lane >= o) incl += u;
        }
        if (lane == 31) sm.wtot[warp] = incl;
        __syncthreads();                                             /* (a) */

        /* ---- phase 2: cross-warp carry, prefix row into the ring */
        if (live) {
            unsigned carry = incl - run;
#pragma unroll
            for (int w = 0; w < K4_WARPS; ++w) carry += (w < warp) ? sm.wtot[w] : 0u;
            uint4* dst = reinterpret_cast<uint4*>(&sm.I[s3][e0]);
#pragma unroll
            for (int v = 0; v < V; ++v) dst[v] = make_uint4(loc[v][0] + carry, loc[v][1] + carry, loc[v][2] + carry, loc[v][3] + carry);
        }
        if (tid == 0) sm.cnt[sl] = 0;
        __syncthreads();                                             /* (b) */

        /* ---- phase 3a: integer prefilter of row r */
        if (live && r >= i0 && r < i1) {
            const unsigned* I = sm.I[s3];
            const K4RowConst& rc = sm.rc[s4];
            unsigned short* list = sm.list[sl];
            int* cnt = &sm.cnt[sl];
            switch (p.nwidths) {
#define K4_CASE(N) case N: if (p.pow2) k4_prefilter<N, true>(I, rc, p, qmax, qfull, nloc, list, cnt, tid, lane); \
                           else k4_prefilter<N, false>(I, rc, p, qmax, qfull, nloc, list, cnt, tid, lane); break;
                K4_CASE(1) K4_CASE(2) K4_CASE(3) K4_CASE(4) K4_CASE(5) K4_CASE(6) K4_CASE(7) K4_CASE(8)
                K4_CASE(9) K4_CASE(10) K4_CASE(11) K4_CASE(12) K4_CASE(13) K4_CASE(14) K4_CASE(15) K4_CASE(16)
#undef K4_CASE
            }
        }

        /* ---- phase 3b: exact S and the 3x3 rule for the flagged positions of row r-1 */
        const int rp = r - 1;
        if (rp >= i0 && rp < i1) {
            const int n = sm.cnt[sl ^ 1];
            const unsigned short* list = sm.list[sl ^ 1];
            const unsigned* Irow[3] = {sm.I[(s + 1) % 3], sm.I[(s + 2) % 3], sm.I[s3]};          /* rows rp-1, rp, rp+1 */
            const K4RowConst* rcs[3] = {&sm.rc[(s + 2) & 3], &sm.rc[(s + 3) & 3], &sm.rc[s4]};
            for (int k0 = 0; k0 < n; k0 += K4_THREADS) {
                const int k = k0 + tid;
                bool is = false; int q = 0, bw = 0; double sc = 0.0;
                if (k < n) {
                    q = list[k];
                    const i64 t = t0 + q;
                    const int e = q + 4;
                    sc = k4_eval<PW>(Irow[1], *rcs[1], p, e, t, bw);
                    if (sc > p.threshold) {
                        is = true;
#pragma unroll
                        for (int dr = -1; dr <= 1; ++dr) {
                            if (!rcs[dr + 1]->live) continue;
#pragma unroll
                            for (int dq = -1; dq <= 1; ++dq) {
                                if (dr == 0 && dq == 0) continue;
                                const i64 tn = t + dq;
                                if (tn < 0 || tn >= p.nt) continue;
                                int dummy;
                                const double v = k4_eval<PW>(Irow[dr + 1], *rcs[dr + 1], p, e + dq, tn, dummy);
                                const bool before = (dr < 0) || (dr == 0 && dq < 0);
                                if (before ? !(sc > v) : !(sc >= v)) is = false;
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
                            aak_candidate c;
                            c.sample = p.chunk_start + (u64)p.bin * (u64)(t0 + q);
                            c.dm = (float)__dadd_rn(p.dm_low, __dmul_rn((double)rp, p.dm_step));
                            c.snr = (float)sc;
                            c.width = (uint32_t)p.bin * (uint32_t)bw;
                            c.range = (uint32_t)p.range_index;
                            c.dm_index = (uint32_t)rp;
                            p.cands[slot] = c;
                        }
                    }
                }
            }
        }
#pragma unroll
        for (int v = 0; v < V; ++v) cur[v] = nxt[v];
        pv_c = pv_n; mu_c = mu_n; sg_c = sg_n;
    }
}

}  // namespace

extern "C" int aak_row_stats(const aak_row_desc* rows, int32_t nrows, double* mu_sigma, int64_t* n_iters, void* stream) {
    if (nrows <= 0) return 0;
    k_row_stats<<<(unsigned)nrows, STAT_THREADS, sizeof(StatSmem), (cudaStream_t)stream>>>(rows, mu_sigma, (i64*)n_iters);
    return (int)cudaGetLastError();
}

extern "C" int aak_row_width_stats(const aak_wstats_args* a, void* stream) {
    if (a->nwidths < 1 || a->nwidths > SPS_MAXW) return (int)cudaErrorInvalidValue;
    if (a->nt <= 0 || a->ndms <= 0) return 0;
    PwParams p;
    p.D = a->D; p.pitch = a->pitch; p.nt = a->nt; p.ntd = a->nt_data > a->nt ? a->nt_data : a->nt; p.nwidths = a->nwidths; p.wmax = 0;
    for (int k = 0; k < SPS_MAXW; ++k) { p.widths[k] = k < a->nwidths ? a->widths[k] : 0; if (p.widths[k] > p.wmax) p.wmax = p.widths[k]; }
    if (p.wmax > PW_MAXW) return (int)cudaErrorInvalidValue;
    p.wstats = a->wstats; p.wpivot = (i64*)a->wpivot; p.wlive = a->wlive;
    cudaStream_t st = (cudaStream_t)stream;
    if (a->nwidths <= 4) k_row_width_stats<4><<<(unsigned)a->ndms, PW_THREADS, 0, st>>>(p);
    else if (a->nwidths <= 8) k_row_width_stats<8><<<(unsigned)a->ndms, PW_THREADS, 0, st>>>(p);
    else if (a->nwidths <= 12) k_row_width_stats<12><<<(unsigned)a->ndms, PW_THREADS, 0, st>>>(p);
    else k_row_width_stats<16><<<(unsigned)a->ndms, PW_THREADS, 0, st>>>(p);
    return (int)cudaGetLastError();
}

extern "C" int aak_sps_init(void) {
    int e;
    if ((e = (int)cudaFuncSetAttribute(k_row_stats, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(StatSmem)))) return e;
    if ((e = (int)cudaFuncSetAttribute(k_sps_peaks<3, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(K4Smem<3>)))) return e;
    if ((e = (int)cudaFuncSetAttribute(k_sps_peaks<4, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(K4Smem<4>)))) return e;
    if ((e = (int)cudaFuncSetAttribute(k_sps_peaks<8, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(K4Smem<8>)))) return e;
    if ((e = (int)cudaFuncSetAttribute(k_sps_peaks<3, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(K4Smem<3>)))) return e;
    if ((e = (int)cudaFuncSetAttribute(k_sps_peaks<4, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(K4Smem<4>)))) return e;
    if ((e = (int)cudaFuncSetAttribute(k_sps_peaks<8, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sizeof(K4Smem<8>)))) return e;
    return 0;
}

extern "C" int aak_sps_peaks(const aak_sps_args* a, void* stream) {
    if (a->nwidths < 1 || a->nwidths > SPS_MAXW) return (int)cudaErrorInvalidValue;
    SpsParams p;
    p.D = a->D; p.pitch = a->pitch; p.nt = a->nt; p.ntd = a->nt_data > a->nt ? a->nt_data : a->nt; p.ndms = a->ndms; p.bin = a->bin; p.range_index = a->range_index;
    p.dm_low = a->dm_low; p.dm_step = a->dm_step; p.mu_sigma = a->mu_sigma; p.chunk_start = a->chunk_start;
    p.nwidths = a->nwidths; p.wmax = 0; p.pow2 = 1;
    for (int k = 0; k < a->nwidths; ++k) if (a->widths[k] != (1 << k)) p.pow2 = 0;
    for (int k = 0; k < SPS_MAXW; ++k) { p.widths[k] = k < a->nwidths ? a->widths[k] : 0; if (p.widths[k] > p.wmax) p.wmax = p.widths[k]; }
    p.threshold = a->threshold; p.cands = a->cands; p.counter = (u64*)a->counter; p.capacity = a->capacity;
    p.wstats = a->wstats; p.wpivot = (const i64*)a->wpivot; p.wlive = a->wlive; p.range_flag = a->range_flag;
    if (a->nt <= 0 || a->ndms <= 0) return 0;
    /* segment = tt + 4 + wmax elements <= 1024 V; the strip keeps at least ~2000 centre samples */
    const int V = p.wmax <= 1024 ? 3 : (p.wmax <= 2048 ? 4 : 8);
    if (p.wmax > 6000) return (int)cudaErrorInvalidValue;
    p.tt = (1024 * V - 4 - p.wmax) & ~3;
    /* each CTA recomputes 2 halo rows, so tall bands are cheaper; small searches take shorter bands to fill the 148 SMs */
    const long long strips = (a->nt + p.tt - 1) / p.tt;
    p.rb = K4_RB;
    while (p.rb > 2 && strips * ((a->ndms + p.rb - 1) / p.rb) < 2 * 148) p.rb /= 2;
    dim3 grid((unsigned)strips, (unsigned)((a->ndms + p.rb - 1) / p.rb));
    cudaStream_t st = (cudaStream_t)stream;
    const bool pw = p.wstats != nullptr;
    switch (V) {
        case 3: if (pw) k_sps_peaks<3, true><<<grid, K4_THREADS, sizeof(K4Smem<3>), st>>>(p); else k_sps_peaks<3, false><<<grid, K4_THREADS, sizeof(K4Smem<3>), st>>>(p); break;
        case 4: if (pw) k_sps_peaks<4, true><<<grid, K4_THREADS, sizeof(K4Smem<4>), st>>>(p); else k_sps_peaks<4, false><<<grid, K4_THREADS, sizeof(K4Smem<4>), st>>>(p); break;
        default: if (pw) k_sps_peaks<8, true><<<grid, K4_THREADS, sizeof(K4Smem<8>), st>>>(p); else k_sps_peaks<8, false><<<grid, K4_THREADS, sizeof(K4Smem<8>), st>>>(p); break;
    }
    return (int)cudaGetLastError();
}
