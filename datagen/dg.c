/*
 * datagen/dg.c — seeded synthetic filterbank generator.
 *
 * Serves BOTH the oracle-side tests and the CUDA path with identical bytes. It holds none of
 * the search method's arithmetic: no dedispersion, binning, statistics, boxcars or peaks, and
 * no delay formula — pulse sweeps arrive as explicit per-channel sample offsets.
 *
 * Recipe (BASELINE.json configs: "uint8 samples drawn as
 * round(N(127, 16)) clipped to [0,255], seed-generated"):
 *   every sample is a pure function of (seed, channel c, absolute sample t):
 *     h      = mix64(seed, c, t >> 1)                     counter-based, no state
 *     (g0,g1)= Box-Muller(h)  ; g = (t & 1) ? g1 : g0     standard normal
 *     v      = mean + sigma*g + sum_p amp_p * [ t0_p + delay_p[c] <= t < t0_p + delay_p[c] + width_p ]
 *     x      = clip(floor(v + 0.5), 0, 255)
 * Because it is a pure function of (seed, c, t) any chunk of a long stream can be regenerated.
 */
#include <math.h>
#include <stdint.h>
#include <stddef.h>

typedef struct {
    int64_t t0;     /* arrival sample at the reference (top) channel */
    int64_t width;  /* samples */
    double  amp;    /* added to the real-valued sample before rounding */
} dg_pulse;

static inline uint64_t dg_mix64(uint64_t z) {
    z += 0x9E3779B97F4A7C15ull;
    z = (z ^ (z >> 30)) * 0xBF58476D1CE4E5B9ull;
    z = (z ^ (z >> 27)) * 0x94D049BB133111EBull;
    return z ^ (z >> 31);
}

static inline uint64_t dg_hash(uint64_t seed, uint64_t c, uint64_t tpair) {
    uint64_t h = dg_mix64(seed ^ 0xD1B54A32D192ED03ull);
    h = dg_mix64(h ^ (c * 0xA0761D6478BD642Full));
    h = dg_mix64(h ^ (tpair * 0xE7037ED1A0B428DBull));
    return h;
}

static inline void dg_normal_pair(uint64_t h, double* g0, double* g1) {
    const double inv24 = 1.0 / 16777216.0;
    double u1 = ((double)(h >> 40) + 0.5) * inv24;                 /* (0,1) */
    double u2 = ((double)((h >> 16) & 0xFFFFFFull) + 0.5) * inv24; /* (0,1) */
    double r = sqrt(-2.0 * log(u1));
    double a = 6.283185307179586476925286766559 * u2;
    *g0 = r * cos(a);
    *g1 = r * sin(a);
}

/* Fill out[c*row_stride + (t - t_begin)] for c in [0,nchans), t in [t_begin, t_begin+nsamp).
 * pulse_delays is [npulses][nchans] (int64, samples); may be NULL when npulses == 0. */
void dg_fill(uint8_t* out, size_t row_stride, int32_t nchans, int64_t t_begin, int64_t nsamp,
             uint64_t seed, double mean, double sigma,
             int32_t npulses, const dg_pulse* pulses, const int64_t* pulse_delays)
{
    #pragma omp parallel for schedule(dynamic, 4)
    for (int32_t c = 0; c < nchans; ++c) {
        uint8_t* row = out + (size_t)c * row_stride;
        int64_t t_end = t_begin + nsamp;
        int64_t tp0 = t_begin >> 1, tp1 = (t_end + 1) >> 1;
        for (int64_t tp = tp0; tp < tp1; ++tp) {
            double g[2];
            dg_normal_pair(dg_hash(seed, (uint64_t)c, (uint64_t)tp), &g[0], &g[1]);
            for (int k = 0; k < 2; ++k) {
                int64_t t = 2 * tp + k;
                if (t < t_begin || t >= t_end) continue;
                double v = mean + sigma * g[k];
                double q = floor(v + 0.5);
                row[t - t_begin] = (uint8_t)(q < 0.0 ? 0.0 : (q > 255.0 ? 255.0 : q));
            }
        }
        /* pulses: re-derive the affected samples with the amplitude added before rounding */
        for (int32_t p = 0; p < npulses; ++p) {
            int64_t a = pulses[p].t0 + pulse_delays[(size_t)p * nchans + c];
            int64_t b = a + pulses[p].width;
            if (a < t_begin) a = t_begin;
            if (b > t_end) b = t_end;
            for (int64_t t = a; t < b; ++t) {
                double g[2];
                dg_normal_pair(dg_hash(seed, (uint64_t)c, (uint64_t)(t >> 1)), &g[0], &g[1]);
                double v = mean + sigma * g[t & 1];
                for (int32_t q = 0; q < npulses; ++q) {   /* all pulses covering t, so overlaps add */
                    int64_t qa = pulses[q].t0 + pulse_delays[(size_t)q * nchans + c];
                    if (t >= qa && t < qa + pulses[q].width) v += pulses[q].amp;
                }
                double r = floor(v + 0.5);
                row[t - t_begin] = (uint8_t)(r < 0.0 ? 0.0 : (r > 255.0 ? 255.0 : r));
            }
        }
    }
}

/* The same recipe for 16-bit samples: x = clip(floor(v + 0.5), 0, max_value), max_value <= 65535 (the stated bit
 * depth, e.g. 4095). out rows are row_stride BYTES apart. */
void dg_fill16(uint16_t* out, size_t row_stride, int32_t nchans, int64_t t_begin, int64_t nsamp,
               uint64_t seed, double mean, double sigma, double max_value,
               int32_t npulses, const dg_pulse* pulses, const int64_t* pulse_delays)
{
    #pragma omp parallel for schedule(dynamic, 4)
    for (int32_t c = 0; c < nchans; ++c) {
        uint16_t* row = (uint16_t*)((uint8_t*)out + (size_t)c * row_stride);
        int64_t t_end = t_begin + nsamp;
        int64_t tp0 = t_begin >> 1, tp1 = (t_end + 1) >> 1;
        for (int64_t tp = tp0; tp < tp1; ++tp) {
            double g[2];
            dg_normal_pair(dg_hash(seed, (uint64_t)c, (uint64_t)tp), &g[0], &g[1]);
            for (int k = 0; k < 2; ++k) {
                int64_t t = 2 * tp + k;
                if (t < t_begin || t >= t_end) continue;
                double q = floor(mean + sigma * g[k] + 0.5);
                row[t - t_begin] = (uint16_t)(q < 0.0 ? 0.0 : (q > max_value ? max_value : q));
            }
        }
        for (int32_t p = 0; p < npulses; ++p) {
            int64_t a = pulses[p].t0 + pulse_delays[(size_t)p * nchans + c];
            int64_t b = a + pulses[p].width;
            if (a < t_begin) a = t_begin;
            if (b > t_end) b = t_end;
            for (int64_t t = a; t < b; ++t) {
                double g[2];
                dg_normal_pair(dg_hash(seed, (uint64_t)c, (uint64_t)(t >> 1)), &g[0], &g[1]);
                double v = mean + sigma * g[t & 1];
                for (int32_t q = 0; q < npulses; ++q) {
                    int64_t qa = pulses[q].t0 + pulse_delays[(size_t)q * nchans + c];
                    if (t >= qa && t < qa + pulses[q].width) v += pulses[q].amp;
                }
                double r = floor(v + 0.5);
                row[t - t_begin] = (uint16_t)(r < 0.0 ? 0.0 : (r > max_value ? max_value : r));
            }
        }
    }
}

/* 64-bit FNV-1a over a strided 2-D byte array; lets tests assert that host input is untouched. */
uint64_t dg_checksum(const uint8_t* x, size_t row_stride, int32_t nchans, int64_t nsamp) {
    uint64_t h = 0xCBF29CE484222325ull;
    for (int32_t c = 0; c < nchans; ++c) {
        const uint8_t* row = x + (size_t)c * row_stride;
        for (int64_t t = 0; t < nsamp; ++t) { h ^= row[t]; h *= 0x100000001B3ull; }
    }
    return h;
}
