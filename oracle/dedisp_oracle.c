/*
 * dedisp_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU statement of brute-force incoherent
 * dedispersion, written from the paper (Sclocco et al., arXiv 1601.01165,
 * /root/reference/PAPER.md) and the readings listed in DESIGN.md "Readings".
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call this file.  It shares no code,
 * header, table or helper with the CUDA path under paper_1601_01165_b200/.
 *
 * Build (see oracle/__init__.py):
 *   gcc -O2 -fopenmp -ffp-contract=off -fno-fast-math -shared -fPIC
 *
 * What is pinned where (tests/test_oracle_pins.py):
 *   - delay / shift table : closed-form properties of Eq. (1), the padding
 *     figures printed in BASELINE.json, exact rational arithmetic, hand value.
 *   - dedisperse (f32, u8): DM=0 row = library channel sum, constant input,
 *     single-channel pure shift, linearity, injected pulse, brute-force gather
 *     with arbitrary hand-made tables.
 *   - *_points            : against the full routine and the brute-force gather.
 *   Performance numbers of the paper: parity unpinned (figures are images).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* ---- Eq. (1), PAPER.md:34-37 ------------------------------------------- */

/* Reading A1: channel c is labelled by f_low + c*bw ...          */
double oracle_channel_freq_MHz(double f_low_MHz, double channel_bw_MHz, int c)
{
    return f_low_MHz + (double)c * channel_bw_MHz;
}

/* ... and f_h, "the highest frequency in a certain band", is the
 * top edge of the band, f_low + C*bw.  This is the one place to switch to the
 * alternative reading f_low + (C-1)*bw.                                       */
double oracle_f_high_MHz(double f_low_MHz, double channel_bw_MHz, int nr_channels)
{
    return f_low_MHz + (double)nr_channels * channel_bw_MHz;
}

/* Trial DM i ("start at 0 and increment by ..."; reading A5:
 * computed, never accumulated).                                              */
double oracle_trial_dm(double dm_first, double dm_step, int i)
{
    return dm_first + (double)i * dm_step;
}

/* Delay in samples before rounding, reading A3 (fixed association):
 *   a = 1/(f*f);  b = 1/(f_h*f_h);  x = ((4150*dm) * (a-b)) * rate           */
double oracle_delay_samples(double f_MHz, double f_h_MHz, double dm, double sample_rate)
{
    double a = 1.0 / (f_MHz * f_MHz);
    double b = 1.0 / (f_h_MHz * f_h_MHz);
    double diff = a - b;
    double k = (4150.0 * dm) * diff;   /* Eq. (1): seconds */
    return k * sample_rate;
}

/* Reading A4: nearest integer, ties up (x >= 0 here).                         */
int64_t oracle_round_half_up(double x)
{
    double fl = floor(x);
    return (int64_t)fl + ((x - fl) >= 0.5 ? 1 : 0);
}

/* Shift table Delta(chan, dm), "can be computed in advance".
 * out is row-major [nr_dms][nr_channels].  Returns 0, or -1 if an entry does
 * not fit int32.                                                             */
int oracle_shift_table(int nr_channels, double f_low_MHz, double channel_bw_MHz,
                       double sample_rate, double dm_first, double dm_step,
                       int nr_dms, int32_t *out)
{
    double f_h = oracle_f_high_MHz(f_low_MHz, channel_bw_MHz, nr_channels);
    for (int i = 0; i < nr_dms; ++i) {
        double dm = oracle_trial_dm(dm_first, dm_step, i);
        for (int c = 0; c < nr_channels; ++c) {
            double f = oracle_channel_freq_MHz(f_low_MHz, channel_bw_MHz, c);
            int64_t s = oracle_round_half_up(oracle_delay_samples(f, f_h, dm, sample_rate));
            if (s < 0 || s > INT32_MAX) return -1;
            out[(size_t)i * nr_channels + c] = (int32_t)s;
        }
    }
    return 0;
}

/* ---- Algorithm 1, PAPER.md:51-55 ---------------------------------------- */
/*
 * in    : [nr_beams][nr_channels][in_pitch]   (channel-major rows)
 * shift : [nr_dms][nr_channels]
 * out   : [nr_beams][nr_dms][nr_samples]
 * Loop order is the paper's: dm -> sample -> chan, channels ascending.
 * OpenMP only spreads (beam, dm) rows over threads; each output is still the
 * sequential channel sum.
 */
void oracle_dedisperse_f32(const float *in, int64_t in_pitch, int nr_channels,
                           int nr_dms, int64_t nr_samples, const int32_t *shift,
                           int nr_beams, double *out, double *sabs)
{
    int64_t rows = (int64_t)nr_beams * nr_dms;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t row = 0; row < rows; ++row) {
        int64_t b = row / nr_dms;
        int dm = (int)(row % nr_dms);
        const float *inb = in + (size_t)b * nr_channels * in_pitch;
        for (int64_t sample = 0; sample < nr_samples; ++sample) {
            double dSample = 0.0;
            double aSample = 0.0;
            for (int chan = 0; chan < nr_channels; ++chan) {
                int64_t delta = shift[(size_t)dm * nr_channels + chan];
                double v = (double)inb[(size_t)chan * in_pitch + sample + delta];
                dSample += v;
                aSample += fabs(v);
            }
            out[(size_t)row * nr_samples + sample] = dSample;
            if (sabs) sabs[(size_t)row * nr_samples + sample] = aSample;
        }
    }
}

void oracle_dedisperse_u8(const uint8_t *in, int64_t in_pitch, int nr_channels,
                          int nr_dms, int64_t nr_samples, const int32_t *shift,
                          int nr_beams, uint64_t *out)
{
    int64_t rows = (int64_t)nr_beams * nr_dms;
#pragma omp parallel for schedule(dynamic, 1)
    for (int64_t row = 0; row < rows; ++row) {
        int64_t b = row / nr_dms;
        int dm = (int)(row % nr_dms);
        const uint8_t *inb = in + (size_t)b * nr_channels * in_pitch;
        for (int64_t sample = 0; sample < nr_samples; ++sample) {
            uint64_t dSample = 0;
            for (int chan = 0; chan < nr_channels; ++chan) {
                int64_t delta = shift[(size_t)dm * nr_channels + chan];
                dSample += inb[(size_t)chan * in_pitch + sample + delta];
            }
            out[(size_t)row * nr_samples + sample] = dSample;
        }
    }
}

/* The same sums at a list of (beam, dm, sample) points, for full-size parity
 * where the whole output is too expensive.  pts is [n][3] int64.             */
void oracle_dedisperse_f32_points(const float *in, int64_t in_pitch, int nr_channels,
                                  const int32_t *shift, const int64_t *pts, int64_t n,
                                  double *out, double *sabs)
{
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        int64_t b = pts[3 * p], dm = pts[3 * p + 1], sample = pts[3 * p + 2];
        const float *inb = in + (size_t)b * nr_channels * in_pitch;
        double dSample = 0.0, aSample = 0.0;
        for (int chan = 0; chan < nr_channels; ++chan) {
            int64_t delta = shift[(size_t)dm * nr_channels + chan];
            double v = (double)inb[(size_t)chan * in_pitch + sample + delta];
            dSample += v;
            aSample += fabs(v);
        }
        out[p] = dSample;
        if (sabs) sabs[p] = aSample;
    }
}

void oracle_dedisperse_u8_points(const uint8_t *in, int64_t in_pitch, int nr_channels,
                                 const int32_t *shift, const int64_t *pts, int64_t n,
                                 uint64_t *out)
{
#pragma omp parallel for schedule(static)
    for (int64_t p = 0; p < n; ++p) {
        int64_t b = pts[3 * p], dm = pts[3 * p + 1], sample = pts[3 * p + 2];
        const uint8_t *inb = in + (size_t)b * nr_channels * in_pitch;
        uint64_t dSample = 0;
        for (int chan = 0; chan < nr_channels; ++chan) {
            int64_t delta = shift[(size_t)dm * nr_channels + chan];
            dSample += inb[(size_t)chan * in_pitch + sample + delta];
        }
        out[p] = dSample;
    }
}

int oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void oracle_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}
