/*
 * dedisp_oracle.c -- CPU ORACLE for direct incoherent dedispersion.
 *
 * TEST INFRASTRUCTURE ONLY.  Nothing in the product path (the package
 * paper_1112_0065_b200/, include/, the CUDA library) may include, link, import
 * or call this file.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs use it.  It shares no code, header,
 * table or constant generator with the CUDA path.
 *
 * What it computes (the plain definition, written out):
 *
 *   out[d][t] = sum_{c=0}^{nchans-1} in[c][ t + delay[c][d] ]
 *   delay[c][d] = round( 4148.808 * DM_d * ( f_c^-2 - f_top^-2 ) / dt ),
 *   f_c = f_top + c*df                       (MHz, seconds, pc cm^-3)
 *
 * Sources: BASELINE.json:north_star (formula, "rounding is to nearest with
 * ties away from zero, evaluated in double", "f_c = f_top + c*df");
 * PAPER.md:44 (Sec. 2.2) "The computation of each dispersion trial involves a
 * complete integration over frequency channels"; PAPER.md:48 (Sec. 2.2) "the
 * most common 'direct' dedispersion algorithm".  The paper prints no formula;
 * the readings taken where it is silent are listed in DESIGN.md ("Readings").
 *
 * Arithmetic: delays in IEEE double, one rounding per operation, no FMA
 * contraction (compile with -ffp-contract=off), C99 round() = ties away from
 * zero.  Sums are exact unsigned integers (max 4096 channels * 255 < 2^24), so
 * the uint32 result is unique and the float32 result is its exact conversion.
 *
 * Parity pins (tests/test_oracle_pins.py, tests/golden/): hand-worked 4-channel
 * example, exact-rational delay table, textbook closed form of the sweep,
 * DM=0 == channel sum, impulse along the sweep, linearity, constant input,
 * time shift, prefix-sum conservation, brute force vs an independent NumPy
 * slice-sum.  Every function below is pinned; nothing here is "parity unpinned".
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

/* Dispersion constant, s MHz^2 / (pc cm^-3): BASELINE.json:north_star. */
static const double ORACLE_KDM = 4148.808;

/* One delay entry.  Order of operations = DESIGN.md reading R4:
 *   fc = f_top + c*df ; a = 1/(fc*fc) - 1/(f_top*f_top) ; x = ((K*DM)*a)/dt . */
static int32_t oracle_delay_one(int c, double dm, double dt, double f_top, double df)
{
    double fc = f_top + (double)c * df;
    double a = 1.0 / (fc * fc) - 1.0 / (f_top * f_top);
    double x = ((ORACLE_KDM * dm) * a) / dt;
    return (int32_t)round(x); /* C99 round(): nearest, ties away from zero */
}

/* delay[c*ndm + d], c in [0,nchans), d in [0,ndm).  Returns max over the table
 * (reading R16), or -1 on a bad argument. */
int64_t oracle_delay_table(int nchans, double dt, double f_top, double df,
                           const double *dms, int ndm, int32_t *delay)
{
    if (nchans < 1 || ndm < 1 || !dms || !delay || !(dt > 0.0) || !(f_top > 0.0))
        return -1;
    int64_t max_delay = 0;
    for (int c = 0; c < nchans; ++c)
        for (int d = 0; d < ndm; ++d) {
            int32_t v = oracle_delay_one(c, dms[d], dt, f_top, df);
            delay[(size_t)c * ndm + d] = v;
            if (v > max_delay) max_delay = v;
        }
    return max_delay;
}

/* Tight row stride in bytes of a packed row of nsamps samples
 * (reading R9). */
int64_t oracle_row_stride_bytes(int64_t nsamps, int nbits)
{
    return (nsamps * nbits + 7) / 8;
}

/* Sample t of a packed row.  2-bit: LSB-first, 4 per byte (reading R10);
 * 8-bit: unsigned byte (reading R11); 1- and 4-bit (row f4, reading R36): the same
 * LSB-first rule, 8 / 2 samples per byte: bits [t*nbits, (t+1)*nbits) of the row read
 * as a little-endian bit string. */
static inline uint32_t oracle_get_sample(const uint8_t *row, int64_t t, int nbits)
{
    if (nbits == 8) return row[t];
    int64_t bit = t * nbits;
    return (row[bit >> 3] >> (bit & 7)) & ((1u << nbits) - 1u);
}

static int oracle_nbits_ok(int nbits) { return nbits == 1 || nbits == 2 || nbits == 4 || nbits == 8; }

/* O1 -- the literal triple loop on the packed bytes.
 *   in  : nchans rows of row_stride bytes, each holding nsamps_out+max_delay samples
 *   out : [ndm][nsamps_out] uint32, t fastest
 * Returns 0, or -1 on a bad argument. */
int oracle_dedisperse_literal(int nchans, int ndm, int64_t nsamps_out,
                              const int32_t *delay, const uint8_t *in,
                              int64_t row_stride, int nbits, uint32_t *out)
{
    if (nchans < 1 || ndm < 1 || nsamps_out < 1 || !delay || !in || !out) return -1;
    if (!oracle_nbits_ok(nbits)) return -1;
    for (int d = 0; d < ndm; ++d)
        for (int64_t t = 0; t < nsamps_out; ++t) {
            uint32_t acc = 0;
            for (int c = 0; c < nchans; ++c)
                acc += oracle_get_sample(in + (size_t)c * row_stride,
                                         t + delay[(size_t)c * ndm + d], nbits);
            out[(size_t)d * nsamps_out + t] = acc;
        }
    return 0;
}

/* O2 -- same definition, rows unpacked to one byte per sample first, trials
 * spread over OpenMP threads, t innermost.  No blocking, no reordering of the
 * sum beyond "for d: for c: for t".  Used for full-size parity and as the
 * timed CPU baseline.  d_begin/d_end select a range of trials so that callers
 * can bound the work (out still indexed by absolute d).
 * nthreads <= 0: use the OpenMP default.  Returns threads used, or -1. */
int oracle_dedisperse(int nchans, int ndm, int64_t nsamps_out,
                      const int32_t *delay, int64_t max_delay,
                      const uint8_t *in, int64_t row_stride, int nbits,
                      uint32_t *out, int d_begin, int d_end, int nthreads)
{
    if (nchans < 1 || ndm < 1 || nsamps_out < 1 || !delay || !in || !out) return -1;
    if (!oracle_nbits_ok(nbits)) return -1;
    if (d_begin < 0 || d_end > ndm || d_begin > d_end || max_delay < 0) return -1;
    int64_t nsamps_in = nsamps_out + max_delay;
    uint8_t *u8 = NULL;
    const uint8_t *rows;
    int64_t rstride;
    if (nbits == 8) {
        rows = in;
        rstride = row_stride;
    } else {
        u8 = (uint8_t *)malloc((size_t)nchans * (size_t)nsamps_in);
        if (!u8) return -1;
        for (int c = 0; c < nchans; ++c)
            for (int64_t t = 0; t < nsamps_in; ++t)
                u8[(size_t)c * nsamps_in + t] =
                    (uint8_t)oracle_get_sample(in + (size_t)c * row_stride, t, nbits);
        rows = u8;
        rstride = nsamps_in;
    }
    int used = 1;
#ifdef _OPENMP
    if (nthreads > 0) omp_set_num_threads(nthreads);
#pragma omp parallel
    {
#pragma omp single
        used = omp_get_num_threads();
    }
#pragma omp parallel for schedule(dynamic, 1)
#endif
    for (int d = d_begin; d < d_end; ++d) {
        uint32_t *acc = out + (size_t)d * nsamps_out;
        memset(acc, 0, (size_t)nsamps_out * sizeof(uint32_t));
        for (int c = 0; c < nchans; ++c) {
            const uint8_t *row = rows + (size_t)c * rstride + delay[(size_t)c * ndm + d];
            for (int64_t t = 0; t < nsamps_out; ++t) acc[t] += row[t];
        }
    }
    free(u8);
    return used;
}

/* float32 view of an exact integer result (every sum < 2^24, so exact). */
void oracle_u32_to_f32(const uint32_t *src, float *dst, int64_t n)
{
    for (int64_t i = 0; i < n; ++i) dst[i] = (float)src[i];
}
