/*
 * dd_oracle.c -- CPU ORACLE for direct incoherent dedispersion.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the plain, slow, obviously-correct statement of what the hot path computes,
 * written from the paper (arXiv:1201.5380, /root/reference/PAPER.md) and nothing else.
 * It shares NO code with the CUDA path (paper_1201_5380_b200/csrc): no headers, helpers,
 * tables or constants.  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may build, load or call it.  The product never does.
 *
 * What it computes (steps O1..O6 of DESIGN.md section 3):
 *
 *   O1  f[c]        = f_top + c*df                                  PAPER.md:62 (eq. 4, "nu_0 + nu*dnu")
 *   O2  x[d][c]     = K*DM[d]*(1/f[c]^2 - 1/f_top^2)/dt             PAPER.md:23-25 (eq. 1), 62-65 (eq. 4-5)
 *   O3  delay[d][c] = floor(x[d][c] + 0.5)                          PAPER.md:64-67 ("rounded to the nearest integer")
 *   O4  a[c][t]     = sample t of packed row c                      PAPER.md:101 (sub-word samples, shift and mask)
 *   O5  out[d][t]   = sum_{c=0}^{nchans-1} a[c][t + delay[d][c]]    PAPER.md:57-60 (eq. 3; sum_i^N means i=0..N-1)
 *   O6  cast to the requested output type (value preserving)        done by the Python wrapper, which asserts it fits
 *   O7  channel kill mask, applied arithmetically:                  PAPER.md:113 ("sum += data * kill_mask[channel]")
 *       out[d][t] = sum_c a[c][t + delay[d][c]] * mask[c],  mask[c] in {0, 1};  no mask = all ones
 *
 * K = k_DM = 4.148808e3 MHz^2 pc^-1 cm^3 s, frequencies in MHz, dt in seconds,
 * DM in pc cm^-3, all floating point in double (fp64).
 *
 * Loop order is d, c, t (t innermost), exactly eq. 3 with the sum over channels performed
 * sequentially (PAPER.md:83 finding (i)).  The only concession to run time is an OpenMP
 * "parallel for" over d (each d is an independent output row); there is no
 * blocking, no bit-level parallelism, no reordering.
 *
 * Parity status: every function here is pinned by tests/test_oracle_pins.py (P1..P11 of DESIGN.md).
 */
#include <math.h>
#include <stddef.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_K_DM 4.148808e3

/* O1-O3.  delay is [ndm][nchans], row-major, int64.  Returns 0, or -1 on a bad argument. */
int oracle_delay_table(int nchans, double dt, double f_top, double df, int ndm, const double *dm,
                       int64_t *delay)
{
    if (nchans <= 0 || ndm <= 0 || !(dt > 0.0) || !(f_top > 0.0) || !dm || !delay)
        return -1;
    for (int d = 0; d < ndm; ++d) {
        for (int c = 0; c < nchans; ++c) {
            double f = f_top + (double)c * df;                                        /* O1 */
            double x = ORACLE_K_DM * dm[d] * (1.0 / (f * f) - 1.0 / (f_top * f_top)) / dt; /* O2 */
            delay[(size_t)d * (size_t)nchans + (size_t)c] = (int64_t)floor(x + 0.5);    /* O3 */
        }
    }
    return 0;
}

/* O4 for one sample: sample t of a packed row, nbits in {1,2,4,8}.
 * Reading R9: byte (t*nbits)/8, bits [(t*nbits)%8, +nbits), least-significant first. */
static unsigned oracle_sample(const uint8_t *row, int nbits, int64_t t)
{
    int64_t bit = t * (int64_t)nbits;
    unsigned byte = row[bit / 8];
    return (byte >> (unsigned)(bit % 8)) % (1u << nbits);
}

/* O4 for a whole row: n samples of `row` into out[0..n). */
void oracle_unpack_row(const uint8_t *row, int nbits, int64_t n, uint8_t *out)
{
    for (int64_t t = 0; t < n; ++t)
        out[t] = (uint8_t)oracle_sample(row, nbits, t);
}

/* Number of OpenMP threads the timed loop will use for a request of `nthreads` (0 = all). */
int oracle_threads(int nthreads)
{
#ifdef _OPENMP
    int m = omp_get_max_threads();
    if (nthreads <= 0 || nthreads > m)
        return m;
    return nthreads;
#else
    (void)nthreads;
    return 1;
#endif
}

/* O5 on unpacked samples a[c][t] (row length a_len >= nsamps + max delay), for the ndm rows of
 * `delay` ([ndm][nchans], int64).  out is [ndm][nsamps] uint32, overwritten.
 * mask: NULL, or nchans ints, nonzero = channel kept (O7).
 * Returns 0; -1 bad argument; -2 a delay is negative or reaches past a_len. */
int oracle_dedisperse_unpacked(int nchans, int64_t nsamps, const uint8_t *a, int64_t a_len, int ndm,
                               const int64_t *delay, const int32_t *mask, uint32_t *out, int nthreads)
{
    if (nchans <= 0 || nsamps <= 0 || ndm <= 0 || !a || !delay || !out)
        return -1;
    for (size_t i = 0; i < (size_t)ndm * (size_t)nchans; ++i)
        if (delay[i] < 0 || delay[i] + nsamps > a_len)
            return -2;
    int nt = oracle_threads(nthreads);
    (void)nt;
#pragma omp parallel for schedule(dynamic, 1) num_threads(nt)
    for (int d = 0; d < ndm; ++d) {
        uint32_t *row = out + (size_t)d * (size_t)nsamps;
        memset(row, 0, (size_t)nsamps * sizeof(uint32_t));
        for (int c = 0; c < nchans; ++c) {
            const uint8_t *src = a + (size_t)c * (size_t)a_len + delay[(size_t)d * nchans + c];
            const uint32_t keep = (mask == NULL || mask[c] != 0) ? 1u : 0u;
            for (int64_t t = 0; t < nsamps; ++t)
                row[t] += src[t] * keep;                                             /* O5, O7 */
        }
    }
    return 0;
}

/* O4 + O5 from the packed input in[c] (rows in_stride bytes apart, each holding at least
 * nsamps + max delay samples).  out as above.  -3 = out of memory, -4 = row too short. */
int oracle_dedisperse(int nchans, int64_t nsamps, int nbits, const uint8_t *in, int64_t in_stride,
                      int ndm, const int64_t *delay, const int32_t *mask, uint32_t *out, int nthreads)
{
    if (nchans <= 0 || nsamps <= 0 || ndm <= 0 || !in || !delay || !out)
        return -1;
    if (nbits != 1 && nbits != 2 && nbits != 4 && nbits != 8)
        return -1;
    int64_t maxd = 0;
    for (size_t i = 0; i < (size_t)ndm * (size_t)nchans; ++i) {
        if (delay[i] < 0)
            return -2;
        if (delay[i] > maxd)
            maxd = delay[i];
    }
    int64_t a_len = nsamps + maxd;
    if ((a_len * nbits + 7) / 8 > in_stride)
        return -4;
    uint8_t *a = (uint8_t *)malloc((size_t)nchans * (size_t)a_len);
    if (!a)
        return -3;
    for (int c = 0; c < nchans; ++c)                                                  /* O4 */
        oracle_unpack_row(in + (size_t)c * (size_t)in_stride, nbits, a_len, a + (size_t)c * (size_t)a_len);
    int rc = oracle_dedisperse_unpacked(nchans, nsamps, a, a_len, ndm, delay, mask, out, nthreads);
    free(a);
    return rc;
}
