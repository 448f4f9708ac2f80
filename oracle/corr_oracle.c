/* corr_oracle.c -- CPU oracle for the X-engine hot path of arXiv 1503.06203.
 *
 * TEST INFRASTRUCTURE, NOT PRODUCT.  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may call this.  It shares no code, header, table or
 * helper with the CUDA path under paper_1503_06203_b200/ and neither includes the other.
 *
 * What it computes (every function cites the passage it follows; PAPER.md is
 * /root/reference/PAPER.md, line numbers of that file):
 *
 *   For every frequency channel f (channels are independent) and every pair of
 *   inputs x <= y ("only the upper triangle needs to be calculated"), the correlation
 *   of Eq. (1)
 *        Corr(X, Y) = X Y* = ( XRe*YRe + XIm*YIm ,  XIm*YRe - XRe*YIm )
 *   accumulated over the T time samples of the call ("These products are accumulated over many
 *   time samples").
 *
 *   Input  (Fig. 2): packed[T][F][N] bytes, one per complex sample, Re and Im
 *          offset-encoded (excess-8): stored nibble = value + 8, value in [-8,7].
 *          Nibble order is fixed by BASELINE.json (the paper's text is silent): Re = high nibble.
 *   Output ("signed 32+32-bit complex correlation products"; layout from
 *          BASELINE.json): vis[F][N(N+1)/2][2] int32 (Re, Im), upper triangle row-major:
 *          index b(x,y) = x*N - x*(x-1)/2 + (y-x), 0 <= x <= y < N.
 *
 * The method is exact integer arithmetic, so the oracle is the definition written out.
 * Pins (tests/test_oracle_pins.py): Eq. 1 worked by hand, closed form for constant input,
 * Hermitian/diagonal invariants, Eq. 3 identity (an independent decode through the stored
 * unsigned nibbles), numpy complex128 matrix product, pure-Python brute force, additivity,
 * multiply-by-i / conjugation / permutation metamorphic relations.  Nothing is "parity unpinned".
 *
 * Two levels:
 *   level 0  corr_oracle_level0 : the loop exactly as written above, straight off the packed
 *            bytes, 64-bit accumulators, single thread.
 *   level 1  corr_oracle_level1 : de-interleave once to planar int8 re[f][n][t], im[f][n][t],
 *            then the same triple loop, int32 accumulators, OpenMP over (f, x).  No blocking,
 *            no reordering beyond the de-interleave; used for the large configs and timed as
 *            the CPU baseline.  Validated bit-for-bit against level 0 in the tests.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define ORACLE_OK 0
#define ORACLE_ERR_ARG 1
#define ORACLE_ERR_RANGE 2 /* a per-call sum does not fit int32 */
#define ORACLE_ERR_ALLOC 3

/* Excess-8 decode: "data with a possible range [-8,7] is shifted by an offset of 8". */
static inline int dec_re(uint8_t w) { return (int)(w >> 4) - 8; }
static inline int dec_im(uint8_t w) { return (int)(w & 15) - 8; }

/* Upper-triangle row-major index (BASELINE.json output layout). */
static inline size_t bidx(size_t N, size_t x, size_t y) { return x * N - x * (x - 1) / 2 + (y - x); }

size_t corr_oracle_baseline_index(int N, int x, int y) { return bidx((size_t)N, (size_t)x, (size_t)y); }

int corr_oracle_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* accumulate != 0: add modulo 2^32 to what is there (two's complement wrap, reading 7);
 * accumulate == 0: overwrite. */
static inline void put(int32_t *dst, int64_t v, int accumulate)
{
    if (accumulate)
        *dst = (int32_t)((uint32_t)*dst + (uint32_t)(int32_t)v);
    else
        *dst = (int32_t)v;
}

/* One ordered pair (x, y) -- ANY order, also x > y -- of channel f, by Eq. (1) summed over t.
 * Used for the Hermitian pin and for sampled checks of full-size runs. */
int corr_oracle_pair(const uint8_t *packed, int N, int F, int T, int f, int x, int y,
                     int64_t *re_out, int64_t *im_out)
{
    if (!packed || N < 1 || F < 1 || T < 1 || f < 0 || f >= F || x < 0 || x >= N || y < 0 || y >= N)
        return ORACLE_ERR_ARG;
    int64_t re = 0, im = 0;
    for (int t = 0; t < T; ++t) {
        uint8_t wx = packed[((size_t)t * F + f) * N + x];
        uint8_t wy = packed[((size_t)t * F + f) * N + y];
        int xr = dec_re(wx), xi = dec_im(wx), yr = dec_re(wy), yi = dec_im(wy);
        re += xr * yr + xi * yi; /* Eq. (1), first component  */
        im += xi * yr - xr * yi; /* Eq. (1), second component */
    }
    *re_out = re;
    *im_out = im;
    return ORACLE_OK;
}

/* Level 0: the definition. */
int corr_oracle_level0(const uint8_t *packed, int N, int F, int T, int32_t *vis, int accumulate)
{
    if (!packed || !vis || N < 1 || F < 1 || T < 1)
        return ORACLE_ERR_ARG;
    const size_t B = (size_t)N * ((size_t)N + 1) / 2;
    for (int f = 0; f < F; ++f)
        for (int x = 0; x < N; ++x)
            for (int y = x; y < N; ++y) {
                int64_t re = 0, im = 0;
                for (int t = 0; t < T; ++t) {
                    uint8_t wx = packed[((size_t)t * F + f) * N + x];
                    uint8_t wy = packed[((size_t)t * F + f) * N + y];
                    int xr = dec_re(wx), xi = dec_im(wx), yr = dec_re(wy), yi = dec_im(wy);
                    re += xr * yr + xi * yi;
                    im += xi * yr - xr * yi;
                }
                if (re > INT32_MAX || re < INT32_MIN || im > INT32_MAX || im < INT32_MIN)
                    return ORACLE_ERR_RANGE;
                int32_t *o = vis + ((size_t)f * B + bidx(N, x, y)) * 2;
                put(o + 0, re, accumulate);
                put(o + 1, im, accumulate);
            }
    return ORACLE_OK;
}

/* Level 1: planar de-interleave, then the same loops.  int32 accumulators are safe because one
 * sample contributes at most 128 to Re ((-8)^2+(-8)^2) and 120 to |Im| (Appendix A of SURVEY.md),
 * and T <= 2^24-1 is enforced: 128*(2^24-1) < 2^31. */
int corr_oracle_level1(const uint8_t *packed, int N, int F, int T, int32_t *vis, int accumulate)
{
    if (!packed || !vis || N < 1 || F < 1 || T < 1 || T > 16777215)
        return ORACLE_ERR_ARG;
    const size_t B = (size_t)N * ((size_t)N + 1) / 2;
    const size_t plane = (size_t)F * N * T;
    int8_t *re = (int8_t *)malloc(plane);
    int8_t *im = (int8_t *)malloc(plane);
    if (!re || !im) {
        free(re);
        free(im);
        return ORACLE_ERR_ALLOC;
    }
    /* de-interleave [T][F][N] packed -> re[f][n][t], im[f][n][t] */
#pragma omp parallel for schedule(static)
    for (int f = 0; f < F; ++f)
        for (int t = 0; t < T; ++t) {
            const uint8_t *src = packed + ((size_t)t * F + f) * N;
            for (int n = 0; n < N; ++n) {
                re[((size_t)f * N + n) * T + t] = (int8_t)dec_re(src[n]);
                im[((size_t)f * N + n) * T + t] = (int8_t)dec_im(src[n]);
            }
        }
    const long rows = (long)F * N;
#pragma omp parallel for schedule(dynamic, 1)
    for (long r = 0; r < rows; ++r) {
        const int f = (int)(r / N), x = (int)(r % N);
        const int8_t *xr = re + ((size_t)f * N + x) * T;
        const int8_t *xi = im + ((size_t)f * N + x) * T;
        for (int y = x; y < N; ++y) {
            const int8_t *yr = re + ((size_t)f * N + y) * T;
            const int8_t *yi = im + ((size_t)f * N + y) * T;
            int32_t sre = 0, sim = 0;
            for (int t = 0; t < T; ++t) {
                sre += xr[t] * yr[t] + xi[t] * yi[t];
                sim += xi[t] * yr[t] - xr[t] * yi[t];
            }
            int32_t *o = vis + ((size_t)f * B + bidx(N, x, y)) * 2;
            put(o + 0, sre, accumulate);
            put(o + 1, sim, accumulate);
        }
    }
    free(re);
    free(im);
    return ORACLE_OK;
}

/* The paper's own route through the STORED (unsigned, offset-encoded) nibbles, PAPER.md:84-91:
 * sum the products of the stored values X', Y' in [0,15] and add the offset term of Eq. (3),
 *     B(X,Y,t) = sum_time ( -8((X're+X'im)+(Y're+Y'im)) + 128 ,  8((X're-X'im)-(Y're-Y'im)) ).
 * DESIGN.md reading 4: X, Y in Eq. (3) are the stored values and "+128" is per time sample.
 * This never subtracts 8 from a nibble, so it is an independent decode of the excess-8 format:
 * agreement with level 0 pins both (pin P4). */
int corr_oracle_eq3_route(const uint8_t *packed, int N, int F, int T, int32_t *vis)
{
    if (!packed || !vis || N < 1 || F < 1 || T < 1)
        return ORACLE_ERR_ARG;
    const size_t B = (size_t)N * ((size_t)N + 1) / 2;
    for (int f = 0; f < F; ++f)
        for (int x = 0; x < N; ++x)
            for (int y = x; y < N; ++y) {
                int64_t raw_re = 0, raw_im = 0, off_re = 0, off_im = 0;
                for (int t = 0; t < T; ++t) {
                    uint8_t wx = packed[((size_t)t * F + f) * N + x];
                    uint8_t wy = packed[((size_t)t * F + f) * N + y];
                    int Xr = wx >> 4, Xi = wx & 15, Yr = wy >> 4, Yi = wy & 15; /* stored, unsigned */
                    raw_re += Xr * Yr + Xi * Yi;
                    raw_im += Xi * Yr - Xr * Yi;
                    off_re += -8 * ((Xr + Xi) + (Yr + Yi)) + 128;
                    off_im += 8 * ((Xr - Xi) - (Yr - Yi));
                }
                int32_t *o = vis + ((size_t)f * B + bidx(N, x, y)) * 2;
                o[0] = (int32_t)(raw_re + off_re);
                o[1] = (int32_t)(raw_im + off_im);
            }
    return ORACLE_OK;
}
