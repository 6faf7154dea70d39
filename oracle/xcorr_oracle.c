/* oracle/xcorr_oracle.c  --  TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, obviously-correct CPU definition of what the X-engine hot path computes.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference legs
 * may build, load or call this file.  It shares no code, header, table or helper with
 * paper_1708_00720_b200/csrc (the CUDA path) and includes nothing from include/.
 *
 * What it computes (BASELINE.json north_star; the paper itself
 * prints no formula for correlation -- PAPER.md:141 "Linear algebra: matrix multiplication
 * and related routines" and PAPER.md:579 list it as back-end / future functionality):
 *
 *   for every channel c and every input pair i >= j
 *       V[c][i][j] = sum_t  x[t][c][i] * conj( x[t][c][j] )
 *         .re = sum_t ( re_i*re_j + im_i*im_j )
 *         .im = sum_t ( im_i*re_j - re_i*im_j )
 *       out[c][ i*(i+1)/2 + j ] = (accumulate ? out : 0) + V        (int32 re, int32 im)
 *
 * The method reaches exactly this result, so the oracle is the definition written out:
 * three nested loops (channel, pair, sample).  Sums are taken in int64 and truncated to
 * 32 bits, which equals the int32 accumulator wrapping mod 2^32 (reading A7); the number
 * of (re or im) sums that did not fit in int32 is reported so tests can assert "no wrap".
 *
 * Input  x : dense [ntime][nchan][ninputs], input fastest (ring spans are contiguous,
 *            PAPER.md:345).
 *   ci8 (dtype 8, "8+8 bit complex"): byte 0 = re, byte 1 = im, both int8   (A5)
 *   ci4 (dtype 4, "4+4 complex signed integers"): one byte, re = high nibble,
 *        im = low nibble, each two's complement in [-8,7]                                   (A4)
 * Output   : [nchan][B][2] int32, B = ninputs*(ninputs+1)/2, packed row-major lower
 *            triangle (A2, A3).
 *
 * Pins (tests/test_oracle_pins.py, all `-m "not gpu"`): hand-worked example, two-constant
 * closed form, Hermitian symmetry of the full matrix, real non-negative autos, trace and
 * beam-power identities, accumulation laws, invariances, numpy complex128 HERK, ci4 == ci8,
 * extreme codes, brute force against a pure-Python evaluation.
 * Parity with the real Bifrost library's byte conventions (nibble order, triangle order)
 * is UNPINNED: the paper does not state them.
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>

/* decode one complex sample at x[t][c][i] -> (re, im) */
static void decode_sample(const uint8_t* in, int dtype, long long N, long long C,
                          long long t, long long c, long long i, int* re, int* im)
{
    long long s = (t * C + c) * N + i;            /* sample index in [T][C][N] */
    if (dtype == 8) {
        *re = (int8_t)in[2 * s + 0];
        *im = (int8_t)in[2 * s + 1];
    } else {
        uint8_t b = in[s];
        int hi = (b >> 4) & 0xF, lo = b & 0xF;
        *re = hi >= 8 ? hi - 16 : hi;
        *im = lo >= 8 ? lo - 16 : lo;
    }
}

/* One visibility, straight from the definition. Returns sums in int64. */
static void visibility(const uint8_t* in, int dtype, long long N, long long C, long long T,
                       long long c, long long i, long long j, int64_t* vre, int64_t* vim)
{
    int64_t sr = 0, si = 0;
    for (long long t = 0; t < T; ++t) {
        int ri, ii, rj, ij;
        decode_sample(in, dtype, N, C, t, c, i, &ri, &ii);
        decode_sample(in, dtype, N, C, t, c, j, &rj, &ij);
        sr += (int64_t)(ri * rj + ii * ij);
        si += (int64_t)(ii * rj - ri * ij);
    }
    *vre = sr;
    *vim = si;
}

static int fits32(int64_t v) { return v >= INT32_MIN && v <= INT32_MAX; }

/* out[k] = (accumulate ? out[k] : 0) + v   with int32 wrap-around */
static void add_wrap(int32_t* dst, int64_t v, int accumulate)
{
    uint32_t old = accumulate ? (uint32_t)*dst : 0u;
    *dst = (int32_t)(old + (uint32_t)(uint64_t)v);
}

/* Selected entries only: entry e is (c[e], i[e], j[e]) with any i, j in [0, N) -- also the
 * upper triangle, which is how the Hermitian-symmetry pin reads the full matrix.
 * vals[2e] = re, vals[2e+1] = im (int64, not wrapped).  Returns 0, or -1 on bad arguments. */
int xcorr_oracle_entries(const uint8_t* in, int ninputs, int nchan, int ntime, int dtype,
                         long long nentries, const int* c, const int* i, const int* j,
                         int64_t* vals)
{
    if (!in || !c || !i || !j || !vals || ninputs <= 0 || nchan <= 0 || ntime <= 0) return -1;
    if (dtype != 4 && dtype != 8) return -1;
    for (long long e = 0; e < nentries; ++e) {
        if (c[e] < 0 || c[e] >= nchan || i[e] < 0 || i[e] >= ninputs || j[e] < 0 || j[e] >= ninputs)
            return -1;
        visibility(in, dtype, ninputs, nchan, ntime, c[e], i[e], j[e], &vals[2 * e], &vals[2 * e + 1]);
    }
    return 0;
}

/* The whole span, definition order: channel, pair (i >= j), sample.
 * Channels are independent and are spread over OpenMP threads when built with -fopenmp.
 * To keep the sample loop contiguous each thread first copies its channel's [T][N] slab
 * into de-interleaved int8 rows re[i][t], im[i][t] (a transposition only; no arithmetic).
 * Returns the number of sums that did not fit in int32 (0 = no wrap), or -1 on bad args. */
long long xcorr_oracle(const uint8_t* in, int32_t* out, int ninputs, int nchan, int ntime,
                       int dtype, int accumulate)
{
    if (!in || !out || ninputs <= 0 || nchan <= 0 || ntime <= 0) return -1;
    if (dtype != 4 && dtype != 8) return -1;
    const long long N = ninputs, C = nchan, T = ntime;
    const long long B = N * (N + 1) / 2;
    long long nwrap = 0;

#pragma omp parallel reduction(+ : nwrap)
    {
        int8_t* re = (int8_t*)malloc((size_t)(N * T));
        int8_t* im = (int8_t*)malloc((size_t)(N * T));
#pragma omp for schedule(dynamic, 1)
        for (long long c = 0; c < C; ++c) {
            for (long long t = 0; t < T; ++t)
                for (long long i = 0; i < N; ++i) {
                    int r, m;
                    decode_sample(in, dtype, N, C, t, c, i, &r, &m);
                    re[i * T + t] = (int8_t)r;
                    im[i * T + t] = (int8_t)m;
                }
            for (long long i = 0; i < N; ++i) {
                const int8_t* ri = re + i * T;
                const int8_t* ii = im + i * T;
                for (long long j = 0; j <= i; ++j) {
                    const int8_t* rj = re + j * T;
                    const int8_t* ij = im + j * T;
                    int64_t sr = 0, si = 0;
                    for (long long t = 0; t < T; ++t) {
                        sr += (int64_t)((int)ri[t] * rj[t] + (int)ii[t] * ij[t]);
                        si += (int64_t)((int)ii[t] * rj[t] - (int)ri[t] * ij[t]);
                    }
                    if (!fits32(sr)) ++nwrap;
                    if (!fits32(si)) ++nwrap;
                    int32_t* dst = out + 2 * (c * B + i * (i + 1) / 2 + j);
                    add_wrap(dst + 0, sr, accumulate);
                    add_wrap(dst + 1, si, accumulate);
                }
            }
        }
        free(re);
        free(im);
    }
    return nwrap;
}

/* Integration dump (the paper's accumulate block hands an integration on when it is
 * complete, and its pipelines convert integer data to floating point for the stages that follow,
 * PAPER.md:549): every int32 component v of the packed visibility buffer becomes the float32
 *        f = (float) v * scale          (int32 -> float32 round-to-nearest-even, then one float32 multiply)
 * in the same [nchan][B][2] order, and, if zero_acc != 0, the accumulator is cleared afterwards so that the next
 * integration can start with accumulate = 1.  Returns the number of components converted, or -1 on bad arguments. */
long long xcorr_oracle_dump(int32_t* acc, float* out, long long ncomponents, float scale, int zero_acc)
{
    long long k;
    if (!acc || !out || ncomponents < 0) return -1;
    for (k = 0; k < ncomponents; ++k) {
        const float f = (float)acc[k];
        out[k] = f * scale;
        if (zero_acc) acc[k] = 0;
    }
    return ncomponents;
}

/* Integration dump with reorder (its optional part; the paper's back end has "efficient data
 * reordering"): the packed lower triangle becomes the FULL Hermitian matrix in float32,
 *        out[c][i][j] = ( (float) V.re * scale ,   (float) V.im * scale  )     for j <= i,  V = acc[c][ i(i+1)/2 + j ]
 *        out[c][i][j] = ( (float) V.re * scale , -((float) V.im * scale) )     for j >  i,  V = acc[c][ j(j+1)/2 + i ]
 * i.e. the upper triangle is the complex conjugate of the mirrored lower entry (the negation is exact; an imaginary
 * part of zero becomes -0.0f).  out: [nchan][ninputs][ninputs][2] float32.  The accumulator is cleared afterwards if
 * zero_acc != 0.  Returns the number of matrix entries written, or -1 on bad arguments. */
long long xcorr_oracle_dump_matrix(int32_t* acc, float* out, int ninputs, int nchan, float scale, int zero_acc)
{
    const long long N = ninputs, C = nchan, B = N * (N + 1) / 2;
    if (!acc || !out || N <= 0 || C <= 0) return -1;
    for (long long c = 0; c < C; ++c)
        for (long long i = 0; i < N; ++i)
            for (long long j = 0; j < N; ++j) {
                const long long hi = i >= j ? i : j, lo = i >= j ? j : i;
                const int32_t* v = acc + 2 * (c * B + hi * (hi + 1) / 2 + lo);
                const float re = (float)v[0] * scale, im = (float)v[1] * scale;
                float* o = out + 2 * ((c * N + i) * N + j);
                o[0] = re;
                o[1] = j > i ? -im : im;
            }
    if (zero_acc)
        for (long long k = 0; k < 2 * C * B; ++k) acc[k] = 0;
    return C * N * N;
}

/* Beamformer on the same span (the GPU stage the paper's deployment runs on the
 * "4+4 complex signed integers"; a "phase-and-sum" of all inputs per beam):
 *
 *   for every sample t, channel c and beam k
 *       b[t][c][k] = sum over inputs i of   w[c][k][i] * x[t][c][i]           (complex product, no conjugate)
 *         .re = sum_i ( wr*xr - wi*xi )
 *         .im = sum_i ( wr*xi + wi*xr )
 *       out[t][c][k] = b            (int32 re, int32 im; sums taken in int64 and truncated to 32 bits)
 *
 * x as above (ci4 or ci8).  Weights w: dense [nchan][nbeam][ninputs], input fastest, always 8+8 bit: byte 0 = re,
 * byte 1 = im, int8.  Every code is legal for both parts, -128 included (reading B4: as for the
 * voltages, reading A6, the extreme code is ordinary input and the result must stay exact).
 * Returns the number of sums that did not fit in int32 (0 for every legal input: 2 * 32768 * 128 * 128 < 2^31
 * holds up to 32768 inputs), -1 on bad arguments. */
long long xcorr_oracle_beamform(const uint8_t* in, const uint8_t* w, int32_t* out, int ninputs, int nchan,
                                int ntime, int nbeam, int dtype)
{
    const long long N = ninputs, C = nchan, T = ntime, K = nbeam;
    long long nwrap = 0;
    if (!in || !w || !out || N <= 0 || C <= 0 || T <= 0 || K <= 0 || (dtype != 4 && dtype != 8)) return -1;
#ifdef _OPENMP
#pragma omp parallel for collapse(2) reduction(+ : nwrap) schedule(static)
#endif
    for (long long t = 0; t < T; ++t) {
        for (long long c = 0; c < C; ++c) {
            for (long long k = 0; k < K; ++k) {
                int64_t sr = 0, si = 0;
                for (long long i = 0; i < N; ++i) {
                    int xr, xi;
                    const uint8_t* wp = w + 2 * ((c * K + k) * N + i);
                    const int wr = (int8_t)wp[0], wi = (int8_t)wp[1];
                    decode_sample(in, dtype, N, C, t, c, i, &xr, &xi);
                    sr += (int64_t)(wr * xr - wi * xi);
                    si += (int64_t)(wr * xi + wi * xr);
                }
                nwrap += !fits32(sr) + !fits32(si);
                out[2 * ((t * C + c) * K + k) + 0] = (int32_t)(uint32_t)(uint64_t)sr;
                out[2 * ((t * C + c) * K + k) + 1] = (int32_t)(uint32_t)(uint64_t)si;
            }
        }
    }
    return nwrap;
}

/* Number of threads the span routines will use (1 when built without OpenMP). */
#ifdef _OPENMP
#include <omp.h>
int xcorr_oracle_threads(void) { return omp_get_max_threads(); }
void xcorr_oracle_set_threads(int n) { if (n > 0) omp_set_num_threads(n); }
#else
int xcorr_oracle_threads(void) { return 1; }
void xcorr_oracle_set_threads(int n) { (void)n; }
#endif
