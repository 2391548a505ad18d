/*
 * xengine_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * Plain, slow, obviously-correct CPU oracle for the X-engine of an FX correlator:
 *
 *     C_ij[k] = sum_{a=0}^{A-1} conj(S_{a,i}[k]) * S_{a,j}[k]          (Sec. 2, Eq. 2)
 *
 * evaluated for every frequency channel k, every station pair including the
 * autocorrelations on the triangle's hypotenuse (Sec. 4, Sec. 4.2)
 * and every polarisation product, as raw sums with no normalisation (Eq. 2 has no 1/A).
 * "Results are usually then accumulated" is the `accumulate` argument.
 *
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference leg
 * may call this.  It shares no code, header, table or helper with the CUDA path under
 * paper_1305_5639_b200/csrc; the layouts below are restated here from DESIGN.md.
 *
 * Readings of the paper taken here:
 *   R1  the FIRST factor is conjugated (Eq. 2), V_ij is stored for i >= j;
 *   R2  autocorrelations are included, B = N(N+1)/2, b(i,j) = i(i+1)/2 + j;
 *   R3  a (station, polarisation) pair is one of the paper's "input streams";
 *       output keeps all P*P products per station pair, also for i == j;
 *   R6  raw sums, no scaling.
 *
 * Layouts (all C-contiguous):
 *   in  [T][C][N][P] complex, (re, im) interleaved; int8 pairs (ci8) or IEEE binary16 pairs (cf16)
 *   out [n_sel][B][P][P] complex, (re, im) interleaved; int64 (ci8) or double (cf16);
 *       p = polarisation of the conjugated station i, q = polarisation of station j;
 *       n_sel = number of selected channels, listed in chans[] (NULL = all C, in order).
 *
 * Arithmetic: ci8 exact in int64; cf16 inputs converted exactly to double, products and
 * sums in double in the order t = 0..T-1.  No blocking, no reordering: the loops are Eq. 2.
 *
 * The rectangular cross-only variant (xo_xengine_cross_*) is at the end of this file; its pins are
 * tests/test_oracle_cross_pins.py (einsum brute force, ZGEMM, the triangle oracle's off-diagonal block,
 * conjugate swap, constant closed form).
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute force against numpy complex128
 * einsum on tiny inputs, reduction to a library ZGEMM, Hermitian symmetry, real non-negative
 * autocorrelations, constant-input closed form with asymmetric constants (pins the sign of
 * Im and which factor is conjugated), identical streams, single delayed tone analytic phase,
 * additivity in time, exact rotation by j, beam-sum identity, station permutation.
 * Nothing in the paper prints a numerical X-engine output, so no paper-printed value is
 * pinned ("parity unpinned" applies only to the paper's own unprinted outputs).
 */
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#include <math.h>
#ifdef _OPENMP
#include <omp.h>
#endif

long long xo_baseline_index(int i, int j) { return (long long)i * (i + 1) / 2 + j; }

int xo_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void xo_set_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* IEEE 754 binary16 bit pattern -> double, exact (every binary16 value is a double). */
static double half_bits_to_double(uint16_t h)
{
    int sign = (h >> 15) & 1;
    int expo = (h >> 10) & 0x1f;
    int frac = h & 0x3ff;
    double v;
    if (expo == 0)
        v = ldexp((double)frac, -24);                 /* zero and subnormals: frac * 2^-24 */
    else if (expo == 31)
        v = frac ? NAN : INFINITY;
    else
        v = ldexp((double)(1024 + frac), expo - 25);  /* (1 + frac/1024) * 2^(expo-15) */
    return sign ? -v : v;
}

double xo_half_to_double(uint16_t h) { return half_bits_to_double(h); }

/* One visibility straight from the un-gathered input: Eq. 2 for channel c, conjugated
 * stream (i,p), second stream (j,q).  vis[0] = Re, vis[1] = Im. */
void xo_pair_ci8(const int8_t* in, int N, int P, int C, int T,
                 int c, int i, int p, int j, int q, int64_t vis[2])
{
    int64_t re = 0, im = 0;
    for (int t = 0; t < T; ++t) {
        const int8_t* a = in + 2 * ((((size_t)t * C + c) * N + i) * P + p);
        const int8_t* b = in + 2 * ((((size_t)t * C + c) * N + j) * P + q);
        int64_t ar = a[0], ai = a[1], br = b[0], bi = b[1];
        re += ar * br + ai * bi;      /* Re conj(a) b */
        im += ar * bi - ai * br;      /* Im conj(a) b */
    }
    vis[0] = re;
    vis[1] = im;
}

void xo_pair_cf16(const uint16_t* in, int N, int P, int C, int T,
                  int c, int i, int p, int j, int q, double vis[2])
{
    double re = 0.0, im = 0.0;
    for (int t = 0; t < T; ++t) {
        const uint16_t* a = in + 2 * ((((size_t)t * C + c) * N + i) * P + p);
        const uint16_t* b = in + 2 * ((((size_t)t * C + c) * N + j) * P + q);
        double ar = half_bits_to_double(a[0]), ai = half_bits_to_double(a[1]);
        double br = half_bits_to_double(b[0]), bi = half_bits_to_double(b[1]);
        re += ar * br + ai * bi;
        im += ar * bi - ai * br;
    }
    vis[0] = re;
    vis[1] = im;
}

/* Whole packed triangle for the selected channels.
 * The only concession to the memory system is a private per-channel gather of
 * x[t][m] (m = s*P + p) into two contiguous arrays before the loops. */
int xo_xengine_ci8(const int8_t* in, int64_t* out, int N, int P, int C, int T,
                   const int* chans, int n_sel, int accumulate)
{
    if (!in || !out || N <= 0 || P <= 0 || C <= 0 || T < 0) return -1;
    if (!chans) n_sel = C;
    const int M = N * P;
    const size_t B = (size_t)N * (N + 1) / 2;
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n_sel; ++k) {
        const int c = chans ? chans[k] : k;
        int32_t* xr = (int32_t*)malloc(sizeof(int32_t) * (size_t)M * (T ? T : 1));
        int32_t* xi = (int32_t*)malloc(sizeof(int32_t) * (size_t)M * (T ? T : 1));
        if (!xr || !xi || c < 0 || c >= C) { fail = 1; free(xr); free(xi); continue; }
        for (int t = 0; t < T; ++t)
            for (int m = 0; m < M; ++m) {
                const int8_t* s = in + 2 * (((size_t)t * C + c) * M + m);
                xr[(size_t)m * T + t] = s[0];
                xi[(size_t)m * T + t] = s[1];
            }
        for (int i = 0; i < N; ++i)
            for (int j = 0; j <= i; ++j)
                for (int p = 0; p < P; ++p)
                    for (int q = 0; q < P; ++q) {
                        const int32_t* ar = xr + (size_t)(i * P + p) * T;
                        const int32_t* ai = xi + (size_t)(i * P + p) * T;
                        const int32_t* br = xr + (size_t)(j * P + q) * T;
                        const int32_t* bi = xi + (size_t)(j * P + q) * T;
                        int64_t re = 0, im = 0;
                        for (int t = 0; t < T; ++t) {
                            re += (int64_t)ar[t] * br[t] + (int64_t)ai[t] * bi[t];
                            im += (int64_t)ar[t] * bi[t] - (int64_t)ai[t] * br[t];
                        }
                        int64_t* o = out + 2 * ((((size_t)k * B + (size_t)xo_baseline_index(i, j)) * P + p) * P + q);
                        if (accumulate) { o[0] += re; o[1] += im; }
                        else            { o[0]  = re; o[1]  = im; }
                    }
        free(xr);
        free(xi);
    }
    return fail ? -2 : 0;
}

int xo_xengine_cf16(const uint16_t* in, double* out, int N, int P, int C, int T,
                    const int* chans, int n_sel, int accumulate)
{
    if (!in || !out || N <= 0 || P <= 0 || C <= 0 || T < 0) return -1;
    if (!chans) n_sel = C;
    const int M = N * P;
    const size_t B = (size_t)N * (N + 1) / 2;
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n_sel; ++k) {
        const int c = chans ? chans[k] : k;
        double* xr = (double*)malloc(sizeof(double) * (size_t)M * (T ? T : 1));
        double* xi = (double*)malloc(sizeof(double) * (size_t)M * (T ? T : 1));
        if (!xr || !xi || c < 0 || c >= C) { fail = 1; free(xr); free(xi); continue; }
        for (int t = 0; t < T; ++t)
            for (int m = 0; m < M; ++m) {
                const uint16_t* s = in + 2 * (((size_t)t * C + c) * M + m);
                xr[(size_t)m * T + t] = half_bits_to_double(s[0]);
                xi[(size_t)m * T + t] = half_bits_to_double(s[1]);
            }
        for (int i = 0; i < N; ++i)
            for (int j = 0; j <= i; ++j)
                for (int p = 0; p < P; ++p)
                    for (int q = 0; q < P; ++q) {
                        const double* ar = xr + (size_t)(i * P + p) * T;
                        const double* ai = xi + (size_t)(i * P + p) * T;
                        const double* br = xr + (size_t)(j * P + q) * T;
                        const double* bi = xi + (size_t)(j * P + q) * T;
                        double re = 0.0, im = 0.0;
                        for (int t = 0; t < T; ++t) {
                            re += ar[t] * br[t] + ai[t] * bi[t];
                            im += ar[t] * bi[t] - ai[t] * br[t];
                        }
                        double* o = out + 2 * ((((size_t)k * B + (size_t)xo_baseline_index(i, j)) * P + p) * P + q);
                        if (accumulate) { o[0] += re; o[1] += im; }
                        else            { o[0]  = re; o[1]  = im; }
                    }
        free(xr);
        free(xi);
    }
    return fail ? -2 : 0;
}

/* ------------------------------------------------------------------------------------------
 * Rectangular, cross-only X-engine (Sec. 4: nodes of the space-division models
 * "process two parts of the input streams in a rectangle pattern for cross-correlations only"):
 *
 *     V[c][i][j][p][q] = sum_t conj(a[t][c][i][p]) * b[t][c][j][q]      i in group A, j in group B
 *
 * Eq. 2 with the conjugated stream taken from group A and the other from group B; every (i, j)
 * is stored (no triangle, no autocorrelations).  Layouts: in_a [T][C][Na][P], in_b [T][C][Nb][P]
 * complex interleaved; out [n_sel][Na][Nb][P][P] complex interleaved (int64 / double).
 * Plain loops, time innermost, no gather, no blocking.
 * ------------------------------------------------------------------------------------------ */
int xo_xengine_cross_ci8(const int8_t* in_a, const int8_t* in_b, int64_t* out, int Na, int Nb, int P,
                         int C, int T, const int* chans, int n_sel, int accumulate)
{
    if (!in_a || !in_b || !out || Na <= 0 || Nb <= 0 || P <= 0 || C <= 0 || T < 0) return -1;
    if (!chans) n_sel = C;
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n_sel; ++k) {
        const int c = chans ? chans[k] : k;
        if (c < 0 || c >= C) { fail = 1; continue; }
        for (int i = 0; i < Na; ++i)
            for (int j = 0; j < Nb; ++j)
                for (int p = 0; p < P; ++p)
                    for (int q = 0; q < P; ++q) {
                        int64_t re = 0, im = 0;
                        for (int t = 0; t < T; ++t) {
                            const int8_t* a = in_a + 2 * ((((size_t)t * C + c) * Na + i) * P + p);
                            const int8_t* b = in_b + 2 * ((((size_t)t * C + c) * Nb + j) * P + q);
                            int64_t ar = a[0], ai = a[1], br = b[0], bi = b[1];
                            re += ar * br + ai * bi;      /* Re conj(a) b */
                            im += ar * bi - ai * br;      /* Im conj(a) b */
                        }
                        int64_t* o = out + 2 * (((((size_t)k * Na + i) * Nb + j) * P + p) * P + q);
                        if (accumulate) { o[0] += re; o[1] += im; }
                        else            { o[0]  = re; o[1]  = im; }
                    }
    }
    return fail ? -2 : 0;
}

int xo_xengine_cross_cf16(const uint16_t* in_a, const uint16_t* in_b, double* out, int Na, int Nb, int P,
                          int C, int T, const int* chans, int n_sel, int accumulate)
{
    if (!in_a || !in_b || !out || Na <= 0 || Nb <= 0 || P <= 0 || C <= 0 || T < 0) return -1;
    if (!chans) n_sel = C;
    int fail = 0;
#pragma omp parallel for schedule(dynamic, 1)
    for (int k = 0; k < n_sel; ++k) {
        const int c = chans ? chans[k] : k;
        if (c < 0 || c >= C) { fail = 1; continue; }
        for (int i = 0; i < Na; ++i)
            for (int j = 0; j < Nb; ++j)
                for (int p = 0; p < P; ++p)
                    for (int q = 0; q < P; ++q) {
                        double re = 0.0, im = 0.0;
                        for (int t = 0; t < T; ++t) {
                            const uint16_t* a = in_a + 2 * ((((size_t)t * C + c) * Na + i) * P + p);
                            const uint16_t* b = in_b + 2 * ((((size_t)t * C + c) * Nb + j) * P + q);
                            double ar = half_bits_to_double(a[0]), ai = half_bits_to_double(a[1]);
                            double br = half_bits_to_double(b[0]), bi = half_bits_to_double(b[1]);
                            re += ar * br + ai * bi;
                            im += ar * bi - ai * br;
                        }
                        double* o = out + 2 * (((((size_t)k * Na + i) * Nb + j) * P + p) * P + q);
                        if (accumulate) { o[0] += re; o[1] += im; }
                        else            { o[0]  = re; o[1]  = im; }
                    }
    }
    return fail ? -2 : 0;
}
