/*
 * fft3d_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, fp64 CPU oracle for the 3D real-to-complex forward DFT and the
 * complex-to-real inverse DFT of "Scalable Multi-node Fast Fourier Transform on
 * GPUs" (arXiv 2202.12756).  Only tests/, __graft_entry__.smoke() and bench.py's
 * cpu_baseline / --impl reference legs may load this file.  It shares no code,
 * header, table or constant generator with the CUDA path under
 * paper_2202_12756_b200/csrc/ and neither side includes the other.
 *
 * What it computes (citations: P:n = /root/reference/PAPER.md line n):
 *
 *   forward  F(kx,ky,kz) = sum_{jx,jy,jz} f(jx,jy,jz)
 *                          exp(-2 pi i [jx kx/Nx + jy ky/Ny + jz kz/Nz])   Eq. (1)
 *            stored for kx in [0,Nx), ky in [0,Ny), kz in [0,Nz/2]        Eq. (4)
 *            (Nz/2+1 entries along z: the FFTW convention the paper adopts)
 *   inverse  f(j) = 1/(Nx Ny Nz) * Re sum_{k over the FULL grid} Ft(k)
 *                          exp(+2 pi i [...])                               Eq. (2)
 *            where Ft extends the stored half by Ft(kx,ky,kz) =
 *            conj F(-kx mod Nx, -ky mod Ny, Nz-kz) for kz > Nz/2            Eq. (3)
 *            The 1/(Nx Ny Nz) is BASELINE.json's reading (forward unnormalised,
 *            inverse normalised); the paper prints Eq. (2) without it but times a
 *            "normalization" step and recovers f after a pair.
 *
 * Two levels:
 *   oracle_dft3d_direct / oracle_idft3d_direct  -- the definitions written out,
 *       O(N^6), for tiny grids; these pin the fast routines below.
 *   oracle_r2c / oracle_c2r -- the same result via separable 1D transforms along
 *       z, then y, then x (forward) / x, y, z (inverse); each 1D transform is a
 *       recursive decimation-in-time mixed-radix Cooley-Tukey FFT (ref [13])
 *       that splits by the smallest prime factor and falls back to the O(n^2) sum
 *       for a prime length.  Full-length complex transforms of the real rows: no
 *       even/odd packing, no Stockham autosort, no fused steps.
 *
 * All arrays are dense, row-major, z fastest, x slowest; complex numbers are
 * interleaved (re, im) doubles; the half spectrum is in NATURAL order
 * [Nx][Ny][Nz/2+1] (the slab layout of the product is a separate index map, see
 * oracle/slab_layout.py).
 *
 * Pins (tests/test_oracle_pins.py): direct O(N^6) on 8^3, 12^3 and 8x12x6; shifted
 * delta; single cosine mode; the paper's worked example Eq. (5) P:100 with its
 * closed-form spikes (tests/golden/eq5_spikes.txt); Parseval; Hermitian planes;
 * round trip; numpy.fft as a second library cross-check.  Nothing here is
 * "parity unpinned".
 */
#define _GNU_SOURCE
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

typedef struct { double re, im; } cplx;

static const double TWO_PI = 6.283185307179586476925286766559;

static inline cplx c_mul(cplx a, cplx b) {
    cplx r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re };
    return r;
}
static inline cplx c_add(cplx a, cplx b) { cplx r = { a.re + b.re, a.im + b.im }; return r; }

/* exp(sign * 2 pi i * num / den) with the fraction reduced to [0,1) in integers first,
 * so the argument handed to sin/cos is never large. */
static cplx root_of_unity(long long num, long long den, int sign) {
    long long m = num % den;
    if (m < 0) m += den;
    /* exact values on the axes keep deltas and Nyquist terms clean */
    cplx r;
    if (m == 0) { r.re = 1.0; r.im = 0.0; return r; }
    if (2 * m == den) { r.re = -1.0; r.im = 0.0; return r; }
    if (4 * m == den) { r.re = 0.0; r.im = sign > 0 ? 1.0 : -1.0; return r; }
    if (4 * m == 3 * den) { r.re = 0.0; r.im = sign > 0 ? -1.0 : 1.0; return r; }
    long double a = (long double)TWO_PI * (long double)m / (long double)den;
    r.re = (double)cosl(a);
    r.im = (double)(sign > 0 ? sinl(a) : -sinl(a));
    return r;
}

/* ------------------------------------------------------------------------------------
 * 1. The definitions written out: O(N^6).  Eq. (1) P:35 and Eq. (2)+(3) P:37-41.
 * ---------------------------------------------------------------------------------- */

/* F[kx][ky][kz], kz = 0..Nz/2, from real f[jx][jy][jz].  Returns 0. */
int oracle_dft3d_direct(const double *f, int Nx, int Ny, int Nz, double *F_out)
{
    cplx *F = (cplx *)F_out;
    const int Nzh = Nz / 2 + 1;
    for (int kx = 0; kx < Nx; ++kx)
    for (int ky = 0; ky < Ny; ++ky)
    for (int kz = 0; kz < Nzh; ++kz) {
        long double sre = 0.0L, sim = 0.0L;
        for (int jx = 0; jx < Nx; ++jx)
        for (int jy = 0; jy < Ny; ++jy)
        for (int jz = 0; jz < Nz; ++jz) {
            /* phase = jx kx/Nx + jy ky/Ny + jz kz/Nz as one fraction over Nx*Ny*Nz */
            long long den = (long long)Nx * Ny * Nz;
            long long num = (long long)jx * kx * ((long long)Ny * Nz)
                          + (long long)jy * ky * ((long long)Nx * Nz)
                          + (long long)jz * kz * ((long long)Nx * Ny);
            cplx w = root_of_unity(num, den, -1);
            double v = f[((size_t)jx * Ny + jy) * Nz + jz];
            sre += (long double)v * w.re;
            sim += (long double)v * w.im;
        }
        cplx r = { (double)sre, (double)sim };
        F[((size_t)kx * Ny + ky) * Nzh + kz] = r;
    }
    return 0;
}

/* f[jx][jy][jz] = 1/(NxNyNz) Re sum over the full kz range of the Hermitian-extended
 * spectrum, literally Eq. (2) with Eq. (3) supplying kz > Nz/2. */
int oracle_idft3d_direct(const double *F_in, int Nx, int Ny, int Nz, double *f)
{
    const cplx *F = (const cplx *)F_in;
    const int Nzh = Nz / 2 + 1;
    const long long den = (long long)Nx * Ny * Nz;
    for (int jx = 0; jx < Nx; ++jx)
    for (int jy = 0; jy < Ny; ++jy)
    for (int jz = 0; jz < Nz; ++jz) {
        long double sre = 0.0L;
        for (int kx = 0; kx < Nx; ++kx)
        for (int ky = 0; ky < Ny; ++ky)
        for (int kz = 0; kz < Nz; ++kz) {
            cplx v;
            if (kz < Nzh) {
                v = F[((size_t)kx * Ny + ky) * Nzh + kz];
            } else {                                   /* Eq. (3): Ft(k) = conj F(-k) */
                int mx = (Nx - kx) % Nx, my = (Ny - ky) % Ny, mz = Nz - kz;
                v = F[((size_t)mx * Ny + my) * Nzh + mz];
                v.im = -v.im;
            }
            long long num = (long long)jx * kx * ((long long)Ny * Nz)
                          + (long long)jy * ky * ((long long)Nx * Nz)
                          + (long long)jz * kz * ((long long)Nx * Ny);
            cplx w = root_of_unity(num, den, +1);
            sre += (long double)v.re * w.re - (long double)v.im * w.im;   /* real part only */
        }
        f[((size_t)jx * Ny + jy) * Nz + jz] = (double)(sre / (long double)den);
    }
    return 0;
}

/* ------------------------------------------------------------------------------------
 * 2. 1D mixed-radix recursive FFT (Cooley-Tukey, decimation in time).
 *
 *    X[k] = sum_{j<n} x[j] w^(jk),  w = exp(sign 2 pi i / n).
 *    With n = r m (r the smallest prime factor of n), j = r a + q:
 *        X[k + s m] = sum_{q<r} w^(q (k + s m)) Y_q[k],   Y_q = DFT_m of x[q], x[q+r], ...
 *    for k < m, s < r.  For prime n this is the plain O(n^2) sum.
 *
 *    tw[t] = exp(sign 2 pi i t / n0) for the top-level length n0; a level of length n
 *    uses tw[(e mod n) * (n0/n)].
 * ---------------------------------------------------------------------------------- */
static long smallest_prime_factor(long n)
{
    if (n % 2 == 0) return 2;
    for (long d = 3; d * d <= n; d += 2)
        if (n % d == 0) return d;
    return n;
}

static void fft_rec(const cplx *in, long istride, cplx *out, long n,
                    const cplx *tw, long n0, cplx *tmp /* >= n0 entries of scratch */)
{
    if (n == 1) { out[0] = in[0]; return; }
    const long r = smallest_prime_factor(n);
    const long m = n / r;
    for (long q = 0; q < r; ++q)
        fft_rec(in + q * istride, istride * r, out + q * m, m, tw, n0, tmp);
    const long tws = n0 / n;
    for (long k = 0; k < m; ++k) {
        for (long s = 0; s < r; ++s) {
            cplx acc = { 0.0, 0.0 };
            for (long q = 0; q < r; ++q) {
                long e = (q * (k + s * m)) % n;
                acc = c_add(acc, c_mul(out[q * m + k], tw[e * tws]));
            }
            tmp[s] = acc;
        }
        for (long s = 0; s < r; ++s) out[k + s * m] = tmp[s];
    }
}

static cplx *make_twiddles(long n, int sign)
{
    cplx *tw = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!tw) return NULL;
    for (long t = 0; t < n; ++t) tw[t] = root_of_unity(t, n, sign);
    return tw;
}

/* Public 1D transform: out[k] = sum_j in[j] exp(sign 2 pi i jk/n), unnormalised. */
int oracle_fft1d(const double *in, double *out, long n, int sign)
{
    cplx *tw = make_twiddles(n, sign);
    cplx *tmp = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!tw || !tmp) { free(tw); free(tmp); return 3; }
    fft_rec((const cplx *)in, 1, (cplx *)out, n, tw, n, tmp);
    free(tw); free(tmp);
    return 0;
}

/* In-place transform of `count` lines of length n inside `a`: line l starts at
 * a + base(l) and has element stride `stride`; base(l) = (l / inner) * outer_stride
 * + (l % inner) * inner_stride.  Lines are independent, so OpenMP may split them. */
static int fft_lines(cplx *a, long n, long stride, long count,
                     long inner, long inner_stride, long outer_stride,
                     int sign, int nthreads)
{
    cplx *tw = make_twiddles(n, sign);
    if (!tw) return 3;
    int err = 0;
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel num_threads(nthreads)
#endif
    {
        cplx *line = (cplx *)malloc(sizeof(cplx) * (size_t)n);
        cplx *res  = (cplx *)malloc(sizeof(cplx) * (size_t)n);
        cplx *tmp  = (cplx *)malloc(sizeof(cplx) * (size_t)n);
        if (!line || !res || !tmp) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
            err = 3;
        } else {
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
            for (long l = 0; l < count; ++l) {
                cplx *p = a + (l / inner) * outer_stride + (l % inner) * inner_stride;
                for (long j = 0; j < n; ++j) line[j] = p[j * stride];
                fft_rec(line, 1, res, n, tw, n, tmp);
                for (long j = 0; j < n; ++j) p[j * stride] = res[j];
            }
        }
        free(line); free(res); free(tmp);
    }
    free(tw);
    return err;
}

/* ------------------------------------------------------------------------------------
 * 3. Separable 3D R2C forward: z, then y, then x (paper step 1 then step 5, P:69-77,
 *    without the data movement in between: natural order in, natural order out).
 * ---------------------------------------------------------------------------------- */
int oracle_r2c(const double *f, long Nx, long Ny, long Nz, double *F_out, int nthreads)
{
    if (Nx < 1 || Ny < 1 || Nz < 2 || (Nz & 1)) return 1;
    cplx *F = (cplx *)F_out;
    const long Nzh = Nz / 2 + 1;
    int err = 0;
    /* z: full-length complex DFT of each real row, keep kz = 0..Nz/2 (Eq. (4)). */
    cplx *tw = make_twiddles(Nz, -1);
    if (!tw) return 3;
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel num_threads(nthreads)
#endif
    {
        cplx *line = (cplx *)malloc(sizeof(cplx) * (size_t)Nz);
        cplx *res  = (cplx *)malloc(sizeof(cplx) * (size_t)Nz);
        cplx *tmp  = (cplx *)malloc(sizeof(cplx) * (size_t)Nz);
        if (!line || !res || !tmp) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
            err = 3;
        } else {
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
            for (long row = 0; row < Nx * Ny; ++row) {
                const double *src = f + (size_t)row * Nz;
                for (long j = 0; j < Nz; ++j) { line[j].re = src[j]; line[j].im = 0.0; }
                fft_rec(line, 1, res, Nz, tw, Nz, tmp);
                cplx *dst = F + (size_t)row * Nzh;
                for (long k = 0; k < Nzh; ++k) dst[k] = res[k];
            }
        }
        free(line); free(res); free(tmp);
    }
    free(tw);
    if (err) return err;
    /* y: for each (x, kz) a line of length Ny with stride Nzh. */
    err = fft_lines(F, Ny, Nzh, Nx * Nzh, Nzh, 1, Ny * Nzh, -1, nthreads);
    if (err) return err;
    /* x: for each (ky, kz) a line of length Nx with stride Ny*Nzh. */
    err = fft_lines(F, Nx, Ny * Nzh, Ny * Nzh, Ny * Nzh, 1, 0, -1, nthreads);
    return err;
}

/* ------------------------------------------------------------------------------------
 * 4. Separable 3D C2R inverse: x, then y, then z ("reverse order"), scaled by
 *    1/(Nx Ny Nz).
 *
 *    Why the half spectrum suffices for x and y: for kz > Nz/2 the extended array is
 *    Ft(kx,ky,kz) = conj F(-kx,-ky,Nz-kz) (Eq. (3)); its inverse transform over (kx,ky)
 *    is sum conj F(-kx,-ky,Nz-kz) e^{+i(..)} = conj[ sum F(k'x,k'y,Nz-kz) e^{+i(..)} ]
 *    = conj G(jx,jy,Nz-kz), with G the x,y-inverse of the stored half.  So each z row
 *    of the full problem is the stored G(jx,jy,0..Nz/2) extended by conj G(.,.,Nz-kz);
 *    the full-length complex inverse of that row is taken and its real part kept.
 *    (tests pin this against oracle_idft3d_direct, which extends the 3D array literally,
 *    including on inputs whose kz=0 / kz=Nz/2 planes are NOT Hermitian-consistent.)
 * ---------------------------------------------------------------------------------- */
int oracle_c2r(const double *F_in, long Nx, long Ny, long Nz, double *f, int nthreads)
{
    if (Nx < 1 || Ny < 1 || Nz < 2 || (Nz & 1)) return 1;
    const long Nzh = Nz / 2 + 1;
    const size_t nspec = (size_t)Nx * Ny * Nzh;
    cplx *G = (cplx *)malloc(sizeof(cplx) * nspec);
    if (!G) return 3;
    memcpy(G, F_in, sizeof(cplx) * nspec);
    int err = fft_lines(G, Nx, Ny * Nzh, Ny * Nzh, Ny * Nzh, 1, 0, +1, nthreads);
    if (!err) err = fft_lines(G, Ny, Nzh, Nx * Nzh, Nzh, 1, Ny * Nzh, +1, nthreads);
    if (err) { free(G); return err; }
    cplx *tw = make_twiddles(Nz, +1);
    if (!tw) { free(G); return 3; }
    const double scale = 1.0 / ((double)Nx * (double)Ny * (double)Nz);
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel num_threads(nthreads)
#endif
    {
        cplx *line = (cplx *)malloc(sizeof(cplx) * (size_t)Nz);
        cplx *res  = (cplx *)malloc(sizeof(cplx) * (size_t)Nz);
        cplx *tmp  = (cplx *)malloc(sizeof(cplx) * (size_t)Nz);
        if (!line || !res || !tmp) {
#ifdef _OPENMP
#pragma omp atomic write
#endif
            err = 3;
        } else {
#ifdef _OPENMP
#pragma omp for schedule(static)
#endif
            for (long row = 0; row < Nx * Ny; ++row) {
                const cplx *src = G + (size_t)row * Nzh;
                for (long k = 0; k < Nzh; ++k) line[k] = src[k];
                for (long k = Nzh; k < Nz; ++k) {          /* conj G(., ., Nz-kz) */
                    line[k].re =  src[Nz - k].re;
                    line[k].im = -src[Nz - k].im;
                }
                fft_rec(line, 1, res, Nz, tw, Nz, tmp);
                double *dst = f + (size_t)row * Nz;
                for (long j = 0; j < Nz; ++j) dst[j] = res[j].re * scale;   /* Re, 1/N */
            }
        }
        free(line); free(res); free(tmp);
    }
    free(tw);
    free(G);
    return err;
}

/* ------------------------------------------------------------------------------------
 * 5. Sampled oracles for grids whose full fp64 transform does not fit the host.
 *
 *    Forward pencil: for K chosen (ky,kz) pairs, all kx, straight from Eq. (1):
 *        g_c(jx) = sum_{jy,jz} f(jx,jy,jz) exp(-2 pi i [jy ky_c/Ny + jz kz_c/Nz])
 *        F(kx,ky_c,kz_c) = sum_{jx} g_c(jx) exp(-2 pi i jx kx/Nx)          (O(Nx^2))
 *    One streaming sweep over f serves all K pairs.  f may be fp32 (promoted, as the
 *    fp32 configs feed both sides the same rounded values) or fp64.
 *
 *    Inverse point: f(j) for chosen grid points straight from Eq. (2)+(3).  Pairing
 *    each kz > Nz/2 term with its mirror (the term at -k is the conjugate of the term
 *    at k) gives
 *        f(j) = 1/(NxNyNz) Re sum_{kx,ky,kz<=Nz/2} w(kz) F(k) exp(+2 pi i [...]),
 *        w = 1 for kz in {0, Nz/2}, 2 otherwise.
 *    (pinned against oracle_idft3d_direct in the tests).  `index` maps (kx,ky,kz) to
 *    the element offset in F so the sweep can read the product's slab layout in place:
 *        offset = ((q*Nx + kx)*(Ny/p) + ky%(Ny/p))*Nzh + kz, q = ky/(Ny/p)  (p=1: natural)
 * ---------------------------------------------------------------------------------- */
static int pencil_generic(const void *f, int is_f32, long Nx, long Ny, long Nz,
                          int K, const long *kys, const long *kzs,
                          double *out /* [K][Nx] complex */, int nthreads)
{
    cplx *ey = (cplx *)malloc(sizeof(cplx) * (size_t)K * Ny);
    cplx *ez = (cplx *)malloc(sizeof(cplx) * (size_t)K * Nz);
    cplx *g  = (cplx *)calloc((size_t)K * Nx, sizeof(cplx));
    if (!ey || !ez || !g) { free(ey); free(ez); free(g); return 3; }
    for (int c = 0; c < K; ++c) {
        for (long y = 0; y < Ny; ++y) ey[(size_t)c * Ny + y] = root_of_unity(y * kys[c], Ny, -1);
        for (long z = 0; z < Nz; ++z) ez[(size_t)c * Nz + z] = root_of_unity(z * kzs[c], Nz, -1);
    }
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
    for (long x = 0; x < Nx; ++x) {
        for (int c = 0; c < K; ++c) {
            long double gre = 0.0L, gim = 0.0L;
            for (long y = 0; y < Ny; ++y) {
                double rre = 0.0, rim = 0.0;
                const cplx *ezc = ez + (size_t)c * Nz;
                size_t base = ((size_t)x * Ny + y) * Nz;
                if (is_f32) {
                    const float *row = (const float *)f + base;
                    for (long z = 0; z < Nz; ++z) { rre += row[z] * ezc[z].re; rim += row[z] * ezc[z].im; }
                } else {
                    const double *row = (const double *)f + base;
                    for (long z = 0; z < Nz; ++z) { rre += row[z] * ezc[z].re; rim += row[z] * ezc[z].im; }
                }
                cplx e = ey[(size_t)c * Ny + y];
                gre += (long double)rre * e.re - (long double)rim * e.im;
                gim += (long double)rre * e.im + (long double)rim * e.re;
            }
            g[(size_t)c * Nx + x].re = (double)gre;
            g[(size_t)c * Nx + x].im = (double)gim;
        }
    }
    cplx *o = (cplx *)out;
    for (int c = 0; c < K; ++c)
        for (long kx = 0; kx < Nx; ++kx) {
            long double sre = 0.0L, sim = 0.0L;
            for (long x = 0; x < Nx; ++x) {
                cplx w = root_of_unity(x * kx, Nx, -1);
                cplx v = g[(size_t)c * Nx + x];
                sre += (long double)v.re * w.re - (long double)v.im * w.im;
                sim += (long double)v.re * w.im + (long double)v.im * w.re;
            }
            o[(size_t)c * Nx + kx].re = (double)sre;
            o[(size_t)c * Nx + kx].im = (double)sim;
        }
    free(ey); free(ez); free(g);
    return 0;
}

int oracle_r2c_pencils_f64(const double *f, long Nx, long Ny, long Nz, int K,
                           const long *kys, const long *kzs, double *out, int nthreads)
{ return pencil_generic(f, 0, Nx, Ny, Nz, K, kys, kzs, out, nthreads); }

int oracle_r2c_pencils_f32(const float *f, long Nx, long Ny, long Nz, int K,
                           const long *kys, const long *kzs, double *out, int nthreads)
{ return pencil_generic(f, 1, Nx, Ny, Nz, K, kys, kzs, out, nthreads); }

static int points_generic(const void *F, int is_f32, long Nx, long Ny, long Nz, long p,
                          int K, const long *jxs, const long *jys, const long *jzs,
                          double *out /* [K] */, int nthreads)
{
    if (p < 1 || Ny % p) return 1;
    const long Nzh = Nz / 2 + 1, L = Ny / p;
    cplx *ex = (cplx *)malloc(sizeof(cplx) * (size_t)K * Nx);
    cplx *ey = (cplx *)malloc(sizeof(cplx) * (size_t)K * Ny);
    cplx *ez = (cplx *)malloc(sizeof(cplx) * (size_t)K * Nzh);
    long double *acc = (long double *)calloc((size_t)K * Nx, sizeof(long double));
    if (!ex || !ey || !ez || !acc) { free(ex); free(ey); free(ez); free(acc); return 3; }
    for (int c = 0; c < K; ++c) {
        for (long k = 0; k < Nx; ++k) ex[(size_t)c * Nx + k] = root_of_unity(k * jxs[c], Nx, +1);
        for (long k = 0; k < Ny; ++k) ey[(size_t)c * Ny + k] = root_of_unity(k * jys[c], Ny, +1);
        for (long k = 0; k < Nzh; ++k) {
            cplx w = root_of_unity(k * jzs[c], Nz, +1);
            double wt = (k == 0 || 2 * k == Nz) ? 1.0 : 2.0;
            w.re *= wt; w.im *= wt;
            ez[(size_t)c * Nzh + k] = w;
        }
    }
#ifdef _OPENMP
    if (nthreads < 1) nthreads = 1;
#pragma omp parallel for schedule(static) num_threads(nthreads)
#endif
    for (long kx = 0; kx < Nx; ++kx) {
        for (int c = 0; c < K; ++c) {
            long double sx = 0.0L;                 /* Re of the (ky,kz) sum times e^{i kx jx} */
            long double pre = 0.0L, pim = 0.0L;
            for (long ky = 0; ky < Ny; ++ky) {
                size_t base = (((size_t)(ky / L) * Nx + kx) * L + (ky % L)) * Nzh;
                double rre = 0.0, rim = 0.0;
                const cplx *ezc = ez + (size_t)c * Nzh;
                if (is_f32) {
                    const float *row = (const float *)F + 2 * base;
                    for (long kz = 0; kz < Nzh; ++kz) {
                        double a = row[2 * kz], b = row[2 * kz + 1];
                        rre += a * ezc[kz].re - b * ezc[kz].im;
                        rim += a * ezc[kz].im + b * ezc[kz].re;
                    }
                } else {
                    const double *row = (const double *)F + 2 * base;
                    for (long kz = 0; kz < Nzh; ++kz) {
                        double a = row[2 * kz], b = row[2 * kz + 1];
                        rre += a * ezc[kz].re - b * ezc[kz].im;
                        rim += a * ezc[kz].im + b * ezc[kz].re;
                    }
                }
                cplx e = ey[(size_t)c * Ny + ky];
                pre += (long double)rre * e.re - (long double)rim * e.im;
                pim += (long double)rre * e.im + (long double)rim * e.re;
            }
            cplx e = ex[(size_t)c * Nx + kx];
            sx = pre * e.re - pim * e.im;
            acc[(size_t)c * Nx + kx] = sx;
        }
    }
    const long double den = (long double)Nx * Ny * Nz;
    for (int c = 0; c < K; ++c) {
        long double s = 0.0L;
        for (long kx = 0; kx < Nx; ++kx) s += acc[(size_t)c * Nx + kx];
        out[c] = (double)(s / den);
    }
    free(ex); free(ey); free(ez); free(acc);
    return 0;
}

int oracle_c2r_points_f64(const double *F, long Nx, long Ny, long Nz, long p, int K,
                          const long *jxs, const long *jys, const long *jzs, double *out, int nthreads)
{ return points_generic(F, 0, Nx, Ny, Nz, p, K, jxs, jys, jzs, out, nthreads); }

int oracle_c2r_points_f32(const float *F, long Nx, long Ny, long Nz, long p, int K,
                          const long *jxs, const long *jys, const long *jzs, double *out, int nthreads)
{ return points_generic(F, 1, Nx, Ny, Nz, p, K, jxs, jys, jzs, out, nthreads); }

/* ------------------------------------------------------------------------------------
 * 6. 3D complex-to-complex transform (the paper's library shares one
 *    workspace between R2C, C2C and C2R).  sign = -1: forward, unnormalised,
 *    F(k) = sum_j f(j) exp(-2 pi i [jx kx/Nx + jy ky/Ny + jz kz/Nz]) (Eq. (1) with complex f,
 *    all kz); sign = +1: inverse, scaled by 1/(NxNyNz) (Eq. (2) with the convention of
 *    reading R1).  oracle_dft3d_c2c_direct is that definition summed term by term,
 *    O(N^6); oracle_c2c is the separable evaluation (z, y, x lines; x, y, z for the
 *    inverse) with the recursive mixed-radix 1D transform above.
 * ---------------------------------------------------------------------------------- */
int oracle_dft3d_c2c_direct(const double *f_in, int Nx, int Ny, int Nz, int sign, double *F_out)
{
    const cplx *f = (const cplx *)f_in;
    cplx *F = (cplx *)F_out;
    if (sign != 1 && sign != -1) return 1;
    const long double scale = sign > 0 ? 1.0L / ((long double)Nx * Ny * Nz) : 1.0L;
    for (int kx = 0; kx < Nx; ++kx)
    for (int ky = 0; ky < Ny; ++ky)
    for (int kz = 0; kz < Nz; ++kz) {
        long double sre = 0.0L, sim = 0.0L;
        for (int jx = 0; jx < Nx; ++jx)
        for (int jy = 0; jy < Ny; ++jy)
        for (int jz = 0; jz < Nz; ++jz) {
            long long den = (long long)Nx * Ny * Nz;
            long long num = (long long)jx * kx * ((long long)Ny * Nz)
                          + (long long)jy * ky * ((long long)Nx * Nz)
                          + (long long)jz * kz * ((long long)Nx * Ny);
            cplx w = root_of_unity(num, den, sign);
            cplx v = f[((size_t)jx * Ny + jy) * Nz + jz];
            sre += (long double)v.re * w.re - (long double)v.im * w.im;
            sim += (long double)v.re * w.im + (long double)v.im * w.re;
        }
        cplx r = { (double)(sre * scale), (double)(sim * scale) };
        F[((size_t)kx * Ny + ky) * Nz + kz] = r;
    }
    return 0;
}

int oracle_c2c(const double *in, long Nx, long Ny, long Nz, int sign, double *out, int nthreads)
{
    if (Nx < 1 || Ny < 1 || Nz < 1 || (sign != 1 && sign != -1)) return 1;
    cplx *a = (cplx *)out;
    const size_t n = (size_t)Nx * Ny * Nz;
    memcpy(a, in, n * sizeof(cplx));
    int err;
    if (sign < 0) {
        /* z rows, then y lines (stride Nz), then x lines (stride Ny*Nz): paper steps 1 and 5 */
        err = fft_lines(a, Nz, 1, Nx * Ny, Nx * Ny, Nz, 0, sign, nthreads);
        if (!err) err = fft_lines(a, Ny, Nz, Nx * Nz, Nz, 1, Ny * Nz, sign, nthreads);
        if (!err) err = fft_lines(a, Nx, Ny * Nz, Ny * Nz, Ny * Nz, 1, 0, sign, nthreads);
    } else {
        /* reverse order */
        err = fft_lines(a, Nx, Ny * Nz, Ny * Nz, Ny * Nz, 1, 0, sign, nthreads);
        if (!err) err = fft_lines(a, Ny, Nz, Nx * Nz, Nz, 1, Ny * Nz, sign, nthreads);
        if (!err) err = fft_lines(a, Nz, 1, Nx * Ny, Nx * Ny, Nz, 0, sign, nthreads);
        if (!err) {
            const double sc = 1.0 / ((double)Nx * (double)Ny * (double)Nz);
            for (size_t i = 0; i < n; ++i) { a[i].re *= sc; a[i].im *= sc; }
        }
    }
    return err;
}

int oracle_max_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
