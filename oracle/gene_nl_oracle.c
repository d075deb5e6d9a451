/*
 * gene_nl_oracle.c -- CPU ORACLE for the GENE ExB nonlinearity.  TEST INFRASTRUCTURE ONLY.
 *
 * This file is the slow, plain, obviously-correct statement of what the hot path computes.
 * It shares NO code with the CUDA path (paper_1310_1485_b200/csrc) and must never be called
 * from the product path: only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may use it.
 *
 * What is computed (sect. 2.1): "the usual approach [14] to avoid the
 * computationally expensive convolutions in spectral space by multiplication of the two fields
 * corresponding to the quadratic term in real space after Fourier transforming them.  [...] the
 * fields are preprocessed ([...] extension [...] for dealiasing according to the 3/2-rule) [...]
 * and a fast Fourier transform to real space is applied.  After multiplication the result is
 * transformed back to the spectral representation, the additional modes are deleted, [...]
 * multiplied with a prefactor, and is finally added to the right-hand side vector."
 * The operator, layout and sizes are BASELINE.json north_star's flux-tube variant (spectral in kx
 * AND ky, 2-D transforms, derivatives formed from g and chi): SURVEY.md sect. 8(c), readings R1-R16.
 *
 * Two independent routes are given:
 *   (1) oracle_nl_convolution_*  -- THE DEFINITION: the truncated spectral convolution
 *         N(a,b) = sum_{k'+k''=k; k',k'' in K} (ky' kx'' - kx' ky'') chi(k') g(k'')
 *       which the pseudo-spectral method reaches exactly up to rounding (3/2 rule, ref. [14],
 *       PAPER.md:202).  O(M^2) per plane; used for tiny grids and for sampled output modes.
 *   (2) oracle_nl_pseudospectral -- the algorithm of PAPER.md:61 step by step in the paper's order
 *       (derivative, pad, to real space, multiply, back, delete modes, prefactor, add to rhs),
 *       with either a naive O(N^2) DFT or a plain recursive radix-2/3 FFT as the 1-D transform.
 * Route (2) is pinned to route (1), and both to closed forms / invariants, in tests/test_oracle_*.py
 * (pins P1-P9 of SURVEY.md sect. 8(c)).  Nothing here is "parity unpinned".
 *
 * Layout (BASELINE.json configs[0]): a plane is nx0*nky0 complex128, kx fastest:
 *   F[i + nx0*j], i = kx index (0..nx0-1), j = ky index (0..nky0-1).
 *   kx_i = kxmin*i (i < nx0/2), kxmin*(i-nx0) (i > nx0/2); row i = nx0/2 is the Nyquist row: it is
 *   IGNORED on input and left UNTOUCHED in rhs (reading R6).  ky_j = kymin*j, ky<0 implied by reality.
 * Padded real grid: Nx = 3*nx0/2, Ny = 3*nky0 (reading R8).
 *
 * Build: gcc -O2 -fopenmp -shared -fPIC (see oracle/gene_nl_oracle.py).  All arithmetic is FP64
 * (the paper's S_c = 16 B double-complex); twiddles are formed in long double.
 */
#include <complex.h>
#include <math.h>
#include <stdlib.h>
#include <string.h>

typedef double complex cplx;

#define ORACLE_DFT_NAIVE 0
#define ORACLE_DFT_RECURSIVE 1

/* Table of the n-th roots of unity, w[t] = exp(sign * 2*pi*i * t/n), t = 0..n-1, formed in
 * long double so that every entry is the correctly rounded double (no recurrences). */
static cplx *root_table(int n, int sign)
{
    cplx *w = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    for (int t = 0; t < n; ++t) {
        long double ang = 2.0L * 3.14159265358979323846264338327950288L * (long double)t / (long double)n;
        w[t] = (double)cosl(ang) + I * (double)(sign * sinl(ang));
    }
    return w;
}

/* ---- 1-D DFT, naive: out[k] = sum_j in[j*istride] * W^{j k}, W = exp(sign*2*pi*i/n), given as
 *      w[t*wstride] = W^t.  Unnormalised.  This is the textbook definition. ---- */
static void dft_naive_w(int n, const cplx *w, int wstride, const cplx *in, int istride, cplx *out)
{
    for (int k = 0; k < n; ++k) {
        cplx acc = 0.0;
        for (int j = 0; j < n; ++j)
            acc += in[(long)j * istride] * w[(((long)j * k) % n) * wstride];
        out[k] = acc;
    }
}

/* ---- 1-D DFT, plain recursive decimation in time: split by 2 if even, by 3 if divisible by 3,
 *      naive otherwise.  Same definition as the naive routine; checked against it (pin P9).
 *      w[t*wstride] = exp(sign*2*pi*i*t/n) for the CURRENT n. ---- */
static void dft_recursive_w(int n, const cplx *w, int wstride, const cplx *in, int istride, cplx *out)
{
    int r = (n % 2 == 0) ? 2 : (n % 3 == 0) ? 3 : 0;
    if (r == 0 || n <= 3) {
        dft_naive_w(n, w, wstride, in, istride, out);
        return;
    }
    int m = n / r;
    cplx *sub = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    for (int q = 0; q < r; ++q) /* sub-sequence x[r*t + q], t = 0..m-1; its root table has stride r */
        dft_recursive_w(m, w, wstride * r, in + (long)q * istride, istride * r, sub + (long)q * m);
    for (int k = 0; k < n; ++k) { /* X[k] = sum_q W_n^{q k} * Sub_q[k mod m] */
        cplx acc = 0.0;
        for (int q = 0; q < r; ++q)
            acc += w[(((long)q * k) % n) * wstride] * sub[(long)q * m + (k % m)];
        out[k] = acc;
    }
    free(sub);
}

/* one 1-D transform with a root table w of the same length n */
static void dft1d(int backend, int n, const cplx *w, const cplx *in, int istride, cplx *out)
{
    if (backend == ORACLE_DFT_NAIVE)
        dft_naive_w(n, w, 1, in, istride, out);
    else
        dft_recursive_w(n, w, 1, in, istride, out);
}

/* exported wrapper so tests can pin the two 1-D routines against each other and against numpy */
void oracle_dft(int backend, int n, int sign, const double *in_ri, double *out_ri)
{
    cplx *w = root_table(n, sign);
    dft1d(backend, n, w, (const cplx *)in_ri, 1, (cplx *)out_ri);
    free(w);
}

/* 2-D DFT of a row-major [n0][n1] array (n1 fastest), in place, row-column. */
static void dft2d(int backend, int n0, int n1, int sign, cplx *a)
{
    int nmax = n0 > n1 ? n0 : n1;
    cplx *tmp = (cplx *)malloc(sizeof(cplx) * (size_t)nmax);
    cplx *w0 = root_table(n0, sign), *w1 = root_table(n1, sign);
    for (int i = 0; i < n0; ++i) { /* along n1 */
        dft1d(backend, n1, w1, a + (long)i * n1, 1, tmp);
        memcpy(a + (long)i * n1, tmp, sizeof(cplx) * (size_t)n1);
    }
    for (int j = 0; j < n1; ++j) { /* along n0 */
        dft1d(backend, n0, w0, a + j, n1, tmp);
        for (int i = 0; i < n0; ++i) a[(long)i * n1 + j] = tmp[i];
    }
    free(tmp); free(w0); free(w1);
}

static double kx_of(int i, int nx0, double kxmin)
{
    if (i < nx0 / 2) return kxmin * i;
    if (i == nx0 / 2) return 0.0; /* Nyquist: wavenumber 0 and data ignored (R6) */
    return kxmin * (i - nx0);
}

/* Steps 1-3 of SURVEY 8(c): real-space field of d/dx (which=0) or d/dy (which=1) of F.
 * out[m*Ny + n], m = x index, n = y index; work is an Nx*Ny complex scratch. */
static void derivative_to_real(int backend, int nx0, int nky0, double kxmin, double kymin,
                               const cplx *F, int which, cplx *work, double *out)
{
    const int Nx = 3 * nx0 / 2, Ny = 3 * nky0;
    memset(work, 0, sizeof(cplx) * (size_t)Nx * Ny);
    for (int j = 0; j < nky0; ++j) {
        for (int i = 0; i < nx0; ++i) {
            if (i == nx0 / 2) continue;
            double k = which == 0 ? kx_of(i, nx0, kxmin) : kymin * j;
            cplx D = (I * k) * F[i + (long)nx0 * j];          /* step 1: i*k*F            */
            int ip = i < nx0 / 2 ? i : i + (Nx - nx0);         /* step 2: 3/2 zero padding */
            work[(long)ip * Ny + j] = D;
            if (j >= 1) work[(long)((Nx - ip) % Nx) * Ny + (Ny - j)] = conj(D); /* reality */
        }
    }
    dft2d(backend, Nx, Ny, +1, work);                          /* step 3: synthesis e^{+i...} */
    for (long t = 0; t < (long)Nx * Ny; ++t) out[t] = creal(work[t]); /* real part (R7)      */
}

/* ---- Route (2): one plane, pseudo-spectral, PAPER.md:61 order.  rhs is updated in place. ---- */
void oracle_nl_pseudospectral_plane(int backend, int nx0, int nky0, double kxmin, double kymin,
                                    const double *chi_ri, const double *g_ri, double *rhs_ri,
                                    double scale)
{
    const int Nx = 3 * nx0 / 2, Ny = 3 * nky0;
    const cplx *X = (const cplx *)chi_ri, *G = (const cplx *)g_ri;
    cplx *rhs = (cplx *)rhs_ri;
    size_t npts = (size_t)Nx * Ny;
    cplx *work = (cplx *)malloc(sizeof(cplx) * npts);
    double *dxX = (double *)malloc(sizeof(double) * npts), *dyX = (double *)malloc(sizeof(double) * npts);
    double *dxG = (double *)malloc(sizeof(double) * npts), *dyG = (double *)malloc(sizeof(double) * npts);

    derivative_to_real(backend, nx0, nky0, kxmin, kymin, X, 0, work, dxX);
    derivative_to_real(backend, nx0, nky0, kxmin, kymin, X, 1, work, dyX);
    derivative_to_real(backend, nx0, nky0, kxmin, kymin, G, 0, work, dxG);
    derivative_to_real(backend, nx0, nky0, kxmin, kymin, G, 1, work, dyG);

    for (size_t t = 0; t < npts; ++t)                          /* step 4: the bracket        */
        work[t] = dxX[t] * dyG[t] - dyX[t] * dxG[t];

    dft2d(backend, Nx, Ny, -1, work);                          /* step 5: analysis e^{-i...} */
    const double norm = 1.0 / ((double)Nx * (double)Ny);

    for (int j = 0; j < nky0; ++j)                             /* step 6: delete modes, prefactor, add */
        for (int i = 0; i < nx0; ++i) {
            if (i == nx0 / 2) continue;
            int ip = i < nx0 / 2 ? i : i + (Nx - nx0);
            rhs[i + (long)nx0 * j] += scale * (norm * work[(long)ip * Ny + j]);
        }
    free(work); free(dxX); free(dyX); free(dxG); free(dyG);
}

/* Batched route (2), OpenMP over planes only.  chi_index[p] selects the chi plane used by g plane p
 * (chi has no v dependence when chi_has_v = 0: several g planes share one chi plane). */
void oracle_nl_pseudospectral(int backend, int nx0, int nky0, double kxmin, double kymin,
                              long nplanes, const double *chi_ri, const long *chi_index,
                              const double *g_ri, double *rhs_ri, double scale)
{
    const long M2 = 2L * nx0 * nky0;
#pragma omp parallel for schedule(dynamic, 1)
    for (long p = 0; p < nplanes; ++p)
        oracle_nl_pseudospectral_plane(backend, nx0, nky0, kxmin, kymin,
                                       chi_ri + chi_index[p] * M2, g_ri + p * M2, rhs_ri + p * M2, scale);
}

/* ---- Route (1): the definition.  Extended spectrum value at signed mode (a,b), |a|<=nx0/2-1,
 *      |b|<=nky0-1, from the stored half plane: b>0 stored; b<0 conj of stored(-a,-b); b=0 the
 *      Hermitian part (F(a,0)+conj F(-a,0))/2, which equals the stored value on Hermitian-
 *      consistent input and is what "real part of the synthesis" (R7) means otherwise. ---- */
static cplx ext_mode(const cplx *F, int nx0, int a, int b)
{
    int ia = a >= 0 ? a : a + nx0, ina = a > 0 ? nx0 - a : -a;
    if (b > 0) return F[ia + (long)nx0 * b];
    if (b < 0) return conj(F[ina + (long)nx0 * (-b)]);
    return 0.5 * (F[ia] + conj(F[ina]));
}

/* N(a,b) for one retained mode (signed a, b >= 0) by direct summation over all pairs in K. */
static cplx convolution_mode(int nx0, int nky0, double kxmin, double kymin,
                             const cplx *X, const cplx *G, int a, int b)
{
    const int amax = nx0 / 2 - 1, bmax = nky0 - 1;
    cplx acc = 0.0;
    for (int b1 = -bmax; b1 <= bmax; ++b1) {
        int b2 = b - b1;
        if (b2 < -bmax || b2 > bmax) continue;
        for (int a1 = -amax; a1 <= amax; ++a1) {
            int a2 = a - a1;
            if (a2 < -amax || a2 > amax) continue;
            double kx1 = kxmin * a1, ky1 = kymin * b1, kx2 = kxmin * a2, ky2 = kymin * b2;
            double C = ky1 * kx2 - kx1 * ky2; /* from (i kx')(i ky'') - (i ky')(i kx'') */
            acc += C * ext_mode(X, nx0, a1, b1) * ext_mode(G, nx0, a2, b2);
        }
    }
    return acc;
}

/* Whole plane by the definition: out[i + nx0*j] = N(a(i), j); Nyquist row set to 0. */
void oracle_nl_convolution_plane(int nx0, int nky0, double kxmin, double kymin,
                                 const double *chi_ri, const double *g_ri, double *out_ri)
{
    cplx *out = (cplx *)out_ri;
#pragma omp parallel for schedule(dynamic, 1)
    for (int j = 0; j < nky0; ++j)
        for (int i = 0; i < nx0; ++i) {
            if (i == nx0 / 2) { out[i + (long)nx0 * j] = 0.0; continue; }
            int a = i < nx0 / 2 ? i : i - nx0;
            out[i + (long)nx0 * j] = convolution_mode(nx0, nky0, kxmin, kymin,
                                                      (const cplx *)chi_ri, (const cplx *)g_ri, a, j);
        }
}

/* Sampled outputs by the definition: nmodes stored indices (i_idx[t], j_idx[t]) of one plane. */
void oracle_nl_convolution_modes(int nx0, int nky0, double kxmin, double kymin,
                                 const double *chi_ri, const double *g_ri,
                                 int nmodes, const int *i_idx, const int *j_idx, double *out_ri)
{
    cplx *out = (cplx *)out_ri;
#pragma omp parallel for schedule(dynamic, 1)
    for (int t = 0; t < nmodes; ++t) {
        int i = i_idx[t], j = j_idx[t];
        if (i == nx0 / 2) { out[t] = 0.0; continue; }
        int a = i < nx0 / 2 ? i : i - nx0;
        out[t] = convolution_mode(nx0, nky0, kxmin, kymin, (const cplx *)chi_ri, (const cplx *)g_ri, a, j);
    }
}

/* =====================================================================================================
 * x-GLOBAL VARIANT -- the operator the paper itself ran and timed.
 *
 * PAPER.md:39 (sect. 2): GENE's x-global version is spectral in y only; "the fields are
 * preprocessed (transposition, extension in y direction for dealiasing according to the 3/2-rule) in a
 * first step, and a fast Fourier transform to real space is applied.  After multiplication the result is
 * transformed back to the spectral representation, the additional modes are deleted, the array is
 * transposed and multiplied with a prefactor, and is finally added to the right-hand side vector."
 * "The nonlinear term needs as input four arrays, the x and y component of the ExB-velocity
 * and the derivatives of the distribution function with respect to x and y.  Additionally it needs the
 * already computed right-hand side" (5 planes in, 1 out: intensity 1/6).
 *
 * A plane is nx*nky0 complex128, x fastest: F[x + nx*j], x a REAL-SPACE point, j the ky index
 * (ky >= 0; ky < 0 implied by reality of the field; Im F[x,0] is ignored, as in reading R7).
 * Per plane and per x:   N(x,y) = vex(x,y)*dxg(x,y) + vey(x,y)*dyg(x,y)   (v_E . grad g) on the padded
 * real grid Ny = 3*nky0, and   rhs[x,j] += scale * pref[x] * N^(x,j),  j < nky0,  N^ = (1/Ny) sum_y N e^{-i..}.
 * Readings (the paper gives no formulas): the sign and any metric factor live in pref/scale; pref is a
 * real array over x ("prefactor", x-dependent in an x-global code); Ny = 3*nky0 as in R8.
 * Two routes, as above: the definition (truncated convolution over ky) and the algorithm step by step.
 * ===================================================================================================== */

/* Hermitian extension in ky of the stored half-spectrum at one x: b in (-nky0, nky0) */
static cplx extx_mode(const cplx *F, int nx, int x, int b)
{
    if (b == 0) return creal(F[x]);
    if (b > 0) return F[x + (long)nx * b];
    return conj(F[x + (long)nx * (-b)]);
}

/* (1) THE DEFINITION: N^(x,k) = sum_{k'+k''=k, |k'|,|k''| < nky0} [vex(k') dxg(k'') + vey(k') dyg(k'')] */
void oracle_nlx_convolution_plane(int nx, int nky0, const double *vex_ri, const double *vey_ri,
                                  const double *dxg_ri, const double *dyg_ri, double *out_ri)
{
    const cplx *vex = (const cplx *)vex_ri, *vey = (const cplx *)vey_ri;
    const cplx *dxg = (const cplx *)dxg_ri, *dyg = (const cplx *)dyg_ri;
    cplx *out = (cplx *)out_ri;
    for (int x = 0; x < nx; ++x)
        for (int k = 0; k < nky0; ++k) {
            cplx acc = 0.0;
            for (int k1 = -(nky0 - 1); k1 <= nky0 - 1; ++k1) {
                int k2 = k - k1;
                if (k2 <= -nky0 || k2 >= nky0) continue;
                acc += extx_mode(vex, nx, x, k1) * extx_mode(dxg, nx, x, k2) +
                       extx_mode(vey, nx, x, k1) * extx_mode(dyg, nx, x, k2);
            }
            out[x + (long)nx * k] = acc;
        }
}

/* to real space at one x: extension to Ny = 3 nky0 (zero modes added), synthesis e^{+i ky y}, real part */
static void nlx_to_real(int backend, int nx, int nky0, int Ny, const cplx *wp, const cplx *F, int x,
                        cplx *S, cplx *T, double *f)
{
    for (int j = 0; j < Ny; ++j) S[j] = 0.0;
    for (int j = 0; j < nky0; ++j) {
        S[j] = F[x + (long)nx * j];
        if (j >= 1) S[Ny - j] = conj(F[x + (long)nx * j]);
    }
    dft1d(backend, Ny, wp, S, 1, T);
    for (int n = 0; n < Ny; ++n) f[n] = creal(T[n]);
}

/* (2) THE ALGORITHM of PAPER.md:61, plane by plane (OpenMP over planes) */
void oracle_nlx_pseudospectral(int backend, int nx, int nky0, long planes, const double *vex_ri,
                               const double *vey_ri, const double *dxg_ri, const double *dyg_ri,
                               const double *pref, double *rhs_ri, double scale)
{
    const int Ny = 3 * nky0;
    const long M = (long)nx * nky0;
    cplx *wp = root_table(Ny, +1), *wm = root_table(Ny, -1);
#pragma omp parallel
    {
        cplx *S = (cplx *)malloc(sizeof(cplx) * (size_t)Ny), *T = (cplx *)malloc(sizeof(cplx) * (size_t)Ny);
        double *a = (double *)malloc(sizeof(double) * (size_t)Ny * 4);
#pragma omp for schedule(static)
        for (long p = 0; p < planes; ++p) {
            const cplx *vex = (const cplx *)vex_ri + p * M, *vey = (const cplx *)vey_ri + p * M;
            const cplx *dxg = (const cplx *)dxg_ri + p * M, *dyg = (const cplx *)dyg_ri + p * M;
            cplx *rhs = (cplx *)rhs_ri + p * M;
            for (int x = 0; x < nx; ++x) {
                nlx_to_real(backend, nx, nky0, Ny, wp, vex, x, S, T, a);
                nlx_to_real(backend, nx, nky0, Ny, wp, vey, x, S, T, a + Ny);
                nlx_to_real(backend, nx, nky0, Ny, wp, dxg, x, S, T, a + 2 * Ny);
                nlx_to_real(backend, nx, nky0, Ny, wp, dyg, x, S, T, a + 3 * Ny);
                for (int n = 0; n < Ny; ++n) /* multiplication in real space */
                    S[n] = a[n] * a[2 * Ny + n] + a[Ny + n] * a[3 * Ny + n];
                dft1d(backend, Ny, wm, S, 1, T);                /* back to the spectral representation */
                for (int j = 0; j < nky0; ++j)                  /* additional modes deleted, prefactor, add */
                    rhs[x + (long)nx * j] += scale * pref[x] * (T[j] / (double)Ny);
            }
        }
        free(S); free(T); free(a);
    }
    free(wp); free(wm);
}
