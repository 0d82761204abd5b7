/*
 * oracle/snref.c -- float64 CPU ORACLE for the Strang split-step Fourier step of the
 * generalized Schroedinger-Newton system.
 *
 * THIS IS TEST INFRASTRUCTURE, NOT THE PRODUCT.  Only tests/, __graft_entry__.smoke() and
 * bench.py's cpu_baseline / --impl reference legs may load it.  It shares no code, header,
 * table or helper with the CUDA path (paper_1909_08354_b200/csrc), and the CUDA path never
 * calls it.  It is deliberately plain and slow: full complex transforms everywhere, its own
 * radix-2 FFT (plus one radix-3 split for N = 3*2^m), one operator at a time in the order the
 * method states, OpenMP over independent lines only.
 *
 * What it computes (section II eq. (1),(2)):
 *      i dpsi/dtau = A lap psi + B phi psi + G(|psi|^2) psi          (1)
 *      lap phi + C phi = D |psi|^2                                    (2)
 * on a periodic d-dimensional box (d = 2,3), advanced by the "Symmetric Split-Step Fourier
 * Method" with eq. (2) "also solved with spectral methods" (section III).
 *
 * The paper states the method by name only; the operator forms below are BASELINE.json's
 * north_star and SURVEY.md 8(c) readings Q1-Q10 (listed in DESIGN.md):
 *      grid   N_a points, h_a = L_a/N_a, dV = prod h_a
 *      k_a[j] = (2 pi/L_a) (j < N_a/2 ? j : j - N_a),   k^2 = sum_a k_a^2
 *      K(s):  psi^ = FFT(psi);  psi^ *= exp(+i A k^2 s);  psi = IFFT(psi^)          [Q2]
 *      N(s):  rho = |psi|^2;  rho^ = FFT(rho);  phi^ = D rho^/(C - k^2) for every mode,
 *             if C == 0: phi^[k=0] = 0;  phi = Re IFFT(phi^);                         [Q4]
 *             psi *= exp(-i s (B phi + sum_j g_j rho^j))                             [Q3,Q6]
 *      step:  K(dtau/2); N(dtau); K(dtau/2)                                          [Q1]
 * FFT convention [Q8]: forward sum_j x_j e^{-2 pi i jk/N}; inverse carries 1/N.
 * Diagnostics [Q10]: norm = sum |psi|^2 dV;
 *      H = -A sum_k k^2 |psi^_k|^2 dV/prod N + (B/2) sum phi rho dV + sum F(rho) dV,
 *      F(rho) = sum_j g_j rho^(j+1)/(j+1).
 * NEXT-1 extension (eq. (15),(16)): G may also carry g_log ln(rho) + g_pow rho^p
 * (pressure potential) and the N phase a fixed external potential V(x) (phi_C); e_local then
 * includes their energies sum (F(rho) + V rho) dV.
 *
 * Pins (tests/test_oracle_pins.py, -m "not gpu"): brute-force DFT, plane wave, free and
 * boosted Gaussian closed forms, single-mode Poisson/Helmholtz, norm conservation, Strang
 * order 2, time reversal, NLS bright soliton, 2D<->3D reduction, translation covariance,
 * momentum and energy.  Every exported function is pinned by at least one of them.
 */
#include <complex.h>
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define SNREF_OK 0
#define SNREF_ERR_NULL -1
#define SNREF_ERR_DIMS -2
#define SNREF_ERR_PARAM -3
#define SNREF_ERR_SINGULAR -4
#define SNREF_ERR_STATE -6
#define SNREF_ERR_NOMEM -8

typedef double complex cplx;

typedef struct {
    double norm, e_kin, e_nonlocal, e_local, e_total;
} snref_diag;

typedef struct snref_ctx {
    int ndim;
    int64_t n[3];
    double L[3];
    double A, B, C, D;
    double g[4];
    int n_g;
    double dtau;
    int64_t cells;
    /* NEXT-1 terms of the local potential (eq. (15),(16)): pressure potential
     * w ln(rho) / (n w/(n-1)) rho^(n-1), and a fixed external potential phi_C(r) (eq. (11)) */
    double g_log, rho_floor, g_pow, p_pow;
    double *vext; /* NULL or cells doubles */
    /* modified Poisson source of eq. (12): lap phi + C phi = D (gamma(x) rho + beta(x) lap rho) */
    double *beta, *gamma; /* both NULL (plain eq. (2)) or both cells doubles */
    /* Bohm quantum potential of eq. (15): coefficient c_B (nu^2 there), V_B = lap sqrt(rho)/(2 sqrt(rho)),
     * with sqrt(rho) clamped from below by sqrt_floor in the denominator (reading Q17 of DESIGN.md) */
    double c_bohm, sqrt_floor;
    double *vb; /* scratch, cells doubles, allocated on first use */
    cplx *psi;   /* state */
    cplx *work;  /* rho^ / phi^ scratch */
    int has_state;
} snref_ctx;

/* ------------------------------------------------------------------ FFT */

static int is_pow2(int64_t n) { return n > 0 && (n & (n - 1)) == 0; }

/* length the oracle's FFT can do: 2^m or 3*2^m */
static int fft_len_ok(int64_t n)
{
    if (n < 1) return 0;
    if (is_pow2(n)) return 1;
    return (n % 3 == 0) && is_pow2(n / 3);
}

/* In-place iterative radix-2 decimation-in-time FFT, n = 2^m.  sign = -1 forward, +1 inverse
 * (no scaling).  Textbook Cooley-Tukey: bit-reversal permutation, then log2(n) butterfly
 * levels with twiddle e^{sign 2 pi i j/len} from cos/sin in double. */
static void fft_pow2(cplx *x, int64_t n, int sign)
{
    for (int64_t i = 1, j = 0; i < n; i++) {
        int64_t bit = n >> 1;
        for (; j & bit; bit >>= 1) j ^= bit;
        j ^= bit;
        if (i < j) { cplx t = x[i]; x[i] = x[j]; x[j] = t; }
    }
    for (int64_t len = 2; len <= n; len <<= 1) {
        int64_t half = len >> 1;
        for (int64_t start = 0; start < n; start += len) {
            for (int64_t j = 0; j < half; j++) {
                double ang = sign * 2.0 * M_PI * (double)j / (double)len;
                cplx w = cos(ang) + I * sin(ang);
                cplx u = x[start + j];
                cplx v = w * x[start + j + half];
                x[start + j] = u + v;
                x[start + j + half] = u - v;
            }
        }
    }
}

/* 1D transform of length n = 2^m or 3*2^m; buf holds n scratch entries.  For n = 3 m one
 * decimation-in-time split:  X[k + q m] = sum_{j=0..2} W_n^{j k} W_3^{j q} F_j[k],
 * F_j = FFT_m(x[3 i + j]),  W_n = e^{sign 2 pi i/n}. */
static void fft_line(cplx *x, int64_t n, int sign, cplx *buf)
{
    if (is_pow2(n)) { fft_pow2(x, n, sign); return; }
    int64_t m = n / 3;
    for (int j = 0; j < 3; j++)
        for (int64_t i = 0; i < m; i++) buf[j * m + i] = x[3 * i + j];
    for (int j = 0; j < 3; j++) fft_pow2(buf + j * m, m, sign);
    for (int64_t k = 0; k < m; k++) {
        for (int q = 0; q < 3; q++) {
            cplx acc = 0.0;
            for (int j = 0; j < 3; j++) {
                double ang = sign * 2.0 * M_PI * ((double)(j * k) / (double)n + (double)(j * q) / 3.0);
                acc += (cos(ang) + I * sin(ang)) * buf[j * m + k];
            }
            x[k + q * m] = acc;
        }
    }
}

/* d-dimensional transform in place: 1D line transforms along each axis in turn.
 * dir = +1 forward (e^{-i..}), dir = -1 inverse (e^{+i..}, scaled by 1/prod N). */
static int fftn(cplx *a, int ndim, const int64_t *n, int dir)
{
    int sign = dir > 0 ? -1 : +1;
    int64_t cells = 1;
    for (int d = 0; d < ndim; d++) cells *= n[d];
    for (int ax = 0; ax < ndim; ax++) {
        int64_t len = n[ax];
        int64_t stride = 1;
        for (int d = ax + 1; d < ndim; d++) stride *= n[d];
        int64_t nlines = cells / len;
        int fail = 0;
#pragma omp parallel
        {
            cplx *line = (cplx *)malloc(sizeof(cplx) * (size_t)len);
            cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)len);
            if (!line || !buf) {
#pragma omp atomic write
                fail = 1;
            }
#pragma omp for schedule(static)
            for (int64_t l = 0; l < nlines; l++) {
                if (!line || !buf) continue;
                int64_t outer = l / stride, inner = l % stride;
                cplx *base = a + outer * len * stride + inner;
                for (int64_t i = 0; i < len; i++) line[i] = base[i * stride];
                fft_line(line, len, sign, buf);
                for (int64_t i = 0; i < len; i++) base[i * stride] = line[i];
            }
            free(line);
            free(buf);
        }
        if (fail) return SNREF_ERR_NOMEM;
    }
    if (dir < 0) {
        double s = 1.0 / (double)cells;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < cells; i++) a[i] *= s;
    }
    return SNREF_OK;
}

/* exported for the brute-force DFT pin (V1) */
int snref_fft1d(cplx *x, int64_t n, int dir)
{
    if (!x) return SNREF_ERR_NULL;
    if (!fft_len_ok(n)) return SNREF_ERR_DIMS;
    cplx *buf = (cplx *)malloc(sizeof(cplx) * (size_t)n);
    if (!buf) return SNREF_ERR_NOMEM;
    fft_line(x, n, dir > 0 ? -1 : +1, buf);
    if (dir < 0)
        for (int64_t i = 0; i < n; i++) x[i] /= (double)n;
    free(buf);
    return SNREF_OK;
}

int snref_fftn(cplx *a, int ndim, const int64_t *dims, int dir)
{
    if (!a || !dims) return SNREF_ERR_NULL;
    if (ndim < 1 || ndim > 3) return SNREF_ERR_DIMS;
    for (int d = 0; d < ndim; d++)
        if (!fft_len_ok(dims[d])) return SNREF_ERR_DIMS;
    return fftn(a, ndim, dims, dir);
}

/* ------------------------------------------------------------------ grid helpers */

/* k_a[j] = (2 pi/L_a)(j < N_a/2 ? j : j - N_a) */
static double kval(int64_t j, int64_t n, double L)
{
    int64_t jj = (j < n / 2) ? j : j - n;
    return 2.0 * M_PI / L * (double)jj;
}

/* k^2 of the mode at flat index idx */
static double ksq_at(const snref_ctx *c, int64_t idx)
{
    double k2 = 0.0;
    for (int d = c->ndim - 1; d >= 0; d--) {
        int64_t j = idx % c->n[d];
        idx /= c->n[d];
        double k = kval(j, c->n[d], c->L[d]);
        k2 += k * k;
    }
    return k2;
}

/* G(rho) = sum_j g_j rho^j  +  g_log ln(rho_f)  +  g_pow rho_f^p,   rho_f = max(rho, rho_floor)
 * (polynomial: PAPER.md:54; logarithmic and power-law terms: V_pressure of eq. (16), PAPER.md:106;
 *  the floor is reading Q15 of DESIGN.md: the paper does not say how ln(0) is avoided) */
static double G_of(const snref_ctx *c, double rho)
{
    double s = 0.0, p = 1.0;
    for (int j = 0; j < c->n_g; j++) { p *= rho; s += c->g[j] * p; }
    if (c->g_log != 0.0 || c->g_pow != 0.0) {
        double rf = fmax(rho, c->rho_floor);
        if (c->g_log != 0.0) s += c->g_log * log(rf);
        if (c->g_pow != 0.0) s += c->g_pow * pow(rf, c->p_pow);
    }
    return s;
}

/* F(rho) with F' = G: sum_j g_j rho^(j+1)/(j+1) + g_log (rho ln rho_f - rho) + g_pow rho rho_f^p/(p+1) */
static double F_of(const snref_ctx *c, double rho)
{
    double s = 0.0, p = rho;
    for (int j = 0; j < c->n_g; j++) { p *= rho; s += c->g[j] * p / (double)(j + 2); }
    if (c->g_log != 0.0 || c->g_pow != 0.0) {
        double rf = fmax(rho, c->rho_floor);
        if (c->g_log != 0.0) s += c->g_log * (rho * log(rf) - rho);
        if (c->g_pow != 0.0) s += c->g_pow * rho * pow(rf, c->p_pow) / (c->p_pow + 1.0);
    }
    return s;
}

/* ------------------------------------------------------------------ life cycle */

int snref_create(snref_ctx **out, int ndim, const int64_t *dims, const double *L, double A, double B,
                 double C, double D, const double *g, int n_g, double dtau)
{
    if (!out || !dims || !L || (n_g > 0 && !g)) return SNREF_ERR_NULL;
    if (ndim != 2 && ndim != 3) return SNREF_ERR_DIMS;
    if (n_g < 0 || n_g > 4) return SNREF_ERR_PARAM;
    if (!isfinite(A) || !isfinite(B) || !isfinite(C) || !isfinite(D) || !isfinite(dtau)) return SNREF_ERR_PARAM;
    int64_t cells = 1;
    for (int d = 0; d < ndim; d++) {
        if (dims[d] < 2 || (dims[d] & 1) || !fft_len_ok(dims[d])) return SNREF_ERR_DIMS; /* Q9: even N only */
        if (!isfinite(L[d]) || L[d] <= 0.0) return SNREF_ERR_PARAM;
        cells *= dims[d];
    }
    for (int j = 0; j < n_g; j++)
        if (!isfinite(g[j])) return SNREF_ERR_PARAM;
    snref_ctx *c = (snref_ctx *)calloc(1, sizeof(snref_ctx));
    if (!c) return SNREF_ERR_NOMEM;
    c->ndim = ndim;
    for (int d = 0; d < ndim; d++) { c->n[d] = dims[d]; c->L[d] = L[d]; }
    c->A = A; c->B = B; c->C = C; c->D = D; c->n_g = n_g; c->dtau = dtau; c->cells = cells;
    c->rho_floor = 1e-30; c->p_pow = 1.0; c->sqrt_floor = 1e-30;
    for (int j = 0; j < n_g; j++) c->g[j] = g[j];
    /* Q5: C > 0 hitting a grid mode makes eq. (2) unsolvable */
    if (C > 0.0) {
        double tol = 1e-12 * fmax(1.0, fabs(C));
        for (int64_t i = 0; i < cells; i++) {
            if (fabs(C - ksq_at(c, i)) < tol) { free(c); return SNREF_ERR_SINGULAR; }
        }
    }
    c->psi = (cplx *)malloc(sizeof(cplx) * (size_t)cells);
    c->work = (cplx *)malloc(sizeof(cplx) * (size_t)cells);
    if (!c->psi || !c->work) { free(c->psi); free(c->work); free(c); return SNREF_ERR_NOMEM; }
    *out = c;
    return SNREF_OK;
}

/* G += g_log ln(max(rho, rho_floor)) + g_pow max(rho, rho_floor)^p_pow   (eq. (16)) */
int snref_set_local_terms(snref_ctx *c, double g_log, double rho_floor, double g_pow, double p_pow)
{
    if (!c) return SNREF_ERR_NULL;
    if (!isfinite(g_log) || !isfinite(rho_floor) || !isfinite(g_pow) || !isfinite(p_pow)) return SNREF_ERR_PARAM;
    if (rho_floor <= 0.0 || p_pow == -1.0) return SNREF_ERR_PARAM;
    c->g_log = g_log; c->rho_floor = rho_floor; c->g_pow = g_pow; c->p_pow = p_pow;
    return SNREF_OK;
}

/* fixed external potential V(x) (cells doubles, copied; NULL removes it): the N sub-step phase becomes
 * exp(-i s (B phi + G(rho) + V))   (phi_C of eq. (11),(15)) */
int snref_set_external_potential(snref_ctx *c, const double *v)
{
    if (!c) return SNREF_ERR_NULL;
    free(c->vext);
    c->vext = NULL;
    if (!v) return SNREF_OK;
    c->vext = (double *)malloc(sizeof(double) * (size_t)c->cells);
    if (!c->vext) return SNREF_ERR_NOMEM;
    memcpy(c->vext, v, sizeof(double) * (size_t)c->cells);
    return SNREF_OK;
}

static int bohm_potential(snref_ctx *c);

/* c_B V_B added to the N sub-step potential (eq. (15): c_B = nu^2); c_B = 0 switches it off */
int snref_set_bohm(snref_ctx *c, double c_bohm, double sqrt_floor)
{
    if (!c) return SNREF_ERR_NULL;
    if (!isfinite(c_bohm) || !isfinite(sqrt_floor) || sqrt_floor <= 0.0) return SNREF_ERR_PARAM;
    c->c_bohm = c_bohm; c->sqrt_floor = sqrt_floor;
    return SNREF_OK;
}

/* V_B of the current state (cells doubles); state unchanged */
int snref_bohm_potential(snref_ctx *c, double *out)
{
    if (!c || !out) return SNREF_ERR_NULL;
    if (!c->has_state) return SNREF_ERR_STATE;
    int rc = bohm_potential(c);
    if (rc) return rc;
    memcpy(out, c->vb, sizeof(double) * (size_t)c->cells);
    return SNREF_OK;
}

/* position-dependent source of eq. (12): lap phi + C phi = D (gamma(x) rho + beta(x) lap rho); tables are copied;
 * two NULLs restore eq. (2) (equivalent to gamma = 1, beta = 0) */
int snref_set_source_tables(snref_ctx *c, const double *beta, const double *gamma)
{
    if (!c) return SNREF_ERR_NULL;
    if ((beta == NULL) != (gamma == NULL)) return SNREF_ERR_NULL;
    free(c->beta); free(c->gamma);
    c->beta = c->gamma = NULL;
    if (!beta) return SNREF_OK;
    c->beta = (double *)malloc(sizeof(double) * (size_t)c->cells);
    c->gamma = (double *)malloc(sizeof(double) * (size_t)c->cells);
    if (!c->beta || !c->gamma) { free(c->beta); free(c->gamma); c->beta = c->gamma = NULL; return SNREF_ERR_NOMEM; }
    memcpy(c->beta, beta, sizeof(double) * (size_t)c->cells);
    memcpy(c->gamma, gamma, sizeof(double) * (size_t)c->cells);
    return SNREF_OK;
}

int snref_destroy(snref_ctx *c)
{
    if (!c) return SNREF_ERR_NULL;
    free(c->vb);
    free(c->beta);
    free(c->gamma);
    free(c->vext);
    free(c->psi);
    free(c->work);
    free(c);
    return SNREF_OK;
}

int snref_set_dtau(snref_ctx *c, double dtau)
{
    if (!c) return SNREF_ERR_NULL;
    if (!isfinite(dtau)) return SNREF_ERR_PARAM;
    c->dtau = dtau;
    return SNREF_OK;
}

int snref_set_state(snref_ctx *c, const cplx *psi)
{
    if (!c || !psi) return SNREF_ERR_NULL;
    memcpy(c->psi, psi, sizeof(cplx) * (size_t)c->cells);
    c->has_state = 1;
    return SNREF_OK;
}

int snref_get_state(snref_ctx *c, cplx *psi_out)
{
    if (!c || !psi_out) return SNREF_ERR_NULL;
    if (!c->has_state) return SNREF_ERR_STATE;
    memcpy(psi_out, c->psi, sizeof(cplx) * (size_t)c->cells);
    return SNREF_OK;
}

/* ------------------------------------------------------------------ operators */

/* K(s): psi^ = FFT(psi); psi^ *= exp(+i A k^2 s); psi = IFFT(psi^) */
static int kinetic(snref_ctx *c, double s)
{
    int rc = fftn(c->psi, c->ndim, c->n, +1);
    if (rc) return rc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) {
        double th = c->A * ksq_at(c, i) * s;
        c->psi[i] *= cos(th) + I * sin(th);
    }
    return fftn(c->psi, c->ndim, c->n, -1);
}

/* phi from the current psi into c->work (real part holds phi):
 * rho^ = FFT(|psi|^2); phi^ = D rho^/(C - k^2); C == 0: phi^[0] = 0; phi = Re IFFT(phi^) */
static int potential(snref_ctx *c)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) {
        double re = creal(c->psi[i]), im = cimag(c->psi[i]);
        c->work[i] = re * re + im * im;
    }
    int rc;
    if (c->beta) {
        /* source s = gamma rho + beta lap rho, lap rho spectrally: F^-1[-k^2 F[rho]]   (eq. (12)) */
        if ((rc = fftn(c->work, c->ndim, c->n, +1))) return rc;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < c->cells; i++) c->work[i] *= -ksq_at(c, i);
        if ((rc = fftn(c->work, c->ndim, c->n, -1))) return rc;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < c->cells; i++) {
            double re = creal(c->psi[i]), im = cimag(c->psi[i]);
            c->work[i] = c->gamma[i] * (re * re + im * im) + c->beta[i] * creal(c->work[i]);
        }
    }
    rc = fftn(c->work, c->ndim, c->n, +1);
    if (rc) return rc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) {
        if (c->C == 0.0 && i == 0) { c->work[i] = 0.0; continue; }
        c->work[i] = c->D * c->work[i] / (c->C - ksq_at(c, i));
    }
    rc = fftn(c->work, c->ndim, c->n, -1);
    if (rc) return rc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) c->work[i] = creal(c->work[i]);
    return SNREF_OK;
}

/* V_B = lap sqrt(rho) / (2 max(sqrt(rho), sqrt_floor)) into c->vb; lap taken spectrally: F^-1[-k^2 F[sqrt(rho)]] */
static int bohm_potential(snref_ctx *c)
{
    if (!c->vb) {
        c->vb = (double *)malloc(sizeof(double) * (size_t)c->cells);
        if (!c->vb) return SNREF_ERR_NOMEM;
    }
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) c->work[i] = cabs(c->psi[i]);
    int rc = fftn(c->work, c->ndim, c->n, +1);
    if (rc) return rc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) c->work[i] *= -ksq_at(c, i);
    if ((rc = fftn(c->work, c->ndim, c->n, -1))) return rc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) c->vb[i] = creal(c->work[i]) / (2.0 * fmax(cabs(c->psi[i]), c->sqrt_floor));
    return SNREF_OK;
}

/* N(s): psi *= exp(-i s (B phi + G(rho) + V + c_B V_B)) with phi, rho, V_B from psi at the start of the sub-step
 * (every factor leaves rho unchanged, so the order of the factors does not matter) */
static int nonlinear(snref_ctx *c, double s)
{
    int rc;
    if (c->c_bohm != 0.0 && (rc = bohm_potential(c))) return rc;
    rc = potential(c);
    if (rc) return rc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) {
        double re = creal(c->psi[i]), im = cimag(c->psi[i]);
        double rho = re * re + im * im;
        double th = -s * (c->B * creal(c->work[i]) + G_of(c, rho) + (c->vext ? c->vext[i] : 0.0) +
                          (c->c_bohm != 0.0 ? c->c_bohm * c->vb[i] : 0.0));
        c->psi[i] *= cos(th) + I * sin(th);
    }
    return SNREF_OK;
}

/* n Strang steps K(dtau/2) N(dtau) K(dtau/2), nothing merged */
int snref_step(snref_ctx *c, int64_t nsteps)
{
    if (!c) return SNREF_ERR_NULL;
    if (!c->has_state) return SNREF_ERR_STATE;
    if (nsteps < 0) return SNREF_ERR_PARAM;
    for (int64_t s = 0; s < nsteps; s++) {
        int rc;
        if ((rc = kinetic(c, 0.5 * c->dtau))) return rc;
        if ((rc = nonlinear(c, c->dtau))) return rc;
        if ((rc = kinetic(c, 0.5 * c->dtau))) return rc;
    }
    return SNREF_OK;
}

/* n fourth-order steps: each is the composition S2(w1 dtau) S2(w0 dtau) S2(w1 dtau) of three Strang steps
 * (Yoshida 1990 triple jump), w1 = 1/(2 - 2^(1/3)), w0 = 1 - 2 w1; written out as three plain Strang steps,
 * nothing merged.  Not in the paper (its scheme is the second-order one); SURVEY.md 8(f) item 4. */
int snref_step_order4(snref_ctx *c, int64_t nsteps)
{
    if (!c) return SNREF_ERR_NULL;
    if (!c->has_state) return SNREF_ERR_STATE;
    if (nsteps < 0) return SNREF_ERR_PARAM;
    const double w1 = 1.0 / (2.0 - cbrt(2.0)), w0 = 1.0 - 2.0 * w1, h = c->dtau;
    const double w[3] = {w1, w0, w1};
    int rc = SNREF_OK;
    for (int64_t s = 0; s < nsteps && !rc; s++)
        for (int i = 0; i < 3 && !rc; i++) {
            c->dtau = w[i] * h;
            rc = snref_step(c, 1);
        }
    c->dtau = h;
    return rc;
}

/* phi (real, cells doubles) from the current state; state unchanged */
int snref_potential(snref_ctx *c, double *phi_out)
{
    if (!c || !phi_out) return SNREF_ERR_NULL;
    if (!c->has_state) return SNREF_ERR_STATE;
    int rc = potential(c);
    if (rc) return rc;
    for (int64_t i = 0; i < c->cells; i++) phi_out[i] = creal(c->work[i]);
    return SNREF_OK;
}

int snref_diagnostics(snref_ctx *c, snref_diag *out)
{
    if (!c || !out) return SNREF_ERR_NULL;
    if (!c->has_state) return SNREF_ERR_STATE;
    double dV = 1.0;
    for (int d = 0; d < c->ndim; d++) dV *= c->L[d] / (double)c->n[d];
    int rc = potential(c);
    if (rc) return rc;
    double norm = 0.0, enl = 0.0, eloc = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : norm, enl, eloc)
    for (int64_t i = 0; i < c->cells; i++) {
        double re = creal(c->psi[i]), im = cimag(c->psi[i]);
        double rho = re * re + im * im;
        norm += rho;
        enl += creal(c->work[i]) * rho;
        eloc += F_of(c, rho) + (c->vext ? c->vext[i] * rho : 0.0);
    }
    /* kinetic part in k-space, on a copy of psi */
    memcpy(c->work, c->psi, sizeof(cplx) * (size_t)c->cells);
    rc = fftn(c->work, c->ndim, c->n, +1);
    if (rc) return rc;
    double ek = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : ek)
    for (int64_t i = 0; i < c->cells; i++) {
        double re = creal(c->work[i]), im = cimag(c->work[i]);
        ek += ksq_at(c, i) * (re * re + im * im);
    }
    out->norm = norm * dV;
    out->e_kin = -c->A * ek * dV / (double)c->cells;
    out->e_nonlocal = 0.5 * c->B * enl * dV;
    out->e_local = eloc * dV;
    out->e_total = out->e_kin + out->e_nonlocal + out->e_local;
    return SNREF_OK;
}

int snref_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

void snref_set_num_threads(int n)
{
#ifdef _OPENMP
    if (n > 0) omp_set_num_threads(n);
#else
    (void)n;
#endif
}

/* ================================================================== NEXT-4b: coupled wave functions
 *
 * PAPER.md:46 (section II): "Equations (1) and (2) can be further generalized if one considers multiple wave
 * functions coupled through the different nonlinearities of the system".  The paper does not write the generalized
 * system down; reading Q18 of DESIGN.md -- M components psi_c, each with its own kinetic and nonlocal constants, coupled
 * through (i) the local (Kerr-type) nonlinearity, a matrix g_cc' acting on the component densities, and (ii) the
 * nonlocal field, sourced by the weighted total density:
 *      i dpsi_c/dtau = A_c lap psi_c + B_c phi psi_c + (sum_c' g_cc' |psi_c'|^2) psi_c          (1')
 *      lap phi + C phi = D sum_c w_c |psi_c|^2                                                   (2')
 * Strang step, same readings as the one-component path (Q1-Q4):
 *      K(s):  psi_c^ *= exp(+i A_c k^2 s) for every c
 *      N(s):  rho_c = |psi_c|^2;  phi from (2') (phi^(0) = 0 when C == 0);
 *             psi_c *= exp(-i s (B_c phi + sum_c' g_cc' rho_c'))   -- exact for the N sub-flow: every rho_c is invariant
 *      step:  K(dtau/2) N(dtau) K(dtau/2)
 * State layout: [M][cells], component-major.  Reuses fftn / kval of this file; everything else is written out here.
 * Pins (tests/test_oracle_pins_mc.py): two plane waves (exact for any dtau), decoupled limit against snref_step,
 * equal split of a one-component state, per-component norm conservation, order 2 under dtau halving. */

#define SNREF_MC_MAX 4

typedef struct snref_mc_ctx {
    int ndim, M;
    int64_t n[3];
    double L[3];
    double A[SNREF_MC_MAX], B[SNREF_MC_MAX], w[SNREF_MC_MAX], g[SNREF_MC_MAX][SNREF_MC_MAX];
    double C, D, dtau;
    int64_t cells;
    cplx *psi;  /* [M][cells] */
    cplx *work; /* cells */
    int has_state;
} snref_mc_ctx;

static double mc_ksq_at(const snref_mc_ctx *c, int64_t idx)
{
    double k2 = 0.0;
    for (int d = c->ndim - 1; d >= 0; d--) {
        int64_t j = idx % c->n[d];
        idx /= c->n[d];
        double k = kval(j, c->n[d], c->L[d]);
        k2 += k * k;
    }
    return k2;
}

int snref_mc_create(snref_mc_ctx **out, int ndim, const int64_t *dims, const double *L, int M, const double *A,
                    const double *B, double C, double D, const double *w, const double *g /* [M][M] row-major */,
                    double dtau)
{
    if (!out || !dims || !L || !A || !B || !w || !g) return SNREF_ERR_NULL;
    if (ndim != 2 && ndim != 3) return SNREF_ERR_DIMS;
    if (M < 1 || M > SNREF_MC_MAX) return SNREF_ERR_PARAM;
    snref_mc_ctx *c = (snref_mc_ctx *)calloc(1, sizeof(*c));
    if (!c) return SNREF_ERR_NOMEM;
    c->ndim = ndim;
    c->M = M;
    c->cells = 1;
    for (int d = 0; d < ndim; d++) {
        if (!fft_len_ok(dims[d]) || !(L[d] > 0.0)) { free(c); return SNREF_ERR_DIMS; }
        c->n[d] = dims[d];
        c->L[d] = L[d];
        c->cells *= dims[d];
    }
    for (int a = 0; a < M; a++) {
        c->A[a] = A[a]; c->B[a] = B[a]; c->w[a] = w[a];
        for (int b = 0; b < M; b++) c->g[a][b] = g[a * M + b];
    }
    c->C = C; c->D = D; c->dtau = dtau;
    c->psi = (cplx *)malloc(sizeof(cplx) * (size_t)c->cells * (size_t)M);
    c->work = (cplx *)malloc(sizeof(cplx) * (size_t)c->cells);
    if (!c->psi || !c->work) { free(c->psi); free(c->work); free(c); return SNREF_ERR_NOMEM; }
    *out = c;
    return SNREF_OK;
}

int snref_mc_destroy(snref_mc_ctx *c)
{
    if (!c) return SNREF_ERR_NULL;
    free(c->psi);
    free(c->work);
    free(c);
    return SNREF_OK;
}

int snref_mc_set_dtau(snref_mc_ctx *c, double dtau)
{
    if (!c) return SNREF_ERR_NULL;
    c->dtau = dtau;
    return SNREF_OK;
}

int snref_mc_set_state(snref_mc_ctx *c, const cplx *psi)
{
    if (!c || !psi) return SNREF_ERR_NULL;
    memcpy(c->psi, psi, sizeof(cplx) * (size_t)c->cells * (size_t)c->M);
    c->has_state = 1;
    return SNREF_OK;
}

int snref_mc_get_state(snref_mc_ctx *c, cplx *out)
{
    if (!c || !out) return SNREF_ERR_NULL;
    if (!c->has_state) return SNREF_ERR_STATE;
    memcpy(out, c->psi, sizeof(cplx) * (size_t)c->cells * (size_t)c->M);
    return SNREF_OK;
}

/* K(s) of (1'): component by component */
static int mc_kinetic(snref_mc_ctx *c, double s)
{
    for (int a = 0; a < c->M; a++) {
        cplx *p = c->psi + (size_t)a * (size_t)c->cells;
        int rc = fftn(p, c->ndim, c->n, +1);
        if (rc) return rc;
#pragma omp parallel for schedule(static)
        for (int64_t i = 0; i < c->cells; i++) {
            double th = c->A[a] * mc_ksq_at(c, i) * s;
            p[i] *= cos(th) + I * sin(th);
        }
        if ((rc = fftn(p, c->ndim, c->n, -1))) return rc;
    }
    return SNREF_OK;
}

/* N(s) of (1'),(2') */
static int mc_nonlinear(snref_mc_ctx *c, double s)
{
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) {
        double src = 0.0;
        for (int a = 0; a < c->M; a++) {
            cplx v = c->psi[(size_t)a * (size_t)c->cells + (size_t)i];
            src += c->w[a] * (creal(v) * creal(v) + cimag(v) * cimag(v));
        }
        c->work[i] = src;
    }
    int rc = fftn(c->work, c->ndim, c->n, +1);
    if (rc) return rc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) {
        if (c->C == 0.0 && i == 0) { c->work[i] = 0.0; continue; }
        c->work[i] = c->D * c->work[i] / (c->C - mc_ksq_at(c, i));
    }
    if ((rc = fftn(c->work, c->ndim, c->n, -1))) return rc;
#pragma omp parallel for schedule(static)
    for (int64_t i = 0; i < c->cells; i++) {
        double rho[SNREF_MC_MAX];
        for (int a = 0; a < c->M; a++) {
            cplx v = c->psi[(size_t)a * (size_t)c->cells + (size_t)i];
            rho[a] = creal(v) * creal(v) + cimag(v) * cimag(v);
        }
        double phi = creal(c->work[i]);
        for (int a = 0; a < c->M; a++) {
            double loc = 0.0;
            for (int b = 0; b < c->M; b++) loc += c->g[a][b] * rho[b];
            double th = -s * (c->B[a] * phi + loc);
            c->psi[(size_t)a * (size_t)c->cells + (size_t)i] *= cos(th) + I * sin(th);
        }
    }
    return SNREF_OK;
}

int snref_mc_step(snref_mc_ctx *c, int64_t nsteps)
{
    if (!c) return SNREF_ERR_NULL;
    if (!c->has_state) return SNREF_ERR_STATE;
    if (nsteps < 0) return SNREF_ERR_PARAM;
    for (int64_t s = 0; s < nsteps; s++) {
        int rc;
        if ((rc = mc_kinetic(c, 0.5 * c->dtau))) return rc;
        if ((rc = mc_nonlinear(c, c->dtau))) return rc;
        if ((rc = mc_kinetic(c, 0.5 * c->dtau))) return rc;
    }
    return SNREF_OK;
}

/* norms[a] = sum |psi_a|^2 dV */
int snref_mc_norms(snref_mc_ctx *c, double *norms)
{
    if (!c || !norms) return SNREF_ERR_NULL;
    if (!c->has_state) return SNREF_ERR_STATE;
    double dV = 1.0;
    for (int d = 0; d < c->ndim; d++) dV *= c->L[d] / (double)c->n[d];
    for (int a = 0; a < c->M; a++) {
        const cplx *p = c->psi + (size_t)a * (size_t)c->cells;
        double s = 0.0;
#pragma omp parallel for schedule(static) reduction(+ : s)
        for (int64_t i = 0; i < c->cells; i++) s += creal(p[i]) * creal(p[i]) + cimag(p[i]) * cimag(p[i]);
        norms[a] = s * dV;
    }
    return SNREF_OK;
}
