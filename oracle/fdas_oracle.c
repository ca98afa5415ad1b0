/*
 * fdas_oracle.c -- TEST INFRASTRUCTURE, NOT THE PRODUCT.
 *
 * Plain, slow, double-precision CPU statement of what the FDAS hot path computes
 * (arXiv:1711.10855).  Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline /
 * --impl reference legs may load this file.  It shares no code, header, table or helper with
 * the CUDA path under paper_1711_10855_b200/csrc/ and neither side includes the other.
 *
 * What is here, and the passage each function follows (P:NN = /root/reference/PAPER.md line NN;
 * S8c = SURVEY.md section 8(c), whose readings are listed in DESIGN.md):
 *
 *   fdas_oracle_dft        eq.(3), P:35   X_m = sum_n x_n exp(-i 2 pi n m / N), O(N^2)
 *   fdas_oracle_fft        P:40           the same transform by radix-2 divide and conquer
 *   fdas_oracle_fresnel    S8c            C(x), S(x) = int_0^x cos|sin(pi t^2 / 2) dt
 *   fdas_oracle_response   P:21, S8c      I(q,z) = int_0^1 exp(i pi (2 q u + z u^2)) du, the
 *                                         Fourier response of a constant-fdot signal
 *   fdas_oracle_templates  P:21, S8c      h_z[j] = H_z(j - m/2) / ||H_z||, H_z(d) = I(d - z/2, z)
 *   fdas_oracle_direct     eq.(2), P:23   A'_{r0} = sum_k A_k conj(H_{r0-k}) by direct summation,
 *                                         and its power |A'|^2 (the authority for parity)
 *   fdas_oracle_ols        P:31           the same plane by overlap-and-save in double, with
 *                                         fdas_oracle_fft (checked against fdas_oracle_direct)
 *   fdas_oracle_spectrum   P:21           "the FFT output of the observation": eq.(3) of the real time series,
 *                                         bins 0 .. n_t/2 - 1, each block of bins scaled to unit variance per
 *                                         component (reading 18) -- the input of the correlation
 *   fdas_oracle_blockmax   P:21, P:50     the detection step that consumes the plane ("FDAS code";
 *                                         the paper leaves it to Dimoudi 2017, reading 17):
 *                                         per row and block of columns, the maximum power and the
 *                                         lowest column that attains it
 *
 * Pins (tests/test_oracle_*.py): brute-force DFT vs FFT; Parseval; scipy.special.fresnel; an
 * independent quadrature of the defining integral; the DFT of a sampled chirp; z=0 -> delta;
 * numpy.convolve; impulse / constant inputs with closed forms; an injected signal peaking in
 * its row; linearity; OLS == direct; block maxima against a Python loop, numpy and the C1 peak.
 * Nothing in this file is "parity unpinned".
 *
 * Complex arrays are interleaved (re, im) doubles.  No function here reorders, blocks or fuses
 * beyond what the cited definition states, except that fdas_oracle_direct walks columns in
 * blocks so that gcc can vectorise the inner loop; the sum over taps for one output is still
 * accumulated tap by tap in increasing j.
 */
#include <math.h>
#include <stdint.h>
#include <stdlib.h>
#include <string.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#ifndef M_PI
#define M_PI 3.14159265358979323846
#endif

int fdas_oracle_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}

/* ------------------------------------------------------------------------------------------
 * eq.(3): X_m = sum_{n=0}^{N-1} x_n exp(-i 2 pi n m / N).  sign = -1 is eq.(3); sign = +1
 * is the unnormalised inverse (S8c reading 9: the 1/N of the inverse is applied by the caller).
 * ------------------------------------------------------------------------------------------ */
void fdas_oracle_dft(const double *x, int64_t n_pts, int sign, double *out)
{
    for (int64_t m = 0; m < n_pts; ++m) {
        double sr = 0.0, si = 0.0;
        for (int64_t n = 0; n < n_pts; ++n) {
            /* reduce n*m mod N exactly in integers before forming the angle */
            int64_t e = (n * m) % n_pts;
            double ang = (double)sign * 2.0 * M_PI * (double)e / (double)n_pts;
            double c = cos(ang), s = sin(ang);
            sr += x[2 * n] * c - x[2 * n + 1] * s;
            si += x[2 * n] * s + x[2 * n + 1] * c;
        }
        out[2 * m] = sr;
        out[2 * m + 1] = si;
    }
}

/* P:40 "each FFT is itself composed from smaller FFTs": recursive radix-2 decimation in time.
 * X_m = E_m + w^m O_m, X_{m+N/2} = E_m - w^m O_m, w = exp(sign i 2 pi / N).  In place on x
 * (length n_pts, a power of two) using scratch of the same length. */
static void fft_rec(double *x, double *scratch, int64_t n_pts, int sign)
{
    if (n_pts == 1) return;
    int64_t h = n_pts / 2;
    for (int64_t i = 0; i < h; ++i) {
        scratch[2 * i] = x[4 * i];
        scratch[2 * i + 1] = x[4 * i + 1];
        scratch[2 * (h + i)] = x[4 * i + 2];
        scratch[2 * (h + i) + 1] = x[4 * i + 3];
    }
    fft_rec(scratch, x, h, sign);
    fft_rec(scratch + 2 * h, x, h, sign);
    for (int64_t m = 0; m < h; ++m) {
        double ang = (double)sign * 2.0 * M_PI * (double)m / (double)n_pts;
        double c = cos(ang), s = sin(ang);
        double er = scratch[2 * m], ei = scratch[2 * m + 1];
        double pr = scratch[2 * (h + m)], pi_ = scratch[2 * (h + m) + 1];
        double tr = pr * c - pi_ * s, ti = pr * s + pi_ * c;
        x[2 * m] = er + tr;
        x[2 * m + 1] = ei + ti;
        x[2 * (m + h)] = er - tr;
        x[2 * (m + h) + 1] = ei - ti;
    }
}

/* returns 0, or -1 if n_pts is not a power of two / allocation failed */
int fdas_oracle_fft(double *x, int64_t n_pts, int sign)
{
    if (n_pts < 1 || (n_pts & (n_pts - 1)) != 0) return -1;
    double *scratch = (double *)malloc(sizeof(double) * 2 * (size_t)n_pts);
    if (!scratch) return -1;
    fft_rec(x, scratch, n_pts, sign);
    free(scratch);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * Fresnel integrals C(x) = int_0^x cos(pi t^2/2) dt, S(x) = int_0^x sin(pi t^2/2) dt  (S8c).
 *
 * |x| <= 1.5 : the Maclaurin series, term by term
 *     C(x) = sum_n (-1)^n (pi/2)^{2n}   x^{4n+1} / ((2n)!   (4n+1))
 *     S(x) = sum_n (-1)^n (pi/2)^{2n+1} x^{4n+3} / ((2n+1)! (4n+3))
 * |x| >  1.5 : C(x) + i S(x) = (1+i)/2 * erf(w), w = (sqrt(pi)/2)(1-i) x, with
 *     erfc(w) = exp(-w^2)/sqrt(pi) * 1/(w + (1/2)/(w + 1/(w + (3/2)/(w + 2/(w + ...)))))
 *     (the classical continued fraction, Re w > 0), evaluated by the modified Lentz recurrence.
 *     Here exp(-w^2) = exp(i pi x^2 / 2) exactly.
 * Both are odd in x.
 * ------------------------------------------------------------------------------------------ */
typedef struct { double re, im; } cplx;
static cplx c_mul(cplx a, cplx b) { cplx r = { a.re * b.re - a.im * b.im, a.re * b.im + a.im * b.re }; return r; }
static cplx c_div(cplx a, cplx b)
{
    double d = b.re * b.re + b.im * b.im;
    cplx r = { (a.re * b.re + a.im * b.im) / d, (a.im * b.re - a.re * b.im) / d };
    return r;
}
static cplx c_add(cplx a, cplx b) { cplx r = { a.re + b.re, a.im + b.im }; return r; }

void fdas_oracle_fresnel(double x, double *c_out, double *s_out)
{
    double ax = fabs(x), C, S;
    if (ax <= 1.5) {
        double t = 0.5 * M_PI * ax * ax; /* pi x^2 / 2 */
        /* C terms: x * (-t^2)^n / ((2n)! (4n+1));  S terms: x * t * (-t^2)^n / ((2n+1)! (4n+3)) */
        double pc = 1.0, ps = t; /* t^{2n}/(2n)!  and  t^{2n+1}/(2n+1)! */
        C = 0.0; S = 0.0;
        for (int n = 0; n < 60; ++n) {
            double sgn = (n & 1) ? -1.0 : 1.0;
            C += sgn * pc / (4.0 * n + 1.0);
            S += sgn * ps / (4.0 * n + 3.0);
            pc = pc * t * t / ((2.0 * n + 1.0) * (2.0 * n + 2.0));
            ps = ps * t * t / ((2.0 * n + 2.0) * (2.0 * n + 3.0));
            if (pc < 1e-20 && ps < 1e-20) break;
        }
        C *= ax; S *= ax;
    } else {
        const double k = 0.5 * sqrt(M_PI);
        cplx w = { k * ax, -k * ax };
        /* continued fraction f = w + a1/(w + a2/(w + ...)), a_n = n/2, by modified Lentz */
        const double tiny = 1e-300;
        cplx f = w, Cn = w, Dn = { 0.0, 0.0 };
        for (int n = 1; n < 200000; ++n) {
            cplx an = { 0.5 * n, 0.0 };
            Dn = c_add(w, c_mul(an, Dn));
            if (Dn.re == 0.0 && Dn.im == 0.0) Dn.re = tiny;
            Cn = c_add(w, c_div(an, Cn));
            if (Cn.re == 0.0 && Cn.im == 0.0) Cn.re = tiny;
            cplx one = { 1.0, 0.0 };
            Dn = c_div(one, Dn);
            cplx delta = c_mul(Cn, Dn);
            f = c_mul(f, delta);
            if (fabs(delta.re - 1.0) + fabs(delta.im) < 1e-17) break;
        }
        double ph = 0.5 * M_PI * ax * ax;
        cplx e = { cos(ph) / sqrt(M_PI), sin(ph) / sqrt(M_PI) };
        cplx erfc_w = c_div(e, f);
        cplx erf_w = { 1.0 - erfc_w.re, -erfc_w.im };
        cplx half1pi = { 0.5, 0.5 };
        cplx r = c_mul(half1pi, erf_w);
        C = r.re; S = r.im;
    }
    if (x < 0) { C = -C; S = -S; }
    *c_out = C; *s_out = S;
}

/* ------------------------------------------------------------------------------------------
 * I(q,z) = int_0^1 exp(i pi (2 q u + z u^2)) du  ("predicted Fourier response"; S8c).
 *   z = 0 : exp(i pi q) sin(pi q)/(pi q), 1 at q = 0
 *   z > 0 : exp(-i pi q^2/z)/sqrt(2z) * ([C(Z)-C(Y)] + i [S(Z)-S(Y)]),
 *           Y = q sqrt(2/z), Z = (q+z) sqrt(2/z)   (complete the square, t = (u+q/z) sqrt(2z))
 *   z < 0 : conj(I(-q,-z))
 * ------------------------------------------------------------------------------------------ */
void fdas_oracle_response(double q, double z, double *re, double *im)
{
    if (z == 0.0) {
        if (q == 0.0) { *re = 1.0; *im = 0.0; return; }
        double s = sin(M_PI * q) / (M_PI * q);
        *re = cos(M_PI * q) * s;
        *im = sin(M_PI * q) * s;
        return;
    }
    if (z < 0.0) {
        fdas_oracle_response(-q, -z, re, im);
        *im = -*im;
        return;
    }
    double Y = q * sqrt(2.0 / z), Z = (q + z) * sqrt(2.0 / z);
    double cy, sy, cz, sz;
    fdas_oracle_fresnel(Y, &cy, &sy);
    fdas_oracle_fresnel(Z, &cz, &sz);
    double ar = cz - cy, ai = sz - sy;
    double ph = -M_PI * q * q / z;
    double pr = cos(ph) / sqrt(2.0 * z), pi_ = sin(ph) / sqrt(2.0 * z);
    *re = pr * ar - pi_ * ai;
    *im = pr * ai + pi_ * ar;
}

/* ------------------------------------------------------------------------------------------
 * Template bank ("predicted, normalized, Fourier response H"; S8c readings 1-4, 7):
 * row i <-> z = -z_max + i z_step, n_z = 2 z_max / z_step + 1; tap j <-> offset d = j - m/2 from
 * the signal's MEAN frequency; H_z(d) = I(d - z/2, z); h_z[j] = H_z(j - m/2) / sqrt(sum |H_z|^2).
 * out: [n_z][m][2].  Returns n_z, or -1 on bad arguments.
 * ------------------------------------------------------------------------------------------ */
int fdas_oracle_templates(int z_max, int z_step, int m, double *out)
{
    if (z_max < 0 || z_step < 1 || z_max % z_step != 0 || m < 2 || (m & 1)) return -1;
    int n_z = 2 * z_max / z_step + 1;
    for (int i = 0; i < n_z; ++i) {
        double z = (double)(-z_max + i * z_step);
        double *row = out + (size_t)i * m * 2;
        double e = 0.0;
        for (int j = 0; j < m; ++j) {
            double d = (double)(j - m / 2);
            fdas_oracle_response(d - 0.5 * z, z, &row[2 * j], &row[2 * j + 1]);
            e += row[2 * j] * row[2 * j] + row[2 * j + 1] * row[2 * j + 1];
        }
        double s = 1.0 / sqrt(e);
        for (int j = 0; j < 2 * m; ++j) row[j] *= s;
    }
    return n_z;
}

/* ------------------------------------------------------------------------------------------
 * eq.(2), by direct summation (S8c "Definition"):
 *   A'[z][r0] = sum_{j=0}^{m-1} A[r0 + m/2 - j] * conj(h_z[j]),  A[k] := 0 outside [0, n_f)
 *   P[z][r0]  = |A'[z][r0]|^2
 * for rows row0 <= z-row < row0+n_rows and columns col0 <= r0 < col0+n_cols.
 * spectrum: [n_f][2]; templates: [n_z_total][m][2] (row index is absolute);
 * power_out: [n_rows][n_cols] or NULL; amp_out: [n_rows][n_cols][2] or NULL.
 * ------------------------------------------------------------------------------------------ */
#define ORACLE_BLOCK 512
int fdas_oracle_direct(const double *spectrum, int64_t n_f, const double *templates, int m,
                       int row0, int n_rows, int64_t col0, int64_t n_cols,
                       double *power_out, double *amp_out)
{
    if (n_f < 1 || m < 2 || (m & 1) || n_rows < 0 || n_cols < 0 || col0 < 0 || col0 + n_cols > n_f)
        return -1;
    /* zero-padded copy of the columns this call can touch: k in [col0 - m/2 + 1, col0+n_cols-1 + m/2] */
    int64_t k_lo = col0 - m / 2 + 1, k_hi = col0 + n_cols - 1 + m / 2;
    int64_t n_pad = k_hi - k_lo + 1;
    if (n_cols == 0 || n_rows == 0) return 0;
    double *ar = (double *)calloc((size_t)n_pad, sizeof(double));
    double *ai = (double *)calloc((size_t)n_pad, sizeof(double));
    if (!ar || !ai) { free(ar); free(ai); return -1; }
    for (int64_t k = k_lo; k <= k_hi; ++k)
        if (k >= 0 && k < n_f) { ar[k - k_lo] = spectrum[2 * k]; ai[k - k_lo] = spectrum[2 * k + 1]; }

    int64_t n_blocks = (n_cols + ORACLE_BLOCK - 1) / ORACLE_BLOCK;
    int64_t n_jobs = (int64_t)n_rows * n_blocks;
#pragma omp parallel for schedule(dynamic, 4)
    for (int64_t job = 0; job < n_jobs; ++job) {
        int row = (int)(job / n_blocks);
        int64_t blk = job % n_blocks;
        int64_t c_lo = blk * ORACLE_BLOCK;
        int64_t c_n = n_cols - c_lo < ORACLE_BLOCK ? n_cols - c_lo : ORACLE_BLOCK;
        const double *h = templates + (size_t)(row0 + row) * m * 2;
        double sr[ORACLE_BLOCK], si[ORACLE_BLOCK];
        for (int64_t i = 0; i < c_n; ++i) { sr[i] = 0.0; si[i] = 0.0; }
        for (int j = 0; j < m; ++j) {
            double hr = h[2 * j], hi = -h[2 * j + 1]; /* conj(h_z[j]) */
            /* column r0 = col0 + c_lo + i reads A[r0 + m/2 - j] = pad[(r0 + m/2 - j) - k_lo] */
            const double *pr = ar + (col0 + c_lo + m / 2 - j - k_lo);
            const double *pi_ = ai + (col0 + c_lo + m / 2 - j - k_lo);
            for (int64_t i = 0; i < c_n; ++i) {
                sr[i] += pr[i] * hr - pi_[i] * hi;
                si[i] += pr[i] * hi + pi_[i] * hr;
            }
        }
        for (int64_t i = 0; i < c_n; ++i) {
            size_t o = (size_t)row * (size_t)n_cols + (size_t)(c_lo + i);
            if (power_out) power_out[o] = sr[i] * sr[i] + si[i] * si[i];
            if (amp_out) { amp_out[2 * o] = sr[i]; amp_out[2 * o + 1] = si[i]; }
        }
    }
    free(ar); free(ai);
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * P:31 overlap-and-save in double (S8c component 4): for segment s the buffer
 *   x[i] = A[s*S - m/2 + 1 + i], i < L (zero outside [0,n_f)); g = conj(h_z) at indices 0..m-1
 *   of a zero length-L buffer; y = IDFT_L(DFT_L(x) .* DFT_L(g)) / L;  P[z][s*S + i] = |y[m-1+i]|^2
 *   for i < min(S, n_f - s*S).  Any step 1 <= S <= L-m+1 gives the linear convolution.
 * power_out: [n_rows][n_f] for template rows row0 .. row0+n_rows-1.
 * ------------------------------------------------------------------------------------------ */
int fdas_oracle_ols(const double *spectrum, int64_t n_f, const double *templates, int m,
                    int row0, int n_rows, int seg_len, int step, double *power_out)
{
    int L = seg_len, S = step;
    if (n_f < 1 || m < 2 || (m & 1) || L < m || (L & (L - 1)) || S < 1 || S > L - m + 1 || n_rows < 0)
        return -1;
    int64_t n_seg = (n_f + S - 1) / S;
    /* DFT_L of the padded conjugated templates, once */
    double *G = (double *)malloc(sizeof(double) * 2 * (size_t)L * (size_t)(n_rows > 0 ? n_rows : 1));
    if (!G) return -1;
    for (int r = 0; r < n_rows; ++r) {
        double *g = G + (size_t)r * 2 * L;
        const double *h = templates + (size_t)(row0 + r) * m * 2;
        memset(g, 0, sizeof(double) * 2 * (size_t)L);
        for (int j = 0; j < m; ++j) { g[2 * j] = h[2 * j]; g[2 * j + 1] = -h[2 * j + 1]; }
        fdas_oracle_fft(g, L, -1);
    }
    int fail = 0;
#pragma omp parallel
    {
        double *X = (double *)malloc(sizeof(double) * 2 * (size_t)L);
        double *Y = (double *)malloc(sizeof(double) * 2 * (size_t)L);
        if (!X || !Y) {
#pragma omp atomic write
            fail = 1;
        } else {
#pragma omp for schedule(dynamic, 1)
            for (int64_t s = 0; s < n_seg; ++s) {
                int64_t base = s * (int64_t)S - m / 2 + 1;
                for (int i = 0; i < L; ++i) {
                    int64_t k = base + i;
                    if (k >= 0 && k < n_f) { X[2 * i] = spectrum[2 * k]; X[2 * i + 1] = spectrum[2 * k + 1]; }
                    else { X[2 * i] = 0.0; X[2 * i + 1] = 0.0; }
                }
                fdas_oracle_fft(X, L, -1);
                for (int r = 0; r < n_rows; ++r) {
                    const double *g = G + (size_t)r * 2 * L;
                    for (int n = 0; n < L; ++n) {
                        Y[2 * n] = X[2 * n] * g[2 * n] - X[2 * n + 1] * g[2 * n + 1];
                        Y[2 * n + 1] = X[2 * n] * g[2 * n + 1] + X[2 * n + 1] * g[2 * n];
                    }
                    fdas_oracle_fft(Y, L, +1);
                    for (int i = 0; i < S; ++i) {
                        int64_t r0 = s * (int64_t)S + i;
                        if (r0 >= n_f) break;
                        double yr = Y[2 * (m - 1 + i)] / L, yi = Y[2 * (m - 1 + i) + 1] / L;
                        power_out[(size_t)r * (size_t)n_f + (size_t)r0] = yr * yr + yi * yi;
                    }
                }
            }
        }
        free(X); free(Y);
    }
    free(G);
    return fail ? -1 : 0;
}

/* ------------------------------------------------------------------------------------------
 * Detection step over a power plane ("detect"; "FDAS code"; reading 17):
 * for every row r and block b of `blk` consecutive columns, [b*blk, min((b+1)*blk, n_cols)),
 *   max_out[r][b] = max_c P[r][c]        arg_out[r][b] = the smallest c - b*blk with P[r][c] = max
 * n_blk = ceil(n_cols / blk).  in_float32 != 0: every power is rounded to IEEE float32 before
 * it is compared (the precision in which the CUDA path takes the same decision); max_out then
 * holds the rounded value.  Plain scan, left to right.
 * ------------------------------------------------------------------------------------------ */
int fdas_oracle_blockmax(const double *power, int n_rows, int64_t n_cols, int64_t blk, int in_float32,
                         double *max_out, int64_t *arg_out)
{
    if (!power || !max_out || !arg_out || n_rows < 0 || n_cols < 1 || blk < 1) return -1;
    int64_t n_blk = (n_cols + blk - 1) / blk;
    for (int r = 0; r < n_rows; ++r) {
        for (int64_t b = 0; b < n_blk; ++b) {
            int64_t c0 = b * blk, c1 = c0 + blk < n_cols ? c0 + blk : n_cols;
            double best = 0.0;
            int64_t arg = -1;
            for (int64_t c = c0; c < c1; ++c) {
                double v = power[(size_t)r * (size_t)n_cols + (size_t)c];
                if (in_float32) v = (double)(float)v;
                if (arg < 0 || v > best) { best = v; arg = c - c0; }
            }
            max_out[(size_t)r * (size_t)n_blk + (size_t)b] = best;
            arg_out[(size_t)r * (size_t)n_blk + (size_t)b] = arg;
        }
    }
    return 0;
}

/* ------------------------------------------------------------------------------------------
 * The step before the correlation ("the FFT output of the observation"; SURVEY.md NEXT-3;
 * DESIGN.md reading 18).  series: n_t real samples, n_t a power of two >= 4.
 *   X_k = sum_n series[n] exp(-i 2 pi n k / n_t)                     eq.(3), k = 0 .. n_t/2 - 1
 *   whitening: bins are cut into blocks of `blk` bins, block b = [b*blk, min((b+1)*blk, n_t/2));
 *     m_b = mean over the block's bins of |X_k|^2, bin 0 (the DC term) counted as 0
 *     A_k = X_k * sqrt(2 / m_b)   (each of re, im then has unit variance where the block is noise),
 *     A_0 = 0, and A_k = 0 in a block with m_b = 0.   blk <= 0: no whitening, A_k = X_k.
 * out: [n_t/2][2].  The transform is fdas_oracle_fft on the zero-imaginary complex sequence.
 * ------------------------------------------------------------------------------------------ */
int fdas_oracle_spectrum(const double *series, int64_t n_t, int64_t blk, double *out)
{
    if (!series || !out || n_t < 4 || (n_t & (n_t - 1))) return -1;
    double *z = (double *)malloc(sizeof(double) * 2 * (size_t)n_t);
    if (!z) return -1;
    for (int64_t n = 0; n < n_t; ++n) { z[2 * n] = series[n]; z[2 * n + 1] = 0.0; }
    if (fdas_oracle_fft(z, n_t, -1) != 0) { free(z); return -1; }
    int64_t n_f = n_t / 2;
    if (blk <= 0) {
        memcpy(out, z, sizeof(double) * 2 * (size_t)n_f);
        free(z);
        return 0;
    }
    for (int64_t b0 = 0; b0 < n_f; b0 += blk) {
        int64_t b1 = b0 + blk < n_f ? b0 + blk : n_f;
        double sum = 0.0;
        for (int64_t k = b0; k < b1; ++k)
            if (k != 0) sum += z[2 * k] * z[2 * k] + z[2 * k + 1] * z[2 * k + 1];
        double mean = sum / (double)(b1 - b0);
        double scale = mean > 0.0 ? sqrt(2.0 / mean) : 0.0;
        for (int64_t k = b0; k < b1; ++k) {
            out[2 * k] = k == 0 ? 0.0 : z[2 * k] * scale;
            out[2 * k + 1] = k == 0 ? 0.0 : z[2 * k + 1] * scale;
        }
    }
    free(z);
    return 0;
}
