/*
 * bioem_oracle.c -- TEST INFRASTRUCTURE, NOT PRODUCT CODE.
 *
 * A plain, slow, double-precision CPU statement of what the BioEM hot path computes
 * (arXiv:1609.06634; citations "P:<line>" are lines of /root/reference/PAPER.md,
 * "R<k>" are the readings listed in DESIGN.md section 3).  It exists so that the CUDA
 * path can be checked against something that can be verified against the paper by eye.
 * Only tests/, __graft_entry__.smoke() and bench.py's cpu_baseline / --impl reference
 * legs may load this file.  It shares no code, header, table or constant with
 * paper_1609_06634_b200/csrc/.
 *
 * What is the definition and what is not:
 *   - cross-correlation: direct circular summation in real space (Eq. 7 semantics,
 *     P:109, R4, R5).  No FFT anywhere in this file.
 *   - DFT: the naive O(N^3) separable sum of Eq. 2/3 under reading R3.
 *   - likelihood: closed form (C1) derived from Eq. 8 with flat priors on
 *     N, mu, lambda (R1); pinned against quadrature of Eq. 8 in tests/.
 *   - "tier B" (bo_cross_corr_dft) is the same correlation through an FP64
 *     output-pruned separable DFT.  It is NOT the definition; tests validate it against
 *     the direct summation and it is only used to extend full-grid goldens.
 *
 * Parity pins (tests/test_oracle_*.py): every function below has at least one pin
 * that is not a restatement of itself.  bo_fourier_slice (R21, a definition the
 * paper does not give) is pinned exactly at general orientations on spectra that
 * are multi-affine in k (which trilinear interpolation reproduces exactly, so the
 * expected slice is a closed form), exactly at the rotations that permute the grid
 * (90 deg about x, y, z; 120 deg about the body diagonal), exactly at the identity
 * against the 2-D DFT of the z-sum, and loosely against analytic Gaussian blobs.
 *
 * Layout: images are row-major [k][j] = [y][x], x fastest (R11).
 */
#include <math.h>
#include <stdlib.h>
#include <string.h>
#include <stdint.h>
#ifdef _OPENMP
#include <omp.h>
#endif

#define BO_PI 3.14159265358979323846264338327950288

/* ------------------------------------------------------------------ rotation (R12) */
/* unit quaternion (w,x,y,z) -> active rotation matrix, r' = R r. */
void bo_quat_to_matrix(const double q[4], double R[9])
{
    double w = q[0], x = q[1], y = q[2], z = q[3];
    double nrm = sqrt(w * w + x * x + y * y + z * z);
    w /= nrm; x /= nrm; y /= nrm; z /= nrm;
    R[0] = 1 - 2 * (y * y + z * z); R[1] = 2 * (x * y - w * z);     R[2] = 2 * (x * z + w * y);
    R[3] = 2 * (x * y + w * z);     R[4] = 1 - 2 * (x * x + z * z); R[5] = 2 * (y * z - w * x);
    R[6] = 2 * (x * z - w * y);     R[7] = 2 * (y * z + w * x);     R[8] = 1 - 2 * (x * x + y * y);
}

/* ------------------------------------------------------------------ Eq. 1 */
/* I0(j,k) = sum_atoms int_pixel dxdy int dz rho.  Atom = uniform sphere radius R_a,
 * total weight w_a (R10): column density 2 sqrt(R^2 - r^2)_+ * w / (4/3 pi R^3).
 * Pixel integral by Kq x Kq midpoint sub-sampling (R10).  Pixel centres
 * x_j = (j - N/2) px, y_k = (k - N/2) px (R11).  Projection along z' after r' = R r. */
void bo_project_atoms(int n_atoms, const double *xyz, const double *radius, const double *weight,
                      const double q[4], int N, double px, int Kq, double *I0)
{
    double R[9];
    bo_quat_to_matrix(q, R);
    memset(I0, 0, sizeof(double) * (size_t)N * N);
    double h = px / Kq;
    for (int a = 0; a < n_atoms; ++a) {
        const double *r = xyz + 3 * a;
        double xr = R[0] * r[0] + R[1] * r[1] + R[2] * r[2];
        double yr = R[3] * r[0] + R[4] * r[1] + R[5] * r[2];
        double Ra = radius[a];
        double dens = weight[a] / (4.0 / 3.0 * BO_PI * Ra * Ra * Ra);
        /* pixels whose extent [x_j - px/2, x_j + px/2] can touch the disc */
        int j0 = (int)floor((xr - Ra) / px + N / 2 - 0.5) - 1, j1 = (int)ceil((xr + Ra) / px + N / 2 + 0.5) + 1;
        int k0 = (int)floor((yr - Ra) / px + N / 2 - 0.5) - 1, k1 = (int)ceil((yr + Ra) / px + N / 2 + 0.5) + 1;
        for (int k = k0; k <= k1; ++k) {
            if (k < 0 || k >= N) continue;      /* atoms outside the box are cropped, not wrapped */
            for (int j = j0; j <= j1; ++j) {
                if (j < 0 || j >= N) continue;
                double xc = (j - N / 2) * px, yc = (k - N / 2) * px;
                double acc = 0.0;
                for (int sy = 0; sy < Kq; ++sy)
                    for (int sx = 0; sx < Kq; ++sx) {
                        double x = xc - 0.5 * px + (sx + 0.5) * h;
                        double y = yc - 0.5 * px + (sy + 0.5) * h;
                        double d2 = Ra * Ra - (x - xr) * (x - xr) - (y - yr) * (y - yr);
                        if (d2 > 0.0) acc += 2.0 * sqrt(d2);
                    }
                I0[(size_t)k * N + j] += dens * acc * h * h;
            }
        }
    }
}

/* ------------------------------------------------------------------ Eqs. 2-3, R3 */
/* out(l,m) = scale * sum_{j,k} in(j,k) exp(sign * 2 pi i (l j / N + m k / N)),
 * arrays [m][l] / [k][j].  sign = -1: forward (Eq. 2 under R3); sign = +1 with
 * scale = 1/N^2: inverse (Eq. 3).  Naive separable sums, no FFT. in_im may be NULL. */
void bo_dft2(int N, const double *in_re, const double *in_im, int sign, double scale,
             double *out_re, double *out_im)
{
    size_t n = (size_t)N * N;
    double *tr = (double *)malloc(sizeof(double) * n), *ti = (double *)malloc(sizeof(double) * n);
    double *cw = (double *)malloc(sizeof(double) * N), *sw = (double *)malloc(sizeof(double) * N);
    for (int t = 0; t < N; ++t) {
        cw[t] = cos(2.0 * BO_PI * t / N);
        sw[t] = sign * sin(2.0 * BO_PI * t / N);
    }
    /* along x: t(l,k) = sum_j in(j,k) w^{l j} */
#pragma omp parallel for schedule(static)
    for (int k = 0; k < N; ++k)
        for (int l = 0; l < N; ++l) {
            double ar = 0, ai = 0;
            for (int j = 0; j < N; ++j) {
                int t = (int)(((long long)l * j) % N);
                double xr = in_re[(size_t)k * N + j], xi = in_im ? in_im[(size_t)k * N + j] : 0.0;
                ar += xr * cw[t] - xi * sw[t];
                ai += xr * sw[t] + xi * cw[t];
            }
            tr[(size_t)k * N + l] = ar; ti[(size_t)k * N + l] = ai;
        }
    /* along y: out(l,m) = sum_k t(l,k) w^{m k} */
#pragma omp parallel for schedule(static)
    for (int m = 0; m < N; ++m)
        for (int l = 0; l < N; ++l) {
            double ar = 0, ai = 0;
            for (int k = 0; k < N; ++k) {
                int t = (int)(((long long)m * k) % N);
                double xr = tr[(size_t)k * N + l], xi = ti[(size_t)k * N + l];
                ar += xr * cw[t] - xi * sw[t];
                ai += xr * sw[t] + xi * cw[t];
            }
            out_re[(size_t)m * N + l] = scale * ar; out_im[(size_t)m * N + l] = scale * ai;
        }
    free(tr); free(ti); free(cw); free(sw);
}

/* ------------------------------------------------------------------ Eqs. 4-5 */
/* CTF(s|a,A) Env(s|b) with s2 = |s|^2:  -A cos(a s^2/2) - sqrt(1-A^2) sin(a s^2/2), times exp(-b s^2/2). */
double bo_ctf_env(double s2, double a, double A, double b)
{
    double ph = 0.5 * a * s2;
    return (-A * cos(ph) - sqrt(1.0 - A * A) * sin(ph)) * exp(-0.5 * b * s2);
}

/* |s|^2 of DFT bin (l,m): s = 2 pi (l'/(N px), m'/(N px)), l' the signed frequency. */
static double bo_s2(int l, int m, int N, double px)
{
    int ls = (l <= N / 2) ? l : l - N, ms = (m <= N / 2) ? m : m - N;
    double f = 2.0 * BO_PI / (N * px);
    return f * f * ((double)ls * ls + (double)ms * ms);
}

/* I1 = Re F^-1( F_hat * CTF * Env )  (Eq. 5) from a full spectrum [m][l]. */
void bo_apply_ctf_spectrum(int N, double px, const double *F_re, const double *F_im,
                           double a, double A, double b, double *I1)
{
    size_t n = (size_t)N * N;
    double *gr = (double *)malloc(sizeof(double) * n), *gi = (double *)malloc(sizeof(double) * n);
    double *or_ = (double *)malloc(sizeof(double) * n), *oi = (double *)malloc(sizeof(double) * n);
    for (int m = 0; m < N; ++m)
        for (int l = 0; l < N; ++l) {
            double c = bo_ctf_env(bo_s2(l, m, N, px), a, A, b);
            gr[(size_t)m * N + l] = F_re[(size_t)m * N + l] * c;
            gi[(size_t)m * N + l] = F_im[(size_t)m * N + l] * c;
        }
    bo_dft2(N, gr, gi, +1, 1.0 / (double)n, or_, oi);
    memcpy(I1, or_, sizeof(double) * n);
    free(gr); free(gi); free(or_); free(oi);
}

/* I1 from a real-space I0: forward DFT (Eq. 2), multiply (Eq. 5), inverse (Eq. 3). */
void bo_apply_ctf(int N, double px, const double *I0, double a, double A, double b, double *I1)
{
    size_t n = (size_t)N * N;
    double *fr = (double *)malloc(sizeof(double) * n), *fi = (double *)malloc(sizeof(double) * n);
    bo_dft2(N, I0, NULL, -1, 1.0, fr, fi);
    bo_apply_ctf_spectrum(N, px, fr, fi, a, A, b, I1);
    free(fr); free(fi);
}

/* Eq. 6: the same I1 by real-space circular convolution with PSF = F^-1(CTF Env).
 * Only used by a pin (Eq. 5 == Eq. 6 on tiny images). */
void bo_apply_psf_realspace(int N, double px, const double *I0, double a, double A, double b, double *I1)
{
    size_t n = (size_t)N * N;
    double *cr = (double *)calloc(n, sizeof(double)), *ci = (double *)calloc(n, sizeof(double));
    double *pr = (double *)malloc(sizeof(double) * n), *pi_ = (double *)malloc(sizeof(double) * n);
    for (int m = 0; m < N; ++m)
        for (int l = 0; l < N; ++l) cr[(size_t)m * N + l] = bo_ctf_env(bo_s2(l, m, N, px), a, A, b);
    bo_dft2(N, cr, ci, +1, 1.0 / (double)n, pr, pi_);
    for (int k = 0; k < N; ++k)
        for (int j = 0; j < N; ++j) {
            double acc = 0;
            for (int kk = 0; kk < N; ++kk)
                for (int jj = 0; jj < N; ++jj)
                    acc += I0[(size_t)kk * N + jj] * pr[(size_t)(((k - kk) % N + N) % N) * N + (((j - jj) % N + N) % N)];
            I1[(size_t)k * N + j] = acc;
        }
    free(cr); free(ci); free(pr); free(pi_);
}

/* ------------------------------------------------------------------ Eq. 7 / Eq. 11-12 */
/* C_co(d) = sum_{j,k} I_obs(j,k) * I1((j+dx) mod N, (k+dy) mod N), |dx|,|dy| <= D   (R4, R5, R6).
 * out[(dy+D)*(2D+1) + (dx+D)].  Direct summation; I1 is tiled periodically first so the
 * inner loop is contiguous (index arithmetic only -- the sum and its order are unchanged). */
void bo_cross_corr_direct(int N, const double *Iobs, const double *I1, int D, double *Cco)
{
    int W = N + 2 * D, S1 = 2 * D + 1;
    double *ext = (double *)malloc(sizeof(double) * (size_t)W * W);
    for (int k = 0; k < W; ++k)
        for (int j = 0; j < W; ++j)
            ext[(size_t)k * W + j] = I1[(size_t)(((k - D) % N + N) % N) * N + (((j - D) % N + N) % N)];
    for (int dy = -D; dy <= D; ++dy)
        for (int dx = -D; dx <= D; ++dx) {
            double acc = 0.0;
            for (int k = 0; k < N; ++k) {
                const double *a = Iobs + (size_t)k * N;
                const double *b = ext + (size_t)(k + dy + D) * W + (dx + D);
                double row = 0.0;
#pragma omp simd reduction(+ : row)
                for (int j = 0; j < N; ++j) row += a[j] * b[j];
                acc += row;
            }
            Cco[(size_t)(dy + D) * S1 + (dx + D)] = acc;
        }
    free(ext);
}

/* Eq. 12 evaluated literally as a naive double sum over (l,n) for every d, under R3:
 * C_co(d) = 1/Npix sum_{l,n} conj(Iobs_hat(l,n)) I1_hat(l,n) exp(+2 pi i (l dx + n dy)/N).
 * O(N^4 S): tiny images only.  Pin for north_star check 1. */
void bo_cross_corr_eq12(int N, const double *Iobs, const double *I1, int D, double *Cco)
{
    size_t n = (size_t)N * N;
    int S1 = 2 * D + 1;
    double *ar = (double *)malloc(sizeof(double) * n), *ai = (double *)malloc(sizeof(double) * n);
    double *br = (double *)malloc(sizeof(double) * n), *bi = (double *)malloc(sizeof(double) * n);
    bo_dft2(N, Iobs, NULL, -1, 1.0, ar, ai);
    bo_dft2(N, I1, NULL, -1, 1.0, br, bi);
    for (int dy = -D; dy <= D; ++dy)
        for (int dx = -D; dx <= D; ++dx) {
            double acc = 0.0;
            for (int m = 0; m < N; ++m)
                for (int l = 0; l < N; ++l) {
                    double pr = ar[m * N + l] * br[m * N + l] + ai[m * N + l] * bi[m * N + l];   /* conj(a) b */
                    double pi_ = ar[m * N + l] * bi[m * N + l] - ai[m * N + l] * br[m * N + l];
                    double ph = 2.0 * BO_PI * ((double)l * dx + (double)m * dy) / N;
                    acc += pr * cos(ph) - pi_ * sin(ph);
                }
            Cco[(size_t)(dy + D) * S1 + (dx + D)] = acc / (double)n;
        }
    free(ar); free(ai); free(br); free(bi);
}

/* Tier B (NOT the definition): the same C_co through an FP64 output-pruned separable DFT of
 * conj(Iobs_hat) I1_hat.  Spectra are full [m][l] arrays.  tw_c/tw_s = cos/sin(2 pi t/N). */
static void bo_cross_corr_dft_spec(int N, const double *ar, const double *ai, const double *br, const double *bi,
                                   int D, const double *tw_c, const double *tw_s, double *Cco, double *wr, double *wi)
{
    int S1 = 2 * D + 1;
    /* pass 1 over m for every l: g(l,dy) = sum_m conj(a) b exp(+2 pi i m dy / N) */
    for (int l = 0; l < N; ++l)
        for (int dy = -D; dy <= D; ++dy) {
            double gr = 0, gi = 0;
            for (int m = 0; m < N; ++m) {
                size_t i = (size_t)m * N + l;
                double pr = ar[i] * br[i] + ai[i] * bi[i], pi_ = ar[i] * bi[i] - ai[i] * br[i];
                int t = (int)((((long long)m * dy) % N + N) % N);
                gr += pr * tw_c[t] - pi_ * tw_s[t];
                gi += pr * tw_s[t] + pi_ * tw_c[t];
            }
            wr[(size_t)(dy + D) * N + l] = gr; wi[(size_t)(dy + D) * N + l] = gi;
        }
    for (int dy = -D; dy <= D; ++dy)
        for (int dx = -D; dx <= D; ++dx) {
            double acc = 0;
            for (int l = 0; l < N; ++l) {
                int t = (int)((((long long)l * dx) % N + N) % N);
                acc += wr[(size_t)(dy + D) * N + l] * tw_c[t] - wi[(size_t)(dy + D) * N + l] * tw_s[t];
            }
            Cco[(size_t)(dy + D) * S1 + (dx + D)] = acc / ((double)N * N);
        }
}

void bo_cross_corr_dft(int N, const double *Iobs, const double *I1, int D, double *Cco)
{
    size_t n = (size_t)N * N;
    double *ar = (double *)malloc(sizeof(double) * n), *ai = (double *)malloc(sizeof(double) * n);
    double *br = (double *)malloc(sizeof(double) * n), *bi = (double *)malloc(sizeof(double) * n);
    double *wr = (double *)malloc(sizeof(double) * (2 * D + 1) * N), *wi = (double *)malloc(sizeof(double) * (2 * D + 1) * N);
    double *tc = (double *)malloc(sizeof(double) * N), *ts = (double *)malloc(sizeof(double) * N);
    for (int t = 0; t < N; ++t) { tc[t] = cos(2.0 * BO_PI * t / N); ts[t] = sin(2.0 * BO_PI * t / N); }
    bo_dft2(N, Iobs, NULL, -1, 1.0, ar, ai);
    bo_dft2(N, I1, NULL, -1, 1.0, br, bi);
    bo_cross_corr_dft_spec(N, ar, ai, br, bi, D, tc, ts, Cco, wr, wi);
    free(ar); free(ai); free(br); free(bi); free(wr); free(wi); free(tc); free(ts);
}

/* ------------------------------------------------------------------ Eq. 8 */
/* log L(omega|m,theta) with I_cal = N_ * I1s - mu (Eq. 7); I1s is I1 already shifted by d. */
double bo_log_lik_eq8(int n, const double *Iobs, const double *I1s, double N_, double mu, double lambda)
{
    double ss = 0.0;
    for (int i = 0; i < n; ++i) {
        double r = Iobs[i] - (N_ * I1s[i] - mu);
        ss += r * r;
    }
    return -ss / (2.0 * lambda * lambda) - 0.5 * n * log(2.0 * BO_PI * lambda * lambda);
}

/* ------------------------------------------------------------------ closed form (stands in for Eq. S8; R1) */
/* (C1): log int dN dmu dlambda L, flat priors on N, mu in (-inf,inf), lambda in (0,inf):
 *   log P = const(n) + (n/2 - 2) log T_c + (3/2 - n/2) log F,
 *   T_c = n C_cc - C_c^2,
 *   F   = n (C_oo C_cc - C_co^2) + 2 C_o C_co C_c - C_cc C_o^2 - C_oo C_c^2,
 *   const(n) = -((n-2)/2) log 2pi + ((n-5)/2) log 2 + lgamma((n-3)/2).
 * C_* are plain sums over pixels (R17).  Evaluated in long double. */
double bo_const_n(double n)
{
    return -0.5 * (n - 2.0) * log(2.0 * BO_PI) + 0.5 * (n - 5.0) * log(2.0) + lgamma(0.5 * (n - 3.0));
}

double bo_log_post_c1(double n_, double Co_, double Coo_, double Cc_, double Ccc_, double Cco_)
{
    long double n = n_, Co = Co_, Coo = Coo_, Cc = Cc_, Ccc = Ccc_, Cco = Cco_;
    long double Tc = n * Ccc - Cc * Cc;
    long double F = n * (Coo * Ccc - Cco * Cco) + 2.0L * Co * Cco * Cc - Ccc * Co * Co - Coo * Cc * Cc;
    /* R14: a noiseless planted image gives F -> 0; clamp 1 - rho^2 >= 1e-300 (F = T_c D (1-rho^2)/n ... ) */
    long double Dn = n * Coo - Co * Co;                 /* n * D */
    long double Fmin = 1e-300L * Tc * Dn / n;
    if (F < Fmin) F = Fmin;
    return (double)((long double)bo_const_n(n_) + (n / 2.0L - 2.0L) * logl(Tc) + (1.5L - n / 2.0L) * logl(F));
}

/* (C2): rho^2 = B^2/(A D), log P = const(n) - 1/2 log T_c - (n-3)/2 [log D + log1p(-rho^2)],
 * A = C_cc - C_c^2/n, B = C_co - C_o C_c/n, D = C_oo - C_o^2/n.  Pin: (C1) == (C2). */
double bo_log_post_c2(double n, double Co, double Coo, double Cc, double Ccc, double Cco)
{
    double A = Ccc - Cc * Cc / n, B = Cco - Co * Cc / n, Dd = Coo - Co * Co / n;
    double rho2 = B * B / (A * Dd);
    double om = -rho2;
    if (1.0 + om < 1e-300) om = -(1.0 - 1e-300);
    return bo_const_n(n) - 0.5 * log(n * A) - 0.5 * (n - 3.0) * (log(Dd) + log1p(om));
}

/* ------------------------------------------------------------------ density-map model (R21) */
/* V(kx,ky,kz) = sum rho(x,y,z) exp(-2 pi i (kx x + ky y + kz z)/N), rho is [z][y][x].  Naive separable. */
void bo_dft3(int N, const double *rho, double *V_re, double *V_im)
{
    size_t n3 = (size_t)N * N * N;
    double *ar = (double *)malloc(sizeof(double) * n3), *ai = (double *)malloc(sizeof(double) * n3);
    double *cw = (double *)malloc(sizeof(double) * N), *sw = (double *)malloc(sizeof(double) * N);
    for (int t = 0; t < N; ++t) { cw[t] = cos(2.0 * BO_PI * t / N); sw[t] = -sin(2.0 * BO_PI * t / N); }
    /* x */
#pragma omp parallel for schedule(static)
    for (long long zy = 0; zy < (long long)N * N; ++zy)
        for (int kx = 0; kx < N; ++kx) {
            double sr = 0, si = 0;
            for (int x = 0; x < N; ++x) {
                int t = (int)(((long long)kx * x) % N);
                sr += rho[zy * N + x] * cw[t]; si += rho[zy * N + x] * sw[t];
            }
            V_re[zy * N + kx] = sr; V_im[zy * N + kx] = si;
        }
    /* y */
#pragma omp parallel for schedule(static)
    for (int z = 0; z < N; ++z)
        for (int ky = 0; ky < N; ++ky)
            for (int kx = 0; kx < N; ++kx) {
                double sr = 0, si = 0;
                for (int y = 0; y < N; ++y) {
                    int t = (int)(((long long)ky * y) % N);
                    size_t i = ((size_t)z * N + y) * N + kx;
                    sr += V_re[i] * cw[t] - V_im[i] * sw[t]; si += V_re[i] * sw[t] + V_im[i] * cw[t];
                }
                ar[((size_t)z * N + ky) * N + kx] = sr; ai[((size_t)z * N + ky) * N + kx] = si;
            }
    /* z */
#pragma omp parallel for schedule(static)
    for (int kz = 0; kz < N; ++kz)
        for (int ky = 0; ky < N; ++ky)
            for (int kx = 0; kx < N; ++kx) {
                double sr = 0, si = 0;
                for (int z = 0; z < N; ++z) {
                    int t = (int)(((long long)kz * z) % N);
                    size_t i = ((size_t)z * N + ky) * N + kx;
                    sr += ar[i] * cw[t] - ai[i] * sw[t]; si += ar[i] * sw[t] + ai[i] * cw[t];
                }
                V_re[((size_t)kz * N + ky) * N + kx] = sr; V_im[((size_t)kz * N + ky) * N + kx] = si;
            }
    free(ar); free(ai); free(cw); free(sw);
}

/* Central section (R21): I0_hat(l,m) = (-1)^(l'+m') * voxel * trilinear[ Vc ]( R^T (l', m', 0) ),
 * Vc(k) = (-1)^(kx+ky+kz) V(k) (origin moved to voxel N/2), l',m' signed frequencies, index units
 * (voxel size = pixel size, same N).  R^T because the model is rotated actively by R (R12):
 * rho'(r) = rho(R^-1 r)  =>  rho'_hat(k) = rho_hat(R^-1 k).  Zero where any |k_i| > N/2 - 1, and zero on
 * the 2-D Nyquist bins |l'| = N/2 or |m'| = N/2 (no unique signed frequency).  The half-plane l' >= 0 is
 * evaluated (for l' = 0 only m' >= 0) and the rest is Hermitian-completed, F(-l,-m) = conj F(l,m), so the
 * image is exactly real.  Output: full spectrum [m][l]. */
void bo_fourier_slice(int N, const double *V_re, const double *V_im, double voxel_A, const double q[4],
                      double *F_re, double *F_im)
{
    double R[9];
    bo_quat_to_matrix(q, R);
    int h = N / 2;
    memset(F_re, 0, sizeof(double) * (size_t)N * N);
    memset(F_im, 0, sizeof(double) * (size_t)N * N);
    for (int ls = 0; ls <= h - 1; ++ls)
        for (int ms = (ls == 0 ? 0 : -h + 1); ms <= h - 1; ++ms) {
            double k[3] = { R[0] * ls + R[3] * ms, R[1] * ls + R[4] * ms, R[2] * ls + R[5] * ms };   /* R^T (ls,ms,0) */
            double vr = 0, vi = 0;
            if (fabs(k[0]) <= h - 1 && fabs(k[1]) <= h - 1 && fabs(k[2]) <= h - 1) {
                int f[3]; double t[3];
                for (int c = 0; c < 3; ++c) { f[c] = (int)floor(k[c]); t[c] = k[c] - f[c]; }
                for (int cz = 0; cz < 2; ++cz)
                    for (int cy = 0; cy < 2; ++cy)
                        for (int cx = 0; cx < 2; ++cx) {
                            int ix = f[0] + cx, iy = f[1] + cy, iz = f[2] + cz;
                            double w = (cx ? t[0] : 1 - t[0]) * (cy ? t[1] : 1 - t[1]) * (cz ? t[2] : 1 - t[2]);
                            double sgn = ((ix + iy + iz) & 1) ? -1.0 : 1.0;
                            size_t i = ((size_t)((iz % N + N) % N) * N + ((iy % N + N) % N)) * N + ((ix % N + N) % N);
                            vr += w * sgn * V_re[i]; vi += w * sgn * V_im[i];
                        }
            }
            double sg = ((ls + ms) & 1) ? -1.0 : 1.0;
            vr *= sg * voxel_A; vi *= sg * voxel_A;
            int l = ls, m = (ms + N) % N;
            int l2 = (N - l) % N, m2 = (N - m) % N;
            if (l2 == l && m2 == m) vi = 0.0;                      /* DC bin is real */
            F_re[(size_t)m * N + l] = vr;   F_im[(size_t)m * N + l] = vi;
            F_re[(size_t)m2 * N + l2] = vr; F_im[(size_t)m2 * N + l2] = -vi;
        }
}

/* ------------------------------------------------------------------ Eq. 9 on the grid (R2, R6, R7, R15, R16) */
typedef struct {
    double m, s;            /* running log-sum-exp: sum = s * exp(m) */
    double best, second;    /* largest and second largest term */
    long long best_flat;    /* flat index ((o*C + c)*S1 + (dy+D))*S1 + (dx+D) of the largest term */
} bo_acc;

static void bo_acc_add(bo_acc *a, double x, long long flat)
{
    if (x == -INFINITY) return;     /* a grid point of weight zero (log-prior -inf, R7) adds nothing to the sum of Eq. 9 */
    if (x > a->m) { a->s = a->s * exp(a->m - x) + 1.0; a->m = x; }
    else a->s += exp(x - a->m);
    if (x > a->best) { a->second = a->best; a->best = x; a->best_flat = flat; }   /* strict: ties keep lowest flat index */
    else if (x > a->second) a->second = x;
}

/* Real-space displacement variant ("in a real space formulation, the cross-correlation is simply calculated for
 * different displacements d"; P:171 it "crops" the borders where the Fourier variant wraps around).  Reading R25
 * (DESIGN.md): the calculated image displaced by d is I_d(r) = I1(r + d) where r + d lies inside the box and 0 elsewhere
 * (the part pushed over the border is cut off, nothing re-enters on the other side), and Eq. 8 is applied to the pair
 * (I_obs, I_d) over all n pixels.  So all three sums that involve the calculated image depend on d:
 *   C_co(d) = sum_{r, r+d in box} I_obs(r) I1(r+d),   C_c(d) = sum_{r, r+d in box} I1(r+d),   C_cc(d) likewise with squares.
 * Output index (dy+D)*(2D+1) + (dx+D), as bo_cross_corr_direct. */
void bo_cropped_sums(int N, const double *obs, const double *I1, int D, double *cco, double *cc, double *ccc)
{
    int S1 = 2 * D + 1;
    for (int dy = -D; dy <= D; ++dy)
        for (int dx = -D; dx <= D; ++dx) {
            long double s_co = 0.0L, s_c = 0.0L, s_cc = 0.0L;
            for (int k = 0; k < N; ++k) {
                int k2 = k + dy;
                if (k2 < 0 || k2 >= N) continue;
                for (int j = 0; j < N; ++j) {
                    int j2 = j + dx;
                    if (j2 < 0 || j2 >= N) continue;
                    double v = I1[(size_t)k2 * N + j2];
                    s_co += (long double)obs[(size_t)k * N + j] * v; s_c += v; s_cc += (long double)v * v;
                }
            }
            size_t d = (size_t)(dy + D) * S1 + (dx + D);
            cco[d] = (double)s_co; cc[d] = (double)s_c; ccc[d] = (double)s_cc;
        }
}

/* Scores images against calc images (orientation o in [o_begin,o_end), all CTFs, all shifts) of ONE model and
 * folds the terms into acc[] in loop order.  lse_m/lse_s/best/second/best_flat are in/out (initialise with
 * -inf, 0, -inf, -inf, -1) so a grid can be processed in orientation chunks with identical results.
 * Per term: log P(C1) + logw,  logw = lp_o + lp_c - log S  (R7; lp_* default to -log O, -log C).
 * model_kind 0: atoms (xyz,radius,weight,Kq);  1: density spectrum (V_re,V_im,voxel_A).
 * tier: 0 = direct summation (the definition), 1 = tier B pruned DFT, 2 = the real-space CROPPING variant (bo_cropped_sums, R25). */
int bo_run(int N, double px, int D, int model_kind,
           int n_atoms, const double *xyz, const double *radius, const double *weight, int Kq,
           const double *V_re, const double *V_im, double voxel_A,
           int n_orient, const double *quats, const double *lp_orient,
           int n_ctf, const double *ctf_a, const double *ctf_A, const double *ctf_b, const double *lp_ctf,
           int n_img, const float *images, int o_begin, int o_end, int tier,
           double *lse_m, double *lse_s, double *best, double *second, long long *best_flat)
{
    size_t n = (size_t)N * N;
    int S1 = 2 * D + 1;
    size_t S = (size_t)S1 * S1;
    double *I0 = (double *)malloc(sizeof(double) * n), *I1 = (double *)malloc(sizeof(double) * n);
    double *fr = (double *)malloc(sizeof(double) * n), *fi = (double *)malloc(sizeof(double) * n);
    double *obs = (double *)malloc(sizeof(double) * n * n_img);
    double *Co = (double *)malloc(sizeof(double) * n_img), *Coo = (double *)malloc(sizeof(double) * n_img);
    double *cco = (double *)malloc(sizeof(double) * S * n_img);
    double *ccd = NULL, *cccd = NULL;                       /* tier 2: C_c(d), C_cc(d) per image and shift */
    if (tier == 2) { ccd = (double *)malloc(sizeof(double) * S * n_img); cccd = (double *)malloc(sizeof(double) * S * n_img); }
    /* tier B scratch */
    double *or_ = NULL, *oi = NULL, *br = NULL, *bi = NULL, *tc = NULL, *ts = NULL;
    for (int w = 0; w < n_img; ++w) {                      /* "Eqs. S3, S5": C_o, C_oo */
        double s1 = 0, s2 = 0;
        for (size_t i = 0; i < n; ++i) {
            double v = (double)images[(size_t)w * n + i];
            obs[(size_t)w * n + i] = v; s1 += v; s2 += v * v;
        }
        Co[w] = s1; Coo[w] = s2;
    }
    if (tier == 1) {
        or_ = (double *)malloc(sizeof(double) * n * n_img); oi = (double *)malloc(sizeof(double) * n * n_img);
        br = (double *)malloc(sizeof(double) * n); bi = (double *)malloc(sizeof(double) * n);
        tc = (double *)malloc(sizeof(double) * N); ts = (double *)malloc(sizeof(double) * N);
        for (int t = 0; t < N; ++t) { tc[t] = cos(2.0 * BO_PI * t / N); ts[t] = sin(2.0 * BO_PI * t / N); }
        for (int w = 0; w < n_img; ++w) bo_dft2(N, obs + (size_t)w * n, NULL, -1, 1.0, or_ + (size_t)w * n, oi + (size_t)w * n);
    }
    double logS = log((double)S);
    for (int o = o_begin; o < o_end; ++o) {
        if (model_kind == 0) {
            bo_project_atoms(n_atoms, xyz, radius, weight, quats + 4 * o, N, px, Kq, I0);   /* Eq. 1 */
            bo_dft2(N, I0, NULL, -1, 1.0, fr, fi);                                           /* Eq. 2 */
        } else {
            bo_fourier_slice(N, V_re, V_im, voxel_A, quats + 4 * o, fr, fi);                /* R21 */
        }
        for (int c = 0; c < n_ctf; ++c) {
            bo_apply_ctf_spectrum(N, px, fr, fi, ctf_a[c], ctf_A[c], ctf_b[c], I1);          /* Eqs. 3-5 */
            double Cc = 0, Ccc = 0;                                                          /* "Eqs. S4, S6" */
            for (size_t i = 0; i < n; ++i) { Cc += I1[i]; Ccc += I1[i] * I1[i]; }
            if (tier == 1) bo_dft2(N, I1, NULL, -1, 1.0, br, bi);
#pragma omp parallel
            {
                double *wr = NULL, *wi = NULL;
                if (tier == 1) { wr = (double *)malloc(sizeof(double) * S1 * N); wi = (double *)malloc(sizeof(double) * S1 * N); }
#pragma omp for schedule(dynamic, 1)
                for (int w = 0; w < n_img; ++w) {
                    if (tier == 0) bo_cross_corr_direct(N, obs + (size_t)w * n, I1, D, cco + (size_t)w * S);
                    else if (tier == 2) bo_cropped_sums(N, obs + (size_t)w * n, I1, D, cco + (size_t)w * S, ccd + (size_t)w * S, cccd + (size_t)w * S);
                    else bo_cross_corr_dft_spec(N, or_ + (size_t)w * n, oi + (size_t)w * n, br, bi, D, tc, ts, cco + (size_t)w * S, wr, wi);
                }
                free(wr); free(wi);
            }
            double logw = (lp_orient ? lp_orient[o] : -log((double)n_orient)) + (lp_ctf ? lp_ctf[c] : -log((double)n_ctf)) - logS;
            for (int w = 0; w < n_img; ++w) {
                bo_acc a = { lse_m[w], lse_s[w], best[w], second[w], best_flat[w] };
                for (size_t d = 0; d < S; ++d) {
                    double lp = tier == 2 ? bo_log_post_c1((double)n, Co[w], Coo[w], ccd[(size_t)w * S + d], cccd[(size_t)w * S + d], cco[(size_t)w * S + d])
                                          : bo_log_post_c1((double)n, Co[w], Coo[w], Cc, Ccc, cco[(size_t)w * S + d]);
                    bo_acc_add(&a, lp + logw, ((long long)o * n_ctf + c) * (long long)S + (long long)d);
                }
                lse_m[w] = a.m; lse_s[w] = a.s; best[w] = a.best; second[w] = a.second; best_flat[w] = a.best_flat;
            }
        }
    }
    free(I0); free(I1); free(fr); free(fi); free(obs); free(Co); free(Coo); free(cco); free(ccd); free(cccd);
    free(or_); free(oi); free(br); free(bi); free(tc); free(ts);
    return 0;
}

/* One (image, calc image) pair: the whole (2D+1)^2 map of log P(C1) + logw.  For sampled-tuple parity. */
void bo_shift_map(int N, int D, const float *image, const double *I1, double logw, int tier, double *out)
{
    size_t n = (size_t)N * N;
    int S1 = 2 * D + 1;
    double *obs = (double *)malloc(sizeof(double) * n), *cco = (double *)malloc(sizeof(double) * S1 * S1);
    double Co = 0, Coo = 0, Cc = 0, Ccc = 0;
    for (size_t i = 0; i < n; ++i) { obs[i] = (double)image[i]; Co += obs[i]; Coo += obs[i] * obs[i]; Cc += I1[i]; Ccc += I1[i] * I1[i]; }
    if (tier == 0) bo_cross_corr_direct(N, obs, I1, D, cco); else bo_cross_corr_dft(N, obs, I1, D, cco);
    for (int d = 0; d < S1 * S1; ++d) out[d] = bo_log_post_c1((double)n, Co, Coo, Cc, Ccc, cco[d]) + logw;
    free(obs); free(cco);
}

int bo_num_threads(void)
{
#ifdef _OPENMP
    return omp_get_max_threads();
#else
    return 1;
#endif
}
