// precompute.cu -- SURVEY section 8 rows a0 (observed images), a1 (atom projection, Eq. 1), a1' (Fourier slice, R21),
// a2 (forward transform, Eq. 2) and a3 (CTF tables, Eq. 5, and the per-calc-image statistics).  Everything here runs
// once per image / per (model, orientation) / per (model, orientation, CTF): <= 1/N_img of the hot loop's work.  It is
// done in FP64 so that (i) the FP32 operands of the hot loop are correctly rounded and (ii) the FP64 re-scoring pass
// (a7) can reuse the same spectra.
#include "common.cuh"
#include <math_constants.h>

namespace bioem {

// deterministic block sum (fixed tree), result valid in thread 0
template <int NT>
__device__ __forceinline__ double block_sum(double v, double *sh)
{
    sh[threadIdx.x] = v;
    __syncthreads();
#pragma unroll
    for (int s = NT / 2; s >= 1; s >>= 1) {
        if ((int)threadIdx.x < s) sh[threadIdx.x] += sh[threadIdx.x + s];
        __syncthreads();
    }
    double r = sh[0];
    __syncthreads();
    return r;
}

// ------------------------------------------------------------------------------------------------ a0: C_o, C_oo
// centered = I_obs - mean (so the correlation with it IS B(d), SURVEY 7 hard part 2);  Dw = sum centered^2 = C_oo - C_o^2/n.
__global__ void __launch_bounds__(256) k_image_stats(const float *img, int n, double *centered, double *Dw)
{
    __shared__ double sh[256];
    const float *src = img + (size_t)blockIdx.x * n;
    double *dst = centered + (size_t)blockIdx.x * n;
    double s = 0;
    for (int i = threadIdx.x; i < n; i += 256) s += (double)src[i];
    double mean = block_sum<256>(s, sh) / n;
    double q = 0;
    for (int i = threadIdx.x; i < n; i += 256) { double v = (double)src[i] - mean; dst[i] = v; q += v * v; }
    q = block_sum<256>(q, sh);
    if (threadIdx.x == 0) Dw[blockIdx.x] = q;
}

cudaError_t launch_image_stats(const float *img, int n_img, int N, double *centered, double *Dw, cudaStream_t st)
{
    k_image_stats<<<n_img, 256, 0, st>>>(img, N * N, centered, Dw);
    return cudaGetLastError();
}

// flags[0] |= 1 when an image has no variance (D_omega = sum o^2 <= 0, or not finite): rho^2 = B^2 / (A D) is undefined for it
__global__ void k_beta(const double *Dw, int n, float *beta, int *flags)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    const double d = Dw[i];
    if (!(d > 0.0) || isinf(d)) atomicOr(flags, 1);
    beta[i] = (float)(1.0 / sqrt(d));
}
cudaError_t launch_beta(const double *Dw, int n_img, float *beta, int *flags, cudaStream_t st)
{
    k_beta<<<(n_img + 255) / 256, 256, 0, st>>>(Dw, n_img, beta, flags);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ generic FP64 1-D transform (two-step)
// y[k] = sum_e x[e] exp(SIGN 2 pi i e k / N), k < kout.  Sequence g: batch b = g / spb, s = g % spb;
// x[e] at in + b*ibs + s*iss + e*ies, y[k] at out + b*obs + s*oss + k*oes.  IN = IN_CPLX: complex input; IN_REAL: real doubles;
// IN_FIXED: the 64-bit fixed-point pixels k_project accumulates, x = (double)q * in_scale (the conversion pass of its own that
// round 2 began with was 4 ms of the Ensemble step).  out32 != NULL: the result is also written as complex<float> at the same
// index (the FP32 copy the hot loop reads; was a pass of its own too).
enum { IN_CPLX = 0, IN_REAL = 1, IN_FIXED = 2 };
template <int N, int SIGN, int IN, int SPB>
__global__ void __launch_bounds__(SPB *(N / n1_of(N))) k_fft1d_f64(const void *in_, double in_scale, long ibs, long iss, long ies, cd *out, cf *out32,
                                                                    long obs, long oss, long oes, int nseq, int spb, int kout)
{
    constexpr int N1 = n1_of(N), N2 = N / N1, ZP = N1 + 1, LB = ilog2(N1), NT = SPB * N2;
    __shared__ cd Z[SPB * N2 * ZP];
    __shared__ cd tw[N];
    const int tid = threadIdx.x;
    for (int i = tid; i < N; i += NT) {
        double sn, cs;
        sincospi(2.0 * i / N, &sn, &cs);
        tw[i] = {cs, SIGN > 0 ? sn : -sn};
    }
    const int sl = tid / N2, t = tid % N2;
    const int g = blockIdx.x * SPB + sl;
    if (g < nseq) {
        const long off = (long)(g / spb) * ibs + (long)(g % spb) * iss;
        cd a[N1];
#pragma unroll
        for (int j = 0; j < N1; ++j) {
            long e = off + (long)(N2 * j + t) * ies;
            if (IN == IN_REAL) a[j] = {reinterpret_cast<const double *>(in_)[e], 0.0};
            else if (IN == IN_FIXED) a[j] = {(double)reinterpret_cast<const long long *>(in_)[e] * in_scale, 0.0};
            else a[j] = reinterpret_cast<const cd *>(in_)[e];
        }
        fft_dif<double, N1, SIGN>(a);
#pragma unroll
        for (int r = 0; r < N1; ++r) Z[(sl * N2 + t) * ZP + bitrev(r, LB)] = a[r];
    }
    __syncthreads();
    for (int idx = tid; idx < SPB * kout; idx += NT) {
        const int s2 = idx / kout, k = idx % kout;
        const int g2 = blockIdx.x * SPB + s2;
        if (g2 >= nseq) break;
        const int k1 = k % N1;
        cd acc = {0.0, 0.0};
#pragma unroll
        for (int tt = 0; tt < N2; ++tt) {
            cd w = tw[(tt * k) % N], z = Z[(s2 * N2 + tt) * ZP + k1];
            acc.x += w.x * z.x - w.y * z.y;
            acc.y += w.x * z.y + w.y * z.x;
        }
        const long oi = (long)(g2 / spb) * obs + (long)(g2 % spb) * oss + (long)k * oes;
        out[oi] = acc;
        if (out32) out32[oi] = {(float)acc.x, (float)acc.y};
    }
}

// sequences per block: as many as keep the Z tile under ~35 KB of static shared memory, so that the block's twiddle table
// (N sincospi) is shared by 8-32 sequences and not by 4 (round 1: 32-thread blocks; the transforms of the 73 728 Ensemble
// projections took 25 ms)
__host__ __device__ constexpr int spb_of(int N) { return N == 64 ? 32 : N == 128 ? 16 : N == 96 ? 16 : N == 170 ? 4 : 8; }

template <int N, int SIGN, int IN>
static cudaError_t fft1d_n(const void *in, double in_scale, long ibs, long iss, long ies, cd *out, cf *out32, long obs, long oss, long oes, int nseq,
                           int spb, int kout, cudaStream_t st)
{
    constexpr int SPB = spb_of(N);
    k_fft1d_f64<N, SIGN, IN, SPB><<<(nseq + SPB - 1) / SPB, SPB * (N / n1_of(N)), 0, st>>>(in, in_scale, ibs, iss, ies, out, out32, obs, oss, oes, nseq,
                                                                                      spb, kout);
    return cudaGetLastError();
}

template <int SIGN, int IN>
static cudaError_t fft1d(int N, const void *in, long ibs, long iss, long ies, cd *out, long obs, long oss, long oes, int nseq,
                         int spb, int kout, cudaStream_t st, double in_scale = 1.0, cf *out32 = nullptr)
{
    switch (N) {
    case 64: return fft1d_n<64, SIGN, IN>(in, in_scale, ibs, iss, ies, out, out32, obs, oss, oes, nseq, spb, kout, st);
    case 96: return fft1d_n<96, SIGN, IN>(in, in_scale, ibs, iss, ies, out, out32, obs, oss, oes, nseq, spb, kout, st);
    case 128: return fft1d_n<128, SIGN, IN>(in, in_scale, ibs, iss, ies, out, out32, obs, oss, oes, nseq, spb, kout, st);
    case 160: return fft1d_n<160, SIGN, IN>(in, in_scale, ibs, iss, ies, out, out32, obs, oss, oes, nseq, spb, kout, st);
    case 170: return fft1d_n<170, SIGN, IN>(in, in_scale, ibs, iss, ies, out, out32, obs, oss, oes, nseq, spb, kout, st);
    case 192: return fft1d_n<192, SIGN, IN>(in, in_scale, ibs, iss, ies, out, out32, obs, oss, oes, nseq, spb, kout, st);
    case 224: return fft1d_n<224, SIGN, IN>(in, in_scale, ibs, iss, ies, out, out32, obs, oss, oes, nseq, spb, kout, st);
    case 256: return fft1d_n<256, SIGN, IN>(in, in_scale, ibs, iss, ies, out, out32, obs, oss, oes, nseq, spb, kout, st);
    default: return cudaErrorInvalidValue;
    }
}

// a0 / a2: real [b][k][j] -> half spectrum [b][l][m], forward sign (Eq. 2 under R3).  tmp: [b][l][k].
cudaError_t launch_fft2_r2c_f64(const double *in, int batch, int N, cd *tmp, cd *out, cudaStream_t st)
{
    const int NC = N / 2 + 1;
    const long H = (long)NC * N;
    // along x: sequence = row k of image b
    cudaError_t e = fft1d<-1, IN_REAL>(N, in, (long)N * N, N, 1, tmp, H, 1, N, batch * N, N, NC, st);
    if (e != cudaSuccess) return e;
    // along y: sequence = column l of image b
    return fft1d<-1, IN_CPLX>(N, tmp, H, N, 1, out, H, N, 1, batch * NC, NC, N, st);
}
// the same for the fixed-point projections of k_project (x = q * in_scale), with the FP32 copy of the spectrum written alongside
cudaError_t launch_fft2_r2c_fixed(const long long *in, double in_scale, int batch, int N, cd *tmp, cd *out, cf *out32, cudaStream_t st)
{
    const int NC = N / 2 + 1;
    const long H = (long)NC * N;
    cudaError_t e = fft1d<-1, IN_FIXED>(N, in, (long)N * N, N, 1, tmp, H, 1, N, batch * N, N, NC, st, in_scale);
    if (e != cudaSuccess) return e;
    return fft1d<-1, IN_CPLX>(N, tmp, H, N, 1, out, H, N, 1, batch * NC, NC, N, st, 1.0, out32);
}

__global__ void k_cast_spec(const cd *in, cf *out, size_t n)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { cd v = in[i]; out[i] = {(float)v.x, (float)v.y}; }
}
cudaError_t launch_cast_spectrum(const cd *in, cf *out, size_t count, cudaStream_t st)
{
    k_cast_spec<<<(unsigned)((count + 255) / 256), 256, 0, st>>>(in, out, count);
    return cudaGetLastError();
}

__global__ void k_zero_dc(cd *spec, int batch, size_t H)
{
    int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i < batch) spec[(size_t)i * H] = {0.0, 0.0};
}
cudaError_t launch_zero_dc(cd *spec, int batch, size_t H, cudaStream_t st)
{
    k_zero_dc<<<(batch + 255) / 256, 256, 0, st>>>(spec, batch, H);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ a1: Eq. 1, R10-R12
// grid = (orientation, block of 256 atoms): one thread per atom, so that a batch of 256 orientations of a 3000-atom model is
// 3072 CTAs and not 256 (round 1: one CTA per orientation, 1.7 CTAs per SM, bound by the latency of the FP64 square roots).  The pixel integral is the 4x4 mid-point sum of the chord length
// 2 sqrt(R^2 - r^2)_+ (R10), accumulated as 64-bit FIXED-POINT integers with atomics: integer addition is associative,
// so the image is bit-identical from run to run whatever the order of the atoms (no float atomics).
__global__ void __launch_bounds__(256) k_project(const double *xyz, const double *rad, const double *wt, int n_atoms, const double *rot,
                                                 int N, double px, double fx_scale, long long *acc)
{
    const double *R = rot + (size_t)blockIdx.x * 9;
    unsigned long long *img = reinterpret_cast<unsigned long long *>(acc) + (size_t)blockIdx.x * N * N;
    constexpr int KQ = 4;
    const double h = px / KQ;
    for (int a = blockIdx.y * 256 + threadIdx.x; a < n_atoms; a += 256 * gridDim.y) {
        const double x0 = xyz[3 * a], y0 = xyz[3 * a + 1], z0 = xyz[3 * a + 2];
        const double xr = R[0] * x0 + R[1] * y0 + R[2] * z0;
        const double yr = R[3] * x0 + R[4] * y0 + R[5] * z0;
        const double Ra = rad[a], R2 = Ra * Ra;
        const double dens = wt[a] / (4.0 / 3.0 * CUDART_PI * Ra * Ra * Ra) * h * h;
        // pixel j covers [(j - N/2 - 1/2) px, (j - N/2 + 1/2) px]: it meets the disc iff A < j < B with A = (xr - Ra)/px + N/2 - 1/2,
        // B = (xr + Ra)/px + N/2 + 1/2, i.e. floor(A) + 1 <= j <= ceil(B) - 1.  No spare pixel is needed against rounding: a pixel
        // that A or B misses by an ulp overlaps the disc by a sliver that holds none of the 4x4 mid-points (they sit px/8 inside
        // the pixel), so it adds exactly 0 on both sides of the parity test.
        const int j0 = (int)floor((xr - Ra) / px + N / 2 - 0.5) + 1, j1 = (int)ceil((xr + Ra) / px + N / 2 + 0.5) - 1;
        const int k0 = (int)floor((yr - Ra) / px + N / 2 - 0.5) + 1, k1 = (int)ceil((yr + Ra) / px + N / 2 + 0.5) - 1;
        for (int k = k0; k <= k1; ++k) {
            if (k < 0 || k >= N) continue;
            const double yc = (k - N / 2) * px - 0.5 * px - yr;
            for (int j = j0; j <= j1; ++j) {
                if (j < 0 || j >= N) continue;
                const double xc = (j - N / 2) * px - 0.5 * px - xr;
                double s = 0.0;
#pragma unroll
                for (int sy = 0; sy < KQ; ++sy) {
                    const double dy = yc + (sy + 0.5) * h;
#pragma unroll
                    for (int sx = 0; sx < KQ; ++sx) {
                        const double dx = xc + (sx + 0.5) * h;
                        const double d2 = R2 - dx * dx - dy * dy;
                        if (d2 > 0.0 && d2 < 1e-30) s += 2.0 * sqrt(d2);           // below the FP32 range of the seed
                        else if (d2 > 0.0) {
                            // sqrt(d2) = d2 r with r = 1/sqrt(d2) from the FP32 unit (relative error 1e-7), one Newton step in FP64
                            // (error 1e-14 relative, far below the 2^-58 fixed-point quantum): a third of DSQRT's FP64 work
                            const double r = (double)rsqrtf((float)d2);
                            const double s0 = d2 * r;
                            s += 2.0 * fma(0.5 * r, fma(-s0, s0, d2), s0);
                        }
                    }
                }
                if (s > 0.0) {
                    long long q = __double2ll_rn(dens * s * fx_scale);
                    atomicAdd(img + (size_t)k * N + j, (unsigned long long)q);
                }
            }
        }
    }
}

// acc: [n_orient][N][N] fixed-point pixels, value = acc / fx_scale (launch_fft2_r2c_fixed converts on load)
cudaError_t launch_project_atoms(const double *xyz, const double *rad, const double *wt, int n_atoms, const double *rot, int n_orient,
                                 int N, double px, double fx_scale, long long *acc, cudaStream_t st)
{
    size_t n = (size_t)n_orient * N * N;
    cudaError_t e = cudaMemsetAsync(acc, 0, n * sizeof(long long), st);
    if (e != cudaSuccess) return e;
    k_project<<<dim3(n_orient, (n_atoms + 255) / 256), 256, 0, st>>>(xyz, rad, wt, n_atoms, rot, N, px, fx_scale, acc);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ a1': density model (R21)
__global__ void k_rho_to_cd(const float *rho, cd *out, size_t n)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) out[i] = {(double)rho[i], 0.0};
}
__global__ void k_centre_sign(cd *V, int N)
{
    size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    size_t n3 = (size_t)N * N * N;
    if (i < n3) {
        int kx = (int)(i % N), ky = (int)((i / N) % N), kz = (int)(i / ((size_t)N * N));
        if ((kx + ky + kz) & 1) { cd v = V[i]; V[i] = {-v.x, -v.y}; }       // (-1)^(kx+ky+kz): parity of the index == parity of the signed frequency (N even)
    }
}

// 3-D forward DFT of rho[z][y][x]; result (with the origin moved to voxel N/2) in work_a.
cudaError_t launch_dft3_f64(const float *rho, int N, cd *work_a, cd *work_b, cudaStream_t st)
{
    const size_t n3 = (size_t)N * N * N;
    const long N2 = (long)N * N;
    k_rho_to_cd<<<(unsigned)((n3 + 255) / 256), 256, 0, st>>>(rho, work_a, n3);
    // x: sequences (z,y) contiguous
    cudaError_t e = fft1d<-1, IN_CPLX>(N, work_a, 0, N, 1, work_b, 0, N, 1, N * N, N * N, N, st);
    if (e != cudaSuccess) return e;
    // y: batch z, sequence kx, element stride N
    e = fft1d<-1, IN_CPLX>(N, work_b, N2, 1, N, work_a, N2, 1, N, N * N, N, N, st);
    if (e != cudaSuccess) return e;
    // z: sequence (ky,kx) flat, element stride N^2
    e = fft1d<-1, IN_CPLX>(N, work_a, 0, 1, N2, work_b, 0, 1, N2, N * N, N * N, N, st);
    if (e != cudaSuccess) return e;
    e = cudaMemcpyAsync(work_a, work_b, n3 * sizeof(cd), cudaMemcpyDeviceToDevice, st);
    if (e != cudaSuccess) return e;
    k_centre_sign<<<(unsigned)((n3 + 255) / 256), 256, 0, st>>>(work_a, N);
    return cudaGetLastError();
}

// Central section: F0(l,m) = (-1)^(l'+m') voxel * trilinear[Vc](R^T (l',m',0)); zero outside |k_i| <= N/2-1 and on the
// 2-D Nyquist bins; column l = 0 is completed from m' >= 0 so that the spectrum is exactly Hermitian.
__global__ void __launch_bounds__(256) k_slice(const cd *Vc, int N, double voxel, const double *rot, cd *out)
{
    const double *R = rot + (size_t)blockIdx.y * 9;
    const int NC = N / 2 + 1, h = N / 2;
    const int idx = blockIdx.x * 256 + threadIdx.x;
    if (idx >= NC * N) return;
    const int l = idx / N, m = idx % N;
    int ls = l, ms = (m <= h) ? m : m - N;
    cd r = {0.0, 0.0};
    bool conj = false;
    if (ls == 0 && ms < 0) { ms = -ms; conj = true; }
    if (ls < h && ms > -h && ms < h) {
        const double k[3] = {R[0] * ls + R[3] * ms, R[1] * ls + R[4] * ms, R[2] * ls + R[5] * ms};
        if (fabs(k[0]) <= h - 1 && fabs(k[1]) <= h - 1 && fabs(k[2]) <= h - 1) {
            int f[3];
            double t[3];
#pragma unroll
            for (int c = 0; c < 3; ++c) { double fl = floor(k[c]); f[c] = (int)fl; t[c] = k[c] - fl; }
#pragma unroll
            for (int cz = 0; cz < 2; ++cz)
#pragma unroll
                for (int cy = 0; cy < 2; ++cy)
#pragma unroll
                    for (int cx_ = 0; cx_ < 2; ++cx_) {
                        const int ix = ((f[0] + cx_) % N + N) % N, iy = ((f[1] + cy) % N + N) % N, iz = ((f[2] + cz) % N + N) % N;
                        const double w = (cx_ ? t[0] : 1 - t[0]) * (cy ? t[1] : 1 - t[1]) * (cz ? t[2] : 1 - t[2]);
                        const cd v = Vc[((size_t)iz * N + iy) * N + ix];
                        r.x += w * v.x; r.y += w * v.y;
                    }
            const double sg = ((ls + ms) & 1) ? -voxel : voxel;
            r.x *= sg; r.y *= sg;
            if (conj) r.y = -r.y;
            if (ls == 0 && ms == 0) r.y = 0.0;
        }
    }
    out[(size_t)blockIdx.y * NC * N + idx] = r;
}

cudaError_t launch_slice_f64(const cd *Vc, int N, double voxel, const double *rot, int n_orient, cd *out, cudaStream_t st)
{
    const int NC = N / 2 + 1;
    dim3 grid((NC * N + 255) / 256, n_orient);
    k_slice<<<grid, 256, 0, st>>>(Vc, N, voxel, rot, out);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ a3: Eqs. 4-5
__global__ void k_ctf_tables(const double *a, const double *A, const double *b, int N, double px, double *K64, float *K32)
{
    const int NC = N / 2 + 1;
    const int idx = blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= NC * N) return;
    const int c = blockIdx.y;
    const int l = idx / N, m = idx % N;
    const int ms = (m <= N / 2) ? m : m - N;
    const double f = 2.0 * CUDART_PI / (N * px);
    const double s2 = f * f * ((double)l * l + (double)ms * ms);
    const double ph = 0.5 * a[c] * s2;
    double sn, cs;
    sincos(ph, &sn, &cs);
    const double v = (-A[c] * cs - sqrt(1.0 - A[c] * A[c]) * sn) * exp(-0.5 * b[c] * s2);
    K64[(size_t)c * NC * N + idx] = v;
    K32[(size_t)c * NC * N + idx] = (float)v;
}

cudaError_t launch_ctf_tables(const double *a, const double *A, const double *b, int n_ctf, int N, double px, double *K64, float *K32,
                              cudaStream_t st)
{
    const int NC = N / 2 + 1;
    dim3 grid((NC * N + 255) / 256, n_ctf);
    k_ctf_tables<<<grid, 256, 0, st>>>(a, A, b, N, px, K64, K32);
    return cudaGetLastError();
}

// T_c = n C_cc - C_c^2 = sum_{s != 0} |F0(s) K_c(s)|^2 (Plancherel; "Eqs. S4, S6"), Hermitian weights:
// columns l = 0 and l = N/2 count once, the others twice.  One CTA per (model, orientation), loop over CTFs.
__global__ void __launch_bounds__(256) k_calc_stats(const cd *F0, const double *K64, int n_orient, int n_orient_total, int n_ctf, int N, const double *lp_orient,
                                                    const double *lp_ctf, double log_shifts, double *Tc64, double *h64, float *alpha32,
                                                    float *h32, int *flags)
{
    __shared__ double sh[256];
    const int NC = N / 2 + 1, H = NC * N;
    const int mo = blockIdx.x, o = mo % n_orient;
    const cd *F = F0 + (size_t)mo * H;
    constexpr int CC = 8;                                             // CTF sets per pass over the spectrum (the power |F0|^2 is formed once per pass)
    for (int c0 = 0; c0 < n_ctf; c0 += CC) {
        const int nc = min(CC, n_ctf - c0);
        double acc[CC];
#pragma unroll
        for (int u = 0; u < CC; ++u) acc[u] = 0.0;
        for (int i = threadIdx.x + 1; i < H; i += 256) {              // i = 0 is the DC bin
            const int l = i / N;
            const cd v = F[i];
            const double pw = ((l == 0 || l == N / 2) ? 1.0 : 2.0) * (v.x * v.x + v.y * v.y);
#pragma unroll
            for (int u = 0; u < CC; ++u)
                if (u < nc) { const double k = K64[(size_t)(c0 + u) * H + i]; acc[u] += pw * k * k; }
        }
        for (int u = 0; u < nc; ++u) {
            const int c = c0 + u;
            const double s = block_sum<256>(acc[u], sh);
            if (threadIdx.x == 0) {
                const size_t moc = (size_t)mo * n_ctf + c;
                const double n = (double)N * N;
                const double lpo = lp_orient ? lp_orient[o] : -log((double)n_orient_total);   // a rank that scores a slice of the grid still weighs with the whole grid (R7)
                const double lpc = lp_ctf ? lp_ctf[c] : -log((double)n_ctf);
                const double h = -0.5 * log(s) + lpo + lpc - log_shifts;
                if (!(s > 0.0) || isinf(s)) atomicOr(flags, 2);          // empty calculated image: T_c = 0, rho^2 undefined
                Tc64[moc] = s; h64[moc] = h;
                alpha32[moc] = (float)(1.0 / sqrt(n * s)); h32[moc] = (float)(h * 1.4426950408889634);   // FP32 path: base-2 units
            }
        }
    }
}

cudaError_t launch_calc_stats(const cd *F0, const double *K64, int n_mo, int n_orient, int n_orient_total, int n_ctf, int N, const double *lp_orient,
                              const double *lp_ctf, double log_shifts, double *Tc64, double *h64, float *alpha32, float *h32,
                              int *flags, cudaStream_t st)
{
    k_calc_stats<<<n_mo, 256, 0, st>>>(F0, K64, n_orient, n_orient_total, n_ctf, N, lp_orient, lp_ctf, log_shifts, Tc64, h64, alpha32, h32, flags);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ debug: I1 = F^-1(F0 K)   (Eq. 3)
__global__ void __launch_bounds__(256) k_calc_image(const cd *F0, const double *K64, int N, double *out)
{
    const int NC = N / 2 + 1;
    const int pix = blockIdx.x * 256 + threadIdx.x;
    if (pix >= N * N) return;
    const int k = pix / N, j = pix % N;
    double acc = 0.0;
    for (int l = 0; l < NC; ++l) {
        const double w = (l == 0 || l == N / 2) ? 1.0 : 2.0;
        for (int m = 0; m < N; ++m) {
            const cd v = F0[(size_t)l * N + m];
            const double kk = K64[(size_t)l * N + m];
            double sn, cs;
            sincospi(2.0 * (double)((l * j + m * k) % N) / N, &sn, &cs);
            acc += w * kk * (v.x * cs - v.y * sn);
        }
    }
    out[pix] = acc / ((double)N * N);
}
cudaError_t launch_calc_image(const cd *F0, const double *K64, int N, double *out, cudaStream_t st)
{
    k_calc_image<<<(N * N + 255) / 256, 256, 0, st>>>(F0, K64, N, out);
    return cudaGetLastError();
}

// ------------------------------------------------------------------------------------------------ synthetic map
// I_cal of Eq. 7 for one parameter set: out = N I_d - mu, I_d(k, j) = I1(k + dy, j + dx), wrapped around the box (crop = 0,
// the Fourier variant, R5) or zero outside it (crop = 1, the real-space variant, R25).  obs = NULL: N = 1, mu = 0; otherwise the
// (N, mu) that maximise Eq. 8 for that image (normal equations of sum (obs - N I_d + mu)^2).  One CTA, FP64, fixed summation
// order: thread t takes pixels t, t + 1024, ...; lanes by xor-tree; warps in order.
__global__ void __launch_bounds__(1024) k_synth_map(const double *I1, const float *obs, int N, int dx, int dy, int crop, float *out, double *norm_offset)
{
    __shared__ double sh[4][32];
    __shared__ double fit[2];
    const int n = N * N, tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    auto displaced = [&](int pix) -> double {
        int k2 = pix / N + dy, j2 = pix % N + dx;
        if (crop) {
            if (k2 < 0 || k2 >= N || j2 < 0 || j2 >= N) return 0.0;
        } else {
            k2 = (k2 % N + N) % N; j2 = (j2 % N + N) % N;
        }
        return I1[(size_t)k2 * N + j2];
    };
    double nn = 1.0, mu = 0.0;
    if (obs) {
        double v[4] = {0.0, 0.0, 0.0, 0.0};                          // C_o, C_c, C_cc, C_co
        for (int pix = tid; pix < n; pix += 1024) {
            const double o = obs[pix], c = displaced(pix);
            v[0] += o; v[1] += c; v[2] += c * c; v[3] += o * c;
        }
#pragma unroll
        for (int q = 0; q < 4; ++q) {
            for (int off = 16; off >= 1; off >>= 1) v[q] += __shfl_xor_sync(0xffffffffu, v[q], off);
            if (lane == 0) sh[q][warp] = v[q];
        }
        __syncthreads();
        if (tid == 0) {
            double s[4] = {0.0, 0.0, 0.0, 0.0};
            for (int q = 0; q < 4; ++q)
                for (int w = 0; w < 32; ++w) s[q] += sh[q][w];
            const double den = (double)n * s[2] - s[1] * s[1];     // T_c of the displaced image
            const double a = den > 0.0 ? ((double)n * s[3] - s[0] * s[1]) / den : 0.0;      // a constant calculated image: only the offset fits
            fit[0] = a; fit[1] = (a * s[1] - s[0]) / (double)n;
        }
        __syncthreads();
        nn = fit[0]; mu = fit[1];
    }
    for (int pix = tid; pix < n; pix += 1024) out[pix] = (float)(nn * displaced(pix) - mu);
    if (tid == 0 && norm_offset) { norm_offset[0] = nn; norm_offset[1] = mu; }
}
cudaError_t launch_synth_map(const double *I1, const float *obs, int N, int dx, int dy, int crop, float *out, double *norm_offset, cudaStream_t st)
{
    k_synth_map<<<1, 1024, 0, st>>>(I1, obs, N, dx, dy, crop, out, norm_offset);
    return cudaGetLastError();
}

}  // namespace bioem
