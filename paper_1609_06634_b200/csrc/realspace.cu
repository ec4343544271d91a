// realspace.cu -- SURVEY section 8(f) #3: the REAL-SPACE, CROPPING displacement variant ("in a real space formulation, the
// cross-correlation is simply calculated for different displacements d"; it crops at the borders where the Fourier
// variant wraps around; the displacement loop innermost).  The paper's route for very few displacements (Fig. 2)
// and a semantic alternative to the wrap-around of the hot path.  Reading R25: the calculated image displaced by d
// is I_d(r) = I1(r + d) where r + d lies inside the box and 0 elsewhere, and Eq. 8 is applied to (I_obs, I_d) over all n pixels,
// so C_co, C_c and C_cc all depend on d.  With the observed image mean-free, o = I_obs - mean,
//     B(d) = sum_{r, r+d in box} o(r) I1(r+d)  ( = C_co - C_o C_c(d) / n ),  A(d) = C_cc(d) - C_c(d)^2 / n,  rho^2 = B^2 / (A D_w),
//     log P = const(n) - 1/2 log(n A(d)) - (n-3)/2 [log D_w + log1p(-rho^2)]                                   (form C2, DESIGN 3).
// FP64 throughout (no FP32 loop, so no re-scoring step): this is the small-shift-set variant, S n multiply-adds per pair against
// the Fourier route's pruned transform, and it is bound by the FP64 pipes; bench.py times it only in the shift sweep.
// Deterministic: fixed-order block sums, terms folded in flat-index order per calculated image, calculated images folded in
// batch order by one thread per image; ties -> lowest flat index (R15).
#include "common.cuh"
#include <math_constants.h>

namespace bioem {

template <int BS>
__device__ __forceinline__ double rs_block_sum(double v, double *sh)
{
    sh[threadIdx.x] = v;
    __syncthreads();
    for (int st = BS / 2; st >= 1; st >>= 1) {
        if ((int)threadIdx.x < st) sh[threadIdx.x] += sh[threadIdx.x + st];
        __syncthreads();
    }
    const double r = sh[0];
    __syncthreads();
    return r;
}

// ---- I1 = F^-1(F0 K) (Eq. 3), separable inverse DFT in FP64, step 1: along m.   T(l, k) = sum_m F0(l,m) K(l,m) e^{+2 pi i m k / N}
// grid (N/2+1, nb), 256 threads
__global__ void __launch_bounds__(256) k_rs_inv_m(const cd *F0, const double *K, int N, cd *T)
{
    extern __shared__ __align__(16) double rs_sm[];
    cd *tw = reinterpret_cast<cd *>(rs_sm), *col = tw + N;
    const int l = blockIdx.x, b = blockIdx.y, NC = N / 2 + 1;
    const cd *F = F0 + ((size_t)b * NC + l) * N;
    const double *Kl = K + (size_t)l * N;
    for (int i = threadIdx.x; i < N; i += 256) {
        double sn, cs;
        sincospi(2.0 * i / N, &sn, &cs);
        tw[i] = {cs, sn};
        const cd v = F[i];
        const double kk = Kl[i];
        col[i] = {v.x * kk, v.y * kk};
    }
    __syncthreads();
    for (int k = threadIdx.x; k < N; k += 256) {
        double ar = 0.0, ai = 0.0;
        for (int m = 0; m < N; ++m) {
            const cd w = tw[(m * k) % N], v = col[m];
            ar += v.x * w.x - v.y * w.y;
            ai += v.x * w.y + v.y * w.x;
        }
        T[((size_t)b * NC + l) * N + k] = {ar, ai};
    }
}
// step 2: along l with the Hermitian weights.   I1(k, j) = 1/n sum_l w_l Re[ T(l, k) e^{+2 pi i l j / N} ]     grid (N, nb)
__global__ void __launch_bounds__(256) k_rs_inv_l(const cd *T, int N, double *I1)
{
    extern __shared__ __align__(16) double rs_sm[];
    cd *tw = reinterpret_cast<cd *>(rs_sm), *row = tw + N;
    const int k = blockIdx.x, b = blockIdx.y, NC = N / 2 + 1;
    for (int i = threadIdx.x; i < N; i += 256) {
        double sn, cs;
        sincospi(2.0 * i / N, &sn, &cs);
        tw[i] = {cs, sn};
    }
    for (int l = threadIdx.x; l < NC; l += 256) row[l] = T[((size_t)b * NC + l) * N + k];
    __syncthreads();
    for (int j = threadIdx.x; j < N; j += 256) {
        double acc = 0.0;
        for (int l = 0; l < NC; ++l) {
            const cd w = tw[(l * j) % N], v = row[l];
            acc += ((l == 0 || l == N / 2) ? 1.0 : 2.0) * (v.x * w.x - v.y * w.y);
        }
        I1[((size_t)b * N + k) * N + j] = acc / ((double)N * N);
    }
}

// ---- C_c(d), C_cc(d): sums of I1 and I1^2 over the part of the calculated image that stays inside the box.   grid (S, nb)
__global__ void __launch_bounds__(256) k_rs_crop_sums(const double *I1, int N, int D, double *cc, double *ccc)
{
    __shared__ double sh[256];
    const int KK = 2 * D + 1, d = blockIdx.x, b = blockIdx.y, dy = d / KK - D, dx = d % KK - D;
    const double *I = I1 + (size_t)b * N * N;
    // pixel p = r + d of I1 survives iff r = p - d is inside the box
    const int k_lo = max(0, dy), k_hi = min(N, N + dy), j_lo = max(0, dx), j_hi = min(N, N + dx);
    const int w = max(0, j_hi - j_lo), cnt = max(0, k_hi - k_lo) * w;
    double s1 = 0.0, s2 = 0.0;
    for (int i = threadIdx.x; i < cnt; i += 256) {
        const double v = I[(size_t)(k_lo + i / w) * N + j_lo + i % w];
        s1 += v; s2 += v * v;
    }
    s1 = rs_block_sum<256>(s1, sh);
    s2 = rs_block_sum<256>(s2, sh);
    if (threadIdx.x == 0) { cc[(size_t)b * KK * KK + d] = s1; ccc[(size_t)b * KK * KK + d] = s2; }
}

// ---- one CTA per (image, calculated image of the batch): B(d) for all shifts, the closed form, log-sum-exp over d in flat order
struct RsPartial { double m, s, best; int shift; int valid; };

__global__ void __launch_bounds__(256) k_rs_score(const double *Oc, const double *Dw, const double *I1, const double *cc, const double *ccc,
                                                  const double *logw, int n_img, int N, int D, RsPartial *part, int *flags)
{
    extern __shared__ __align__(16) double rs_sm[];
    __shared__ double sh[256];
    const int KK = 2 * D + 1, S = KK * KK, img = blockIdx.x, b = blockIdx.y;
    double *Bs = rs_sm, *gs = rs_sm + S;
    const double *o = Oc + (size_t)img * N * N, *I = I1 + (size_t)b * N * N;
    for (int dy = -D; dy <= D; ++dy) {
        const int k_lo = max(0, -dy), k_hi = min(N, N - dy);           // rows r with r + dy inside
        for (int dx0 = -D; dx0 <= D; dx0 += 8) {
            double acc[8] = {0, 0, 0, 0, 0, 0, 0, 0};
            const int nd = min(8, D - dx0 + 1);
            for (int i = threadIdx.x; i < (k_hi - k_lo) * N; i += 256) {
                const int k = k_lo + i / N, j = i % N;
                const double ov = o[(size_t)k * N + j];
                const double *Irow = I + (size_t)(k + dy) * N;
#pragma unroll
                for (int u = 0; u < 8; ++u) {
                    const int j2 = j + dx0 + u;
                    if (u < nd && j2 >= 0 && j2 < N) acc[u] += ov * Irow[j2];
                }
            }
            for (int u = 0; u < nd; ++u) {
                const double r = rs_block_sum<256>(acc[u], sh);
                if (threadIdx.x == 0) Bs[(dy + D) * KK + (dx0 + u + D)] = r;
            }
        }
    }
    __syncthreads();
    const double n = (double)N * N, dw = Dw[img], lw = logw[b];
    for (int d = threadIdx.x; d < S; d += 256) {
        const double c1 = cc[(size_t)b * S + d], c2 = ccc[(size_t)b * S + d];
        const double A = c2 - c1 * c1 / n;
        double g = -CUDART_INF;
        if (A > 0.0 && lw > -CUDART_INF) {
            const double Bv = Bs[d], rho2 = Bv * Bv / (A * dw);
            const double l1 = rho2 < 0.5 ? log1p(-rho2) : log(fmax(1.0 - rho2, 1e-300));          // R14
            g = -0.5 * log(n * A) - 0.5 * (n - 3.0) * l1 + lw;
        } else if (!(A > 0.0)) atomicOr(flags, 2);                        // the displaced calculated image is empty or constant
        gs[d] = g;
    }
    __syncthreads();
    if (threadIdx.x == 0) {
        double M = -CUDART_INF, Ssum = 0.0, best = -CUDART_INF;
        int bs = -1;
        for (int d = 0; d < S; ++d) {
            const double g = gs[d];
            if (g == -CUDART_INF) continue;
            if (g > M) { Ssum = Ssum * exp(M - g) + 1.0; M = g; } else Ssum += exp(g - M);
            if (g > best) { best = g; bs = d; }                           // strict: ties keep the lowest flat index (R15)
        }
        RsPartial p = {M, Ssum, best, bs, bs >= 0};
        part[(size_t)b * n_img + img] = p;
    }
}

// ---- fold the batch into the running sums, calculated images in batch order; one thread per image.  po_m != NULL (posterior per
// orientation): calculated image b of the batch belongs to orientation o0 + b, whose own running sum
// po[(img * n_model + model) * n_orient + o] takes the same term (the batches of the other CTFs of that orientation follow in stream order).
__global__ void k_rs_merge(const RsPartial *part, const long long *pair_of, int nb, int n_img, int n_model, int model, double *acc_m, double *acc_s,
                           double *acc_best, long long *acc_pair, int *acc_shift, double *po_m, double *po_s, int n_orient, int o0)
{
    const int img = blockIdx.x * blockDim.x + threadIdx.x;
    if (img >= n_img) return;
    const size_t im = (size_t)img * n_model + model;
    double M = acc_m[im], Ssum = acc_s[im], best = acc_best[im];
    long long bp = acc_pair[im];
    int bsft = acc_shift[im];
    for (int b = 0; b < nb; ++b) {
        const RsPartial p = part[(size_t)b * n_img + img];
        if (!p.valid) continue;
        if (p.m > M) { Ssum = Ssum * exp(M - p.m) + p.s; M = p.m; } else Ssum += p.s * exp(p.m - M);
        if (po_m) {
            const size_t io = im * n_orient + o0 + b;
            const double m0 = po_m[io], s0 = po_s[io];
            if (p.m > m0) { po_s[io] = s0 * exp(m0 - p.m) + p.s; po_m[io] = p.m; } else po_s[io] = s0 + p.s * exp(p.m - m0);
        }
        const long long pr = pair_of[b];
        if (p.best > best || (p.best == best && (bp < 0 || pr < bp))) { best = p.best; bp = pr; bsft = p.shift; }
    }
    acc_m[im] = M; acc_s[im] = Ssum; acc_best[im] = best; acc_pair[im] = bp; acc_shift[im] = bsft;
}

__global__ void k_rs_init(int n, double *acc_m, double *acc_s, double *acc_best, long long *acc_pair, int *acc_shift)
{
    const int i = blockIdx.x * blockDim.x + threadIdx.x;
    if (i >= n) return;
    acc_m[i] = -CUDART_INF; acc_s[i] = 0.0; acc_best[i] = -CUDART_INF; acc_pair[i] = -1; acc_shift[i] = 0;
}

__global__ void k_rs_orient_init(size_t n, double *po_m, double *po_s)
{
    const size_t i = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (i < n) { po_m[i] = -CUDART_INF; po_s[i] = 0.0; }
}

// out[img][model][o] = log sum_{ctf, d} w P of orientation o (FP64 throughout: nothing to re-score)
__global__ void k_rs_orient_final(const double *po_m, const double *po_s, const double *Dw, int n_img, int n_model, int n_orient, int N, double const_n,
                                  double *out)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (size_t)n_img * n_model * n_orient) return;
    const int img = (int)(idx / ((size_t)n_model * n_orient));
    const double n = (double)N * N;
    out[idx] = po_s[idx] > 0.0 ? const_n - 0.5 * (n - 3.0) * log(Dw[img]) + po_m[idx] + log(po_s[idx]) : -CUDART_INF;
}

__global__ void k_rs_final(const double *acc_m, const double *acc_s, const double *acc_best, const long long *acc_pair, const int *acc_shift,
                           const double *Dw, int n_img, int n_model, int n_ctf, int N, int D, double const_n, double *logp, double *logp32,
                           int32_t *best, double *best_logp)
{
    const int im = blockIdx.x * blockDim.x + threadIdx.x;
    if (im >= n_img * n_model) return;
    const int img = im / n_model, KK = 2 * D + 1;
    const double n = (double)N * N, base = const_n - 0.5 * (n - 3.0) * log(Dw[img]);
    logp[im] = logp32[im] = base + acc_m[im] + log(acc_s[im]);
    const long long pr = acc_pair[im];
    if (pr >= 0) {
        best[4 * im + 0] = (int32_t)(pr / n_ctf); best[4 * im + 1] = (int32_t)(pr % n_ctf);
        best[4 * im + 2] = acc_shift[im] % KK - D; best[4 * im + 3] = acc_shift[im] / KK - D;
        best_logp[im] = base + acc_best[im];
    } else {
        best[4 * im + 0] = best[4 * im + 1] = -1; best[4 * im + 2] = best[4 * im + 3] = 0;
        best_logp[im] = -CUDART_INF;
    }
}

// log-weight and flat pair index of the calculated images of a batch, from what a3 left: h64 = -1/2 log T_c + log w (global T_c)
__global__ void k_rs_batch_meta(const double *h64, const double *Tc64, int model, int n_orient, int n_ctf, int o0, int c, int nb, double *logw,
                                long long *pair_of)
{
    const int b = blockIdx.x * blockDim.x + threadIdx.x;
    if (b >= nb) return;
    const size_t moc = ((size_t)model * n_orient + o0 + b) * n_ctf + c;
    logw[b] = h64[moc] + 0.5 * log(Tc64[moc]);
    pair_of[b] = (long long)(o0 + b) * n_ctf + c;
}

// ---- host side: one batch = calculated images (orientation o0 + b, CTF c) of one model, b = 0..nb-1
size_t rs_partial_bytes(int nb, int n_img) { return (size_t)nb * n_img * sizeof(RsPartial); }

cudaError_t launch_rs_calc_images(const cd *F0, const double *K, int nb, int N, cd *T, double *I1, cudaStream_t st)
{
    const int NC = N / 2 + 1;
    const size_t sm = (size_t)2 * N * sizeof(cd);
    k_rs_inv_m<<<dim3(NC, nb), 256, sm, st>>>(F0, K, N, T);
    k_rs_inv_l<<<dim3(N, nb), 256, sm, st>>>(T, N, I1);
    return cudaGetLastError();
}

cudaError_t launch_rs_batch_meta(const double *h64, const double *Tc64, int model, int n_orient, int n_ctf, int o0, int c, int nb, double *logw,
                                 long long *pair_of, cudaStream_t st)
{
    k_rs_batch_meta<<<(nb + 63) / 64, 64, 0, st>>>(h64, Tc64, model, n_orient, n_ctf, o0, c, nb, logw, pair_of);
    return cudaGetLastError();
}

cudaError_t launch_rs_score(const double *Oc, const double *Dw, const double *I1, const double *logw, const long long *pair_of, int nb, int n_img,
                            int n_model, int model, int N, int D, double *cc, double *ccc, void *part, double *acc_m, double *acc_s,
                            double *acc_best, long long *acc_pair, int *acc_shift, int *flags, double *po_m, double *po_s, int n_orient, int o0,
                            cudaStream_t st)
{
    const int S = (2 * D + 1) * (2 * D + 1);
    k_rs_crop_sums<<<dim3(S, nb), 256, 0, st>>>(I1, N, D, cc, ccc);
    const size_t sm = (size_t)2 * S * sizeof(double);
    if (sm > 48 * 1024) {
        cudaError_t e = cudaFuncSetAttribute(k_rs_score, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)sm);
        if (e != cudaSuccess) return e;
    }
    k_rs_score<<<dim3(n_img, nb), 256, sm, st>>>(Oc, Dw, I1, cc, ccc, logw, n_img, N, D, static_cast<RsPartial *>(part), flags);
    k_rs_merge<<<(n_img + 127) / 128, 128, 0, st>>>(static_cast<const RsPartial *>(part), pair_of, nb, n_img, n_model, model, acc_m, acc_s, acc_best,
                                                     acc_pair, acc_shift, po_m, po_s, n_orient, o0);
    return cudaGetLastError();
}

cudaError_t launch_rs_orient_init(size_t n, double *po_m, double *po_s, cudaStream_t st)
{
    k_rs_orient_init<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(n, po_m, po_s);
    return cudaGetLastError();
}

cudaError_t launch_rs_orient_final(const double *po_m, const double *po_s, const double *Dw, int n_img, int n_model, int n_orient, int N, double const_n,
                                   double *out, cudaStream_t st)
{
    const size_t n = (size_t)n_img * n_model * n_orient;
    k_rs_orient_final<<<(unsigned)((n + 255) / 256), 256, 0, st>>>(po_m, po_s, Dw, n_img, n_model, n_orient, N, const_n, out);
    return cudaGetLastError();
}

cudaError_t launch_rs_init(int n, double *acc_m, double *acc_s, double *acc_best, long long *acc_pair, int *acc_shift, cudaStream_t st)
{
    k_rs_init<<<(n + 127) / 128, 128, 0, st>>>(n, acc_m, acc_s, acc_best, acc_pair, acc_shift);
    return cudaGetLastError();
}

cudaError_t launch_rs_final(const double *acc_m, const double *acc_s, const double *acc_best, const long long *acc_pair, const int *acc_shift,
                            const double *Dw, int n_img, int n_model, int n_ctf, int N, int D, double const_n, double *logp, double *logp32,
                            int32_t *best, double *best_logp, cudaStream_t st)
{
    const int n = n_img * n_model;
    k_rs_final<<<(n + 127) / 128, 128, 0, st>>>(acc_m, acc_s, acc_best, acc_pair, acc_shift, Dw, n_img, n_model, n_ctf, N, D, const_n, logp, logp32,
                                                best, best_logp);
    return cudaGetLastError();
}

}  // namespace bioem
