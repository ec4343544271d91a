// finalize.cu -- SURVEY section 8 rows a6 (fixed-order combine of the per-chunk partials) and a7 (FP64 re-scoring of
// the K best terms per (image, model), corrected log-sum-exp, argmax, constants).  Not in the paper: the paper runs
// single precision and states it gives "the same numerical result"; the 1e-3 absolute parity bar on
// log-posteriors of magnitude 1e4-1e5 needs the dominant terms in FP64 (hard part 1; DESIGN 6).
#include "common.cuh"
#include <math_constants.h>

namespace bioem {

__device__ __forceinline__ bool before(const TopEntry &a, const TopEntry &b)
{
    return a.g > b.g || (a.g == b.g && (a.pair < b.pair || (a.pair == b.pair && a.shift < b.shift)));
}

// One WARP per (image, model): combine the per-work-item partials (bit-reproducible: the result is a fixed function of the
// sequence of chunks).  The partials arrive as `n_blobs` blobs of `stride` bytes (one per rank when the orientation grid is sharded,
// P:199; one otherwise), blob r holding chunks_of_blob[r] chunks per model: float m[n_r], float s[n_r], TopEntry
// top[n_r][TOPK], n_r = n_model * chunks * n_img, item = (model * chunks + chunk) * n_img + img.  Blobs in rank order = chunks in
// grid order; lane i takes the chunks whose index in that ONE sequence is i, i + 32, ... -- where the blobs are cut does not
// enter, so the sums and the candidate lists come out exactly as on one GPU with the same chunking.
//   sums:       each lane adds its chunks in order, then a butterfly over the lanes (both partners compute the same a + b)
//   candidates: the K best of all lists under the strict total order `before` -- a set that does not depend on any order of
//               evaluation -- picked one after the other: round k takes the best entry that comes after pick k - 1.
// (As one thread per (image, model) walking the chunks it took 0.20 ms on Tiny, 2.5 x the fused kernel: 64 dependent rounds of
// loads and an insertion sort in local memory.)
__global__ void __launch_bounds__(128) k_merge(const unsigned char *blobs, size_t stride, const int *chunks_of_blob, int n_blobs, int n_img, int n_model,
                                               double *m32, double *s32, TopEntry *top)
{
    constexpr unsigned FULL = 0xffffffffu;
    const int im = blockIdx.x * 4 + (threadIdx.x >> 5), lane = threadIdx.x & 31;
    if (im >= n_img * n_model) return;                               // warp-uniform
    const int img = im / n_model, model = im % n_model;
    // ---- sums
    double M = -CUDART_INF, S = 0.0;
    for (int r = 0, g0 = 0; r < n_blobs; ++r) {
        const int cpm = chunks_of_blob[r];
        const size_t n_r = (size_t)n_model * cpm * n_img;
        const float *part_m = reinterpret_cast<const float *>(blobs + (size_t)r * stride), *part_s = part_m + n_r;
        for (int ch = ((lane - g0) % 32 + 32) % 32; ch < cpm; ch += 32) {
            const size_t item = ((size_t)model * cpm + ch) * n_img + img;
            const double m = part_m[item], s = part_s[item];
            if (m != -CUDART_INF) {
                if (M == -CUDART_INF) { M = m; S = s; }
                else if (m > M) { S = S * exp2(M - m) + s; M = m; }          // base-2 units
                else S += s * exp2(m - M);
            }
        }
        g0 += cpm;
    }
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const double m2 = __shfl_xor_sync(FULL, M, off), s2 = __shfl_xor_sync(FULL, S, off);
        const double Mx = fmax(M, m2);
        const double a = M == -CUDART_INF ? 0.0 : S * exp2(M - Mx), b = m2 == -CUDART_INF ? 0.0 : s2 * exp2(m2 - Mx);
        S = a + b; M = Mx;                                           // a + b == b + a: both partners hold the same bits
    }
    if (lane == 0) { m32[im] = M; s32[im] = S; }
    // ---- candidates
    const TopEntry none = {-CUDART_INF_F, 0xffffffffu, 0xffffffffu};
    TopEntry prev = none;
    for (int k = 0; k < BIOEM_TOPK; ++k) {
        TopEntry cand = none;
        for (int r = 0, g0 = 0; r < n_blobs; ++r) {
            const int cpm = chunks_of_blob[r];
            const size_t n_r = (size_t)n_model * cpm * n_img;
            const TopEntry *part_top = reinterpret_cast<const TopEntry *>(reinterpret_cast<const float *>(blobs + (size_t)r * stride) + 2 * n_r);
            for (int ch = ((lane - g0) % 32 + 32) % 32; ch < cpm; ch += 32) {
                const TopEntry *list = part_top + (((size_t)model * cpm + ch) * n_img + img) * BIOEM_TOPK;
                for (int j = 0; j < BIOEM_TOPK; ++j) {               // every entry: a list need not be in `before` order among equal g
                    const TopEntry e = list[j];
                    if (e.pair == 0xffffffffu) break;
                    if (e.g != e.g || (k > 0 && !before(prev, e))) continue;
                    if (cand.pair == 0xffffffffu || before(e, cand)) cand = e;
                }
            }
            g0 += cpm;
        }
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            TopEntry o;
            o.g = __shfl_xor_sync(FULL, cand.g, off); o.pair = __shfl_xor_sync(FULL, cand.pair, off); o.shift = __shfl_xor_sync(FULL, cand.shift, off);
            if (o.pair != 0xffffffffu && (cand.pair == 0xffffffffu || before(o, cand))) cand = o;
        }
        if (lane == 0) top[(size_t)im * BIOEM_TOPK + k] = cand;      // `none` once the lists are exhausted
        prev = cand;
        if (cand.pair == 0xffffffffu) {
            if (lane == 0) for (int kk = k + 1; kk < BIOEM_TOPK; ++kk) top[(size_t)im * BIOEM_TOPK + kk] = none;
            break;
        }
    }
}

cudaError_t launch_merge(const unsigned char *blobs, size_t stride, const int *chunks_of_blob, int n_blobs, int n_img, int n_model, double *m32,
                         double *s32, TopEntry *top, cudaStream_t st)
{
    int n = n_img * n_model;
    k_merge<<<(n + 3) / 4, 128, 0, st>>>(blobs, stride, chunks_of_blob, n_blobs, n_img, n_model, m32, s32, top);
    return cudaGetLastError();
}

// a7: one CTA per candidate.  B(d) = 1/n sum_s conj(Ohat(s)) F0(s) K_c(s) exp(+2 pi i (l dx + m dy)/N)  (Eq. 12, R3/R4),
// summed over the Hermitian half with weights (1 | 2) in FP64 in a fixed order.
// g = -(n-3)/2 log1p(-rho^2) + h,  rho^2 = B_fft^2 / (n T_c D_w)  (form C2).
__global__ void __launch_bounds__(256) k_rescore(const cd *Ohat, const cd *F0, const double *K64, const double *Tc64, const double *h64,
                                                 const double *Dw, const TopEntry *cand, int ncp, int n_img, int n_model, int n_orient,
                                                 int n_ctf, int N, int D, int model_fixed, int o_first, double *g64)
{
    __shared__ double sh[256];
    __shared__ cd tw[256];
    const int NC = N / 2 + 1, H = NC * N, KK = 2 * D + 1;
    const size_t ci = blockIdx.x;                       // candidate index = (img*n_model + model)*ncp + k
    const TopEntry e = cand[ci];
    if (e.pair == 0xffffffffu) { if (threadIdx.x == 0) g64[ci] = -CUDART_INF; return; }
    const int im = (int)(ci / ncp);
    const int img = model_fixed >= 0 ? im : im / n_model, model = model_fixed >= 0 ? model_fixed : im % n_model;
    // n_orient orientations starting at o_first of the full grid are resident (orientation sharding): a candidate of
    // another rank's slice gets 0 here, so that the SUM over ranks is exactly the owner's value
    const int o = (int)(e.pair / n_ctf) - o_first, c = e.pair % n_ctf;
    if (o < 0 || o >= n_orient) { if (threadIdx.x == 0) g64[ci] = 0.0; return; }
    const int dy = (int)(e.shift / KK) - D, dx = (int)(e.shift % KK) - D;
    for (int i = threadIdx.x; i < N; i += 256) {
        double sn, cs;
        sincospi(2.0 * i / N, &sn, &cs);
        tw[i] = {cs, sn};
    }
    __syncthreads();
    const cd *Oi = Ohat + (size_t)img * H;
    const cd *F = F0 + ((size_t)model * n_orient + o) * H;
    const double *K = K64 + (size_t)c * H;
    double s = 0.0;
    for (int i = threadIdx.x; i < H; i += 256) {
        const int l = i / N, m = i % N;
        const double w = (l == 0 || l == N / 2) ? 1.0 : 2.0;
        const cd a = Oi[i], b = F[i];
        const double pr = a.x * b.x + a.y * b.y, pi = a.x * b.y - a.y * b.x;      // conj(a) b
        const cd ph = tw[(((l * dx + m * dy) % N) + N) % N];
        s += w * K[i] * (pr * ph.x - pi * ph.y);
    }
    __syncthreads();
    sh[threadIdx.x] = s;
    __syncthreads();
    for (int st = 128; st >= 1; st >>= 1) {
        if ((int)threadIdx.x < st) sh[threadIdx.x] += sh[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) {
        const size_t moc = ((size_t)model * n_orient + o) * n_ctf + c;
        const double n = (double)N * N;
        const double B = sh[0];
        const double rho2 = B * B / (n * Tc64[moc] * Dw[img]);
        // R14 (DESIGN 3): 1 - rho^2 >= 1e-300 (1.0 - 1e-300 == 1.0 in double, so the clamp has to sit on
        // the difference: a noiseless planted image then gives a large finite term instead of +inf)
        const double g = rho2 < 0.5 ? log1p(-rho2) : log(fmax(1.0 - rho2, 1e-300));
        g64[ci] = -0.5 * (n - 3.0) * g + h64[moc];
    }
}

cudaError_t launch_rescore(const cd *Ohat64, const cd *F064, const double *K64, const double *Tc64, const double *h64, const double *Dw,
                           const TopEntry *cand, int n_cand_per, int n_img, int n_model, int n_orient, int n_ctf, int N, int D,
                           int cand_model_fixed, int o_first, double *g64, cudaStream_t st)
{
    size_t total = (size_t)n_img * (cand_model_fixed >= 0 ? 1 : n_model) * n_cand_per;
    k_rescore<<<(unsigned)total, 256, 0, st>>>(Ohat64, F064, K64, Tc64, h64, Dw, cand, n_cand_per, n_img, n_model, n_orient, n_ctf, N, D,
                                               cand_model_fixed, o_first, g64);
    return cudaGetLastError();
}

// One thread per (image, model): replace the K best FP32 terms by their FP64 values, argmax among them, constants.
__global__ void k_final(const double *m32, const double *s32, const TopEntry *top, const double *g64, const double *Dw, int n_img,
                        int n_model, int n_ctf, int N, int D, double const_n, double *logp, double *logp32, int32_t *best,
                        double *best_logp)
{
    const int im = blockIdx.x * blockDim.x + threadIdx.x;
    if (im >= n_img * n_model) return;
    const int img = im / n_model, KK = 2 * D + 1;
    const double n = (double)N * N;
    const double base = const_n - 0.5 * (n - 3.0) * log(Dw[img]);
    const TopEntry *t = top + (size_t)im * BIOEM_TOPK;
    const double *g = g64 + (size_t)im * BIOEM_TOPK;
    const double LN2 = 0.6931471805599453;
    const double m32n = m32[im] * LN2;                     // FP32 partials are in base-2 units; convert in double
    double M = m32n;
    int kb = -1;
    for (int k = 0; k < BIOEM_TOPK; ++k) {
        if (t[k].pair == 0xffffffffu) break;
        if (g[k] > M) M = g[k];
        if (kb < 0 || g[k] > g[kb] || (g[k] == g[kb] && (t[k].pair < t[kb].pair || (t[k].pair == t[kb].pair && t[k].shift < t[kb].shift))))
            kb = k;
    }
    double tot32 = s32[im] * exp(m32n - M), top32 = 0.0, top64 = 0.0;
    for (int k = 0; k < BIOEM_TOPK; ++k) {
        if (t[k].pair == 0xffffffffu) break;
        top32 += exp((double)t[k].g * LN2 - M);
        top64 += exp(g[k] - M);
    }
    double rest = tot32 - top32;
    if (rest < 0.0) rest = 0.0;
    logp[im] = base + M + log(top64 + rest);
    logp32[im] = base + m32n + log(s32[im]);
    if (kb >= 0) {
        best[4 * im + 0] = (int32_t)(t[kb].pair / n_ctf);
        best[4 * im + 1] = (int32_t)(t[kb].pair % n_ctf);
        best[4 * im + 2] = (int32_t)(t[kb].shift % KK) - D;
        best[4 * im + 3] = (int32_t)(t[kb].shift / KK) - D;
        best_logp[im] = base + g[kb];
    } else {
        best[4 * im + 0] = best[4 * im + 1] = -1; best[4 * im + 2] = best[4 * im + 3] = 0;
        best_logp[im] = -CUDART_INF;
    }
}

cudaError_t launch_final(const double *m32, const double *s32, const TopEntry *top, const double *g64, const double *Dw, int n_img,
                         int n_model, int n_ctf, int N, int D, double const_n, double *logp, double *logp32, int32_t *best,
                         double *best_logp, cudaStream_t st)
{
    int n = n_img * n_model;
    k_final<<<(n + 63) / 64, 64, 0, st>>>(m32, s32, top, g64, Dw, n_img, n_model, n_ctf, N, D, const_n, logp, logp32, best, best_logp);
    return cudaGetLastError();
}

// Posterior per orientation from the per-orientation (m, s) the fused kernels wrote (the folded table, ppo = 1; or, cluster
// kernel with one orientation per work item, its two partials, ppo = 2).  One thread per (image, model, resident orientation):
// combine in order, replace the re-scored terms of this orientation -- candidates carry GLOBAL orientation indices, local
// orientation o is o + o_first of the grid -- by their FP64 values, add the constants.  out [img][model][o].
__global__ void k_orient_final(const float *part_m, const float *part_s, int ppo, const TopEntry *top, const double *g64, const double *Dw,
                               int n_img, int n_model, int n_orient, int o_first, int n_ctf, int N, double const_n, double *out)
{
    const size_t idx = (size_t)blockIdx.x * blockDim.x + threadIdx.x;
    if (idx >= (size_t)n_img * n_model * n_orient) return;
    const int o = (int)(idx % n_orient), im = (int)(idx / n_orient), img = im / n_model, model = im % n_model;
    const double LN2 = 0.6931471805599453, n = (double)N * N;
    double M = -CUDART_INF, S = 0.0;                       // base-2 units, as the fused kernels write them
    for (int k = 0; k < ppo; ++k) {
        const size_t item = (((size_t)model * n_orient + o) * ppo + k) * n_img + img;
        const double m = part_m[item], s = part_s[item];
        if (m == -CUDART_INF) continue;
        if (M == -CUDART_INF) { M = m; S = s; }
        else if (m > M) { S = S * exp2(M - m) + s; M = m; }
        else S += s * exp2(m - M);
    }
    if (M == -CUDART_INF) { out[idx] = -CUDART_INF; return; }
    double Mn = M * LN2;
    const TopEntry *t = top + (size_t)im * BIOEM_TOPK;
    const double *g = g64 + (size_t)im * BIOEM_TOPK;
    double ref = Mn;
    for (int k = 0; k < BIOEM_TOPK; ++k)
        if (t[k].pair != 0xffffffffu && (int)(t[k].pair / n_ctf) == o + o_first && g[k] > ref) ref = g[k];
    double tot = S * exp(Mn - ref), t32 = 0.0, t64 = 0.0;
    for (int k = 0; k < BIOEM_TOPK; ++k)
        if (t[k].pair != 0xffffffffu && (int)(t[k].pair / n_ctf) == o + o_first) {
            t32 += exp((double)t[k].g * LN2 - ref);
            t64 += exp(g[k] - ref);
        }
    double rest = tot - t32;
    if (rest < 0.0) rest = 0.0;
    out[idx] = const_n - 0.5 * (n - 3.0) * log(Dw[img]) + ref + log(t64 + rest);
}

cudaError_t launch_orient_final(const float *part_m, const float *part_s, int parts_per_orient, const TopEntry *top, const double *g64,
                                const double *Dw, int n_img, int n_model, int n_orient, int o_first, int n_ctf, int N, double const_n,
                                double *logp_orient, cudaStream_t st)
{
    const size_t n = (size_t)n_img * n_model * n_orient;
    k_orient_final<<<(unsigned)((n + 127) / 128), 128, 0, st>>>(part_m, part_s, parts_per_orient, top, g64, Dw, n_img, n_model, n_orient, o_first, n_ctf, N,
                                                                const_n, logp_orient);
    return cudaGetLastError();
}

// Eq. 10: per image the log of the weighted sum over models, then the sum over images (the log of the product).
// One CTA, fixed order: thread i takes images i, i + 256, ... in order, then a fixed tree over the 256 partial sums.
__global__ void __launch_bounds__(256) k_ensemble(const double *logp, const double *logw, int n_img, int n_model, double *per_image, double *total)
{
    __shared__ double sh[256];
    double acc = 0.0;
    for (int img = threadIdx.x; img < n_img; img += 256) {
        const double *lp = logp + (size_t)img * n_model;
        double M = -CUDART_INF;
        for (int m = 0; m < n_model; ++m) M = fmax(M, lp[m] + logw[m]);
        double v = M;
        if (M != -CUDART_INF) {
            double S = 0.0;
            for (int m = 0; m < n_model; ++m) S += exp(lp[m] + logw[m] - M);
            v = M + log(S);
        }
        per_image[img] = v;
        acc += v;
    }
    sh[threadIdx.x] = acc;
    __syncthreads();
    for (int st = 128; st >= 1; st >>= 1) {
        if ((int)threadIdx.x < st) sh[threadIdx.x] += sh[threadIdx.x + st];
        __syncthreads();
    }
    if (threadIdx.x == 0) *total = sh[0];
}

cudaError_t launch_ensemble(const double *logp, const double *logw, int n_img, int n_model, double *per_image, double *total, cudaStream_t st)
{
    k_ensemble<<<1, 256, 0, st>>>(logp, logw, n_img, n_model, per_image, total);
    return cudaGetLastError();
}

}  // namespace bioem
