// common.cuh -- shared declarations of the bioem_b200 library (device-side layouts and host launchers).
//
// Device layouts:
//   half-spectrum  [l][m]   l = 0..N/2 (x frequency, Hermitian half), m = 0..N-1 (y frequency), m fastest:
//                  a column of fixed l is contiguous -> pass 1 of the pruned inverse transform streams it coalesced.
//   Ohat32/64      [image][l][m]        spectrum of the mean-free observed image (a0), DC bin exactly 0
//   F0_32/64       [model*O + o][l][m]  spectrum of the projection I0 (a1/a1'+a2)
//   K32/64         [c][l][m]            CTF(s)Env(s) of CTF set c (a3; the paper's "precalculated radially symmetric images")
//   alpha/hterm    [(model*O + o)*C + c]
#pragma once
#include <cuda_runtime.h>
#include <stdint.h>
#include "fft_core.cuh"

#ifndef BIOEM_TOPK
#define BIOEM_TOPK 8
#endif

namespace bioem {

typedef cx<float> cf;
typedef cx<double> cd;

struct TopEntry { float g; uint32_t pair; uint32_t shift; };   // g in BASE-2 units (log2 of the term); pair = o*C + c within the model, shift = (dy+D)*S1 + (dx+D)

// choice of the two-step factorisation N = N1 * N2 per supported image size
// (N1 a power of two for the register transform, N2 = N / N1 any; 170 = 2 x 85, the GroEL box of the paper's Table 1, P:229,
// runs as a short radix-2 stage plus 85-term direct sums: correct for any even size, fast only where N1 is large)
__host__ __device__ constexpr int n1_of(int N)
{
    return N == 64 ? 16 : N == 128 ? 16 : N == 224 ? 32 : N == 256 ? 32 : N == 96 ? 32 : N == 160 ? 32 : N == 192 ? 32 : N == 170 ? 2 : 0;
}

struct FusedParams {
    // inputs
    const cf *Ohat;        // [I][H]
    const cf *F0;          // [M*O][H]
    const float *K;        // [C][H]
    const float *alpha;    // [M*O*C]   1/sqrt(n T_c)
    const float *hterm;    // [M*O*C]   (-1/2 log T_c + log w) * log2(e)   -- the fused kernels work in base-2 units
    const float *beta;     // [I]       1/sqrt(D_omega)
    int n_img, n_model, n_orient, n_ctf, D;
    int oc;                // orientations per work item (chunk)
    int o_first;           // index in the FULL orientation grid of local orientation 0 (orientation sharding); candidates carry global indices
    int chunks_per_model;
    float cA;              // -(n-3)/2 * log2(e)
    // outputs: one partial per work item = (model, chunk, image)
    float *part_m, *part_s;      // [items]   partial sum = part_s * 2^part_m
    TopEntry *part_top;          // [items][TOPK]
    // posterior per orientation, folded into the chunked work items: NULL, or [(model*O + o)*I + img] (m, s) of the sum over
    // the CTFs and shifts of orientation o, written by the work item that holds o (k_fused_pk / k_fused_tm <.., ORIENT = true>, k_fused)
    float *orient_m, *orient_s;
    // debug dump of one pair (DUMP instantiation only)
    float *dump;                 // [S1*S1]
    int dump_img, dump_model, dump_orient, dump_ctf;
};

// host launchers (each enqueues on `st`); return cudaError_t
cudaError_t launch_fused(int N, const FusedParams &p, bool dump, cudaStream_t st, int *n_launches);
size_t fused_smem_bytes(int N, int D);
// register-resident-Q, packed-f32x2 variant (N = 64, 128; D <= 16)
bool pk_supported(int N, int D);
size_t pk_kt_bytes(int N, int n_ctf);
cudaError_t launch_relayout_K(int N, const float *K32, float *Kt, int n_ctf, cudaStream_t st);
cudaError_t launch_fused_pk(int N, const FusedParams &p, const float *Kt, bool dump, cudaStream_t st);
// two-CTA-cluster variant (N = 224; D <= 31): Q register-resident across a CTA pair; writes TWO partials per work item
bool c2_supported(int N, int D);
size_t c2_kt_bytes(int n_ctf);
cudaError_t launch_relayout_K_c2(const float *K32, float *Kt, int n_ctf, cudaStream_t st);
cudaError_t launch_fused_c2(const FusedParams &p, const float *Kt, bool dump, cudaStream_t st);

// tensor-memory variant (N = 224; D <= 31): Q resident in TMEM, one CTA per work item, one partial per work item
bool tm_supported(int N, int D);
size_t tm_kt_bytes(int n_ctf);
cudaError_t launch_relayout_K_tm(const float *K32, float *Kt, int n_ctf, cudaStream_t st);
cudaError_t launch_fused_tm(const FusedParams &p, const float *Kt, bool dump, cudaStream_t st);

// precompute
cudaError_t launch_image_stats(const float *img, int n_img, int N, double *centered, double *Dw, cudaStream_t st);
cudaError_t launch_fft2_r2c_f64(const double *in, int batch, int N, cd *tmp, cd *out, cudaStream_t st);   // out [b][l][m]
cudaError_t launch_fft2_r2c_fixed(const long long *in, double in_scale, int batch, int N, cd *tmp, cd *out, cf *out32, cudaStream_t st);
cudaError_t launch_cast_spectrum(const cd *in, cf *out, size_t count, cudaStream_t st);
cudaError_t launch_zero_dc(cd *spec, int batch, size_t H, cudaStream_t st);
cudaError_t launch_project_atoms(const double *xyz, const double *rad, const double *wt, int n_atoms, const double *rot,
                                 int n_orient, int N, double px, double fx_scale, long long *acc, cudaStream_t st);
cudaError_t launch_dft3_f64(const float *rho, int N, cd *work_a, cd *work_b, cudaStream_t st);           // result in work_a, centred sign applied
cudaError_t launch_slice_f64(const cd *Vc, int N, double voxel, const double *rot, int n_orient, cd *out, cudaStream_t st);
cudaError_t launch_ctf_tables(const double *a, const double *A, const double *b, int n_ctf, int N, double px,
                              double *K64, float *K32, cudaStream_t st);
cudaError_t launch_calc_stats(const cd *F0, const double *K64, int n_mo, int n_orient, int n_orient_total, int n_ctf, int N,
                              const double *lp_orient, const double *lp_ctf, double log_shifts,
                              double *Tc64, double *h64, float *alpha32, float *h32, int *flags, cudaStream_t st);
cudaError_t launch_beta(const double *Dw, int n_img, float *beta, int *flags, cudaStream_t st);

// finalise
// per-work-item partials travel as one blob: float m[n], float s[n], TopEntry top[n][TOPK], n = n_model * chunks * n_img
inline size_t partial_blob_bytes(size_t n_items) { return n_items * (2 * sizeof(float) + BIOEM_TOPK * sizeof(TopEntry)); }
cudaError_t launch_merge(const unsigned char *blobs, size_t stride, const int *chunks_of_blob, int n_blobs, int n_img, int n_model,
                         double *m32, double *s32, TopEntry *top, cudaStream_t st);
cudaError_t launch_rescore(const cd *Ohat64, const cd *F064, const double *K64, const double *Tc64, const double *h64,
                           const double *Dw, const TopEntry *cand, int n_cand_per, int n_img, int n_model, int n_orient,
                           int n_ctf, int N, int D, int cand_model_fixed, int o_first, double *g64, cudaStream_t st);
cudaError_t launch_final(const double *m32, const double *s32, const TopEntry *top, const double *g64, const double *Dw,
                         int n_img, int n_model, int n_ctf, int N, int D, double const_n, double *logp, double *logp32,
                         int32_t *best, double *best_logp, cudaStream_t st);
cudaError_t launch_orient_final(const float *part_m, const float *part_s, int parts_per_orient, const TopEntry *top, const double *g64,
                                const double *Dw, int n_img, int n_model, int n_orient, int o_first, int n_ctf, int N, double const_n,
                                double *logp_orient, cudaStream_t st);
cudaError_t launch_ensemble(const double *logp, const double *logw, int n_img, int n_model, double *per_image, double *total, cudaStream_t st);
cudaError_t launch_calc_image(const cd *F0, const double *K64, int N, double *out, cudaStream_t st);
cudaError_t launch_synth_map(const double *I1, const float *obs, int N, int dx, int dy, int crop, float *out, double *norm_offset, cudaStream_t st);
cudaError_t launch_fp32_peak(float *sink, int iters, cudaStream_t st);

// real-space, cropping displacement variant (realspace.cu)
size_t rs_partial_bytes(int nb, int n_img);
cudaError_t launch_rs_calc_images(const cd *F0, const double *K, int nb, int N, cd *T, double *I1, cudaStream_t st);
cudaError_t launch_rs_batch_meta(const double *h64, const double *Tc64, int model, int n_orient, int n_ctf, int o0, int c, int nb, double *logw,
                                 long long *pair_of, cudaStream_t st);
cudaError_t launch_rs_score(const double *Oc, const double *Dw, const double *I1, const double *logw, const long long *pair_of, int nb, int n_img,
                            int n_model, int model, int N, int D, double *cc, double *ccc, void *part, double *acc_m, double *acc_s,
                            double *acc_best, long long *acc_pair, int *acc_shift, int *flags, double *po_m, double *po_s, int n_orient, int o0,
                            cudaStream_t st);
cudaError_t launch_rs_orient_init(size_t n, double *po_m, double *po_s, cudaStream_t st);
cudaError_t launch_rs_orient_final(const double *po_m, const double *po_s, const double *Dw, int n_img, int n_model, int n_orient, int N, double const_n,
                                   double *out, cudaStream_t st);
cudaError_t launch_rs_init(int n, double *acc_m, double *acc_s, double *acc_best, long long *acc_pair, int *acc_shift, cudaStream_t st);
cudaError_t launch_rs_final(const double *acc_m, const double *acc_s, const double *acc_best, const long long *acc_pair, const int *acc_shift,
                            const double *Dw, int n_img, int n_model, int n_ctf, int N, int D, double const_n, double *logp, double *logp32,
                            int32_t *best, double *best_logp, cudaStream_t st);

}  // namespace bioem
