// bioem_api.cu -- the C ABI declared in include/bioem.h: context, argument checking, device buffers, and the
// orchestration of one bioem_run (precompute a1-a3 -> fused a4-a6 -> merge -> FP64 re-score a7 -> results).
#include "../../include/bioem.h"
#include "common.cuh"

#include <cmath>
#include <cstdio>
#include <cstring>
#include <string>
#include <vector>

using namespace bioem;

namespace {

struct DBuf {
    void *p = nullptr;
    size_t cap = 0;
    cudaError_t ensure(size_t bytes)
    {
        if (bytes <= cap) return cudaSuccess;
        if (p) { cudaFree(p); p = nullptr; cap = 0; }
        cudaError_t e = cudaMalloc(&p, bytes ? bytes : 1);
        if (e == cudaSuccess) cap = bytes;
        return e;
    }
    void release() { if (p) cudaFree(p); p = nullptr; cap = 0; }
    template <typename T> T *as() const { return reinterpret_cast<T *>(p); }
};

struct Model {
    int kind = 0;                 // 0 atoms, 1 density
    int n_atoms = 0;
    DBuf xyz, rad, wt;            // double
    double sum_abs_w = 0.0;
    int n_vox = 0;
    double voxel = 0.0;
    DBuf rho;                     // float [n_vox^3]
};

}  // namespace

struct bioem_ctx {
    int device = 0;
    cudaStream_t stream = nullptr;
    std::string err;
    int N = 0;
    double px = 0.0;
    int D = -1;
    std::vector<Model> models;
    int n_orient = 0;
    DBuf rot, lp_orient;          // double [O][9], double [O]
    bool has_lp_orient = false;
    int n_ctf = 0;
    DBuf ctf_a, ctf_A, ctf_b, lp_ctf;
    bool has_lp_ctf = false;
    int n_img = 0;
    DBuf Ohat64, Ohat32, Dw, beta;
    // run state
    bool ran = false;
    bool pre_valid = false;                            // a1-a3 outputs (F0, K, T_c, h, alpha) match the current models / grids / shift range
    bool want_orient = false, ran_orient = false;      // per-orientation posterior: requested / produced by the last run
    int oc_user = 0;                                   // orientations per work item (0 = automatic)
    int variant = 0, img_variant = 0;                                   // displacement variant: 0 Fourier / circular (the hot path), 1 real space / cropping
    DBuf Oreal64, rs_T, rs_I1, rs_cc, rs_ccc, rs_part, rs_logw, rs_pair, rs_m, rs_s, rs_best, rs_bpair, rs_bshift;
    int slice_begin = 0, slice_end = -1;               // orientation slice this context scores; end < 0 = the whole grid
    int phase = 0;                                     // of the phased run: 0 nothing, 1 partials, 2 merged, 3 re-scored, 4 finished (= ran)
    int run_o_first = 0, run_o_local = 0, run_chunks = 0;     // slice and chunk count (per model, partials per item included) of the last partial run
    DBuf blob, gathered, blob_chunks;                  // this context's partials (one blob); blobs handed to bioem_merge_partials; their chunk counts
    int kernel_user = 0;                               // BIOEM_KERNEL_*: which fused kernel bioem_run may pick (0 = automatic)
    int n_sm = 148;
    DBuf flags;                                        // int[2]: [0] bit 0 = an image without variance (a0); [1] bit 1 = an empty calculated image (a3)
    int run_kernel = 0, run_oc = 0;
    bool flags_checked = true;
    DBuf logp_orient;
    DBuf orient_m, orient_s;      // float [M*O][I]: per-orientation (m, s) written by the fused kernel (posterior per orientation, folded)
    bool run_want_orient = false, run_orient_folded = false;      // the option as the last run_partial saw it
    int run_models = 0, run_orient = 0, run_ctf = 0, run_D = 0, run_img = 0;
    DBuf F064, F032, K64, K32, Kt, Tc64, h64, alpha32, h32;
    DBuf m32, s32, top, g64;
    DBuf logp, logp32, best, best_logp;
    DBuf scratch_a, scratch_b, scratch_c, dump, staging;
    cudaEvent_t ev[4] = {nullptr, nullptr, nullptr, nullptr};
    int64_t launches = 0, fused_launches = 0, push_launches = 0;
};

#define CK(call)                                                                                     \
    do {                                                                                             \
        cudaError_t e__ = (call);                                                                    \
        if (e__ != cudaSuccess) {                                                                    \
            ctx->err = std::string(#call) + ": " + cudaGetErrorString(e__);                          \
            cudaGetLastError();                                                                      \
            return e__ == cudaErrorMemoryAllocation ? BIOEM_EOOM : BIOEM_ECUDA;                      \
        }                                                                                            \
    } while (0)

#define FAIL(code, msg)          \
    do {                         \
        ctx->err = (msg);        \
        return (code);           \
    } while (0)

static bool supported_n(int n) { return n == 64 || n == 96 || n == 128 || n == 160 || n == 170 || n == 192 || n == 224 || n == 256; }

extern "C" {

int bioem_create(bioem_ctx **out, int device, void *cuda_stream)
{
    if (!out) return BIOEM_EBADARG;
    *out = nullptr;
    int count = 0;
    if (cudaGetDeviceCount(&count) != cudaSuccess || device < 0 || device >= count) { cudaGetLastError(); return BIOEM_ECUDA; }
    if (cudaSetDevice(device) != cudaSuccess) { cudaGetLastError(); return BIOEM_ECUDA; }
    bioem_ctx *ctx = new bioem_ctx();
    ctx->device = device;
    ctx->stream = reinterpret_cast<cudaStream_t>(cuda_stream);
    for (int i = 0; i < 4; ++i)
        if (cudaEventCreate(&ctx->ev[i]) != cudaSuccess) { delete ctx; return BIOEM_ECUDA; }
    if (cudaDeviceGetAttribute(&ctx->n_sm, cudaDevAttrMultiProcessorCount, device) != cudaSuccess || ctx->n_sm < 1) ctx->n_sm = 148;
    if (ctx->flags.ensure(2 * sizeof(int)) != cudaSuccess || cudaMemset(ctx->flags.p, 0, 2 * sizeof(int)) != cudaSuccess) {
        cudaGetLastError();
        for (int i = 0; i < 4; ++i) cudaEventDestroy(ctx->ev[i]);
        delete ctx;
        return BIOEM_ECUDA;
    }
    *out = ctx;
    return BIOEM_OK;
}

int bioem_destroy(bioem_ctx *ctx)
{
    if (!ctx) return BIOEM_EBADARG;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (auto &m : ctx->models) { m.xyz.release(); m.rad.release(); m.wt.release(); m.rho.release(); }
    DBuf *all[] = {&ctx->rot, &ctx->lp_orient, &ctx->ctf_a, &ctx->ctf_A, &ctx->ctf_b, &ctx->lp_ctf, &ctx->Ohat64, &ctx->Ohat32, &ctx->Dw,
                   &ctx->beta, &ctx->F064, &ctx->F032, &ctx->K64, &ctx->K32, &ctx->Kt, &ctx->Tc64, &ctx->h64, &ctx->alpha32, &ctx->h32,
                   &ctx->blob, &ctx->gathered, &ctx->blob_chunks, &ctx->Oreal64, &ctx->rs_T, &ctx->rs_I1, &ctx->rs_cc, &ctx->rs_ccc, &ctx->rs_part, &ctx->rs_logw,
                   &ctx->rs_pair, &ctx->rs_m, &ctx->rs_s, &ctx->rs_best, &ctx->rs_bpair, &ctx->rs_bshift, &ctx->m32, &ctx->s32, &ctx->top, &ctx->g64, &ctx->logp, &ctx->logp_orient, &ctx->orient_m, &ctx->orient_s, &ctx->logp32,
                   &ctx->best, &ctx->best_logp, &ctx->scratch_a, &ctx->scratch_b, &ctx->scratch_c, &ctx->dump, &ctx->flags, &ctx->staging};
    for (DBuf *b : all) b->release();
    for (int i = 0; i < 4; ++i) if (ctx->ev[i]) cudaEventDestroy(ctx->ev[i]);
    delete ctx;
    return BIOEM_OK;
}

const char *bioem_last_error(const bioem_ctx *ctx) { return ctx ? ctx->err.c_str() : "null context"; }

int bioem_set_image_geometry(bioem_ctx *ctx, int n_pix, float pixel_size_A)
{
    if (!ctx) return BIOEM_EBADARG;
    if (!(pixel_size_A > 0.f)) FAIL(BIOEM_EBADARG, "pixel_size_A must be > 0");
    if (!supported_n(n_pix)) FAIL(BIOEM_EUNSUPPORTED, "n_pix must be one of 64, 96, 128, 160, 170, 192, 224, 256");
    ctx->N = n_pix;
    ctx->px = (double)pixel_size_A;
    ctx->n_img = 0;
    ctx->ran = false; ctx->phase = 0; ctx->pre_valid = false;
    return BIOEM_OK;
}

int bioem_clear_models(bioem_ctx *ctx)
{
    if (!ctx) return BIOEM_EBADARG;
    cudaSetDevice(ctx->device);
    cudaStreamSynchronize(ctx->stream);
    for (auto &m : ctx->models) { m.xyz.release(); m.rad.release(); m.wt.release(); m.rho.release(); }
    ctx->models.clear();
    ctx->ran = false; ctx->phase = 0; ctx->pre_valid = false;
    return BIOEM_OK;
}

static int upload_doubles(bioem_ctx *ctx, DBuf &buf, const std::vector<double> &v)
{
    CK(buf.ensure(v.size() * sizeof(double)));
    CK(cudaMemcpyAsync(buf.p, v.data(), v.size() * sizeof(double), cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));       // v is a temporary
    return BIOEM_OK;
}

int bioem_add_model_atoms(bioem_ctx *ctx, int n_atoms, const float *xyz_A, const float *radius_A, const float *weight, int *model_id)
{
    if (!ctx) return BIOEM_EBADARG;
    if (n_atoms <= 0 || !xyz_A || !radius_A || !weight) FAIL(BIOEM_EBADARG, "add_model_atoms: empty model or NULL array");
    CK(cudaSetDevice(ctx->device));
    std::vector<double> x(3 * (size_t)n_atoms), r(n_atoms), w(n_atoms);
    double sw = 0.0;
    for (int i = 0; i < n_atoms; ++i) {
        if (!(radius_A[i] > 0.f)) FAIL(BIOEM_EBADARG, "add_model_atoms: radius must be > 0");
        x[3 * i] = xyz_A[3 * i]; x[3 * i + 1] = xyz_A[3 * i + 1]; x[3 * i + 2] = xyz_A[3 * i + 2];
        r[i] = radius_A[i]; w[i] = weight[i];
        sw += std::fabs((double)weight[i]);
    }
    ctx->models.emplace_back();
    Model &m = ctx->models.back();
    m.kind = 0; m.n_atoms = n_atoms; m.sum_abs_w = sw;
    int rc;
    if ((rc = upload_doubles(ctx, m.xyz, x)) || (rc = upload_doubles(ctx, m.rad, r)) || (rc = upload_doubles(ctx, m.wt, w))) {
        ctx->models.pop_back();
        return rc;
    }
    if (model_id) *model_id = (int)ctx->models.size() - 1;
    ctx->ran = false; ctx->phase = 0; ctx->pre_valid = false;
    return BIOEM_OK;
}

int bioem_add_model_density(bioem_ctx *ctx, int n_vox, float voxel_A, const float *rho, int *model_id)
{
    if (!ctx) return BIOEM_EBADARG;
    if (!rho || !(voxel_A > 0.f)) FAIL(BIOEM_EBADARG, "add_model_density: NULL map or voxel size <= 0");
    if (!supported_n(n_vox)) FAIL(BIOEM_EUNSUPPORTED, "add_model_density: n_vox must be one of 64, 96, 128, 160, 170, 192, 224, 256");
    CK(cudaSetDevice(ctx->device));
    ctx->models.emplace_back();
    Model &m = ctx->models.back();
    m.kind = 1; m.n_vox = n_vox; m.voxel = (double)voxel_A;
    size_t bytes = (size_t)n_vox * n_vox * n_vox * sizeof(float);
    cudaError_t e = m.rho.ensure(bytes);
    if (e == cudaSuccess) e = cudaMemcpyAsync(m.rho.p, rho, bytes, cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    if (e != cudaSuccess) { m.rho.release(); ctx->models.pop_back(); CK(e); }
    if (model_id) *model_id = (int)ctx->models.size() - 1;
    ctx->ran = false; ctx->phase = 0; ctx->pre_valid = false;
    return BIOEM_OK;
}

int bioem_set_orientations_quat(bioem_ctx *ctx, int n, const float *q, const float *log_prior)
{
    if (!ctx) return BIOEM_EBADARG;
    if (n <= 0 || !q) FAIL(BIOEM_EBADARG, "set_orientations_quat: n <= 0 or NULL");
    CK(cudaSetDevice(ctx->device));
    std::vector<double> R(9 * (size_t)n), lp;
    for (int i = 0; i < n; ++i) {
        double w = q[4 * i], x = q[4 * i + 1], y = q[4 * i + 2], z = q[4 * i + 3];
        double nr = std::sqrt(w * w + x * x + y * y + z * z);
        if (!(nr > 0.0)) FAIL(BIOEM_EBADARG, "set_orientations_quat: zero quaternion");
        w /= nr; x /= nr; y /= nr; z /= nr;
        double *r = &R[9 * (size_t)i];                       // active rotation r' = R r (R12)
        r[0] = 1 - 2 * (y * y + z * z); r[1] = 2 * (x * y - w * z);     r[2] = 2 * (x * z + w * y);
        r[3] = 2 * (x * y + w * z);     r[4] = 1 - 2 * (x * x + z * z); r[5] = 2 * (y * z - w * x);
        r[6] = 2 * (x * z - w * y);     r[7] = 2 * (y * z + w * x);     r[8] = 1 - 2 * (x * x + y * y);
    }
    int rc = upload_doubles(ctx, ctx->rot, R);
    if (rc) return rc;
    ctx->has_lp_orient = log_prior != nullptr;
    if (log_prior) {
        lp.assign(log_prior, log_prior + n);
        if ((rc = upload_doubles(ctx, ctx->lp_orient, lp))) return rc;
    }
    ctx->n_orient = n;
    ctx->ran = false; ctx->phase = 0; ctx->pre_valid = false;
    return BIOEM_OK;
}

int bioem_set_ctf_grid(bioem_ctx *ctx, int n, const float *a, const float *A, const float *b, const float *log_prior)
{
    if (!ctx) return BIOEM_EBADARG;
    if (n <= 0 || !a || !A || !b) FAIL(BIOEM_EBADARG, "set_ctf_grid: n <= 0 or NULL");
    CK(cudaSetDevice(ctx->device));
    std::vector<double> va(n), vA(n), vb(n), lp;
    for (int i = 0; i < n; ++i) {
        if (!(A[i] >= 0.f && A[i] <= 1.f)) FAIL(BIOEM_EBADARG, "set_ctf_grid: amplitude contrast A must be in [0,1]");
        va[i] = a[i]; vA[i] = A[i]; vb[i] = b[i];
    }
    int rc;
    if ((rc = upload_doubles(ctx, ctx->ctf_a, va)) || (rc = upload_doubles(ctx, ctx->ctf_A, vA)) || (rc = upload_doubles(ctx, ctx->ctf_b, vb)))
        return rc;
    ctx->has_lp_ctf = log_prior != nullptr;
    if (log_prior) {
        lp.assign(log_prior, log_prior + n);
        if ((rc = upload_doubles(ctx, ctx->lp_ctf, lp))) return rc;
    }
    ctx->n_ctf = n;
    ctx->ran = false; ctx->phase = 0; ctx->pre_valid = false;
    return BIOEM_OK;
}

int bioem_ctf_from_defocus(float defocus_um, float bfactor_A2, float kV, float *a_A2, float *b_A2)
{
    if (!a_A2 || !b_A2 || !(kV > 0.f)) return BIOEM_EBADARG;
    const double V = (double)kV * 1e3;
    const double lambda = 12.2643 / std::sqrt(V + 0.97845e-6 * V * V);          // electron wavelength [A]
    *a_A2 = (float)(lambda * (double)defocus_um * 1e4 / (2.0 * M_PI));            // R8
    *b_A2 = (float)((double)bfactor_A2 / (8.0 * M_PI * M_PI));                    // R9
    return BIOEM_OK;
}

int bioem_set_shift_range(bioem_ctx *ctx, int max_shift_px)
{
    if (!ctx) return BIOEM_EBADARG;
    if (max_shift_px < 0) FAIL(BIOEM_EBADARG, "set_shift_range: negative");
    if (ctx->N && 2 * max_shift_px + 1 > ctx->N) FAIL(BIOEM_EBADARG, "set_shift_range: 2D+1 exceeds n_pix");
    ctx->D = max_shift_px;
    ctx->ran = false; ctx->phase = 0; ctx->pre_valid = false;
    return BIOEM_OK;
}

int bioem_push_images(bioem_ctx *ctx, int n_img, const float *pixels, int is_device)
{
    if (!ctx) return BIOEM_EBADARG;
    if (!ctx->N) FAIL(BIOEM_EBADSTATE, "push_images: set_image_geometry first");
    if (n_img <= 0 || !pixels) FAIL(BIOEM_EBADARG, "push_images: n_img <= 0 or NULL");
    CK(cudaSetDevice(ctx->device));
    const int N = ctx->N;
    const size_t n = (size_t)N * N, H = (size_t)(N / 2 + 1) * N;
    cudaStream_t st = ctx->stream;
    // process in slabs so that scratch stays bounded
    const int slab = 256;
    CK(ctx->Ohat64.ensure((size_t)n_img * H * sizeof(cd)));
    CK(ctx->Ohat32.ensure((size_t)n_img * H * sizeof(cf)));
    CK(ctx->Dw.ensure((size_t)n_img * sizeof(double)));
    CK(ctx->beta.ensure((size_t)n_img * sizeof(float)));
    CK(ctx->scratch_a.ensure((size_t)slab * n * sizeof(double)));       // centred images
    if (ctx->variant == 1) CK(ctx->Oreal64.ensure((size_t)n_img * n * sizeof(double)));     // the real-space variant keeps them
    CK(ctx->scratch_b.ensure((size_t)slab * H * sizeof(cd)));           // transform intermediate
    const float *dsrc = pixels;
    if (!is_device) {
        // grow-only staging buffer owned by the context: no cudaMalloc / cudaFree (both synchronise the device) per call
        CK(ctx->staging.ensure((size_t)n_img * n * sizeof(float)));
        CK(cudaMemcpyAsync(ctx->staging.p, pixels, (size_t)n_img * n * sizeof(float), cudaMemcpyHostToDevice, st));
        dsrc = ctx->staging.as<float>();
    }
    CK(cudaMemsetAsync(ctx->flags.p, 0, sizeof(int), st));
    for (int i0 = 0; i0 < n_img; i0 += slab) {
        const int nb = std::min(slab, n_img - i0);
        double *cent = ctx->variant == 1 ? ctx->Oreal64.as<double>() + (size_t)i0 * n : ctx->scratch_a.as<double>();
        CK(launch_image_stats(dsrc + (size_t)i0 * n, nb, N, cent, ctx->Dw.as<double>() + i0, st));
        CK(launch_fft2_r2c_f64(cent, nb, N, ctx->scratch_b.as<cd>(), ctx->Ohat64.as<cd>() + (size_t)i0 * H, st));
        CK(launch_zero_dc(ctx->Ohat64.as<cd>() + (size_t)i0 * H, nb, H, st));
    }
    CK(launch_cast_spectrum(ctx->Ohat64.as<cd>(), ctx->Ohat32.as<cf>(), (size_t)n_img * H, st));
    CK(launch_beta(ctx->Dw.as<double>(), n_img, ctx->beta.as<float>(), ctx->flags.as<int>(), st));
    int fl = 0;
    CK(cudaMemcpyAsync(&fl, ctx->flags.p, sizeof(int), cudaMemcpyDeviceToHost, st));
    CK(cudaStreamSynchronize(st));                            // inputs are copied: the caller may free `pixels` after return
    if (fl & 1) {
        ctx->n_img = 0;
        FAIL(BIOEM_EBADARG, "push_images: an image is constant or not finite (sum of squared deviations from its mean is not > 0): its posterior is undefined");
    }
    ctx->push_launches = 4 * (int64_t)((n_img + slab - 1) / slab) + 2;
    ctx->n_img = n_img;
    ctx->img_variant = ctx->variant;
    ctx->ran = false; ctx->phase = 0;
    return BIOEM_OK;
}

// Orientations per work item: aim at >= 32 work items per SM, at most 32 orientations per item.
static int choose_oc(long long n_img, long long n_model, long long n_orient, int n_sm)
{
    long long oc = n_img * n_model * n_orient / (32LL * n_sm);
    if (oc < 1) oc = 1;
    if (oc > 32) oc = 32;
    if (oc > n_orient) oc = n_orient;
    return (int)oc;
}

enum { KERNEL_AUTO = 0, KERNEL_GENERIC = 1, KERNEL_PK = 2, KERNEL_C2 = 3, KERNEL_TM = 4, KERNEL_DFT = 5, KERNEL_REALSPACE = 6 };

// the fused kernel a run of (N, D) uses: the one asked for if it supports the shape, else the automatic choice
static int choose_kernel(int N, int D, int user)
{
    if (user == KERNEL_GENERIC) return KERNEL_GENERIC;
    if (user == KERNEL_C2 && c2_supported(N, D)) return KERNEL_C2;
    if (pk_supported(N, D)) return KERNEL_PK;
    if (tm_supported(N, D)) return KERNEL_TM;
    return KERNEL_GENERIC;
}

// ---- the run in phases.  bioem_run = all four on one context; ranks that shard the ORIENTATION grid (the paper's MPI axis,
// P:199) run phase 1 on their slice, exchange the partials, run phase 2 on all of them, phase 3 on the candidates they
// own, exchange the re-scored values, and phase 4 (paper_1609_06634_b200/shard.py: run_orientation_sharded).
static int run_checks(bioem_ctx *ctx)
{
    if (!ctx->N) FAIL(BIOEM_EBADSTATE, "run: image geometry not set");
    if (ctx->models.empty()) FAIL(BIOEM_EBADSTATE, "run: no model");
    if (!ctx->n_orient) FAIL(BIOEM_EBADSTATE, "run: no orientations");
    if (!ctx->n_ctf) FAIL(BIOEM_EBADSTATE, "run: no CTF grid");
    if (ctx->D < 0) FAIL(BIOEM_EBADSTATE, "run: shift range not set");
    if (!ctx->n_img) FAIL(BIOEM_EBADSTATE, "run: no images");
    const int N = ctx->N, D = ctx->D;
    if (2 * D + 1 > N) FAIL(BIOEM_EBADARG, "run: 2D+1 exceeds n_pix");
    if ((long long)ctx->n_orient * ctx->n_ctf > 0x7fffffffLL) FAIL(BIOEM_EUNSUPPORTED, "run: orientations x CTFs exceeds 2^31");
    if (fused_smem_bytes(N, D) == 0) FAIL(BIOEM_EUNSUPPORTED, "run: shift range too large for the shared-memory plan at this n_pix");
    for (auto &m : ctx->models)
        if (m.kind == 1 && (m.n_vox != N || std::fabs(m.voxel - ctx->px) > 1e-9 * ctx->px))
            FAIL(BIOEM_EUNSUPPORTED, "run: density model needs n_vox == n_pix and voxel_A == pixel_size_A (R21)");
    return BIOEM_OK;
}

int bioem_run_partial(bioem_ctx *ctx)
{
    if (!ctx) return BIOEM_EBADARG;
    int rc = run_checks(ctx);
    if (rc) return rc;
    const int N = ctx->N, D = ctx->D, Ofull = ctx->n_orient, C = ctx->n_ctf, I = ctx->n_img, M = (int)ctx->models.size();
    const bool sliced = ctx->slice_end >= 0;
    const int o_first = sliced ? ctx->slice_begin : 0, O = (sliced ? ctx->slice_end : Ofull) - o_first;      // resident orientations
    if (sliced && (o_first < 0 || O < 0 || o_first + O > Ofull)) FAIL(BIOEM_EBADARG, "run: orientation slice outside the grid");
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const size_t n = (size_t)N * N, H = (size_t)(N / 2 + 1) * N;
    const size_t MO = (size_t)M * O, MOC = MO * C;
    ctx->ran = false; ctx->phase = 0;
    ctx->launches = 0; ctx->fused_launches = 0;
    if (ctx->run_o_first != o_first || ctx->run_o_local != O) ctx->pre_valid = false;     // the cache holds another slice

    CK(ctx->F064.ensure(MO * H * sizeof(cd)));
    CK(ctx->F032.ensure(MO * H * sizeof(cf)));
    CK(ctx->K64.ensure((size_t)C * H * sizeof(double)));
    CK(ctx->K32.ensure((size_t)C * H * sizeof(float)));
    CK(ctx->Tc64.ensure(MOC * sizeof(double)));
    CK(ctx->h64.ensure(MOC * sizeof(double)));
    CK(ctx->alpha32.ensure(MOC * sizeof(float)));
    CK(ctx->h32.ensure(MOC * sizeof(float)));
    const int kern = choose_kernel(N, D, ctx->kernel_user);
    const bool use_pk = kern == KERNEL_PK, use_c2 = kern == KERNEL_C2, use_tm = kern == KERNEL_TM;
    // an orientation slice leaves the chunk size to the caller: every rank must cut the grid at the same places
    if (sliced && ctx->oc_user <= 0) FAIL(BIOEM_EBADSTATE, "run: set_orientation_chunk before scoring an orientation slice (all ranks the same value)");
    int oc = ctx->oc_user > 0 ? std::min(ctx->oc_user, Ofull) : choose_oc(I, M, Ofull, ctx->n_sm);
    // posterior per orientation: the chunked kernels close their sums per orientation in a shared-memory table of 32 rows;
    // the cluster kernel (a cross-check, never chosen automatically) has no such table and runs one orientation per work item
    const bool fold = ctx->want_orient && !use_c2;
    if (sliced && ctx->want_orient && !fold) FAIL(BIOEM_EUNSUPPORTED, "run: the per-orientation posterior on an orientation slice needs a kernel that folds it (not the cluster kernel)");
    if (ctx->want_orient && !fold) oc = 1;
    if (fold && oc > 32) oc = 32;
    // (an EMPTY slice -- a rank beyond the last chunk, [n_orient, n_orient) -- begins wherever the grid ends)
    if (sliced && O > 0 && o_first % oc != 0) FAIL(BIOEM_EBADARG, "run: an orientation slice must begin at a multiple of the orientation chunk");
    const int cpm = (O + oc - 1) / oc;
    const int ppi = use_c2 ? 2 : 1;                                       // partials per work item (the cluster kernel writes one per CTA)
    const size_t items = (size_t)I * M * cpm * ppi;
    CK(ctx->blob.ensure(partial_blob_bytes(items)));
    if (fold) {
        CK(ctx->orient_m.ensure(MO * I * sizeof(float)));
        CK(ctx->orient_s.ensure(MO * I * sizeof(float)));
    }

    CK(cudaEventRecord(ctx->ev[0], st));
    if (!ctx->pre_valid) CK(cudaMemsetAsync(ctx->flags.as<int>() + 1, 0, sizeof(int), st));

    if (!ctx->pre_valid) {
        // ---- a3: CTF tables
        CK(launch_ctf_tables(ctx->ctf_a.as<double>(), ctx->ctf_A.as<double>(), ctx->ctf_b.as<double>(), C, N, ctx->px, ctx->K64.as<double>(),
                             ctx->K32.as<float>(), st));
        ctx->launches += 1;
        if (use_pk) {
            CK(ctx->Kt.ensure(pk_kt_bytes(N, C)));
            CK(launch_relayout_K(N, ctx->K32.as<float>(), ctx->Kt.as<float>(), C, st));
            ctx->launches += 1;
        } else if (use_c2) {
            CK(ctx->Kt.ensure(c2_kt_bytes(C)));
            CK(launch_relayout_K_c2(ctx->K32.as<float>(), ctx->Kt.as<float>(), C, st));
            ctx->launches += 1;
        } else if (use_tm) {
            CK(ctx->Kt.ensure(tm_kt_bytes(C)));
            CK(launch_relayout_K_tm(ctx->K32.as<float>(), ctx->Kt.as<float>(), C, st));
            ctx->launches += 1;
        }

        // ---- a1/a1' + a2: spectra of the projections of the resident orientations, model by model, batch by batch
        const int OB = 2048;                                          // orientations per projection batch (scratch: 32 bytes per pixel and orientation: 1.6 GB at 224^2)
        const double *rot = ctx->rot.as<double>() + (size_t)o_first * 9;
        for (int mi = 0; mi < M && O > 0; ++mi) {
            Model &m = ctx->models[mi];
            cd *F64m = ctx->F064.as<cd>() + (size_t)mi * O * H;
            cf *F32m = ctx->F032.as<cf>() + (size_t)mi * O * H;
            if (m.kind == 0) {
                CK(ctx->scratch_b.ensure((size_t)OB * H * sizeof(cd)));          // transform intermediate
                CK(ctx->scratch_c.ensure((size_t)OB * n * sizeof(long long)));   // fixed-point accumulator
                // fixed-point scale: a pixel can never hold more than the total |weight| of the model
                int ex = 0;
                std::frexp(m.sum_abs_w > 0 ? m.sum_abs_w : 1.0, &ex);
                const double fx_scale = std::ldexp(1.0, 60 - ex);
                for (int o0 = 0; o0 < O; o0 += OB) {
                    const int nb = std::min(OB, O - o0);
                    CK(launch_project_atoms(m.xyz.as<double>(), m.rad.as<double>(), m.wt.as<double>(), m.n_atoms, rot + (size_t)o0 * 9,
                                            nb, N, ctx->px, fx_scale, ctx->scratch_c.as<long long>(), st));
                    // I0 = fixed-point / scale, converted as the row transform loads it; the FP32 spectrum is written with the FP64 one
                    CK(launch_fft2_r2c_fixed(ctx->scratch_c.as<long long>(), 1.0 / fx_scale, nb, N, ctx->scratch_b.as<cd>(), F64m + (size_t)o0 * H,
                                             F32m + (size_t)o0 * H, st));
                    ctx->launches += 3;
                }
            } else {
                const size_t n3 = (size_t)N * N * N;
                CK(ctx->scratch_a.ensure(n3 * sizeof(cd)));
                CK(ctx->scratch_b.ensure(n3 * sizeof(cd)));
                CK(launch_dft3_f64(m.rho.as<float>(), N, ctx->scratch_a.as<cd>(), ctx->scratch_b.as<cd>(), st));
                CK(launch_slice_f64(ctx->scratch_a.as<cd>(), N, m.voxel, rot, O, F64m, st));
                CK(launch_cast_spectrum(F64m, F32m, (size_t)O * H, st));
                ctx->launches += 7;
            }
        }
        if (O > 0) {
            CK(launch_calc_stats(ctx->F064.as<cd>(), ctx->K64.as<double>(), (int)MO, O, Ofull, C, N,
                                 ctx->has_lp_orient ? ctx->lp_orient.as<double>() + o_first : nullptr,
                                 ctx->has_lp_ctf ? ctx->lp_ctf.as<double>() : nullptr, std::log((double)(2 * D + 1) * (2 * D + 1)),
                                 ctx->Tc64.as<double>(), ctx->h64.as<double>(), ctx->alpha32.as<float>(), ctx->h32.as<float>(), ctx->flags.as<int>() + 1, st));
            ctx->launches += 1;
        }
    }

    if (ctx->variant == 1) {
        // ---- the real-space, cropping variant: FP64 scoring of every calculated image against every image
        if (sliced) FAIL(BIOEM_EUNSUPPORTED, "run: the real-space variant does not support orientation slices");
        if (ctx->img_variant != 1) FAIL(BIOEM_EBADSTATE, "run: set the displacement variant before bioem_push_images (the real-space variant keeps the images in real space)");
        const int S = (2 * D + 1) * (2 * D + 1), RB = 64;                 // calculated images per batch
        const size_t IM = (size_t)I * M;
        CK(ctx->rs_T.ensure((size_t)RB * H * sizeof(cd)));
        CK(ctx->rs_I1.ensure((size_t)RB * n * sizeof(double)));
        CK(ctx->rs_cc.ensure((size_t)RB * S * sizeof(double)));
        CK(ctx->rs_ccc.ensure((size_t)RB * S * sizeof(double)));
        CK(ctx->rs_part.ensure(rs_partial_bytes(RB, I)));
        CK(ctx->rs_logw.ensure(RB * sizeof(double)));
        CK(ctx->rs_pair.ensure(RB * sizeof(long long)));
        CK(ctx->rs_m.ensure(IM * sizeof(double)));
        CK(ctx->rs_s.ensure(IM * sizeof(double)));
        CK(ctx->rs_best.ensure(IM * sizeof(double)));
        CK(ctx->rs_bpair.ensure(IM * sizeof(long long)));
        CK(ctx->rs_bshift.ensure(IM * sizeof(int)));
        CK(ctx->logp.ensure(IM * sizeof(double)));
        CK(ctx->logp32.ensure(IM * sizeof(double)));
        CK(ctx->best.ensure(IM * 4 * sizeof(int32_t)));
        CK(ctx->best_logp.ensure(IM * sizeof(double)));
        double *po_m = nullptr, *po_s = nullptr;                         // posterior per orientation: running (m, s) per (image, model, orientation)
        if (ctx->want_orient) {
            CK(ctx->orient_m.ensure(IM * O * sizeof(double)));
            CK(ctx->orient_s.ensure(IM * O * sizeof(double)));
            CK(ctx->logp_orient.ensure(IM * O * sizeof(double)));
            po_m = ctx->orient_m.as<double>(); po_s = ctx->orient_s.as<double>();
        }
        CK(cudaEventRecord(ctx->ev[1], st));
        if (po_m) { CK(launch_rs_orient_init(IM * O, po_m, po_s, st)); ctx->launches += 1; }
        CK(launch_rs_init((int)IM, ctx->rs_m.as<double>(), ctx->rs_s.as<double>(), ctx->rs_best.as<double>(), ctx->rs_bpair.as<long long>(),
                          ctx->rs_bshift.as<int>(), st));
        ctx->launches += 1;
        for (int mi = 0; mi < M; ++mi)
            for (int o0 = 0; o0 < O; o0 += RB) {
                const int nb = std::min(RB, O - o0);
                for (int c = 0; c < C; ++c) {
                    CK(launch_rs_calc_images(ctx->F064.as<cd>() + ((size_t)mi * O + o0) * H, ctx->K64.as<double>() + (size_t)c * H, nb, N,
                                             ctx->rs_T.as<cd>(), ctx->rs_I1.as<double>(), st));
                    CK(launch_rs_batch_meta(ctx->h64.as<double>(), ctx->Tc64.as<double>(), mi, O, C, o0, c, nb, ctx->rs_logw.as<double>(),
                                            ctx->rs_pair.as<long long>(), st));
                    CK(launch_rs_score(ctx->Oreal64.as<double>(), ctx->Dw.as<double>(), ctx->rs_I1.as<double>(), ctx->rs_logw.as<double>(),
                                       ctx->rs_pair.as<long long>(), nb, I, M, mi, N, D, ctx->rs_cc.as<double>(), ctx->rs_ccc.as<double>(), ctx->rs_part.p,
                                       ctx->rs_m.as<double>(), ctx->rs_s.as<double>(), ctx->rs_best.as<double>(), ctx->rs_bpair.as<long long>(),
                                       ctx->rs_bshift.as<int>(), ctx->flags.as<int>() + 1, po_m, po_s, O, o0, st));
                    ctx->launches += 6; ctx->fused_launches += 1;
                }
            }
        CK(cudaEventRecord(ctx->ev[2], st));
        const double nn = (double)n;
        const double const_n = -0.5 * (nn - 2.0) * std::log(2.0 * M_PI) + 0.5 * (nn - 5.0) * std::log(2.0) + std::lgamma(0.5 * (nn - 3.0));
        CK(launch_rs_final(ctx->rs_m.as<double>(), ctx->rs_s.as<double>(), ctx->rs_best.as<double>(), ctx->rs_bpair.as<long long>(),
                           ctx->rs_bshift.as<int>(), ctx->Dw.as<double>(), I, M, C, N, D, const_n, ctx->logp.as<double>(), ctx->logp32.as<double>(),
                           ctx->best.as<int32_t>(), ctx->best_logp.as<double>(), st));
        ctx->launches += 1;
        if (po_m) {
            CK(launch_rs_orient_final(po_m, po_s, ctx->Dw.as<double>(), I, M, O, N, const_n, ctx->logp_orient.as<double>(), st));
            ctx->launches += 1;
        }
        CK(cudaEventRecord(ctx->ev[3], st));
        ctx->pre_valid = true; ctx->flags_checked = false;
        ctx->run_kernel = KERNEL_REALSPACE; ctx->run_oc = 0; ctx->run_o_first = 0; ctx->run_o_local = O; ctx->run_chunks = 0;
        ctx->run_models = M; ctx->run_orient = Ofull; ctx->run_ctf = C; ctx->run_D = D; ctx->run_img = I;
        ctx->ran = true; ctx->ran_orient = po_m != nullptr; ctx->phase = 4;
        return BIOEM_OK;
    }

    // ---- a4-a6: the fused kernel
    FusedParams p{};
    p.Ohat = ctx->Ohat32.as<cf>(); p.F0 = ctx->F032.as<cf>(); p.K = ctx->K32.as<float>();
    p.alpha = ctx->alpha32.as<float>(); p.hterm = ctx->h32.as<float>(); p.beta = ctx->beta.as<float>();
    p.n_img = I; p.n_model = M; p.n_orient = O; p.n_ctf = C; p.D = D; p.oc = oc; p.chunks_per_model = cpm; p.o_first = o_first;
    p.cA = (float)(-0.5 * ((double)n - 3.0) * 1.4426950408889634);
    p.part_m = ctx->blob.as<float>(); p.part_s = p.part_m + items; p.part_top = reinterpret_cast<TopEntry *>(p.part_s + items);
    if (fold) { p.orient_m = ctx->orient_m.as<float>(); p.orient_s = ctx->orient_s.as<float>(); }
    CK(cudaEventRecord(ctx->ev[1], st));
    int nl = 1;
    if (items == 0) nl = 0;
    else if (use_pk) CK(launch_fused_pk(N, p, ctx->Kt.as<float>(), false, st));
    else if (use_c2) CK(launch_fused_c2(p, ctx->Kt.as<float>(), false, st));
    else if (use_tm) CK(launch_fused_tm(p, ctx->Kt.as<float>(), false, st));
    else CK(launch_fused(N, p, false, st, &nl));
    CK(cudaEventRecord(ctx->ev[2], st));
    ctx->launches += nl; ctx->fused_launches += nl;
    ctx->pre_valid = true;
    ctx->flags_checked = false;
    ctx->run_kernel = kern; ctx->run_oc = oc; ctx->run_o_first = o_first; ctx->run_o_local = O; ctx->run_chunks = cpm * ppi;
    ctx->run_models = M; ctx->run_orient = Ofull; ctx->run_ctf = C; ctx->run_D = D; ctx->run_img = I;
    ctx->run_orient_folded = fold; ctx->run_want_orient = ctx->want_orient;
    ctx->phase = 1;
    return BIOEM_OK;
}

int bioem_get_partials_size(bioem_ctx *ctx, int64_t *n_bytes, int32_t *n_chunks)
{
    if (!ctx) return BIOEM_EBADARG;
    if (ctx->phase < 1) FAIL(BIOEM_EBADSTATE, "get_partials_size: call bioem_run_partial first");
    if (ctx->run_kernel == KERNEL_REALSPACE) FAIL(BIOEM_EBADSTATE, "the real-space variant has no partials");
    if (n_bytes) *n_bytes = (int64_t)partial_blob_bytes((size_t)ctx->run_img * ctx->run_models * ctx->run_chunks);
    if (n_chunks) *n_chunks = ctx->run_chunks;
    return BIOEM_OK;
}

int bioem_export_partials(bioem_ctx *ctx, void *dst, int is_device)
{
    if (!ctx || !dst) return BIOEM_EBADARG;
    if (ctx->phase < 1) FAIL(BIOEM_EBADSTATE, "export_partials: call bioem_run_partial first");
    if (ctx->run_kernel == KERNEL_REALSPACE) FAIL(BIOEM_EBADSTATE, "the real-space variant has no partials");
    CK(cudaSetDevice(ctx->device));
    const size_t bytes = partial_blob_bytes((size_t)ctx->run_img * ctx->run_models * ctx->run_chunks);
    if (bytes) CK(cudaMemcpyAsync(dst, ctx->blob.p, bytes, is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return BIOEM_OK;
}

// a6: the fixed-order combine over `n_blobs` blobs (NULL = this context's own partials)
int bioem_merge_partials(bioem_ctx *ctx, int n_blobs, const void *blobs, int64_t stride_bytes, const int32_t *chunks_of_blob, int is_device)
{
    if (!ctx) return BIOEM_EBADARG;
    if (ctx->phase < 1) FAIL(BIOEM_EBADSTATE, "merge_partials: call bioem_run_partial first");
    if (ctx->run_kernel == KERNEL_REALSPACE) FAIL(BIOEM_EBADSTATE, "the real-space variant has no partials");
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const int I = ctx->run_img, M = ctx->run_models;
    const size_t IM = (size_t)I * M;
    CK(ctx->m32.ensure(IM * sizeof(double)));
    CK(ctx->s32.ensure(IM * sizeof(double)));
    CK(ctx->top.ensure(IM * BIOEM_TOPK * sizeof(TopEntry)));
    const unsigned char *src = nullptr;
    std::vector<int> chunks;
    if (!blobs) {
        n_blobs = 1; stride_bytes = 0; chunks.assign(1, ctx->run_chunks);
        src = ctx->blob.as<unsigned char>();
    } else {
        if (n_blobs < 1 || !chunks_of_blob || stride_bytes < 0 || stride_bytes % 4) FAIL(BIOEM_EBADARG, "merge_partials: n_blobs < 1, NULL chunk counts or a stride that is not a multiple of 4");
        long long tot = 0;
        for (int r = 0; r < n_blobs; ++r) {
            if (chunks_of_blob[r] < 0 || (int64_t)partial_blob_bytes(IM * chunks_of_blob[r]) > stride_bytes) FAIL(BIOEM_EBADARG, "merge_partials: a blob does not fit its stride");
            chunks.push_back(chunks_of_blob[r]);
            tot += chunks_of_blob[r];
        }
        if (is_device) src = static_cast<const unsigned char *>(blobs);
        else {
            CK(ctx->gathered.ensure((size_t)n_blobs * stride_bytes));
            CK(cudaMemcpyAsync(ctx->gathered.p, blobs, (size_t)n_blobs * stride_bytes, cudaMemcpyHostToDevice, st));
            src = ctx->gathered.as<unsigned char>();
        }
    }
    CK(ctx->blob_chunks.ensure(chunks.size() * sizeof(int)));
    CK(cudaMemcpyAsync(ctx->blob_chunks.p, chunks.data(), chunks.size() * sizeof(int), cudaMemcpyHostToDevice, st));
    CK(launch_merge(src, (size_t)stride_bytes, ctx->blob_chunks.as<int>(), n_blobs, I, M, ctx->m32.as<double>(), ctx->s32.as<double>(),
                    ctx->top.as<TopEntry>(), st));
    if (blobs && !is_device) CK(cudaStreamSynchronize(st));      // a host `blobs` may go away (the small `chunks` array is pageable: its copy is staged before cudaMemcpyAsync returns)
    ctx->launches += 1;
    ctx->phase = 2;
    return BIOEM_OK;
}

// a7, first half: FP64 values of the merged candidates whose orientation is resident here; 0 for the others
int bioem_rescore_local(bioem_ctx *ctx)
{
    if (!ctx) return BIOEM_EBADARG;
    if (ctx->phase < 2) FAIL(BIOEM_EBADSTATE, "rescore_local: call bioem_merge_partials first");
    if (ctx->run_kernel == KERNEL_REALSPACE) FAIL(BIOEM_EBADSTATE, "the real-space variant has no re-scoring step");
    CK(cudaSetDevice(ctx->device));
    const int I = ctx->run_img, M = ctx->run_models;
    CK(ctx->g64.ensure((size_t)I * M * BIOEM_TOPK * sizeof(double)));
    CK(launch_rescore(ctx->Ohat64.as<cd>(), ctx->F064.as<cd>(), ctx->K64.as<double>(), ctx->Tc64.as<double>(), ctx->h64.as<double>(),
                      ctx->Dw.as<double>(), ctx->top.as<TopEntry>(), BIOEM_TOPK, I, M, ctx->run_o_local, ctx->run_ctf, ctx->N, ctx->run_D, -1,
                      ctx->run_o_first, ctx->g64.as<double>(), ctx->stream));
    ctx->launches += 1;
    ctx->phase = 3;
    return BIOEM_OK;
}

int bioem_export_rescore(bioem_ctx *ctx, double *dst, int is_device)
{
    if (!ctx || !dst) return BIOEM_EBADARG;
    if (ctx->phase < 3) FAIL(BIOEM_EBADSTATE, "export_rescore: call bioem_rescore_local first");
    CK(cudaSetDevice(ctx->device));
    CK(cudaMemcpyAsync(dst, ctx->g64.p, (size_t)ctx->run_img * ctx->run_models * BIOEM_TOPK * sizeof(double),
                       is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return BIOEM_OK;
}

int bioem_import_rescore(bioem_ctx *ctx, const double *src, int is_device)
{
    if (!ctx || !src) return BIOEM_EBADARG;
    if (ctx->phase < 3) FAIL(BIOEM_EBADSTATE, "import_rescore: call bioem_rescore_local first");
    CK(cudaSetDevice(ctx->device));
    CK(cudaMemcpyAsync(ctx->g64.p, src, (size_t)ctx->run_img * ctx->run_models * BIOEM_TOPK * sizeof(double),
                       is_device ? cudaMemcpyDeviceToDevice : cudaMemcpyHostToDevice, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return BIOEM_OK;
}

// a7, second half: corrected log-sum-exp, argmax, constants
int bioem_finish(bioem_ctx *ctx)
{
    if (!ctx) return BIOEM_EBADARG;
    if (ctx->phase < 3) FAIL(BIOEM_EBADSTATE, "finish: call bioem_rescore_local first");
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const int I = ctx->run_img, M = ctx->run_models, N = ctx->N;
    const size_t IM = (size_t)I * M;
    CK(ctx->logp.ensure(IM * sizeof(double)));
    CK(ctx->logp32.ensure(IM * sizeof(double)));
    CK(ctx->best.ensure(IM * 4 * sizeof(int32_t)));
    CK(ctx->best_logp.ensure(IM * sizeof(double)));
    const double nn = (double)N * N;
    const double const_n = -0.5 * (nn - 2.0) * std::log(2.0 * M_PI) + 0.5 * (nn - 5.0) * std::log(2.0) + std::lgamma(0.5 * (nn - 3.0));
    CK(launch_final(ctx->m32.as<double>(), ctx->s32.as<double>(), ctx->top.as<TopEntry>(), ctx->g64.as<double>(), ctx->Dw.as<double>(), I, M,
                    ctx->run_ctf, N, ctx->run_D, const_n, ctx->logp.as<double>(), ctx->logp32.as<double>(), ctx->best.as<int32_t>(),
                    ctx->best_logp.as<double>(), st));
    ctx->launches += 1;
    ctx->ran_orient = false;
    if (ctx->run_want_orient) {
        // the per-orientation (m, s): the folded table, or (cluster kernel, one orientation per work item) the partials themselves
        const size_t items = IM * ctx->run_chunks;
        const float *part_m = ctx->run_orient_folded ? ctx->orient_m.as<float>() : ctx->blob.as<float>();
        const float *part_s = ctx->run_orient_folded ? ctx->orient_s.as<float>() : part_m + items;
        // the resident orientations only: a rank of an orientation-sharded run produces its slice of the output
        CK(ctx->logp_orient.ensure(IM * std::max(ctx->run_o_local, 1) * sizeof(double)));
        if (ctx->run_o_local > 0)
            CK(launch_orient_final(part_m, part_s, ctx->run_orient_folded ? 1 : 2, ctx->top.as<TopEntry>(), ctx->g64.as<double>(), ctx->Dw.as<double>(), I, M,
                                   ctx->run_o_local, ctx->run_o_first, ctx->run_ctf, N, const_n, ctx->logp_orient.as<double>(), st));
        ctx->launches += 1;
        ctx->ran_orient = true;
    }
    CK(cudaEventRecord(ctx->ev[3], st));
    ctx->ran = true;
    ctx->phase = 4;
    return BIOEM_OK;
}

int bioem_run(bioem_ctx *ctx)
{
    if (!ctx) return BIOEM_EBADARG;
    if (ctx->slice_end >= 0 && !(ctx->slice_begin == 0 && ctx->slice_end == ctx->n_orient))
        FAIL(BIOEM_EBADSTATE, "run: an orientation slice is set: this context holds part of the grid (use the phased calls, or clear the slice)");
    int rc = bioem_run_partial(ctx);
    if (!rc && ctx->variant == 1) return BIOEM_OK;                       // the real-space variant has no partials: run_partial finished the run
    if (!rc) rc = bioem_merge_partials(ctx, 0, nullptr, 0, nullptr, 1);
    if (!rc) rc = bioem_rescore_local(ctx);
    if (!rc) rc = bioem_finish(ctx);
    return rc;
}

int bioem_set_displacement_variant(bioem_ctx *ctx, int variant)
{
    if (!ctx) return BIOEM_EBADARG;
    if (variant != 0 && variant != 1) FAIL(BIOEM_EBADARG, "set_displacement_variant: 0 (Fourier space, circular) or 1 (real space, cropping)");
    ctx->variant = variant;
    ctx->ran = false; ctx->phase = 0;
    return BIOEM_OK;
}

int bioem_set_orientation_slice(bioem_ctx *ctx, int o_begin, int o_end)
{
    if (!ctx) return BIOEM_EBADARG;
    if (o_end >= 0 && (o_begin < 0 || o_begin > o_end)) FAIL(BIOEM_EBADARG, "set_orientation_slice: need 0 <= o_begin <= o_end (o_end < 0 clears the slice)");
    ctx->slice_begin = o_end < 0 ? 0 : o_begin;
    ctx->slice_end = o_end < 0 ? -1 : o_end;
    ctx->ran = false; ctx->phase = 0; ctx->pre_valid = false;
    return BIOEM_OK;
}

// bioem_run only enqueues: a degenerate calculated image (T_c = 0: the model projects to nothing inside the box, or the CTF
// table is all zero) is seen by the device and reported by the first call that synchronises.
static int check_run_flags(bioem_ctx *ctx)
{
    if (ctx->flags_checked) return BIOEM_OK;
    int fl = 0;
    CK(cudaMemcpyAsync(&fl, ctx->flags.as<int>() + 1, sizeof(int), cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    if (fl & 2) {
        ctx->ran = false; ctx->phase = 0; ctx->pre_valid = false;
        FAIL(BIOEM_EBADARG, "run: a calculated image is empty or not finite (T_c = sum |I1|^2 is not > 0): its posterior is undefined");
    }
    ctx->flags_checked = true;
    return BIOEM_OK;
}

static int fetch(bioem_ctx *ctx, void *dst, const void *src, size_t bytes)
{
    CK(cudaSetDevice(ctx->device));
    if (ctx->ran) { int rc = check_run_flags(ctx); if (rc) return rc; }
    CK(cudaMemcpyAsync(dst, src, bytes, cudaMemcpyDeviceToHost, ctx->stream));
    CK(cudaStreamSynchronize(ctx->stream));
    return BIOEM_OK;
}

int bioem_get_log_posterior(bioem_ctx *ctx, double *out)
{
    if (!ctx || !out) return BIOEM_EBADARG;
    if (!ctx->ran) FAIL(BIOEM_EBADSTATE, "get_log_posterior: no completed run");
    return fetch(ctx, out, ctx->logp.p, (size_t)ctx->run_img * ctx->run_models * sizeof(double));
}

int bioem_set_orientation_posterior(bioem_ctx *ctx, int enable)
{
    if (!ctx) return BIOEM_EBADARG;
    if (enable != 0 && enable != 1) FAIL(BIOEM_EBADARG, "set_orientation_posterior: enable must be 0 or 1");
    ctx->want_orient = enable != 0;
    return BIOEM_OK;
}

int bioem_get_orientation_log_posterior(bioem_ctx *ctx, double *out)
{
    if (!ctx || !out) return BIOEM_EBADARG;
    if (!ctx->ran || !ctx->ran_orient) FAIL(BIOEM_EBADSTATE, "get_orientation_log_posterior: no completed run with the option enabled");
    return fetch(ctx, out, ctx->logp_orient.p, (size_t)ctx->run_img * ctx->run_models * ctx->run_o_local * sizeof(double));
}

int bioem_get_ensemble_log_posterior(bioem_ctx *ctx, const double *weights, double *out_total, double *out_per_image)
{
    if (!ctx || !out_total) return BIOEM_EBADARG;
    if (!ctx->ran) FAIL(BIOEM_EBADSTATE, "get_ensemble_log_posterior: no completed run");
    CK(cudaSetDevice(ctx->device));
    const int I = ctx->run_img, M = ctx->run_models;
    std::vector<double> lw(M);
    for (int m = 0; m < M; ++m) {
        const double w = weights ? weights[m] : 1.0 / M;
        if (!(w >= 0.0)) FAIL(BIOEM_EBADARG, "get_ensemble_log_posterior: weights must be >= 0");
        lw[m] = std::log(w);                                          // w = 0 -> -inf: the model drops out of the sum
    }
    DBuf dlw, dpi, dt;
    cudaError_t e = dlw.ensure(M * sizeof(double));
    if (e == cudaSuccess) e = dpi.ensure((size_t)I * sizeof(double));
    if (e == cudaSuccess) e = dt.ensure(sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpyAsync(dlw.p, lw.data(), M * sizeof(double), cudaMemcpyHostToDevice, ctx->stream);
    if (e == cudaSuccess) e = launch_ensemble(ctx->logp.as<double>(), dlw.as<double>(), I, M, dpi.as<double>(), dt.as<double>(), ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(out_total, dt.p, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess && out_per_image) e = cudaMemcpyAsync(out_per_image, dpi.p, (size_t)I * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    dlw.release(); dpi.release(); dt.release();
    CK(e);
    return BIOEM_OK;
}

int bioem_debug_log_posterior_f32(bioem_ctx *ctx, double *out)
{
    if (!ctx || !out) return BIOEM_EBADARG;
    if (!ctx->ran) FAIL(BIOEM_EBADSTATE, "debug_log_posterior_f32: no completed run");
    return fetch(ctx, out, ctx->logp32.p, (size_t)ctx->run_img * ctx->run_models * sizeof(double));
}

int bioem_get_best(bioem_ctx *ctx, int32_t *orient_idx, int32_t *ctf_idx, int32_t *dx, int32_t *dy, double *best_log_p)
{
    if (!ctx) return BIOEM_EBADARG;
    if (!ctx->ran) FAIL(BIOEM_EBADSTATE, "get_best: no completed run");
    const size_t IM = (size_t)ctx->run_img * ctx->run_models;
    std::vector<int32_t> b(4 * IM);
    int rc = fetch(ctx, b.data(), ctx->best.p, 4 * IM * sizeof(int32_t));
    if (rc) return rc;
    for (size_t i = 0; i < IM; ++i) {
        if (orient_idx) orient_idx[i] = b[4 * i];
        if (ctf_idx) ctf_idx[i] = b[4 * i + 1];
        if (dx) dx[i] = b[4 * i + 2];
        if (dy) dy[i] = b[4 * i + 3];
    }
    if (best_log_p) return fetch(ctx, best_log_p, ctx->best_logp.p, IM * sizeof(double));
    return BIOEM_OK;
}

static int check_tuple(bioem_ctx *ctx, int img, int model, int orient, int ctf)
{
    if (!ctx->ran) FAIL(BIOEM_EBADSTATE, "debug: call bioem_run first (the precomputed spectra are reused)");
    if (img < 0 || img >= ctx->run_img || model < 0 || model >= ctx->run_models || orient < ctx->run_o_first ||
        orient >= ctx->run_o_first + ctx->run_o_local || ctf < 0 || ctf >= ctx->run_ctf)
        FAIL(BIOEM_EBADARG, "debug: index out of range (or an orientation outside this context's slice)");
    return BIOEM_OK;
}

int bioem_debug_calc_image(bioem_ctx *ctx, int model, int orient, int ctf, float *out_real)
{
    if (!ctx || !out_real) return BIOEM_EBADARG;
    int rc = check_tuple(ctx, 0, model, orient, ctf);
    if (rc) return rc;
    CK(cudaSetDevice(ctx->device));
    const int N = ctx->N;
    const size_t n = (size_t)N * N, H = (size_t)(N / 2 + 1) * N;
    CK(ctx->dump.ensure(n * sizeof(double)));
    CK(launch_calc_image(ctx->F064.as<cd>() + ((size_t)model * ctx->run_o_local + (orient - ctx->run_o_first)) * H, ctx->K64.as<double>() + (size_t)ctf * H, N,
                         ctx->dump.as<double>(), ctx->stream));
    std::vector<double> tmp(n);
    rc = fetch(ctx, tmp.data(), ctx->dump.p, n * sizeof(double));
    if (rc) return rc;
    for (size_t i = 0; i < n; ++i) out_real[i] = (float)tmp[i];
    return BIOEM_OK;
}

// the synthetic map of a parameter set -- the calculated image of (model, orient, ctf), displaced, scaled and offset (Eq. 7)
int bioem_get_synthetic_map(bioem_ctx *ctx, int model, int orient, int ctf, int dx, int dy, const float *fit_to_image, float *out,
                            double *out_norm_offset)
{
    if (!ctx || !out) return BIOEM_EBADARG;
    int rc = check_tuple(ctx, 0, model, orient, ctf);
    if (rc) return rc;
    const int N = ctx->N;
    if (dx <= -N || dx >= N || dy <= -N || dy >= N) FAIL(BIOEM_EBADARG, "get_synthetic_map: |dx|, |dy| must be < n_pix");
    CK(cudaSetDevice(ctx->device));
    cudaStream_t st = ctx->stream;
    const size_t n = (size_t)N * N, H = (size_t)(N / 2 + 1) * N;
    CK(ctx->dump.ensure((n + 2) * sizeof(double) + n * sizeof(float)));
    double *I1 = ctx->dump.as<double>(), *no = I1 + n;
    float *dout = reinterpret_cast<float *>(no + 2);
    const float *dobs = nullptr;
    if (fit_to_image) {
        CK(ctx->staging.ensure(n * sizeof(float)));
        CK(cudaMemcpyAsync(ctx->staging.p, fit_to_image, n * sizeof(float), cudaMemcpyHostToDevice, st));
        dobs = ctx->staging.as<float>();
    }
    CK(launch_calc_image(ctx->F064.as<cd>() + ((size_t)model * ctx->run_o_local + (orient - ctx->run_o_first)) * H, ctx->K64.as<double>() + (size_t)ctf * H, N, I1, st));
    CK(launch_synth_map(I1, dobs, N, dx, dy, ctx->variant == 1, dout, no, st));
    rc = fetch(ctx, out, dout, n * sizeof(float));
    if (rc) return rc;
    if (out_norm_offset) CK(cudaMemcpy(out_norm_offset, no, 2 * sizeof(double), cudaMemcpyDeviceToHost));
    return BIOEM_OK;
}

int bioem_debug_shift_map(bioem_ctx *ctx, int img, int model, int orient, int ctf, double *out)
{
    if (!ctx || !out) return BIOEM_EBADARG;
    int rc = check_tuple(ctx, img, model, orient, ctf);
    if (rc) return rc;
    if (ctx->run_kernel == KERNEL_REALSPACE) FAIL(BIOEM_EUNSUPPORTED, "debug_shift_map: the last run used the real-space variant (FP64 throughout, no FP32 map)");
    CK(cudaSetDevice(ctx->device));
    const int N = ctx->N, D = ctx->run_D, KK = 2 * D + 1;
    const size_t n = (size_t)N * N;
    CK(ctx->dump.ensure((size_t)KK * KK * sizeof(float)));
    FusedParams p{};
    p.Ohat = ctx->Ohat32.as<cf>(); p.F0 = ctx->F032.as<cf>(); p.K = ctx->K32.as<float>();
    p.alpha = ctx->alpha32.as<float>(); p.hterm = ctx->h32.as<float>(); p.beta = ctx->beta.as<float>();
    p.n_img = ctx->run_img; p.n_model = ctx->run_models; p.n_orient = ctx->run_o_local; p.n_ctf = ctx->run_ctf; p.D = D; p.oc = 1;
    p.o_first = ctx->run_o_first;
    p.chunks_per_model = 1;
    p.cA = (float)(-0.5 * ((double)n - 3.0) * 1.4426950408889634);
    p.dump = ctx->dump.as<float>(); p.dump_img = img; p.dump_model = model; p.dump_orient = orient - ctx->run_o_first; p.dump_ctf = ctf;
    if (ctx->run_kernel == KERNEL_PK) CK(launch_fused_pk(N, p, ctx->Kt.as<float>(), true, ctx->stream));
    else if (ctx->run_kernel == KERNEL_C2) CK(launch_fused_c2(p, ctx->Kt.as<float>(), true, ctx->stream));
    else if (ctx->run_kernel == KERNEL_TM) CK(launch_fused_tm(p, ctx->Kt.as<float>(), true, ctx->stream));
    else CK(launch_fused(N, p, true, ctx->stream, nullptr));
    std::vector<float> tmp((size_t)KK * KK);
    rc = fetch(ctx, tmp.data(), ctx->dump.p, tmp.size() * sizeof(float));
    if (rc) return rc;
    std::vector<double> dw(1);
    rc = fetch(ctx, dw.data(), ctx->Dw.as<double>() + img, sizeof(double));
    if (rc) return rc;
    const double nn = (double)n;
    const double base = -0.5 * (nn - 2.0) * std::log(2.0 * M_PI) + 0.5 * (nn - 5.0) * std::log(2.0) + std::lgamma(0.5 * (nn - 3.0)) -
                        0.5 * (nn - 3.0) * std::log(dw[0]);
    for (size_t i = 0; i < tmp.size(); ++i) out[i] = base + (double)tmp[i] * 0.6931471805599453;   // kernel units are base 2
    return BIOEM_OK;
}

int bioem_debug_shift_map_f64(bioem_ctx *ctx, int img, int model, int orient, int ctf, double *out)
{
    if (!ctx || !out) return BIOEM_EBADARG;
    int rc = check_tuple(ctx, img, model, orient, ctf);
    if (rc) return rc;
    CK(cudaSetDevice(ctx->device));
    const int N = ctx->N, D = ctx->run_D, KK = 2 * D + 1, S = KK * KK;
    const size_t n = (size_t)N * N;
    std::vector<TopEntry> cand(S);
    for (int s = 0; s < S; ++s) cand[s] = {0.f, (uint32_t)(orient * ctx->run_ctf + ctf), (uint32_t)s};
    DBuf dc, dg;
    cudaError_t e = dc.ensure(S * sizeof(TopEntry));
    if (e == cudaSuccess) e = dg.ensure(S * sizeof(double));
    if (e == cudaSuccess) e = cudaMemcpyAsync(dc.p, cand.data(), S * sizeof(TopEntry), cudaMemcpyHostToDevice, ctx->stream);
    // one "image" slot = img: pass pointers offset so that candidate block 0 maps to (img, model)
    if (e == cudaSuccess)
        e = launch_rescore(ctx->Ohat64.as<cd>() + (size_t)img * (size_t)(N / 2 + 1) * N, ctx->F064.as<cd>(), ctx->K64.as<double>(),
                           ctx->Tc64.as<double>(), ctx->h64.as<double>(), ctx->Dw.as<double>() + img, dc.as<TopEntry>(), S, 1, ctx->run_models,
                           ctx->run_o_local, ctx->run_ctf, N, D, model, ctx->run_o_first, dg.as<double>(), ctx->stream);
    std::vector<double> g(S), dw(1);
    if (e == cudaSuccess) e = cudaMemcpyAsync(g.data(), dg.p, S * sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaMemcpyAsync(dw.data(), ctx->Dw.as<double>() + img, sizeof(double), cudaMemcpyDeviceToHost, ctx->stream);
    if (e == cudaSuccess) e = cudaStreamSynchronize(ctx->stream);
    dc.release(); dg.release();
    CK(e);
    const double nn = (double)n;
    const double base = -0.5 * (nn - 2.0) * std::log(2.0 * M_PI) + 0.5 * (nn - 5.0) * std::log(2.0) + std::lgamma(0.5 * (nn - 3.0)) -
                        0.5 * (nn - 3.0) * std::log(dw[0]);
    for (int s = 0; s < S; ++s) out[s] = base + g[s];
    return BIOEM_OK;
}

int bioem_set_orientation_chunk(bioem_ctx *ctx, int n_orient_per_item)
{
    if (!ctx) return BIOEM_EBADARG;
    if (n_orient_per_item < 0) FAIL(BIOEM_EBADARG, "set_orientation_chunk: negative");
    ctx->oc_user = n_orient_per_item;
    return BIOEM_OK;
}

int bioem_debug_set_kernel(bioem_ctx *ctx, int which)
{
    if (!ctx) return BIOEM_EBADARG;
    if (which != KERNEL_AUTO && which != KERNEL_GENERIC && which != KERNEL_C2) FAIL(BIOEM_EBADARG, "debug_set_kernel: 0 (automatic), 1 (generic) or 3 (two-CTA cluster, n_pix = 224)");
    ctx->kernel_user = which;
    return BIOEM_OK;
}

int bioem_invalidate_precompute(bioem_ctx *ctx)
{
    if (!ctx) return BIOEM_EBADARG;
    ctx->pre_valid = false;
    return BIOEM_OK;
}

int bioem_get_run_plan(bioem_ctx *ctx, int *kernel, int *n_orient_per_item)
{
    if (!ctx) return BIOEM_EBADARG;
    if (!ctx->ran && ctx->phase < 1) FAIL(BIOEM_EBADSTATE, "get_run_plan: no run yet");
    if (kernel) *kernel = ctx->run_kernel;
    if (n_orient_per_item) *n_orient_per_item = ctx->run_oc;
    return BIOEM_OK;
}

int bioem_get_timing(bioem_ctx *ctx, double *ms_total, double *ms_fused_kernel)
{
    if (!ctx) return BIOEM_EBADARG;
    if (!ctx->ran) FAIL(BIOEM_EBADSTATE, "get_timing: no completed run");
    CK(cudaSetDevice(ctx->device));
    CK(cudaEventSynchronize(ctx->ev[3]));
    float a = 0.f, b = 0.f;
    CK(cudaEventElapsedTime(&a, ctx->ev[0], ctx->ev[3]));
    CK(cudaEventElapsedTime(&b, ctx->ev[1], ctx->ev[2]));
    if (ms_total) *ms_total = a;
    if (ms_fused_kernel) *ms_fused_kernel = b;
    return BIOEM_OK;
}

int bioem_get_launch_count(bioem_ctx *ctx, int64_t *n_launches, int64_t *n_fused_launches)
{
    if (!ctx) return BIOEM_EBADARG;
    if (n_launches) *n_launches = ctx->launches + ctx->push_launches;       /* last push_images + last run */
    if (n_fused_launches) *n_fused_launches = ctx->fused_launches;
    return BIOEM_OK;
}

int bioem_measure_fp32_peak(bioem_ctx *ctx, double *tflops, double *sm_mhz)
{
    if (!ctx) return BIOEM_EBADARG;
    CK(cudaSetDevice(ctx->device));
    DBuf sink;
    CK(sink.ensure(64));
    const int iters = 4096;
    cudaEvent_t a, b;
    CK(cudaEventCreate(&a));
    CK(cudaEventCreate(&b));
    cudaError_t e = launch_fp32_peak(sink.as<float>(), 256, ctx->stream);        // warm-up
    float best = 1e30f;
    for (int r = 0; r < 5 && e == cudaSuccess; ++r) {
        cudaEventRecord(a, ctx->stream);
        e = launch_fp32_peak(sink.as<float>(), iters, ctx->stream);
        cudaEventRecord(b, ctx->stream);
        if (e == cudaSuccess) e = cudaEventSynchronize(b);
        float ms = 0.f;
        if (e == cudaSuccess) e = cudaEventElapsedTime(&ms, a, b);
        if (ms < best) best = ms;
    }
    cudaEventDestroy(a); cudaEventDestroy(b);
    sink.release();
    CK(e);
    const double flops = 148.0 * 8 * 256 * (double)iters * 128.0 * 2.0;
    if (tflops) *tflops = flops / (best * 1e-3) / 1e12;
    int khz = 0;
    cudaDeviceGetAttribute(&khz, cudaDevAttrClockRate, ctx->device);
    if (sm_mhz) *sm_mhz = khz / 1000.0;
    return BIOEM_OK;
}

}  // extern "C"
