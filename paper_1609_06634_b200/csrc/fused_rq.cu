// fused_rq.cu -- the hot loop for N = 64 and N = 128: "register-resident Q".
//
// Work item = (image w, model, chunk of orientations).  For one (w, o) the product Q(l,m) = conj(Ohat_w) F0_o
// (Eq. 12) is formed ONCE and kept in registers (16 complex per thread, thread = (column l, residue t of the
// two-step factorisation m = N2 j + t)).  The CTF loop ("for each pair of model orientation and particle image a
// loop over the PSF convolution kernels") then only streams the real radial table K_c (Eq. 5) -- 4 coalesced
// 16-byte loads per thread per CTF, prefetched one CTF ahead -- so per pair the kernel moves H*4 bytes from L2 instead of
// 3 arrays (the v1 kernel was L1/LSU-bound at 85 %, profiles/r1_v1_fused_small_full.csv).
//
//   pass 1 (per column, WARP-LOCAL: a warp owns 32/N2 whole columns, only __syncwarp):
//       A1  a = Q*K_c, 16-point DIF FFT in registers, spill to the warp's private shared-memory tile Z
//       B1  the 2D+1 pruned outputs by a Horner sum over the N2 residues: y[k] = sum_t (w^k)^t Z_t[k mod 16] -> G[c][dy][l]
//   CTA barrier (all columns of the CG CTFs of a group are in G)
//   pass 2 (per pair of rows dy, also warp-local): Hermitian completion, two real rows packed as one complex transform,
//       A2  16-point FFT, B2 Horner sum -> B(dx,dy) for two dy at once
//       a5  rho^2 = B^2 alpha_c^2 beta_w^2, g = cA log1p(-rho^2) + h_c (form C2; base-2 units inside the kernel)
//       a6  running log-sum-exp in registers, K best terms in per-warp sorted lists
// No float atomics, fixed reduction orders: bit-reproducible.
#include "common.cuh"
#include <math_constants.h>

namespace bioem {

static constexpr unsigned FULLM = 0xffffffffu;

template <int N> struct RQ {
    static constexpr int N1 = 16, N2 = N / 16, NC = N / 2 + 1, NTASK = NC * N2, NW = (NTASK + 31) / 32, NT = NW * 32;
    static constexpr int ZP = 17, ZW = 32 * ZP, CPW = 32 / N2;      // Z pitch, Z words per warp, columns per warp
};

__device__ __forceinline__ float ex2f(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ bool entry_before_rq(float ga, uint32_t pa, uint32_t sa, float gb, uint32_t pb, uint32_t sb)
{
    return ga > gb || (ga == gb && (pa < pb || (pa == pb && sa < sb)));
}

__device__ __forceinline__ void warp_topk_insert_rq(float g, uint32_t pair, uint32_t sh, bool valid, float &thr, TopEntry *list)
{
    unsigned m = __ballot_sync(FULLM, valid && g >= thr);
    if (m == 0) return;
    const int lane = threadIdx.x & 31;
    while (m) {
        int src = __ffs(m) - 1;
        m &= m - 1;
        float gv = __shfl_sync(FULLM, g, src);
        uint32_t pv = __shfl_sync(FULLM, pair, src), sv = __shfl_sync(FULLM, sh, src);
        TopEntry e = {0.f, 0u, 0u};
        if (lane < BIOEM_TOPK) e = list[lane];
        bool before = lane < BIOEM_TOPK && entry_before_rq(e.g, e.pair, e.shift, gv, pv, sv);
        int pos = __popc(__ballot_sync(FULLM, before));
        if (pos < BIOEM_TOPK) {
            if (lane >= pos && lane < BIOEM_TOPK - 1) list[lane + 1] = e;
            if (lane == pos) { TopEntry n = {gv, pv, sv}; list[pos] = n; }
            __syncwarp();
            thr = list[BIOEM_TOPK - 1].g;
        }
    }
}

// log1p(-x) for 0 <= x < 1: 5-term series below 2^-6 (truncation < 2e-10 relative), libdevice log1pf above.
__device__ __forceinline__ float log1p_neg(float x)
{
    if (x < 0.015625f) {
        float p = fmaf(x, 0.2f, 0.25f);
        p = fmaf(x, p, 0.33333334f);
        p = fmaf(x, p, 0.5f);
        p = fmaf(x, p, 1.0f);
        return -x * p;
    }
    return log1pf(-x);
}

// Horner sum over the N2 residues: sum_t r^t z[t*ZP]
template <int N2, int ZP>
__device__ __forceinline__ cf horner(const cf *zc, cf r)
{
    cf acc = zc[(N2 - 1) * ZP];
#pragma unroll
    for (int t = N2 - 2; t >= 0; --t) {
        cf z = zc[t * ZP];
        float nx = fmaf(r.x, acc.x, fmaf(-r.y, acc.y, z.x));
        float ny = fmaf(r.x, acc.y, fmaf(r.y, acc.x, z.y));
        acc.x = nx; acc.y = ny;
    }
    return acc;
}

template <int N, bool DUMP>
__global__ void __launch_bounds__(RQ<N>::NT, 1) k_fused_rq(FusedParams p, const float4 *__restrict__ Kt, int CG, int GP, unsigned magicKK)
{
    typedef RQ<N> C_;
    constexpr int N1 = C_::N1, N2 = C_::N2, NC = C_::NC, NTASK = C_::NTASK, NW = C_::NW, NT = C_::NT, ZP = C_::ZP, ZW = C_::ZW, CPW = C_::CPW;
    constexpr size_t H = (size_t)NC * N;
    const int D = p.D, KK = 2 * D + 1, NP = (KK + 1) / 2;
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    cf *Z = reinterpret_cast<cf *>(smem_raw);                        // [NW][32][ZP]  warp-private tiles
    cf *G = Z + (size_t)NW * ZW;                                     // [CG][KK][GP]
    cf *twH = G + (size_t)CG * KK * GP;                              // [KK]  w_N^{k}, k = kk - D
    float2 *sc = reinterpret_cast<float2 *>(twH + KK);               // [CG]  (alpha*beta, h) of the group's CTFs
    TopEntry *tops = reinterpret_cast<TopEntry *>(sc + CG);          // [NW][TOPK]
    float *red = reinterpret_cast<float *>(tops + NW * BIOEM_TOPK);  // [2 NW]

    int img, model, o_begin, o_end, item;
    if (DUMP) { img = p.dump_img; model = p.dump_model; o_begin = p.dump_orient; o_end = o_begin + 1; item = 0; }
    else {
        item = blockIdx.x;
        img = item % p.n_img;
        const int chunk = item / p.n_img;
        model = chunk / p.chunks_per_model;
        o_begin = (chunk % p.chunks_per_model) * p.oc;
        o_end = min(o_begin + p.oc, p.n_orient);
    }
    const float beta = p.beta[img];
    for (int i = tid; i < KK; i += NT) {
        float sn, cs;
        sincospif(2.0f * (float)(((i - D) % N + N) % N) / (float)N, &sn, &cs);
        twH[i] = {cs, sn};
    }
    if (tid < NW * BIOEM_TOPK) { TopEntry e0 = {-CUDART_INF_F, 0xffffffffu, 0xffffffffu}; tops[tid] = e0; }
    __syncthreads();

    // ---- per-thread constants
    const bool act1 = tid < NTASK;
    const int col = act1 ? tid / N2 : 0, t = tid % N2;
    const size_t qbase = (size_t)col * N + t;
    cf *Zw = Z + (size_t)warp * ZW;
    cf *zst = Zw + lane * ZP;
    const int ncols_w = max(0, min(CPW, NC - warp * CPW));           // whole columns owned by this warp
    const int nout1 = ncols_w * KK;
    const cf *Oimg = p.Ohat + (size_t)img * H;
    float lse_m = -CUDART_INF_F, lse_s = 0.f, thr = -CUDART_INF_F;
    TopEntry *mylist = tops + warp * BIOEM_TOPK;
    const int c_lo = DUMP ? p.dump_ctf : 0, c_hi = DUMP ? p.dump_ctf + 1 : p.n_ctf;

    // K of the first CTF
    float4 kq[N1 / 4];
#pragma unroll
    for (int g4 = 0; g4 < N1 / 4; ++g4) kq[g4] = Kt[((size_t)c_lo * (N1 / 4) + g4) * NT + tid];

    for (int o = o_begin; o < o_end; ++o) {
        // ---- Q = conj(Ohat) F0 for this thread's 16 bins (Eq. 12)
        cf q[N1];
        {
            const cf *F0 = p.F0 + ((size_t)model * p.n_orient + o) * H;
#pragma unroll
            for (int j = 0; j < N1; ++j) {
                cf ov = Oimg[qbase + (size_t)N2 * j], fv = F0[qbase + (size_t)N2 * j];
                q[j] = act1 ? cmulc(ov, fv) : cf{0.f, 0.f};
            }
        }
        for (int c0 = c_lo; c0 < c_hi; c0 += CG) {
            const int nc = min(CG, c_hi - c0);
            // ================= pass 1, one CTF at a time, warp-local
            for (int ci = 0; ci < nc; ++ci) {
                cf a[N1];
#pragma unroll
                for (int g4 = 0; g4 < N1 / 4; ++g4) {
                    a[4 * g4 + 0] = {q[4 * g4 + 0].x * kq[g4].x, q[4 * g4 + 0].y * kq[g4].x};
                    a[4 * g4 + 1] = {q[4 * g4 + 1].x * kq[g4].y, q[4 * g4 + 1].y * kq[g4].y};
                    a[4 * g4 + 2] = {q[4 * g4 + 2].x * kq[g4].z, q[4 * g4 + 2].y * kq[g4].z};
                    a[4 * g4 + 3] = {q[4 * g4 + 3].x * kq[g4].w, q[4 * g4 + 3].y * kq[g4].w};
                }
                {   // prefetch K of the next CTF (wraps to the first CTF for the next orientation)
                    int cn = c0 + ci + 1;
                    if (cn >= c_hi) cn = c_lo;
#pragma unroll
                    for (int g4 = 0; g4 < N1 / 4; ++g4) kq[g4] = Kt[((size_t)cn * (N1 / 4) + g4) * NT + tid];
                }
                fft_dif<float, N1, +1>(a);
#pragma unroll
                for (int r = 0; r < N1; ++r) zst[bitrev(r, 4)] = a[r];
                __syncwarp();
                cf *Gc = G + (size_t)ci * KK * GP + warp * CPW;
                for (int idx0 = 0; idx0 < nout1; idx0 += 32) {
                    const int idx = idx0 + lane;
                    const int cl = magicKK ? (int)__umulhi((unsigned)idx, magicKK) : idx, kk = idx - cl * KK;   // idx / KK (magic = 0: KK == 1)
                    const bool valid = idx < nout1;
                    const int k1 = (kk - D) & (N1 - 1);
                    const cf y = horner<N2, ZP>(Zw + (valid ? cl * N2 * ZP + k1 : 0), twH[valid ? kk : 0]);
                    if (valid) Gc[kk * GP + cl] = y;
                }
                __syncwarp();
            }
            if (tid < nc) {
                const size_t moc = ((size_t)model * p.n_orient + o) * p.n_ctf + c0 + tid;
                sc[tid] = make_float2(p.alpha[moc] * beta, p.hterm[moc]);
            }
            __syncthreads();
            // ================= pass 2: (CTF, row pair) combos, CPW per warp, warp-local
            {
                const int ncombo = nc * NP;
                const int combo = tid / N2;                        // this thread's A2 task
                if (combo < ncombo) {                                // whole (combo, t) groups: N2 lanes each
                    const int cl = combo / NP, pr = combo - cl * NP;
                    const int ra = 2 * pr, rb = 2 * pr + 1;
                    const cf *ga = G + ((size_t)cl * KK + ra) * GP;
                    const cf *gb = G + ((size_t)cl * KK + (rb < KK ? rb : ra)) * GP;
                    const float bsel = rb < KK ? 1.f : 0.f;
                    cf a[N1];
#pragma unroll
                    for (int j = 0; j < N1; ++j) {
                        // l = N2 j + t; direct for l <= N/2, mirrored (conjugate) above
                        const bool direct = (N2 * j < N / 2) || (N2 * j == N / 2 && t == 0);
                        const int l = N2 * j + t;
                        const int ll = direct ? l : N - l;
                        cf va = ga[ll], vb = gb[ll];
                        const float sg = direct ? 1.f : -1.f;
                        a[j] = {va.x - bsel * sg * vb.y, sg * va.y + bsel * vb.x};
                    }
                    fft_dif<float, N1, +1>(a);
#pragma unroll
                    for (int r = 0; r < N1; ++r) zst[bitrev(r, 4)] = a[r];
                }
                __syncwarp();
                const int cb0 = warp * CPW;
                const int nout2 = max(0, min(CPW, ncombo - cb0)) * KK;
                for (int idx0 = 0; idx0 < nout2; idx0 += 32) {
                    const int idx = idx0 + lane;
                    const bool valid = idx < nout2;
                    const int cw = magicKK ? (int)__umulhi((unsigned)idx, magicKK) : idx, kk = idx - cw * KK;     // combo within warp, dx index
                    const int k1 = (kk - D) & (N1 - 1);
                    const cf y = horner<N2, ZP>(Zw + (valid ? cw * N2 * ZP + k1 : 0), twH[valid ? kk : 0]);
                    const int combo2 = cb0 + (valid ? cw : 0);
                    const int cl = combo2 / NP, pr = combo2 - cl * NP;
                    const int ra = 2 * pr, rb = ra + 1;
                    const float2 s2 = sc[cl];
                    const float r0 = y.x * s2.x, r1 = y.y * s2.x;
                    const float x0 = fminf(r0 * r0, 0.99999994f), x1 = fminf(r1 * r1, 0.99999994f);          // R14 clamp
                    const float g0 = fmaf(p.cA, log1p_neg(x0), s2.y), g1 = fmaf(p.cA, log1p_neg(x1), s2.y);  // base-2 units
                    const bool v0 = valid, v1 = valid && rb < KK;
                    if (DUMP) {
                        if (v0) p.dump[ra * KK + kk] = g0;
                        if (v1) p.dump[rb * KK + kk] = g1;
                    }
                    if (v0) {
                        const float gb1 = v1 ? g1 : -CUDART_INF_F;
                        const float mn = fmaxf(lse_m, fmaxf(g0, gb1));
                        lse_s = lse_s * ex2f(lse_m - mn) + ex2f(g0 - mn) + ex2f(gb1 - mn);
                        lse_m = mn;
                    }
                    const uint32_t pair = (uint32_t)(o * p.n_ctf + c0 + cl);
                    warp_topk_insert_rq(g0, pair, (uint32_t)(ra * KK + kk), v0, thr, mylist);
                    warp_topk_insert_rq(g1, pair, (uint32_t)(rb * KK + kk), v1, thr, mylist);
                }
            }
            __syncthreads();
        }
    }
    if (DUMP) return;

    // ---- block reduction, fixed order
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const float m2 = __shfl_xor_sync(FULLM, lse_m, off), s2 = __shfl_xor_sync(FULLM, lse_s, off);
        const float M = fmaxf(lse_m, m2);
        const float sa = (lse_m == -CUDART_INF_F) ? 0.f : lse_s * ex2f(lse_m - M);
        const float sb = (m2 == -CUDART_INF_F) ? 0.f : s2 * ex2f(m2 - M);
        lse_s = sa + sb;
        lse_m = M;
    }
    if (lane == 0) { red[2 * warp] = lse_m; red[2 * warp + 1] = lse_s; }
    __syncthreads();
    if (warp == 0) {
        float m = -CUDART_INF_F, s = 0.f;
        for (int w = 0; w < NW; ++w) {
            const float m2 = red[2 * w], s2 = red[2 * w + 1];
            if (m2 == -CUDART_INF_F) continue;
            if (m == -CUDART_INF_F) { m = m2; s = s2; continue; }
            const float M = fmaxf(m, m2);
            s = s * ex2f(m - M) + s2 * ex2f(m2 - M);
            m = M;
        }
        float th0 = tops[BIOEM_TOPK - 1].g;
        for (int w = 1; w < NW; ++w)
            for (int k = 0; k < BIOEM_TOPK; ++k) {
                TopEntry e = tops[w * BIOEM_TOPK + k];
                warp_topk_insert_rq(e.g, e.pair, e.shift, lane == 0 && e.pair != 0xffffffffu, th0, tops);
            }
        __syncwarp();
        if (lane == 0) { p.part_m[item] = m; p.part_s[item] = s; }
        if (lane < BIOEM_TOPK) p.part_top[(size_t)item * BIOEM_TOPK + lane] = tops[lane];
    }
}

// ------------------------------------------------------------------------------------------------ K in task order
// Kt[c][g4][tid][e] = K_c(l = tid / N2, m = N2 (4 g4 + e) + tid % N2): the 16 values a thread needs are 4 coalesced float4.
template <int N>
__global__ void k_relayout_K(const float *K32, float4 *Kt, int n_ctf)
{
    typedef RQ<N> C_;
    const int c = blockIdx.y, i = blockIdx.x * blockDim.x + threadIdx.x;       // i = g4 * NT + tid
    if (i >= (C_::N1 / 4) * C_::NT) return;
    const int g4 = i / C_::NT, tid = i % C_::NT;
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    if (tid < C_::NTASK) {
        const int col = tid / C_::N2, t = tid % C_::N2;
        for (int e = 0; e < 4; ++e) v[e] = K32[(size_t)c * C_::NC * N + (size_t)col * N + C_::N2 * (4 * g4 + e) + t];
    }
    Kt[(size_t)c * (C_::N1 / 4) * C_::NT + i] = make_float4(v[0], v[1], v[2], v[3]);
}

bool rq_supported(int N) { return N == 64 || N == 128; }
size_t rq_kt_bytes(int N, int n_ctf) { return N == 64 ? (size_t)n_ctf * 4 * RQ<64>::NT * 16 : (size_t)n_ctf * 4 * RQ<128>::NT * 16; }

cudaError_t launch_relayout_K(int N, const float *K32, float *Kt, int n_ctf, cudaStream_t st)
{
    if (N == 64) {
        dim3 g((4 * RQ<64>::NT + 255) / 256, n_ctf);
        k_relayout_K<64><<<g, 256, 0, st>>>(K32, reinterpret_cast<float4 *>(Kt), n_ctf);
    } else {
        dim3 g((4 * RQ<128>::NT + 255) / 256, n_ctf);
        k_relayout_K<128><<<g, 256, 0, st>>>(K32, reinterpret_cast<float4 *>(Kt), n_ctf);
    }
    return cudaGetLastError();
}

template <int N>
static void rq_plan(int D, int n_ctf, int &CG, int &GP, size_t &bytes)
{
    typedef RQ<N> C_;
    const int KK = 2 * D + 1, NP = (KK + 1) / 2;
    GP = C_::NC | 1;
    CG = C_::NT / (NP * C_::N2);
    if (CG < 1) CG = 1;
    if (CG > n_ctf) CG = n_ctf;
    const size_t budget = 220 * 1024;
    for (;;) {
        bytes = (size_t)C_::NW * C_::ZW * 8 + (size_t)CG * KK * GP * 8 + (size_t)KK * 8 + (size_t)CG * 8 +
                (size_t)C_::NW * BIOEM_TOPK * sizeof(TopEntry) + 2 * C_::NW * 4 + 64;
        if (bytes <= budget || CG == 1) break;
        --CG;
    }
}

template <int N>
static cudaError_t launch_rq_t(const FusedParams &p, const float *Kt, bool dump, cudaStream_t st)
{
    int CG, GP;
    size_t bytes;
    rq_plan<N>(p.D, p.n_ctf, CG, GP, bytes);
    if (bytes > 227 * 1024) return cudaErrorInvalidConfiguration;
    const int KK = 2 * p.D + 1;
    const unsigned magic = KK == 1 ? 0u : (unsigned)((0x100000000ull + KK - 1) / KK);     // exact idx / KK for idx < 2^16
    cudaError_t e;
    if (dump) {
        e = cudaFuncSetAttribute(k_fused_rq<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        k_fused_rq<N, true><<<1, RQ<N>::NT, bytes, st>>>(p, reinterpret_cast<const float4 *>(Kt), CG, GP, magic);
    } else {
        e = cudaFuncSetAttribute(k_fused_rq<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        const int items = p.n_img * p.n_model * p.chunks_per_model;
        k_fused_rq<N, false><<<items, RQ<N>::NT, bytes, st>>>(p, reinterpret_cast<const float4 *>(Kt), CG, GP, magic);
    }
    return cudaGetLastError();
}

cudaError_t launch_fused_rq(int N, const FusedParams &p, const float *Kt, bool dump, cudaStream_t st)
{
    if (N == 64) return launch_rq_t<64>(p, Kt, dump, st);
    if (N == 128) return launch_rq_t<128>(p, Kt, dump, st);
    return cudaErrorInvalidValue;
}

}  // namespace bioem
