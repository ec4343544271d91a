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
// B-phase mapping (v3): a lane owns one residue k1 = lane % 16 of one column (or row pair) per round and forms BOTH pruned
// outputs k = k1 - 16 and k = k1 from the same N2 shared-memory loads (two Horner chains, twiddles in registers); the single
// k = +16 output of D = 16 is an extra round.  No index arithmetic is left in the CTF loop.  Requires D <= 16.
// No float atomics, fixed reduction orders: bit-reproducible.
#include "common.cuh"
#include <math_constants.h>

namespace bioem {

static constexpr unsigned FULLM = 0xffffffffu;

template <int N> struct RQ {
    static constexpr int N1 = 16, N2 = N / 16, NC = N / 2 + 1, NTASK = NC * N2, NW = (NTASK + 31) / 32, NT = NW * 32;
    static constexpr int ZP = 18, CPW = 32 / N2;      // Z pitch (even: 16-byte aligned pairs), columns per warp
    static constexpr int CS = N2 * ZP + 2;            // column-tile pitch: +2 keeps the k = +16 round (one lane per column) conflict-free
    static constexpr int ZW = CPW * CS;               // Z words (complex) per warp
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

// log1p(-x), 0 <= x < 2^-6: 5-term series (truncation < 2e-10 relative)
__device__ __forceinline__ float log1p_neg_small(float x)
{
    float p = fmaf(x, 0.2f, 0.25f);
    p = fmaf(x, p, 0.33333334f);
    p = fmaf(x, p, 0.5f);
    p = fmaf(x, p, 1.0f);
    return -x * p;
}

// Two Horner sums over the N2 residues sharing their loads: ylo = sum_t rlo^t z[t], yhi = sum_t rhi^t z[t]
template <int N2, int ZP>
__device__ __forceinline__ void horner2(const cf *zc, cf rlo, cf rhi, cf &ylo, cf &yhi)
{
    cf z = zc[(N2 - 1) * ZP];
    ylo = z; yhi = z;
#pragma unroll
    for (int t = N2 - 2; t >= 0; --t) {
        z = zc[t * ZP];
        float ax = fmaf(rlo.x, ylo.x, fmaf(-rlo.y, ylo.y, z.x));
        float ay = fmaf(rlo.x, ylo.y, fmaf(rlo.y, ylo.x, z.y));
        float bx = fmaf(rhi.x, yhi.x, fmaf(-rhi.y, yhi.y, z.x));
        float by = fmaf(rhi.x, yhi.y, fmaf(rhi.y, yhi.x, z.y));
        ylo.x = ax; ylo.y = ay; yhi.x = bx; yhi.y = by;
    }
}
template <int N2, int ZP>
__device__ __forceinline__ cf horner1(const cf *zc, cf r)
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

// spill the bit-reversed FFT output as 8 16-byte stores: a[r] = y[bitrev4(r)], so (a[r], a[r+8]) = (y[2b], y[2b+1]), b = bitrev3(r)
__device__ __forceinline__ void spill16(cf *zst, const cf (&a)[16])
{
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int b = bitrev(r, 3);
        *reinterpret_cast<float4 *>(zst + 2 * b) = make_float4(a[r].x, a[r].y, a[r + 8].x, a[r + 8].y);
    }
}

// per-shift closed form for the (up to) four values a lane produces per round, running log-sum-exp and candidates
struct LseState { float m, s, thr; };

template <bool DUMP>
__device__ __forceinline__ void score4(const FusedParams &p, LseState &st, TopEntry *mylist, const float (&b)[4], const bool (&v)[4],
                                       const uint32_t (&sh)[4], float ab, float hterm, uint32_t pair)
{
    float g[4];
    float xmax = 0.f;
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        const float r = b[i] * ab;
        const float x = fminf(r * r, 0.99999994f);                         // rho^2, R14 clamp
        xmax = fmaxf(xmax, x);
        g[i] = fmaf(p.cA, log1p_neg_small(x), hterm);                       // form C2, base-2 units
    }
    if (__any_sync(FULLM, xmax >= 0.015625f)) {                             // rare (near the posterior peak): accurate log1p
#pragma unroll
        for (int i = 0; i < 4; ++i) {
            const float r = b[i] * ab;
            const float x = fminf(r * r, 0.99999994f);
            if (x >= 0.015625f) g[i] = fmaf(p.cA, log1pf(-x), hterm);
        }
    }
#pragma unroll
    for (int i = 0; i < 4; ++i) {
        if (!v[i]) g[i] = -CUDART_INF_F;
        if (DUMP && v[i]) p.dump[sh[i]] = g[i];
    }
    const float gmax = fmaxf(fmaxf(g[0], g[1]), fmaxf(g[2], g[3]));
    if (gmax > -CUDART_INF_F) {
        const float mn = fmaxf(st.m, gmax);
        st.s = st.s * ex2f(st.m - mn) + ((ex2f(g[0] - mn) + ex2f(g[1] - mn)) + (ex2f(g[2] - mn) + ex2f(g[3] - mn)));
        st.m = mn;
    }
    if (__any_sync(FULLM, gmax >= st.thr)) {
#pragma unroll
        for (int i = 0; i < 4; ++i) warp_topk_insert_rq(g[i], pair, sh[i], v[i], st.thr, mylist);
    }
}

template <int N, bool DUMP>
__global__ void __launch_bounds__(RQ<N>::NT, 1) k_fused_rq(FusedParams p, const float4 *__restrict__ Kt, int CG, int GP, unsigned magicNP, int NBUF)
{
    typedef RQ<N> C_;
    constexpr int N1 = C_::N1, N2 = C_::N2, NC = C_::NC, NTASK = C_::NTASK, NW = C_::NW, NT = C_::NT, ZP = C_::ZP, ZW = C_::ZW, CPW = C_::CPW, CS = C_::CS;
    constexpr size_t H = (size_t)NC * N;
    const int D = p.D, KK = 2 * D + 1, NP = (KK + 1) / 2;                 // host guarantees D <= 16
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    cf *Z = reinterpret_cast<cf *>(smem_raw);                        // [NW][32][ZP]  warp-private tiles
    cf *G = Z + (size_t)NW * ZW;                                     // [2][CG][KK][GP]  double-buffered over CTF groups
    const int GSZ = CG * KK * GP;
    float2 *sc = reinterpret_cast<float2 *>(G + (size_t)NBUF * GSZ); // [2][CG]  (alpha*beta, h) of the group's CTFs
    TopEntry *tops = reinterpret_cast<TopEntry *>(sc + 2 * CG);      // [NW][TOPK]
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
    if (tid < NW * BIOEM_TOPK) { TopEntry e0 = {-CUDART_INF_F, 0xffffffffu, 0xffffffffu}; tops[tid] = e0; }
    __syncthreads();

    // ---- A-phase constants: thread = (column, residue t)
    const bool act1 = tid < NTASK;
    const int col = act1 ? tid / N2 : 0, t = tid % N2;
    const size_t qbase = (size_t)col * N + t;
    cf *Zw = Z + (size_t)warp * ZW;
    cf *zst = Zw + (lane / N2) * CS + (lane % N2) * ZP;
    const int ncols_w = max(0, min(CPW, NC - warp * CPW));           // whole columns owned by this warp
    // ---- B-phase constants: lane = (half, k1); outputs k = k1 - 16 ("lo") and k = k1 ("hi")
    const int half = lane >> 4, k1 = lane & 15;
    const bool vlo = k1 >= 16 - D, vhi = k1 <= D;
    const int kk_lo = k1 - 16 + D, kk_hi = k1 + D;                    // row / dx index of the two outputs
    cf rlo, rhi;
    {
        float sn, cs;
        sincospif(2.0f * (float)(k1 - 16 + N) / (float)N, &sn, &cs); rlo = {cs, sn};
        sincospif(2.0f * (float)k1 / (float)N, &sn, &cs);            rhi = {cs, sn};
    }
    const cf rx = {(float)cos32(512 / N), (float)cos32(8 - 512 / N)};        // w_N^{16} = exp(2 pi i 16/N), k = +16 (only when D == 16)
    const bool has_x = D == 16;
    const cf *zrd = Zw + half * CS + k1;                              // + cp * 2 * CS per round
    const int a2combo = tid / N2;                                     // this thread's A2 task: (CTF in group) x (row pair)

    const cf *Oimg = p.Ohat + (size_t)img * H;
    LseState st = {-CUDART_INF_F, 0.f, -CUDART_INF_F};
    TopEntry *mylist = tops + warp * BIOEM_TOPK;
    const int c_lo = DUMP ? p.dump_ctf : 0, c_hi = DUMP ? p.dump_ctf + 1 : p.n_ctf;
    const float4 *Kt_t = Kt + tid;
    constexpr size_t KSTR = (size_t)(N1 / 4) * NT;                   // float4 per CTF

    float4 kq[N1 / 4];
#pragma unroll
    for (int g4 = 0; g4 < N1 / 4; ++g4) kq[g4] = Kt_t[(size_t)c_lo * KSTR + (size_t)g4 * NT];
    int gbuf = 0;

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
            cf *Gb = G + (size_t)gbuf * GSZ;
            float2 *scb = sc + gbuf * CG;
            gbuf ^= (NBUF - 1);
            float2 schold = make_float2(0.f, 0.f);                 // (alpha*beta, h) of CTF c0 + tid: fetched now, published before the barrier
            if (tid < nc) {
                const size_t moc = ((size_t)model * p.n_orient + o) * p.n_ctf + c0 + tid;
                schold = make_float2(p.alpha[moc] * beta, p.hterm[moc]);
            }
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
                fft_dif<float, N1, +1>(a);
                spill16(zst, a);
                {   // prefetch K of the next CTF (wraps to the first CTF for the next orientation)
                    int cn = c0 + ci + 1;
                    if (cn >= c_hi) cn = c_lo;
                    const float4 *kp = Kt_t + (size_t)cn * KSTR;
#pragma unroll
                    for (int g4 = 0; g4 < N1 / 4; ++g4) kq[g4] = kp[(size_t)g4 * NT];
                }
                __syncwarp();
                cf *Gc = Gb + (size_t)ci * KK * GP + warp * CPW + half;
#pragma unroll
                for (int cp = 0; cp < CPW / 2; ++cp) {
                    if (2 * cp < ncols_w) {                                       // warp-uniform
                        cf ylo, yhi;
                        horner2<N2, ZP>(zrd + cp * 2 * CS, rlo, rhi, ylo, yhi);
                        const bool cv = 2 * cp + half < ncols_w;
                        if (cv && vlo) Gc[kk_lo * GP + 2 * cp] = ylo;
                        if (cv && vhi) Gc[kk_hi * GP + 2 * cp] = yhi;
                    }
                }
                if (has_x) {                                                      // k = +16: one output per column, k1 = 0
                    const int cl = lane < ncols_w ? lane : 0;
                    const cf y = horner1<N2, ZP>(Zw + cl * CS, rx);
                    if (lane < ncols_w) Gb[(size_t)ci * KK * GP + (KK - 1) * GP + warp * CPW + lane] = y;
                }
                __syncwarp();
            }
            if (tid < nc) scb[tid] = schold;
            __syncthreads();
            // ================= pass 2: (CTF, row pair) combos, CPW per warp, warp-local
            {
                const int ncombo = nc * NP;
                if (a2combo < ncombo) {                              // whole (combo, t) groups: N2 lanes each
                    const int a2cl = magicNP ? (int)__umulhi((unsigned)a2combo, magicNP) : a2combo, a2pr = a2combo - a2cl * NP;     // a2combo / NP
                    const bool a2two = 2 * a2pr + 1 < KK;
                    const cf *ga = Gb + (a2cl * KK + 2 * a2pr) * GP, *gb = ga + (a2two ? GP : 0);
                    const float a2bsel = a2two ? 1.f : 0.f;
                    cf a[N1];
#pragma unroll
                    for (int j = 0; j < N1; ++j) {
                        // l = N2 j + t; direct for l <= N/2, mirrored (conjugate) above
                        const bool direct = (N2 * j < N / 2) || (N2 * j == N / 2 && t == 0);
                        const int l = N2 * j + t;
                        const int ll = direct ? l : N - l;
                        cf va = ga[ll], vb = gb[ll];
                        const float sg = direct ? 1.f : -1.f;
                        a[j] = {va.x - a2bsel * sg * vb.y, sg * va.y + a2bsel * vb.x};
                    }
                    fft_dif<float, N1, +1>(a);
                    spill16(zst, a);
                }
                __syncwarp();
                const int cb0 = warp * CPW;
                const int ncw = max(0, min(CPW, ncombo - cb0));     // combos of this warp
#pragma unroll
                for (int cp = 0; cp < CPW / 2; ++cp) {
                    if (2 * cp < ncw) {                              // warp-uniform
                        cf ylo, yhi;
                        horner2<N2, ZP>(zrd + cp * 2 * CS, rlo, rhi, ylo, yhi);
                        const int combo = cb0 + 2 * cp + half;
                        const bool cv = combo < ncombo;
                        const int cl = cv ? (magicNP ? (int)__umulhi((unsigned)combo, magicNP) : combo) : 0, pr = cv ? combo - cl * NP : 0;
                        const float2 s2 = scb[cl];
                        const int sha = 2 * pr * KK, shb = sha + KK;
                        const bool rbv = 2 * pr + 1 < KK;
                        const float b[4] = {ylo.x, ylo.y, yhi.x, yhi.y};
                        const bool v[4] = {cv && vlo, cv && vlo && rbv, cv && vhi, cv && vhi && rbv};
                        const uint32_t sh[4] = {(uint32_t)(sha + kk_lo), (uint32_t)(shb + kk_lo), (uint32_t)(sha + kk_hi), (uint32_t)(shb + kk_hi)};
                        score4<DUMP>(p, st, mylist, b, v, sh, s2.x, s2.y, (uint32_t)(o * p.n_ctf + c0 + cl));
                    }
                }
                if (has_x && ncw > 0) {                              // dx = +16
                    const bool cv = lane < ncw;
                    const cf y = horner1<N2, ZP>(Zw + (cv ? lane : 0) * CS, rx);
                    const int combo = cb0 + (cv ? lane : 0);
                    const int cl = magicNP ? (int)__umulhi((unsigned)combo, magicNP) : combo, pr = combo - cl * NP, xsha = 2 * pr * KK;
                    const float2 s2 = scb[cl];
                    const float b[4] = {y.x, y.y, 0.f, 0.f};
                    const bool v[4] = {cv, cv && 2 * pr + 1 < KK, false, false};
                    const uint32_t sh[4] = {(uint32_t)(xsha + KK - 1), (uint32_t)(xsha + 2 * KK - 1), 0u, 0u};
                    score4<DUMP>(p, st, mylist, b, v, sh, s2.x, s2.y, (uint32_t)(o * p.n_ctf + c0 + cl));
                }
            }
            if (NBUF == 1) __syncthreads();      // single G buffer: pass 2 must drain before the next group's pass 1 (with 2 buffers the next barrier orders the reuse)
        }
    }
    if (DUMP) return;

    // ---- block reduction, fixed order
    float lse_m = st.m, lse_s = st.s;
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

bool rq_supported(int N, int D) { return (N == 64 || N == 128) && D <= 16; }
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
static void rq_plan(int D, int n_ctf, int nbuf, int &CG, int &GP, size_t &bytes)
{
    typedef RQ<N> C_;
    const int KK = 2 * D + 1, NP = (KK + 1) / 2;
    GP = C_::NC | 1;
    CG = C_::NT / (NP * C_::N2);
    if (CG < 1) CG = 1;
    if (CG > n_ctf) CG = n_ctf;
    const size_t budget = 226 * 1024;
    for (;;) {
        bytes = (size_t)C_::NW * C_::ZW * 8 + (size_t)nbuf * CG * KK * GP * 8 + 2 * (size_t)CG * 8 +
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
    const int nbuf = 1;      // G buffers: 2 removes one CTA barrier per group but shrinks L1 to ~30 KB; measured equal on B200 (DESIGN 7)
    rq_plan<N>(p.D, p.n_ctf, nbuf, CG, GP, bytes);
    if (bytes > 227 * 1024) return cudaErrorInvalidConfiguration;
    const int NP = p.D + 1;                                                    // (2D+1+1)/2 row pairs
    const unsigned magic = NP == 1 ? 0u : (unsigned)((0x100000000ull + NP - 1) / NP);   // exact x / NP for x < 2^16 (NP = 1 never divides: D = 0 has one combo per CTF)
    cudaError_t e;
    if (dump) {
        e = cudaFuncSetAttribute(k_fused_rq<N, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        k_fused_rq<N, true><<<1, RQ<N>::NT, bytes, st>>>(p, reinterpret_cast<const float4 *>(Kt), CG, GP, magic, nbuf);
    } else {
        e = cudaFuncSetAttribute(k_fused_rq<N, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        const int items = p.n_img * p.n_model * p.chunks_per_model;
        k_fused_rq<N, false><<<items, RQ<N>::NT, bytes, st>>>(p, reinterpret_cast<const float4 *>(Kt), CG, GP, magic, nbuf);
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
