// fused_pk.cu -- the hot loop for N = 64 and N = 128, D <= 16: register-resident Q,
// PACKED f32x2 arithmetic (sm_100a FFMA2 / FADD2 / FMUL2) and ONE software pipeline over CTF groups.
//
// Work item = (image w, model, chunk of orientations).  For one (w, o) the product Q(l,m) = conj(Ohat_w) F0_o (Eq. 12,
// P:166) is formed ONCE and kept in registers (16 complex per thread; thread = (column l, residue t) of the two-step
// factorisation m = N2 j + t).  The CTF loop then streams only the real radial table K_c (Eq. 5).
//
// Why packed: a complex number is one 64-bit register pair, and sm_100a issues one FFMA2/FADD2/FMUL2 per pair with free
// operand swizzles (swap, per-half negate, scalar broadcast).  A complex add is 1 instruction instead of 2, a complex
// multiply-add 2 instead of 4: the FP32 pipes see the same work, the ISSUE slots see half of it (DESIGN 7).
//
// Why N/2 columns: the CTA is N/2 * N2 threads = 16 warps at N = 128, i.e. exactly 4 warps on each of the SM's 4
// schedulers with 128 registers each (17 warps put 5 on one scheduler: 96 registers, spills, and 3 schedulers waiting
// for the 4th at every barrier -- profiles/r1_v5_*).  The Nyquist column l = N/2 rides on column 0: both are Hermitian
// in m, so the transform of Q(0,.)K(0,.) + i Q(N/2,.)K(N/2,.) is G(.,0) + i G(.,N/2) with both parts real.
//
// Every "slot" is [A-op: 16 complex into registers, 16-point DIF FFT] || [H-op: Horner sums over the Z tile the previous
// slot spilled], then __syncwarp, spill, __syncwarp.  The two halves of a slot share no data, sit in one basic block, and
// the H-op's shared-memory latency hides under the A-op's register-only arithmetic:
//   slot A   F(0)   a = Q K_c0                 ||  H'(group gi-2): B(dx,dy) -> a5 likelihood -> a6 log-sum-exp, candidates
//   slot B   F(ci)  a = Q K_ci                 ||  H(ci-1): the 2D+1 pruned outputs per column -> rows of G[gi & 1]
//   slot C   F'(group gi-1): rows of G[gi-1 & 1], Hermitian completion, two real rows per transform  ||  H(nc-1)
//   G is double-buffered over groups and the Z tiles are warp-private.  There is NO CTA barrier in the loop: two shared-memory
//   mbarriers in split phase hand G over ("rows of group g written": arrive after the last G store, wait before F' reads them;
//   "rows of group g read": arrive right after the F' loads, wait before the next store into that buffer), so warps drift.
//   Pass-2 tasks (CTF in group, row pair) come from a host-built table (pk_build_map): conflict-free G row loads per
//   half-warp, idle slots as whole warps (warp 0, which carries the Nyquist column, always; two more rotating over the
//   schedulers from group to group).
// The k = +16 output (D = 16 only) is the DC bin of the 16-point transforms: a twiddle and a shuffle-reduction over the
// N2 lanes of a column.  The pipeline is primed and drained with masked groups (2 per work item, < 1 % of the work).
//   a5  rho^2 = B^2 alpha_c^2 beta_w^2, g = cA log1p(-rho^2) + h_c (form C2; base-2 units inside the kernel)
//   a6  running log-sum-exp in registers (branch-free), K best terms in per-warp sorted lists
// No float atomics, fixed reduction orders: bit-reproducible.
#include "pk_math.cuh"
#include <vector>

namespace bioem {


template <int N> struct PK {
    static constexpr int N1 = 16, N2 = N / 16, NCH = N / 2, NT = NCH * N2, NW = NT / 32;   // NCH columns: l = 0 carries l = N/2 packed with it
    static constexpr int ZP = 18, CPW = 32 / N2, NR = CPW / 2;   // Z pitch (even: 16-byte aligned pairs), columns per warp, H-phase rounds
    static constexpr int CS = N2 * ZP + 2;                        // column-tile pitch
    static constexpr int ZW = CPW * CS;                           // Z words (complex) per warp
    static constexpr int NCOMBO = NT / N2;                        // (CTF, row pair) tasks of pass 2 per sweep
};
// Two sums over the N2 residues sharing their loads: ylo = sum_t rlo^t z[t], yhi = sum_t rhi^t z[t], where rlo = rhi w_N^-16, so
// that rlo^(N2/2) = -rhi^(N2/2) =: -rh.  With P_a = z_a + rh z_(a+N2/2) and M_a = z_a - rh z_(a+N2/2) = 2 z_a - P_a:
// yhi = sum_a rhi^a P_a, ylo = sum_a rlo^a M_a: two half-length Horner chains (24 instead of 28 packed instructions at N2 = 8).
template <int N2, int ZP>
__device__ __forceinline__ void pk_horner2(const c2 *zc, c2 rlo, c2 rhi, c2 rh, c2 &ylo, c2 &yhi)
{
    constexpr int HF = N2 / 2;
    c2 P[HF], M[HF];
#pragma unroll
    for (int a = 0; a < HF; ++a) {
        const c2 z0 = zc[a * ZP], z1 = zc[(a + HF) * ZP];
        P[a] = pk_cmadd(z1, rh, z0);
        M[a] = __ffma2_rn(z0, pk_bc(2.0f), make_float2(-P[a].x, -P[a].y));
    }
    yhi = P[HF - 1]; ylo = M[HF - 1];
#pragma unroll
    for (int a = HF - 2; a >= 0; --a) {
        yhi = pk_cmadd(yhi, rhi, P[a]);
        ylo = pk_cmadd(ylo, rlo, M[a]);
    }
}

// sum over the N2 lanes of a column (lanes are contiguous and N2-aligned): fixed xor tree, every lane gets the sum
template <int N2>
__device__ __forceinline__ c2 pk_colsum(c2 v)
{
#pragma unroll
    for (int off = 1; off < N2; off <<= 1) {
        c2 w;
        w.x = __shfl_xor_sync(FULLP, v.x, off);
        w.y = __shfl_xor_sync(FULLP, v.y, off);
        v = pk_add(v, w);
    }
    return v;
}
// Pass-2 task table: slot (= tid / N2) -> (CTF in group << 8 | row pair), 0xffff = idle.  Built on the host (pk_plan) so that
// the slots of a half-warp read rows whose shared-memory bank offsets tile the 16 eight-byte banks (conflict-free G loads),
// and so that the idle slots fill whole warps starting at warp 0 (which carries the extra Nyquist-column work of pass 1).
struct PkMap { uint16_t e[3][64]; int nvar; };     // nvar variants, used round-robin over the CTF groups (see pk_build_map)
// ORIENT = true (bioem_set_orientation_posterior): each warp also closes its running sums at the end of every orientation of the
// work item into otab[orientation][warp]; the epilogue combines warps -> orientation (p.orient_m / p.orient_s) -> work item in
// fixed order.  A template parameter: as a run-time flag in the group loop it cost the default path 7 % (DESIGN 7).
template <int N, bool DUMP, bool ORIENT>
__global__ void __launch_bounds__(PK<N>::NT, 1) k_fused_pk(FusedParams p, const float4 *__restrict__ Kt, const float4 *__restrict__ KtN, int CG, int GP, const __grid_constant__ PkMap map)
{
    typedef PK<N> C_;
    constexpr int N1 = C_::N1, N2 = C_::N2, NW = C_::NW, NT = C_::NT, ZP = C_::ZP, ZW = C_::ZW, CPW = C_::CPW, CS = C_::CS,
                  NR = C_::NR;
    constexpr size_t H = (size_t)(N / 2 + 1) * N;
    const int D = p.D, KK = 2 * D + 1, NP = D + 1;                    // host guarantees D <= 16; NP row pairs (the last one is a single row)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    c2 *Z = reinterpret_cast<c2 *>(smem_raw);                         // [NW][ZW]         warp-private tiles
    c2 *G = Z + (size_t)NW * ZW;                                      // [2][CG][KK][GP]  pass-1 output rows of a CTF group, double-buffered over groups
    const int GSZ = CG * KK * GP;
    c2 *qn = G + (size_t)2 * GSZ;                                     // [8][N2][2]       Q of the Nyquist column l = N/2 (warp 0, lanes < N2)
    float4 *kn = reinterpret_cast<float4 *>(qn + 16 * N2);            // [2][4][N2]       K_c(N/2, .) of the current / next CTF  (+ one zero float4)
    float2 *sc = reinterpret_cast<float2 *>(kn + 8 * N2 + 1);         // [4][CG]          (alpha*beta, h) of the CTFs of the last 4 groups
    TopEntry *tops = reinterpret_cast<TopEntry *>(sc + 4 * CG);       // [NW][TOPK]
    float *red = reinterpret_cast<float *>(tops + NW * BIOEM_TOPK);   // [2 NW]
    float2 *otab = reinterpret_cast<float2 *>(red + 2 * NW);          // [32][NW]         ORIENT only: (m, s) per orientation of the item and warp
    __shared__ uint64_t mbar[2];                                      // [0] "G rows of group gi written", [1] "G rows of group gi-1 read"

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
    // the pipeline runs two masked warm-up / drain groups: everything it may read must be finite
    for (int i = tid; i < (NW * ZW + 2 * GSZ + 16 * N2) * 2; i += NT) reinterpret_cast<float *>(Z)[i] = 0.f;
    for (int i = tid; i < (8 * N2 + 1) * 4; i += NT) reinterpret_cast<float *>(kn)[i] = 0.f;
    for (int i = tid; i < 4 * CG; i += NT) sc[i] = make_float2(0.f, 0.f);
    if (tid < NW * BIOEM_TOPK) { TopEntry e0 = {-CUDART_INF_F, 0xffffffffu, 0xffffffffu}; tops[tid] = e0; }
    if (tid == 0) { pk_mbar_init(&mbar[0], NW); pk_mbar_init(&mbar[1], NW); }
    __syncthreads();

    // ---- F-phase constants: thread = (column, residue t); column 0 also carries column N/2 (both are Hermitian in m, so
    //      the transform of Q(0,.) + i Q(N/2,.) has G(.,0) as its real and G(.,N/2) as its imaginary part)
    const int col = tid / N2, t = tid % N2;
    const size_t qbase = (size_t)col * N + t;
    c2 *const Zw = Z + (size_t)warp * ZW;
    const int zst_off = (lane / N2) * CS + (lane % N2) * ZP;
    const bool has_x = D == 16;
    c2 wx;                                                            // exp(2 pi i t / N2) = w_N^{16 t}: the k = +16 output
    sincospif(2.0f * (float)t / (float)N2, &wx.y, &wx.x);
    const bool xlane = has_x && t == 0;
    const bool nyq = warp == 0 && lane < N2;                          // threads of column 0
    const float4 *knp = nyq ? kn + t : kn + 8 * N2;                   // other lanes of warp 0 read the zero float4
    const int kn_str = nyq ? N2 : 0, kn_boff = nyq ? 4 * N2 : 0;
    // ---- H-phase constants: lane = (half, k1); outputs k = k1 - 16 ("lo") and k = k1 ("hi")
    const int half = lane >> 4, k1 = lane & 15;
    const bool vlo = k1 >= 16 - D, vhi = k1 <= D;
    const int kk_lo = k1 - 16 + D, kk_hi = k1 + D;                    // row / dx index of the two outputs
    c2 rlo, rhi;
    sincospif(2.0f * (float)(k1 - 16 + N) / (float)N, &rlo.y, &rlo.x);
    sincospif(2.0f * (float)k1 / (float)N, &rhi.y, &rhi.x);
    c2 rh;                                                            // rhi^(N2/2) = exp(2 pi i k1 / 32)
    sincospif(2.0f * (float)k1 / 32.0f, &rh.y, &rh.x);
    const int zrd_off = half * CS + k1;                               // + cp * 2 * CS per round
    // ---- pass-2 tasks come from the task table, variant (group index mod nvar): slot a2combo is this thread's F' task, slots
    //      warp * CPW + 2 cp + half are this lane's H' tasks.  Entry = CTF in group << 8 | row pair; 0xffff = idle (cl = 255).
    const int a2combo = tid / N2;
    const int l8 = (t == 0) ? 0 : N / 2 - t;                          // j = 8: l = N/2 + t -> mirrored N/2 - t; t = 0: the packed entry
    int var0 = 0, var1 = 0, var2 = 0;                                 // variants of groups gi, gi-1, gi-2
    int eX = 0xffff;                                                  // this thread's F' entry of group gi-2 (owner of xs2)

    const cf *Oimg = p.Ohat + (size_t)img * H;
    PkLse st = {LSE_EMPTY, 0.f, -CUDART_INF_F};
    TopEntry *mylist = tops + warp * BIOEM_TOPK;
    const int c_lo = DUMP ? p.dump_ctf : 0, c_hi = DUMP ? p.dump_ctf + 1 : p.n_ctf;
    const float4 *Kt_t = Kt + tid;
    constexpr size_t KSTR = (size_t)(N1 / 4) * NT;                    // float4 per CTF
    const int gpo = (c_hi - c_lo + CG - 1) / CG;                      // groups per orientation
    const int total = (o_end - o_begin) * gpo;

    float4 kq[N1 / 4];
#pragma unroll
    for (int g4 = 0; g4 < N1 / 4; ++g4) kq[g4] = Kt_t[(size_t)c_lo * KSTR + (size_t)g4 * NT];
    int knb = 0;
    if (nyq) {
#pragma unroll
        for (int g4 = 0; g4 < 4; ++g4) pk_cp_async16(kn + g4 * N2 + t, KtN + ((size_t)c_lo * 4 + g4) * N2 + t);
    }
    pk_cp_async_commit();

    // a = Q K_c (consumes kq; column 0 adds i Q(N/2,.) K_c(N/2,.)), then prefetch K of CTF `cn`
#define PK_LOAD_A(cn)                                                                                         \
    c2 a[N1];                                                                                                 \
    _Pragma("unroll") for (int g4 = 0; g4 < N1 / 4; ++g4) {                                                   \
        a[4 * g4 + 0] = __fmul2_rn(q[4 * g4 + 0], pk_bc(kq[g4].x));                                           \
        a[4 * g4 + 1] = __fmul2_rn(q[4 * g4 + 1], pk_bc(kq[g4].y));                                           \
        a[4 * g4 + 2] = __fmul2_rn(q[4 * g4 + 2], pk_bc(kq[g4].z));                                           \
        a[4 * g4 + 3] = __fmul2_rn(q[4 * g4 + 3], pk_bc(kq[g4].w));                                           \
    }                                                                                                         \
    {                                                                                                         \
        const float4 *kp = Kt_t + (size_t)(cn) * KSTR;                                                        \
        _Pragma("unroll") for (int g4 = 0; g4 < N1 / 4; ++g4) kq[g4] = kp[(size_t)g4 * NT];                   \
    }                                                                                                         \
    if (warp == 0) {                                                                                          \
        pk_cp_async_wait_all();                                                                               \
        _Pragma("unroll") for (int g4 = 0; g4 < 4; ++g4) {                                                    \
            const float4 k4 = knp[knb * kn_boff + g4 * kn_str];                                                \
            const float4 qa = *reinterpret_cast<const float4 *>(qn + ((2 * g4) * N2 + t) * 2);                \
            const float4 qb = *reinterpret_cast<const float4 *>(qn + ((2 * g4 + 1) * N2 + t) * 2);            \
            a[4 * g4 + 0] = __ffma2_rn(make_float2(-qa.y, qa.x), pk_bc(k4.x), a[4 * g4 + 0]);                 \
            a[4 * g4 + 1] = __ffma2_rn(make_float2(-qa.w, qa.z), pk_bc(k4.y), a[4 * g4 + 1]);                 \
            a[4 * g4 + 2] = __ffma2_rn(make_float2(-qb.y, qb.x), pk_bc(k4.z), a[4 * g4 + 2]);                 \
            a[4 * g4 + 3] = __ffma2_rn(make_float2(-qb.w, qb.z), pk_bc(k4.w), a[4 * g4 + 3]);                 \
        }                                                                                                     \
        knb ^= 1;                                                                                             \
        if (nyq) {                                                                                            \
            _Pragma("unroll") for (int g4 = 0; g4 < 4; ++g4)                                                  \
                pk_cp_async16(kn + (knb * 4 + g4) * N2 + t, KtN + ((size_t)(cn) * 4 + g4) * N2 + t);          \
        }                                                                                                     \
        pk_cp_async_commit();                                                                                 \
    }
    // H(ci): pruned outputs of the columns in the Z tile -> rows of G
#define PK_HORNER_G(Gb, ci)                                                                                   \
    {                                                                                                         \
        c2 *Gc = (Gb) + (size_t)(ci) * KK * GP + warp * CPW + half;                                           \
        _Pragma("unroll") for (int cp = 0; cp < NR; ++cp) {                                                   \
            c2 ylo, yhi;                                                                                      \
            pk_horner2<N2, ZP>(Zw + zrd_off + cp * 2 * CS, rlo, rhi, rh, ylo, yhi);                               \
            if (vlo) Gc[kk_lo * GP + 2 * cp] = ylo;                                                           \
            if (vhi) Gc[kk_hi * GP + 2 * cp] = yhi;                                                           \
        }                                                                                                     \
    }
    // tail of a slot: FFT of a, the k = +16 output from the DC bins (xs), then the tile hand-over
#define PK_FFT_XS()                                                                                           \
    pk_fft16(a);                                                                                              \
    const c2 xs = pk_colsum<N2>(pk_cmul(a[0], wx));
#define PK_SPILL()                                                                                            \
    __syncwarp();                         /* every lane has read the previous tile */                         \
    pk_spill16(Zw + zst_off, a);                                                                              \
    __syncwarp();

    // ---- the flat, software-pipelined loop over CTF groups (group gi: pass 1 now, F' one group later, H' two groups later)
    int o = o_begin, c0 = c_lo;
    int nc1 = 0, nc2 = 0;                                             // CTFs in groups gi-1, gi-2 (0 = no such group)
    uint32_t pair1 = 0, pair2 = 0;                                    // o * n_ctf + c0 of those groups
    bool last1 = false, last2 = false;                                // ORIENT: that group is the last one of its orientation ...
    int ol1 = 0, ol2 = 0;                                             // ... which is orientation o_begin + ol of the grid
    c2 xs2 = make_float2(0.f, 0.f);                                   // B(dx = +16) of this thread's pass-2 task, from F' to H'
    c2 q[N1];
#pragma unroll
    for (int j = 0; j < N1; ++j) q[j] = make_float2(0.f, 0.f);
    float2 scn = make_float2(0.f, 0.f);                               // (alpha, h) of the NEXT group's CTF c0 + tid (threads tid < CG)
    if (tid < CG && total > 0 && c_lo + tid < c_hi) {
        const size_t moc = ((size_t)model * p.n_orient + o_begin) * p.n_ctf + c_lo + tid;
        scn = make_float2(p.alpha[moc], p.hterm[moc]);
    }
    for (int gi = 0; gi < total + 2; ++gi) {
        const bool live = gi < total;
        const int nc = live ? min(CG, c_hi - c0) : 1;
        c2 *const Gw = G + (size_t)(gi & 1) * GSZ;                    // written by this group's pass 1
        const c2 *const Gr = G + (size_t)((gi & 1) ^ 1) * GSZ;        // group gi-1: read by F'
        if (live && c0 == c_lo) {
            // ---- Q = conj(Ohat) F0 for this thread's 16 bins (Eq. 12), new orientation
            const cf *F0 = p.F0 + ((size_t)model * p.n_orient + o) * H;
#pragma unroll
            for (int j = 0; j < N1; ++j) {
                const cf ov = Oimg[qbase + (size_t)N2 * j], fv = F0[qbase + (size_t)N2 * j];
                const cf pr = cmulc(ov, fv);
                q[j] = make_float2(pr.x, pr.y);
            }
            if (nyq) {
#pragma unroll
                for (int j = 0; j < N1; ++j) {
                    const size_t e = (size_t)(N / 2) * N + N2 * j + t;
                    const cf pr = cmulc(Oimg[e], F0[e]);
                    qn[((j >> 1) * N2 + t) * 2 + (j & 1)] = make_float2(pr.x, pr.y);
                }
            }
            __syncwarp();
        }
        if (tid < CG) {                                               // (alpha*beta, h) of CTF c0 + tid: stored now, fetched a group ahead
            if (tid < nc && live) sc[(gi & 3) * CG + tid] = make_float2(scn.x * beta, scn.y);
            int c0n = c0 + CG, on = o;
            if (c0n >= c_hi) { c0n = c_lo; ++on; }
            if (gi + 1 < total && c0n + tid < c_hi) {
                const size_t moc = ((size_t)model * p.n_orient + on) * p.n_ctf + c0n + tid;
                scn = make_float2(p.alpha[moc], p.hterm[moc]);
            }
        }
        // ================= slot A: F(0) of this group  ||  H' of group gi-2 (a5 + a6)
        {
            int cn = c0 + 1;
            if (cn >= c_hi) cn = c_lo;
            // H' first: it does not touch Q, so at a new orientation the Q loads issued above are in flight underneath it
            int h2e[NR];
#pragma unroll
            for (int cp = 0; cp < NR; ++cp) h2e[cp] = map.e[var2][warp * CPW + 2 * cp + half];
            int h2all = 0xffff;
#pragma unroll
            for (int cp = 0; cp < NR; ++cp) h2all &= h2e[cp];
            if (nc2 > 0 && __any_sync(FULLP, h2all != 0xffff)) {      // warp-uniform: some H' task in this warp
                const float2 *scb = sc + ((gi + 2) & 3) * CG;
#pragma unroll
                for (int cp = 0; cp < NR; ++cp) {
                    c2 y[2];
                    pk_horner2<N2, ZP>(Zw + zrd_off + cp * 2 * CS, rlo, rhi, rh, y[0], y[1]);
                    const int cl = h2e[cp] >> 8, pr = h2e[cp] == 0xffff ? 0 : h2e[cp] & 255;
                    const bool cv = cl < nc2, two = 2 * pr + 1 < KK;
                    const float2 s2 = scb[cv ? cl : 0];
                    const int sha = 2 * pr * KK, shb = sha + KK;
                    const bool v[4] = {cv && vlo, cv && vlo && two, cv && vhi, cv && vhi && two};
                    const uint32_t sh[4] = {(uint32_t)(sha + kk_lo), (uint32_t)(shb + kk_lo), (uint32_t)(sha + kk_hi), (uint32_t)(shb + kk_hi)};
                    pk_score<DUMP, 4>(p, st, mylist, y, v, sh, s2.x, s2.y, pair2 + (uint32_t)cl);
                }
                if (has_x) {                                          // dx = +16: one lane per task holds the two rows' values
                    const int xcl = eX >> 8, xpr = eX == 0xffff ? 0 : eX & 255;
                    const bool cv = t == 0 && xcl < nc2;
                    const float2 s2 = scb[xcl < nc2 ? xcl : 0];
                    const c2 y[1] = {xs2};
                    const int xsha = 2 * xpr * KK + KK - 1;
                    const bool v[2] = {cv, cv && 2 * xpr + 1 < KK};
                    const uint32_t sh[2] = {(uint32_t)xsha, (uint32_t)(xsha + KK)};
                    pk_score<DUMP, 2>(p, st, mylist, y, v, sh, s2.x, s2.y, pair2 + (uint32_t)xcl);
                }
            }
            if (!DUMP && ORIENT && nc2 > 0 && last2) {
                // group gi-2 was the last of its orientation: close this warp's sums for it
                float lse_m = st.m, lse_s = st.s;
#pragma unroll
                for (int off = 16; off >= 1; off >>= 1) {
                    const float m2 = __shfl_xor_sync(FULLP, lse_m, off), s2 = __shfl_xor_sync(FULLP, lse_s, off);
                    const float M = fmaxf(lse_m, m2);
                    lse_s = lse_s * pk_ex2(lse_m - M) + s2 * pk_ex2(m2 - M);
                    lse_m = M;
                }
                if (lane == 0) otab[ol2 * NW + warp] = make_float2(lse_m, lse_s);
                st.m = LSE_EMPTY; st.s = 0.f;
            }
            PK_LOAD_A(cn)
            PK_FFT_XS()
            if (gi > 0) pk_mbar_wait(&mbar[1], (unsigned)(gi - 1) & 1u);   // every warp has read G[gi & 1] (F' of group gi-2): first write below
            if (xlane) Gw[(size_t)(KK - 1) * GP + col] = xs;
            PK_SPILL()
        }
        // ================= slots B: F(ci)  ||  H(ci-1) -> G
        for (int ci = 1; ci < nc; ++ci) {
            int cn = c0 + ci + 1;
            if (cn >= c_hi) cn = c_lo;
            PK_LOAD_A(cn)
            PK_HORNER_G(Gw, ci - 1)
            PK_FFT_XS()
            if (xlane) Gw[(size_t)ci * KK * GP + (size_t)(KK - 1) * GP + col] = xs;
            PK_SPILL()
        }
        // ================= slot C: F' of group gi-1 (rows of Gr)  ||  H(nc-1) -> G
        if (gi > 0) pk_mbar_wait(&mbar[0], (unsigned)(gi - 1) & 1u);       // G rows of group gi-1 are complete
        const int eF = map.e[var1][a2combo];                          // this thread's F' task of group gi-1
        if (!(nc1 > 0 && __any_sync(FULLP, eF != 0xffff))) {
            if (lane == 0) pk_mbar_arrive(&mbar[1]);
            PK_HORNER_G(Gw, nc - 1)
            __syncwarp();
            if (lane == 0) pk_mbar_arrive(&mbar[0]);
        } else {
            const int a2cl = eF >> 8, a2pr = eF == 0xffff ? 0 : eF & 255;
            const bool a2two = 2 * a2pr + 1 < KK;
            const float a2bsel = a2two ? 1.f : 0.f;
            const c2 *ga = Gr + (size_t)(a2cl < nc1 ? a2cl : 0) * KK * GP + 2 * a2pr * GP, *gb = ga + (a2two ? GP : 0);
            c2 a[N1];
#pragma unroll
            for (int j = 0; j < N1; ++j) {
                // l = N2 j + t; direct for l < N/2, mirrored (conjugate) above: a = A + i B of the two real rows
                if (j > 0 && j < 8) {
                    const c2 va = ga[N2 * j + t], vb = gb[N2 * j + t];
                    a[j] = __ffma2_rn(pk_rot90(vb), pk_bc(a2bsel), va);
                } else if (j > 8) {
                    const c2 va = ga[N - N2 * j - t], vb = gb[N - N2 * j - t];
                    a[j] = __ffma2_rn(make_float2(vb.y, vb.x), pk_bc(a2bsel), make_float2(va.x, -va.y));
                } else if (j == 0) {                                  // t = 0: the packed entry holds (G(.,0), G(.,N/2)), both real
                    const c2 va = ga[t], vb = gb[t];
                    const c2 gen = __ffma2_rn(pk_rot90(vb), pk_bc(a2bsel), va);
                    a[j] = (t == 0) ? make_float2(va.x, a2bsel * vb.x) : gen;
                } else {
                    const c2 va = ga[l8], vb = gb[l8];
                    const c2 gen = __ffma2_rn(make_float2(vb.y, vb.x), pk_bc(a2bsel), make_float2(va.x, -va.y));
                    a[j] = (t == 0) ? make_float2(va.y, a2bsel * vb.y) : gen;
                }
            }
            __syncwarp();                                             // every lane's loads of G[(gi-1) & 1] are in registers
            if (lane == 0) pk_mbar_arrive(&mbar[1]);
            PK_HORNER_G(Gw, nc - 1)
            PK_FFT_XS()
            xs2 = xs;
            PK_SPILL()                                                // its __syncwarp orders every lane's G writes before the arrival
            if (lane == 0) pk_mbar_arrive(&mbar[0]);
        }
        nc2 = nc1; pair2 = pair1; eX = eF;
        var2 = var1; var1 = var0; var0 = var0 + 1 == map.nvar ? 0 : var0 + 1;
        nc1 = live ? nc : 0; pair1 = (uint32_t)((o + p.o_first) * p.n_ctf + c0);
        if (ORIENT) { last2 = last1; ol2 = ol1; last1 = live && c0 + CG >= c_hi; ol1 = o - o_begin; }
        c0 += CG;
        if (c0 >= c_hi) { c0 = c_lo; ++o; }
    }
#undef PK_LOAD_A
#undef PK_HORNER_G
#undef PK_FFT_XS
#undef PK_SPILL
    pk_cp_async_wait_all();
    if (DUMP) return;

    // ---- block reduction, fixed order
    if (ORIENT) {
        // warps -> orientation: thread i of warp 0 combines the NW entries of orientation i in warp order and writes its
        // (m, s), kept in otab[i * NW]: the work item's partial below is then the combination of its orientations, in order
        __syncthreads();
        if (warp == 0 && lane < o_end - o_begin) {
            float m = LSE_EMPTY, sm = 0.f;
            for (int w = 0; w < NW; ++w) {
                const float2 e = otab[lane * NW + w];
                const float M = fmaxf(m, e.x);
                sm = sm * pk_ex2(m - M) + e.y * pk_ex2(e.x - M);
                m = M;
            }
            otab[lane * NW] = make_float2(m, sm);
            const size_t oi = ((size_t)model * p.n_orient + o_begin + lane) * p.n_img + img;
            p.orient_m[oi] = sm > 0.f ? m : -CUDART_INF_F;
            p.orient_s[oi] = sm;
        }
    } else {
        float lse_m = st.m, lse_s = st.s;
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            const float m2 = __shfl_xor_sync(FULLP, lse_m, off), s2 = __shfl_xor_sync(FULLP, lse_s, off);
            const float M = fmaxf(lse_m, m2);
            lse_s = lse_s * pk_ex2(lse_m - M) + s2 * pk_ex2(m2 - M);
            lse_m = M;
        }
        if (lane == 0) { red[2 * warp] = lse_m; red[2 * warp + 1] = lse_s; }
    }
    __syncthreads();
    if (warp == 0) {
        float m = LSE_EMPTY, s = 0.f;
        const int nred = ORIENT ? o_end - o_begin : NW;
        for (int w = 0; w < nred; ++w) {
            const float m2 = ORIENT ? otab[w * NW].x : red[2 * w], s2 = ORIENT ? otab[w * NW].y : red[2 * w + 1];
            const float M = fmaxf(m, m2);
            s = s * pk_ex2(m - M) + s2 * pk_ex2(m2 - M);
            m = M;
        }
        if (!(s > 0.f)) m = -CUDART_INF_F;                            // the merge kernel's "empty partial"
        float th0 = tops[BIOEM_TOPK - 1].g;
        for (int w = 1; w < NW; ++w)
            for (int k = 0; k < BIOEM_TOPK; ++k) {
                TopEntry e = tops[w * BIOEM_TOPK + k];
                if (e.pair == 0xffffffffu || e.g < th0) break;        // lists are sorted: nothing further down can enter (warp-uniform)
                pk_topk_insert(e.g, e.pair, e.shift, lane == 0, th0, tops);
            }
        __syncwarp();
        if (lane == 0) { p.part_m[item] = m; p.part_s[item] = s; }
        if (lane < BIOEM_TOPK) p.part_top[(size_t)item * BIOEM_TOPK + lane] = tops[lane];
    }
}

// ------------------------------------------------------------------------------------------------ K in task order
// Kt[c][g4][tid][e]  = K_c(l = tid / N2, m = N2 (4 g4 + e) + tid % N2): the 16 values a thread needs are 4 coalesced float4.
// KtN[c][g4][t][e]   = K_c(l = N/2,      m = N2 (4 g4 + e) + t): the Nyquist column, read by the threads of column 0.
template <int N>
__global__ void k_relayout_K(const float *K32, float4 *Kt, float4 *KtN, int n_ctf)
{
    typedef PK<N> C_;
    const int c = blockIdx.y, i = blockIdx.x * blockDim.x + threadIdx.x;       // i = g4 * NT + tid
    if (i >= (C_::N1 / 4) * C_::NT) return;
    const int g4 = i / C_::NT, tid = i % C_::NT;
    const int col = tid / C_::N2, t = tid % C_::N2;
    const float *Kc = K32 + (size_t)c * (N / 2 + 1) * N;
    float v[4];
    for (int e = 0; e < 4; ++e) v[e] = Kc[(size_t)col * N + C_::N2 * (4 * g4 + e) + t];
    Kt[(size_t)c * (C_::N1 / 4) * C_::NT + i] = make_float4(v[0], v[1], v[2], v[3]);
    if (col == 0) {
        for (int e = 0; e < 4; ++e) v[e] = Kc[(size_t)(N / 2) * N + C_::N2 * (4 * g4 + e) + t];
        KtN[((size_t)c * 4 + g4) * C_::N2 + t] = make_float4(v[0], v[1], v[2], v[3]);
    }
}

bool pk_supported(int N, int D) { return (N == 64 || N == 128) && D <= 16; }
// Kt followed by KtN
size_t pk_kt_bytes(int N, int n_ctf)
{
    const size_t nt = N == 64 ? PK<64>::NT : PK<128>::NT, n2 = N / 16;
    return (size_t)n_ctf * 4 * nt * 16 + (size_t)n_ctf * 4 * n2 * 16;
}
static const float *pk_ktn(int N, const float *Kt, int n_ctf)
{
    const size_t nt = N == 64 ? PK<64>::NT : PK<128>::NT;
    return Kt + (size_t)n_ctf * 4 * nt * 4;
}

cudaError_t launch_relayout_K(int N, const float *K32, float *Kt, int n_ctf, cudaStream_t st)
{
    float4 *ktn = reinterpret_cast<float4 *>(const_cast<float *>(pk_ktn(N, Kt, n_ctf)));
    if (N == 64) {
        dim3 g((4 * PK<64>::NT + 255) / 256, n_ctf);
        k_relayout_K<64><<<g, 256, 0, st>>>(K32, reinterpret_cast<float4 *>(Kt), ktn, n_ctf);
    } else {
        dim3 g((4 * PK<128>::NT + 255) / 256, n_ctf);
        k_relayout_K<128><<<g, 256, 0, st>>>(K32, reinterpret_cast<float4 *>(Kt), ktn, n_ctf);
    }
    return cudaGetLastError();
}

// Assign the CG * NP pass-2 tasks (CTF in group, row pair) to the NCOMBO slots.  A half-warp holds G = 16 / N2 slots, each
// reading N2 consecutive complex words of one G row per load: the load is conflict-free when the rows' offsets (in 8-byte
// banks, mod 16) are o, o + N2, o + 2 N2, ...  Tasks are bucketed by offset and drawn accordingly; leftovers fill up in any
// order.  Groups are placed at the END of the slot range, so the idle slots make warps 0, 1, ... idle in pass 2.
static bool pk_build_map(int N2, int NCOMBO, int CG, int NP, int KK, int GP, PkMap &map)
{
    const int G = 16 / N2;
    std::vector<std::vector<uint16_t>> bucket(16);
    for (int cl = 0; cl < CG; ++cl)
        for (int pr = 0; pr < NP; ++pr) bucket[((long)cl * KK * GP + 2L * pr * GP) % 16].push_back((uint16_t)(cl << 8 | pr));
    std::vector<uint16_t> slots;
    for (int o = 0; o < 16; ++o)
        for (;;) {
            bool full = true;
            for (int e = 0; e < G; ++e) full = full && !bucket[(o + e * N2) % 16].empty();
            if (!full) break;
            for (int e = 0; e < G; ++e) { auto &b = bucket[(o + e * N2) % 16]; slots.push_back(b.back()); b.pop_back(); }
        }
    for (auto &b : bucket)
        for (uint16_t v : b) slots.push_back(v);
    while (slots.size() % G) slots.push_back(0xffff);
    if ((int)slots.size() > NCOMBO) return false;
    // Idle slots: whole warps are idle in pass 2.  With 16 warps (4 per scheduler) warp 0 is always one of them (it carries the
    // Nyquist column in pass 1) and the others rotate over warps 1..3 from group to group (3 variants), so that over three
    // groups every scheduler sees the same pass-2 load; otherwise one variant with the idle warps first.
    const int CPW = 32 / N2, NW = NCOMBO / CPW, idle = NCOMBO - (int)slots.size(), idle_w = idle / CPW, rem = idle % CPW;
    map.nvar = (NW == 16 && idle_w >= 2 && idle_w <= 4) ? 3 : 1;
    for (int v = 0; v < 3; ++v) {
        bool iw[64] = {false};
        if (map.nvar == 3) {
            iw[0] = true;
            for (int i = 0; i + 1 < idle_w; ++i) iw[1 + (v + i) % 3] = true;
        } else
            for (int w = 0; w < idle_w; ++w) iw[w] = true;
        for (int i = 0; i < 64; ++i) map.e[v][i] = 0xffff;
        int skip = rem;
        size_t k = 0;
        for (int i = 0; i < NCOMBO; ++i) {
            if (iw[i / CPW]) continue;
            if (skip > 0) { --skip; continue; }
            map.e[v][i] = slots[k++];
        }
    }
    return true;
}

template <int N>
static void pk_plan(int D, int n_ctf, bool orient, int &CG, int &GP, size_t &bytes, PkMap &map)
{
    typedef PK<N> C_;
    const int KK = 2 * D + 1, NP = D + 1;
    GP = C_::NCH | 1;
    CG = C_::NCOMBO / NP;                               // CTFs per group: every (CTF, row pair, residue) task of pass 2 has a thread
    if (CG < 1) CG = 1;
    if (CG > n_ctf) CG = n_ctf;
    const size_t budget = 227 * 1024;
    for (;;) {
        bytes = (size_t)C_::NW * C_::ZW * 8 + (size_t)2 * CG * KK * GP * 8 + 16 * C_::N2 * 8 + (8 * C_::N2 + 1) * 16 + 4 * (size_t)CG * 8 +
                (size_t)C_::NW * BIOEM_TOPK * sizeof(TopEntry) + 2 * C_::NW * 4 + 64 + (orient ? (size_t)32 * C_::NW * sizeof(float2) : 0);
        if ((bytes <= budget && pk_build_map(C_::N2, C_::NCOMBO, CG, NP, KK, GP, map)) || CG == 1) break;
        --CG;
    }
    if (CG == 1) pk_build_map(C_::N2, C_::NCOMBO, CG, NP, KK, GP, map);
}

template <int N>
static cudaError_t launch_pk_t(const FusedParams &p, const float *Kt, bool dump, cudaStream_t st)
{
    int CG, GP;
    size_t bytes;
    PkMap map;
    const bool orient = p.orient_m != nullptr && !dump;
    pk_plan<N>(p.D, p.n_ctf, orient, CG, GP, bytes, map);
    if (bytes > 227 * 1024) return cudaErrorInvalidConfiguration;
    if (orient && p.oc > 32) return cudaErrorInvalidValue;            // otab holds 32 orientations per work item
    const float4 *kt = reinterpret_cast<const float4 *>(Kt), *ktn = reinterpret_cast<const float4 *>(pk_ktn(N, Kt, p.n_ctf));
    cudaError_t e;
    if (dump) {
        e = cudaFuncSetAttribute(k_fused_pk<N, true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        k_fused_pk<N, true, false><<<1, PK<N>::NT, bytes, st>>>(p, kt, ktn, CG, GP, map);
    } else if (orient) {
        e = cudaFuncSetAttribute(k_fused_pk<N, false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        const int items = p.n_img * p.n_model * p.chunks_per_model;
        k_fused_pk<N, false, true><<<items, PK<N>::NT, bytes, st>>>(p, kt, ktn, CG, GP, map);
    } else {
        e = cudaFuncSetAttribute(k_fused_pk<N, false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        const int items = p.n_img * p.n_model * p.chunks_per_model;
        k_fused_pk<N, false, false><<<items, PK<N>::NT, bytes, st>>>(p, kt, ktn, CG, GP, map);
    }
    return cudaGetLastError();
}

cudaError_t launch_fused_pk(int N, const FusedParams &p, const float *Kt, bool dump, cudaStream_t st)
{
    if (N == 64) return launch_pk_t<64>(p, Kt, dump, st);
    if (N == 128) return launch_pk_t<128>(p, Kt, dump, st);
    return cudaErrorInvalidValue;
}

}  // namespace bioem
