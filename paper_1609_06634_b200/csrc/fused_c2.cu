// fused_c2.cu -- the hot loop for N = 224 (the paper's box size): a thread-block
// CLUSTER OF TWO CTAs (two SMs) per (image, model, chunk of orientations), Q = conj(Ohat) F0 register-resident across the
// pair, G rows exchanged through distributed shared memory.
//
// Why a cluster: at 224^2 the half spectrum is 113 x 224 complex = 202 KB.  One SM cannot hold Q next to the transform's
// working set (256 KB of registers, 227 KB of shared memory), and re-reading Ohat, F0, K from L2 for every CTF (what the
// generic kernel does: 20 bytes per bin per pair = 506 KB per pair) is bound by the SM's L2 port at twice the FP32 time.
// Split over two SMs each CTA keeps 56 of the 112 packed columns (column 0 carries the Nyquist column l = 112, both are
// Hermitian in m) = 12544 complex = 98 KB in registers, and per CTF only the real table K_c streams from L2 (4 bytes per bin).
//
// Factorisation 224 = 32 x 7: thread = (column l, residue t), m = 7 j + t, j = 0..31.  The 32-point register transform is one
// radix-2 decimation-in-frequency stage and two 16-point transforms run one after the other (u_j = x_j + x_(j+16) gives the
// even outputs, v_j = (x_j - x_(j+16)) w32^j the odd ones; the differences wait in the thread's own shared-memory row), so
// that only 16 complex values are live next to the 32 of Q.  Pass 1 stage 2: lane = output index k1, Horner sums over the 7
// residues for the two needed outputs k1 - 32 and k1 (|k| <= D <= 31), written into the G tile OF THE CTA THAT OWNS THE ROW
// (rank 0: row pairs 0..P0-1, rank 1: the rest), locally or with st.shared::cluster.  Pass 2 (along l, two real rows per complex
// transform, Hermitian completion on load) runs one step later on 4 of the 14 warps, rotating from step to step, and scores
// its outputs at once (a5, a6).  Hand-over: per buffer a "full" mbarrier whose phase completes when every byte of the tile has
// landed (the stores are st.async with complete_tx on the owner's barrier: no fence; a release at cluster scope costs a
// MEMBAR.ALL.GPU per arrival) and an "empty" mbarrier (8 relaxed arrivals: the pass-2 warps of both CTAs).
// No float atomics, fixed reduction orders: bit-reproducible.
#include "pk_math.cuh"

namespace bioem {

struct C2 {
    static constexpr int N = 224, N2 = 7, NCOL = 56, NW = 14, NT = NW * 32;      // 56 packed columns per CTA, 4 columns x 7 residues per warp
    static constexpr int ZP = 34, ZW = 28 * ZP;                                   // Z row pitch (16-byte units odd: conflict-free 128-bit rows); one row per lane with a column
    static constexpr int RP = 34;                                                 // G_T row pitch: [column][local row]
    static constexpr int GSZ = 2 * NCOL * RP;                                     // one G_T buffer: 112 packed columns
    static constexpr int P2W = 4;                                                 // warps running pass 2 in a step
    static constexpr int NB = 2;                                                  // G_T buffers (3 fits shared memory too; measured no faster: the L1 left for the register spills shrinks)
};

// ---- cluster helpers
__device__ __forceinline__ unsigned c2_rank()
{
    unsigned r;
    asm volatile("mov.u32 %0, %%cluster_ctarank;" : "=r"(r));
    return r;
}
__device__ __forceinline__ unsigned c2_map(const void *smem_ptr, unsigned rank)       // shared::cluster address of the same variable in CTA `rank`
{
    unsigned a = (unsigned)__cvta_generic_to_shared(smem_ptr), r;
    asm volatile("mapa.shared::cluster.u32 %0, %1, %2;" : "=r"(r) : "r"(a), "r"(rank));
    return r;
}
// 8-byte store into the shared memory of a CTA of the cluster that also counts its bytes on an mbarrier OF THAT CTA: the
// barrier's phase completes when every expected byte has landed, so the hand-over needs no fence (a release at cluster scope
// costs MEMBAR.ALL.GPU per arrival, an acquire at cluster scope an L1 invalidation per wait).
__device__ __forceinline__ void c2_st_async(unsigned cluster_addr, c2 v, unsigned cluster_mbar)
{
    asm volatile("st.async.weak.shared::cluster.mbarrier::complete_tx::bytes.v2.f32 [%0], {%1, %2}, [%3];" ::"r"(cluster_addr), "f"(v.x),
                 "f"(v.y), "r"(cluster_mbar) : "memory");
}
__device__ __forceinline__ void c2_expect_tx(uint64_t *bar, unsigned bytes)            // one arrival + the bytes this phase will receive
{
    asm volatile("mbarrier.arrive.expect_tx.shared::cta.b64 _, [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(bytes) : "memory");
}
__device__ __forceinline__ void c2_arrive(unsigned cluster_addr)                       // "my reads are done": no data flows with it
{
    asm volatile("mbarrier.arrive.relaxed.cluster.shared::cluster.b64 _, [%0];" ::"r"(cluster_addr) : "memory");
}
__device__ __forceinline__ void c2_wait(uint64_t *bar, unsigned parity)                // sleeps between probes
{
    const unsigned b = (unsigned)__cvta_generic_to_shared(bar);
    while (!pk_mbar_test(b, parity)) __nanosleep(1000);
}
__device__ __forceinline__ void c2_cluster_sync()
{
    asm volatile("barrier.cluster.arrive.release.aligned;\n" "barrier.cluster.wait.acquire.aligned;\n" ::: "memory");
}

// y = sum_t r^t z[t] for both roots, sharing the 7 loads (Horner, t = 6..0)
__device__ __forceinline__ void c2_horner7(const c2 *zc, c2 rlo, c2 rhi, c2 &ylo, c2 &yhi)
{
    c2 z = zc[6 * C2::ZP];
    ylo = z; yhi = z;
#pragma unroll
    for (int t = 5; t >= 0; --t) {
        z = zc[t * C2::ZP];
        ylo = pk_cmadd(ylo, rlo, z);
        yhi = pk_cmadd(yhi, rhi, z);
    }
}

// Second half of a 32-point transform whose first radix-2 stage has been applied: FFT16 of u -> even outputs at row words
// 0..15, then v_j = d_j w32^j (d read back from row words 16..31), FFT16 -> odd outputs at row words 16..31.
__device__ __forceinline__ void c2_spill16(c2 *zst, const c2 (&a)[16], bool act)
{
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int b = bitrev(r, 3);
        if (act) *reinterpret_cast<float4 *>(zst + 2 * b) = make_float4(a[r].x, a[r].y, a[r + 8].x, a[r + 8].y);
    }
}
__device__ __forceinline__ void c2_fft32_tail(c2 (&a)[16], c2 *zrow, bool act)
{
    pk_fft16(a);
    c2_spill16(zrow, a, act);
#pragma unroll
    for (int j = 0; j < 16; j += 2) {
        float4 d = make_float4(0.f, 0.f, 0.f, 0.f);
        if (act) d = *reinterpret_cast<const float4 *>(zrow + 16 + j);
        a[j] = pk_twid(make_float2(d.x, d.y), j);
        a[j + 1] = pk_twid(make_float2(d.z, d.w), j + 1);
    }
    pk_fft16(a);
    c2_spill16(zrow + 16, a, act);
}

// F-phase of pass 1 for one CTF: x_j = Q_j K_j (m = 7 j + t), first radix-2 stage on the fly, two 16-point transforms.
// NYQ: the threads of packed column 0 add i Q(112, m) K(112, m) (both columns are Hermitian in m, so the transform of the sum
// is G(., 0) + i G(., 112) with both parts real).
template <bool NYQ>
__device__ __forceinline__ void c2_pass1_f(const c2 (&q)[16], const float4 *qs, const float4 *__restrict__ kt, c2 *zrow, bool act, bool nyq,
                                           const c2 *qn, const float *__restrict__ kn)
{
    c2 a[16];
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        const float4 kA = kt[(size_t)g * C2::NT], kB = kt[(size_t)(g + 4) * C2::NT];
        const float4 qh0 = qs[(size_t)(2 * g) * C2::NT], qh1 = qs[(size_t)(2 * g + 1) * C2::NT];     // Q_(16 + 4g .. 16 + 4g + 3) of this thread
        const float ka[4] = {kA.x, kA.y, kA.z, kA.w}, kb[4] = {kB.x, kB.y, kB.z, kB.w};
        const c2 qh[4] = {make_float2(qh0.x, qh0.y), make_float2(qh0.z, qh0.w), make_float2(qh1.x, qh1.y), make_float2(qh1.z, qh1.w)};
        c2 d[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int j = 4 * g + e;
            c2 xA = __fmul2_rn(q[j], pk_bc(ka[e]));
            c2 xB = __fmul2_rn(qh[e], pk_bc(kb[e]));
            if (NYQ && nyq) {
                xA = __ffma2_rn(pk_rot90(qn[j * 7]), pk_bc(kn[j * 7]), xA);
                xB = __ffma2_rn(pk_rot90(qn[(j + 16) * 7]), pk_bc(kn[(j + 16) * 7]), xB);
            }
            a[j] = pk_add(xA, xB);
            d[e] = pk_sub(xA, xB);
        }
        if (act) {
            *reinterpret_cast<float4 *>(zrow + 16 + 4 * g) = make_float4(d[0].x, d[0].y, d[1].x, d[1].y);
            *reinterpret_cast<float4 *>(zrow + 16 + 4 * g + 2) = make_float4(d[2].x, d[2].y, d[3].x, d[3].y);
        }
    }
    c2_fft32_tail(a, zrow, act);
}

// F' of pass 2 for one row pair: the 224-point transform along l of A + i B (rows A, B of this CTA's G_T tile, read as one
// 128-bit word per column), thread = (pair, residue t), l = 7 j + t.  Columns l = 1..111 are stored, l = 113..223 are their
// conjugates (Hermitian half), packed column 0 holds (G(., 0), G(., 112)), both real.
__device__ __forceinline__ void c2_pass2_f(const c2 *gt, int t, float bsel, c2 *zrow, bool act)
{
    c2 a[16];
    const c2 bs = pk_bc(bsel);
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        c2 d[4];
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int j = 4 * g + e;
            // low half: l = 7 j + t (direct); high half: l = 112 + 7 j + t -> mirrored column 112 - 7 j - t
            const int cl = 7 * j + t, ch = (j == 0 && t == 0) ? 0 : 112 - 7 * j - t;
            const float4 vl = *reinterpret_cast<const float4 *>(gt + (size_t)cl * C2::RP);
            const float4 vh = *reinterpret_cast<const float4 *>(gt + (size_t)ch * C2::RP);
            // direct: A + i B = (A.x - B.y, A.y + B.x); mirrored: conj(A) + i conj(B) = (A.x + B.y, -A.y + B.x)
            c2 xl = __ffma2_rn(make_float2(-vl.w, vl.z), bs, make_float2(vl.x, vl.y));
            c2 xh = __ffma2_rn(make_float2(vh.w, vh.z), bs, make_float2(vh.x, -vh.y));
            if (j == 0 && t == 0) {                       // packed column: l = 0 -> (A.x, B.x), l = 112 -> (A.y, B.y)
                xl = make_float2(vl.x, bsel * vl.z);
                xh = make_float2(vl.y, bsel * vl.w);
            }
            a[j] = pk_add(xl, xh);
            d[e] = pk_sub(xl, xh);
        }
        if (act) {
            *reinterpret_cast<float4 *>(zrow + 16 + 4 * g) = make_float4(d[0].x, d[0].y, d[1].x, d[1].y);
            *reinterpret_cast<float4 *>(zrow + 16 + 4 * g + 2) = make_float4(d[2].x, d[2].y, d[3].x, d[3].y);
        }
    }
    c2_fft32_tail(a, zrow, act);
}

template <bool DUMP>
__global__ void __cluster_dims__(2, 1, 1) __launch_bounds__(C2::NT, 1)
k_fused_c2(FusedParams p, const float4 *__restrict__ Kt, const float *__restrict__ KtN, int P0)
{
    constexpr int N = C2::N, NW = C2::NW, NT = C2::NT, ZP = C2::ZP, ZW = C2::ZW, RP = C2::RP, GSZ = C2::GSZ, P2W = C2::P2W, NB = C2::NB;
    constexpr size_t H = (size_t)(N / 2 + 1) * N;
    const int D = p.D, KK = 2 * D + 1, NP = D + 1;                    // host guarantees D <= 31; NP row pairs (the last one is a single row)
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;
    const unsigned rank = c2_rank(), peer = rank ^ 1u;
    const int my_p0 = rank ? P0 : 0, my_np = rank ? NP - P0 : P0;     // this CTA's row pairs [my_p0, my_p0 + my_np)

    extern __shared__ __align__(16) unsigned char smem_raw[];
    c2 *Z = reinterpret_cast<c2 *>(smem_raw);                         // [NW][28][ZP]   warp-private tiles, one row per lane with a column
    c2 *G = Z + (size_t)NW * ZW;                                      // [NB][112][RP]  G_T: pass-1 outputs of this CTA's rows, all columns
    float4 *Qs = reinterpret_cast<float4 *>(G + (size_t)NB * GSZ);    // [8][NT]        upper half of Q (j = 16..31): 2 complex per word, own thread's only
    c2 *qn = reinterpret_cast<c2 *>(Qs + 8 * NT);                                   // [32][7]        Q of the Nyquist column (rank 0, warp 0)
    TopEntry *tops = reinterpret_cast<TopEntry *>(qn + 224);          // [NW][TOPK]
    float *red = reinterpret_cast<float *>(tops + NW * BIOEM_TOPK);   // [2 NW]
    __shared__ uint64_t bar_full[NB], bar_empty[NB];

    int img, model, o_begin, o_end, item;
    if (DUMP) { img = p.dump_img; model = p.dump_model; o_begin = p.dump_orient; o_end = o_begin + 1; item = 0; }
    else {
        item = blockIdx.x >> 1;
        img = item % p.n_img;
        const int chunk = item / p.n_img;
        model = chunk / p.chunks_per_model;
        o_begin = (chunk % p.chunks_per_model) * p.oc;
        o_end = min(o_begin + p.oc, p.n_orient);
    }
    const float beta = p.beta[img];
    for (int i = tid; i < (NW * ZW + NB * GSZ + 16 * NT + 224) * 2; i += NT) reinterpret_cast<float *>(Z)[i] = 0.f;
    if (tid < NW * BIOEM_TOPK) { TopEntry e0 = {-CUDART_INF_F, 0xffffffffu, 0xffffffffu}; tops[tid] = e0; }
    if (tid == 0) {
        for (int i = 0; i < NB; ++i) { pk_mbar_init(&bar_full[i], 1); pk_mbar_init(&bar_empty[i], 2 * P2W); }
    }
    __syncthreads();
    c2_cluster_sync();                                                // both CTAs' tiles are zeroed and barriers initialised before any remote access

    // ---- pass-1 F-phase: lane < 28 -> (column 4 warp + lane / 7, residue lane % 7); lanes 28..31 carry zeros
    const bool has_col = lane < 28;
    const int colw = has_col ? lane / 7 : 0, t = has_col ? lane % 7 : 0;
    const int l = 56 * (int)rank + 4 * warp + colw;                   // packed column 0..111
    const size_t qbase = (size_t)l * N + t;
    c2 *const Zw = Z + (size_t)warp * ZW, *const zrow = Zw + (has_col ? lane : 0) * ZP;
    const bool warp_nyq = rank == 0 && warp == 0, nyq = warp_nyq && lane < 7;
    // ---- H-phase: lane -> output index k1 (each half-warp holds one of every pair {2k', 2k'+1} and 16 distinct k1 mod 16)
    const int hw = lane >> 4, q16 = lane & 15, k1 = q16 < 8 ? 2 * q16 + hw : 2 * q16 + 1 - hw;
    const int zpos = (k1 & 1) * 16 + (k1 >> 1);
    const bool vlo = k1 >= 32 - D, vhi = k1 <= D;
    const int kk_lo = vlo ? k1 - 32 + D : 0, kk_hi = vhi ? k1 + D : 0;
    c2 rlo, rhi;
    sincospif(2.0f * (float)(k1 - 32 + N) / (float)N, &rlo.y, &rlo.x);
    sincospif(2.0f * (float)k1 / (float)N, &rhi.y, &rhi.x);
    // owner CTA and local row of the two outputs; cluster addresses of G_T[0][0][row] there
    const unsigned own_lo = (kk_lo >> 1) >= P0, own_hi = (kk_hi >> 1) >= P0;
    const unsigned g_lo = c2_map(G, own_lo) + 8u * (unsigned)(kk_lo - (own_lo ? 2 * P0 : 0));
    const unsigned g_hi = c2_map(G, own_hi) + 8u * (unsigned)(kk_hi - (own_hi ? 2 * P0 : 0));
    const unsigned f_lo = c2_map(&bar_full[0], own_lo), f_hi = c2_map(&bar_full[0], own_hi);       // + 8 b: "full" barrier of buffer b in the owning CTA
    const unsigned empty_l = c2_map(&bar_empty[0], rank), empty_p = c2_map(&bar_empty[0], peer);
    const int rows0 = min(2 * P0, KK);
    const unsigned full_bytes = 8u * 112u * (unsigned)(rank ? KK - rows0 : rows0);      // bytes one step stores into this CTA's G_T tile

    const cf *Oimg = p.Ohat + (size_t)img * H;
    PkLse st = {LSE_EMPTY, 0.f, -CUDART_INF_F};
    TopEntry *mylist = tops + warp * BIOEM_TOPK;
    const int c_lo = DUMP ? p.dump_ctf : 0, c_hi = DUMP ? p.dump_ctf + 1 : p.n_ctf, ncf = c_hi - c_lo;
    const int S = (o_end - o_begin) * ncf;                            // steps = (orientation, CTF) pairs of this work item
    constexpr size_t KSTR = (size_t)2 * 8 * NT;                       // float4 per CTF in Kt: [c][rank][g 0..7][tid]
    const float4 *kt_t = Kt + (size_t)rank * 8 * NT + tid;

    c2 q[16];
#pragma unroll
    for (int j = 0; j < 16; ++j) q[j] = make_float2(0.f, 0.f);
    int o = o_begin, c = c_lo, o1 = o_begin, c1 = c_lo;               // (o, c) of step s; (o1, c1) of step s - 1
    unsigned b = 0, ph = 0, b1 = 0, ph1 = 0;                          // buffer s % NB and phase parity (s / NB) & 1 of steps s and s - 1
    for (int s = 0; s <= S; ++s) {
        if (s < S) {
            if (c == c_lo) {
                // ---- Q = conj(Ohat) F0 for this thread's 32 bins (Eq. 12), new orientation
                const cf *F0 = p.F0 + ((size_t)model * p.n_orient + o) * H;
                if (has_col) {
#pragma unroll
                    for (int j = 0; j < 16; ++j) {
                        const cf pr = cmulc(Oimg[qbase + 7 * j], F0[qbase + 7 * j]);
                        q[j] = make_float2(pr.x, pr.y);
                    }
#pragma unroll
                    for (int i = 0; i < 8; ++i) {
                        const cf p0 = cmulc(Oimg[qbase + 7 * (16 + 2 * i)], F0[qbase + 7 * (16 + 2 * i)]);
                        const cf p1 = cmulc(Oimg[qbase + 7 * (17 + 2 * i)], F0[qbase + 7 * (17 + 2 * i)]);
                        Qs[(size_t)i * NT + tid] = make_float4(p0.x, p0.y, p1.x, p1.y);
                    }
                }
                if (nyq) {
                    for (int j = 0; j < 32; ++j) {
                        const size_t e = (size_t)(N / 2) * N + 7 * j + t;
                        const cf pr = cmulc(Oimg[e], F0[e]);
                        qn[7 * j + t] = make_float2(pr.x, pr.y);
                    }
                }
            }
            // ---- pass 1, F-phase (a4): 32-point transforms along m into the warp's tile
            __syncwarp();                                             // every lane has read the previous tile
            const float4 *kt = kt_t + (size_t)c * KSTR;
            if (warp_nyq) c2_pass1_f<true>(q, Qs + tid, kt, zrow, has_col, nyq, qn + t, KtN + (size_t)c * 224 + t);
            else c2_pass1_f<false>(q, Qs + tid, kt, zrow, has_col, false, nullptr, nullptr);
            __syncwarp();
            // ---- pass 1, H-phase: the 2D+1 needed outputs of each of the warp's 4 columns -> G_T of the owning CTA
            if (s >= NB) c2_wait(&bar_empty[b], ph ^ 1u);                    // both CTAs have read buffer b (step s - NB)
            {
                const unsigned cb = 8u * (b * (unsigned)GSZ + (unsigned)((56 * (int)rank + 4 * warp) * RP));
#pragma unroll
                for (int cw = 0; cw < 4; ++cw) {
                    c2 ylo, yhi;
                    c2_horner7(Zw + cw * 7 * ZP + zpos, rlo, rhi, ylo, yhi);
                    if (vlo) c2_st_async(g_lo + cb + 8u * (unsigned)(cw * RP), ylo, f_lo + 8u * b);
                    if (vhi) c2_st_async(g_hi + cb + 8u * (unsigned)(cw * RP), yhi, f_hi + 8u * b);
                }
            }
        }
        // ---- pass 2 of step s - 1 (a4 along l, a5, a6) on P2W warps, rotating with the step
        if (s >= 1) {
            const int s1 = s - 1;
            int w2 = warp - (P2W * s1) % NW;
            if (w2 < 0) w2 += NW;
            if (w2 < P2W) {
                const int pl = 4 * w2 + colw;                         // this thread's local row pair (F'), lanes < 28
                const bool pv = has_col && pl < my_np;
                const int prf = my_p0 + (pv ? pl : 0);
                const float bsel = 2 * prf + 1 < KK ? 1.f : 0.f;
                if (w2 == 0 && lane == 0) c2_expect_tx(&bar_full[b1], full_bytes);   // this phase: one arrival + every byte of the tile
                c2_wait(&bar_full[b1], ph1);    // all 28 warps of the cluster have stored their part of buffer b1
                __syncwarp();                                         // the H-phase reads of this warp's tile are done
                c2_pass2_f(G + (size_t)b1 * GSZ + 2 * (pv ? pl : 0), t, bsel, zrow, has_col);
                __syncwarp();                                         // tile complete; every lane's G_T loads are in registers
                if (lane == 0) { c2_arrive(empty_l + 8u * b1); c2_arrive(empty_p + 8u * b1); }
                const size_t moc = ((size_t)model * p.n_orient + o1) * p.n_ctf + c1;
                const float ab = p.alpha[moc] * beta, hterm = p.hterm[moc];
                const uint32_t pair = (uint32_t)((o1 + p.o_first) * p.n_ctf + c1);
#pragma unroll
                for (int cw = 0; cw < 4; ++cw) {
                    c2 y[2];
                    c2_horner7(Zw + cw * 7 * ZP + zpos, rlo, rhi, y[0], y[1]);
                    const int plh = 4 * w2 + cw, pr = my_p0 + plh;
                    const bool cv = plh < my_np, two = 2 * pr + 1 < KK;
                    const int sha = 2 * pr * KK, shb = sha + KK;
                    const bool v[4] = {cv && vlo, cv && vlo && two, cv && vhi, cv && vhi && two};
                    const uint32_t sh[4] = {(uint32_t)(sha + kk_lo), (uint32_t)(shb + kk_lo), (uint32_t)(sha + kk_hi), (uint32_t)(shb + kk_hi)};
                    pk_score<DUMP, 4>(p, st, mylist, y, v, sh, ab, hterm, pair);
                }
            }
        }
        o1 = o; c1 = c; b1 = b; ph1 = ph;
        if (++c >= c_hi) { c = c_lo; ++o; }
        if (++b == NB) { b = 0; ph ^= 1u; }
    }
    c2_cluster_sync();                                                // no CTA leaves while its peer may still store to it or arrive on its barriers
    if (DUMP) return;

    // ---- block reduction, fixed order
    float lse_m = st.m, lse_s = st.s;
#pragma unroll
    for (int off = 16; off >= 1; off >>= 1) {
        const float m2 = __shfl_xor_sync(FULLP, lse_m, off), s2 = __shfl_xor_sync(FULLP, lse_s, off);
        const float M = fmaxf(lse_m, m2);
        lse_s = lse_s * pk_ex2(lse_m - M) + s2 * pk_ex2(m2 - M);
        lse_m = M;
    }
    if (lane == 0) { red[2 * warp] = lse_m; red[2 * warp + 1] = lse_s; }
    __syncthreads();
    if (warp == 0) {
        float m = LSE_EMPTY, s = 0.f;
        for (int w = 0; w < NW; ++w) {
            const float m2 = red[2 * w], s2 = red[2 * w + 1];
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
        // the two CTAs of the cluster are two partials of the same (image, model): chunk' = 2 chunk + rank
        const size_t out = ((size_t)(item / p.n_img) * 2 + rank) * p.n_img + (size_t)(item % p.n_img);
        if (lane == 0) { p.part_m[out] = m; p.part_s[out] = s; }
        if (lane < BIOEM_TOPK) p.part_top[out * BIOEM_TOPK + lane] = tops[lane];
    }
}

// ------------------------------------------------------------------------------------------------ K in task order
// Kt[c][rank][g][tid] (float4, g = 0..7): K_c(l = 56 rank + 4 (tid / 32) + (tid % 32) / 7, m = 7 (4 g + e) + (tid % 32) % 7), e = 0..3;
// lanes 28..31 of a warp have no column: zeros.  KtN[c][7 j + t] = K_c(l = 112, m = 7 j + t).
__global__ void k_relayout_K_c2(const float *K32, float4 *Kt, float *KtN, int n_ctf)
{
    constexpr int N = C2::N, NT = C2::NT;
    const int c = blockIdx.y, i = blockIdx.x * blockDim.x + threadIdx.x;       // i = (rank * 8 + g) * NT + tid
    if (i >= 2 * 8 * NT) return;
    const int tid = i % NT, g = (i / NT) % 8, rank = i / (8 * NT);
    const int lane = tid & 31, warp = tid >> 5;
    const float *Kc = K32 + (size_t)c * (N / 2 + 1) * N;
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    if (lane < 28) {
        const int l = 56 * rank + 4 * warp + lane / 7, t = lane % 7;
        for (int e = 0; e < 4; ++e) v[e] = Kc[(size_t)l * N + 7 * (4 * g + e) + t];
    }
    Kt[(size_t)c * 2 * 8 * NT + i] = make_float4(v[0], v[1], v[2], v[3]);
    if (i < N) KtN[(size_t)c * N + i] = Kc[(size_t)(N / 2) * N + i];
}

bool c2_supported(int N, int D) { return N == 224 && D <= 31; }
size_t c2_kt_bytes(int n_ctf) { return (size_t)n_ctf * 2 * 8 * C2::NT * 16 + (size_t)n_ctf * C2::N * 4; }
static const float *c2_ktn(const float *Kt, int n_ctf) { return Kt + (size_t)n_ctf * 2 * 8 * C2::NT * 4; }

cudaError_t launch_relayout_K_c2(const float *K32, float *Kt, int n_ctf, cudaStream_t st)
{
    dim3 g((2 * 8 * C2::NT + 255) / 256, n_ctf);
    k_relayout_K_c2<<<g, 256, 0, st>>>(K32, reinterpret_cast<float4 *>(Kt), const_cast<float *>(c2_ktn(Kt, n_ctf)), n_ctf);
    return cudaGetLastError();
}

// Work items: one cluster (2 CTAs) per (image, model, chunk); partial results: 2 per work item (see the kernel's epilogue).
cudaError_t launch_fused_c2(const FusedParams &p, const float *Kt, bool dump, cudaStream_t st)
{
    const size_t bytes = ((size_t)C2::NW * C2::ZW + C2::NB * C2::GSZ + 16 * C2::NT + 224) * 8 + (size_t)C2::NW * BIOEM_TOPK * sizeof(TopEntry) + 2 * C2::NW * 4 + 64;
    const int P0 = (p.D + 2) / 2;                                     // rank 0 takes ceil(NP / 2) of the NP = D + 1 row pairs
    const float4 *kt = reinterpret_cast<const float4 *>(Kt);
    const float *ktn = c2_ktn(Kt, p.n_ctf);
    cudaError_t e;
    if (dump) {
        e = cudaFuncSetAttribute(k_fused_c2<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        k_fused_c2<true><<<2, C2::NT, bytes, st>>>(p, kt, ktn, P0);
    } else {
        e = cudaFuncSetAttribute(k_fused_c2<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        const int items = p.n_img * p.n_model * p.chunks_per_model;
        k_fused_c2<false><<<2 * items, C2::NT, bytes, st>>>(p, kt, ktn, P0);
    }
    return cudaGetLastError();
}

}  // namespace bioem
