// fused_tm.cu -- the hot loop for N = 224 (the paper's box size), D <= 31:
// ONE CTA per SM with Q = conj(Ohat) F0 resident in TENSOR MEMORY, warp-specialised into pass-1 and pass-2 warps.
//
// Why tensor memory: at 224^2 the half spectrum is 113 x 224 complex = 202 KB.  It fits neither the register file next to a
// transform's working set nor shared memory next to the Z / G tiles -- but the SM has a third 256 KB store, TMEM, which
// tcgen05.ld / tcgen05.st (shape 32x32b) expose as 512 private 32-bit words per (warp quadrant, lane): measured on this pool
// at > 800 B/clk/SM with ~50 cycles latency (shared memory: 128 B/clk).  No tensor-core instruction is issued: the path has
// no dense contraction at the precision the parity bar needs (DESIGN 7).  Each pass-1 thread keeps the bins of Q it owns
// (32 per task) in TMEM for the C CTF sets of an orientation (the CTF loop inside the orientation loop), so per CTF
// only the real table K_c streams from L2 (Eq. 5) and nothing of the product conj(Ohat) F0 K_c (Eq. 12) ever
// touches shared or global memory.
//
// Factorisation 224 = 32 x 7: pass-1 thread = (packed column l, residue t), m = 7 j + t.  The 32-point transform over j is a
// radix-2 stage and two 16-point register transforms: slot E forms u_j = x_j + x_(j+16) (even outputs k1), slot O forms
// v_j = (x_j - x_(j+16)) w32^j (odd outputs); x = Q K is RECOMPUTED from TMEM in slot O instead of being parked anywhere.
// After each 16-point transform the warp spills its 28 x 16 outputs to a warp-private Z tile and, one slot later, forms ONLY
// the |k| <= D outputs of every column by 7-term Horner sums (lane = output index), storing them as rows of G_T (transposed,
// rows grouped by parity of k so that a warp's store is one contiguous run).  Each slot is one basic block
// [radix stage + FFT16 in registers || Horner sums over the tile of the previous slot]: shared-memory latency hides under
// register arithmetic inside a warp, not only across warps.
// Pass-2 warps run one CTF behind on the other G_T buffer: thread = (row pair, residue), the same two slots along l (two real
// rows per complex transform, Hermitian completion on load), Horner sums -> B(dx, dy), scored at once (a5: form C2; a6:
// running log-sum-exp + K best).  Hand-over of G_T between the 12 pass-1 and 4 pass-2 warps: a "full" and an "empty"
// mbarrier per buffer, one arrival per warp, waits by mbarrier.try_wait (the hardware suspends the warp; no polling loop in
// the issue slots).  No CTA barrier in the loop, no float atomics, fixed reduction orders: bit-reproducible.
//
// Warp plan: 16 warps x 128 registers = the whole register file, 4 warps on each of the SM's 4 schedulers (the register
// file is per scheduler: a 5th warp on one of them would cap every thread at 96 registers).  The 112 packed columns are 28
// tasks of 4 columns x 7 residues (28 lanes of a warp); pass-1 warp w (0..11) takes tasks w, w + 12 and, for w < 4, w + 24:
// every scheduler carries 7 pass-1 tasks and one pass-2 warp (2 tasks of 4 row pairs) per CTF.  TMEM columns per quadrant:
// 192 + 128 + 128 of 512.
#include "pk_math.cuh"

namespace bioem {

struct TM {
    static constexpr int N = 224, NCOLP = 112, NTASK = 28;        // packed columns (column 0 carries the Nyquist column l = 112); tasks of 4 columns
    static constexpr int NW1 = 12, NW2 = 4, NW = NW1 + NW2, NT = NW * 32;
    static constexpr int ZP = 18, ZW = 28 * ZP;                   // Z tile: one row of 16 outputs per lane with a column (pitch even: 16-byte rows)
    static constexpr int RP = 62, GSZ = NCOLP * RP;               // G_T [column][row'] pitch (even: 16-byte row pairs)
};

// ---- tensor memory as per-thread scratch (32x32b: thread i of warp w owns lane 32 (w % 4) + i, all 512 columns)
__device__ __forceinline__ void tm_ld8(uint32_t taddr, uint32_t (&r)[8])
{
    asm volatile("tcgen05.ld.sync.aligned.32x32b.x8.b32 {%0,%1,%2,%3,%4,%5,%6,%7}, [%8];"
                 : "=r"(r[0]), "=r"(r[1]), "=r"(r[2]), "=r"(r[3]), "=r"(r[4]), "=r"(r[5]), "=r"(r[6]), "=r"(r[7]) : "r"(taddr));
}
__device__ __forceinline__ void tm_st8(uint32_t taddr, const uint32_t (&r)[8])
{
    asm volatile("tcgen05.st.sync.aligned.32x32b.x8.b32 [%0], {%1,%2,%3,%4,%5,%6,%7,%8};" ::"r"(taddr), "r"(r[0]), "r"(r[1]), "r"(r[2]), "r"(r[3]),
                 "r"(r[4]), "r"(r[5]), "r"(r[6]), "r"(r[7]) : "memory");
}
__device__ __forceinline__ void tm_wait_ld() { asm volatile("tcgen05.wait::ld.sync.aligned;" ::: "memory"); }
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// the hardware suspends the warp until the phase completes or a time limit passes; no sleep / poll instructions in between
__device__ __forceinline__ void tm_mbar_wait(uint64_t *bar, unsigned parity)
{
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "TM_WAIT:\n"
        "mbarrier.try_wait.parity.shared::cta.b64 P1, [%0], %1;\n"
        "@P1 bra TM_DONE;\n"
        "bra TM_WAIT;\n"
        "TM_DONE:\n"
        "}" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(parity) : "memory");
}

// y = sum_t r^t z[t], t = 0..6 (Horner from t = 6); z[t] at zc[t * ZP]
__device__ __forceinline__ c2 tm_horner7(const c2 *zc, c2 r)
{
    c2 y = zc[6 * TM::ZP];
#pragma unroll
    for (int t = 5; t >= 0; --t) y = pk_cmadd(y, r, zc[t * TM::ZP]);
    return y;
}

// Radix-2 stage of pass 1 for one (CTF, task): x_j = Q_j K_j re-read from TMEM; ODD = false: a_j = x_j + x_(j+16);
// ODD = true: a_j = (x_j - x_(j+16)) w32^j.  The next 8-word chunk of Q is in flight under the arithmetic of the current one.
// NYQ: the threads of packed column 0 add i Q(112, m) K(112, m) (both columns are Hermitian in m, so the transform of the sum
// is G(., 0) + i G(., 112) with both parts real).
template <bool ODD, bool NYQ>
__device__ __forceinline__ void tm_p1_radix(c2 (&a)[16], uint32_t qaddr, const float4 (&kq)[8], bool nyq, const c2 *qn, const float *__restrict__ kn)
{
    uint32_t qa[2][8], qb[2][8];
    tm_ld8(qaddr, qa[0]);
    tm_ld8(qaddr + 32, qb[0]);
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        tm_wait_ld();
        if (g < 3) {
            tm_ld8(qaddr + 8 * (g + 1), qa[(g + 1) & 1]);
            tm_ld8(qaddr + 32 + 8 * (g + 1), qb[(g + 1) & 1]);
        }
        const float ka[4] = {kq[g].x, kq[g].y, kq[g].z, kq[g].w}, kb[4] = {kq[g + 4].x, kq[g + 4].y, kq[g + 4].z, kq[g + 4].w};
#pragma unroll
        for (int e = 0; e < 4; ++e) {
            const int j = 4 * g + e;
            const c2 A = make_float2(__uint_as_float(qa[g & 1][2 * e]), __uint_as_float(qa[g & 1][2 * e + 1]));
            const c2 B = make_float2(__uint_as_float(qb[g & 1][2 * e]), __uint_as_float(qb[g & 1][2 * e + 1]));
            const c2 x = __fmul2_rn(A, pk_bc(ka[e]));
            c2 r = __ffma2_rn(B, pk_bc(ODD ? -kb[e] : kb[e]), x);
            if (NYQ && nyq) {
                r = __ffma2_rn(pk_rot90(qn[j * 7]), pk_bc(kn[j * 7]), r);
                r = __ffma2_rn(pk_rot90(qn[(j + 16) * 7]), pk_bc(ODD ? -kn[(j + 16) * 7] : kn[(j + 16) * 7]), r);
            }
            a[j] = ODD ? pk_twid(r, j) : r;
        }
    }
}

// Radix-2 stage of pass 2 for one row pair: the 224-point transform along l of A + i B (rows' 2p, 2p+1 of G_T, one 128-bit
// word per column), thread = (pair, residue t), l = 7 j + t.  Columns l = 1..111 are stored, l = 113..223 are their
// conjugates (Hermitian half); packed column 0 holds (G(., 0), G(., 112)), both real.  a_j = x_j + x_(j+16) feeds the even
// outputs now; d_j = x_j - x_(j+16) waits in registers for the odd ones.
__device__ __forceinline__ void tm_p2_radix(c2 (&a)[16], c2 (&d)[16], const c2 *gt, int t, float bsel)
{
    const c2 bs = pk_bc(bsel);
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        // low half: l = 7 j + t (direct); high half: l = 112 + 7 j + t -> mirrored column 112 - 7 j - t
        const int cl = 7 * j + t, ch = (j == 0 && t == 0) ? 0 : 112 - 7 * j - t;
        const float4 vl = *reinterpret_cast<const float4 *>(gt + (size_t)cl * TM::RP);
        const float4 vh = *reinterpret_cast<const float4 *>(gt + (size_t)ch * TM::RP);
        // direct: A + i B = (A.x - B.y, A.y + B.x); mirrored: conj(A) + i conj(B) = (A.x + B.y, -A.y + B.x)
        c2 xl = __ffma2_rn(make_float2(-vl.w, vl.z), bs, make_float2(vl.x, vl.y));
        c2 xh = __ffma2_rn(make_float2(vh.w, vh.z), bs, make_float2(vh.x, -vh.y));
        if (j == 0 && t == 0) {                           // packed column: l = 0 -> (A.x, B.x), l = 112 -> (A.y, B.y)
            xl = make_float2(vl.x, bsel * vl.z);
            xh = make_float2(vl.y, bsel * vl.w);
        }
        a[j] = pk_add(xl, xh);
        d[j] = pk_sub(xl, xh);
    }
}

template <bool DUMP>
__global__ void __launch_bounds__(TM::NT, 1) k_fused_tm(FusedParams p, const float4 *__restrict__ Kt, const float *__restrict__ KtN)
{
    constexpr int N = TM::N, NW1 = TM::NW1, NW2 = TM::NW2, ZP = TM::ZP, ZW = TM::ZW, RP = TM::RP, GSZ = TM::GSZ;
    constexpr size_t H = (size_t)(N / 2 + 1) * N;
    const int D = p.D, KK = 2 * D + 1, NP = D + 1;                    // host guarantees D <= 31; NP row pairs (the last one is a single row)
    const int De = D / 2, Do = (D + 1) / 2, n_even = 2 * De + 1;      // rows' 0..n_even-1: k = -2 De, .., 2 De; then the odd k = -(2 Do - 1), .., 2 Do - 1
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    c2 *Z = reinterpret_cast<c2 *>(smem_raw);                         // [NW][28][ZP]   warp-private tiles
    c2 *G = Z + (size_t)TM::NW * ZW;                                  // [2][112][RP]   G_T: pass-1 outputs of one CTF, all columns, double-buffered
    c2 *qn = G + (size_t)2 * GSZ;                                     // [32][7]        Q of the Nyquist column (warp 0)
    TopEntry *tops = reinterpret_cast<TopEntry *>(qn + 224);          // [NW2][TOPK]
    float *red = reinterpret_cast<float *>(tops + NW2 * BIOEM_TOPK);  // [2 NW2]
    __shared__ uint64_t bar_full[2], bar_empty[2];
    __shared__ uint32_t tm_base_s;

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
    if (warp == 0) {
        asm volatile("tcgen05.alloc.cta_group::1.sync.aligned.shared::cta.b32 [%0], 512;" ::"r"((unsigned)__cvta_generic_to_shared(&tm_base_s)) : "memory");
        asm volatile("tcgen05.relinquish_alloc_permit.cta_group::1.sync.aligned;" ::: "memory");
    }
    for (int i = tid; i < (TM::NW * ZW + 2 * GSZ + 224) * 2; i += TM::NT) reinterpret_cast<float *>(Z)[i] = 0.f;
    if (tid < NW2 * BIOEM_TOPK) { TopEntry e0 = {-CUDART_INF_F, 0xffffffffu, 0xffffffffu}; tops[tid] = e0; }
    if (tid == 0) {
        for (int i = 0; i < 2; ++i) { pk_mbar_init(&bar_full[i], NW1); pk_mbar_init(&bar_empty[i], NW2); }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tm_base = tm_base_s;

    // ---- lane roles shared by both kinds of warp
    const bool has_col = lane < 28;                                   // F-phase: lane -> (column or row pair lane / 7, residue lane % 7)
    const int colw = has_col ? lane / 7 : 0, t = has_col ? lane % 7 : 0;
    c2 *const Zw = Z + (size_t)warp * ZW, *const zrow = Zw + (has_col ? lane : 0) * ZP;
    // H-phase: lane = (e, h) -> outputs k = 2 e - 32 (1 - h) (tile of even k1) and k + 1 (tile of odd k1)
    const int e16 = lane & 15, hh = lane >> 4;
    const int k_ev = 2 * e16 - 32 * (1 - hh), k_od = k_ev + 1;
    const bool v_ev = abs(k_ev) <= D, v_od = abs(k_od) <= D;
    const int row_ev = v_ev ? (k_ev + 2 * De) / 2 : 0, row_od = v_od ? n_even + (k_od + 2 * Do - 1) / 2 : 0;
    c2 r_ev, r_od;
    sincospif(2.0f * (float)(k_ev + N) / (float)N, &r_ev.y, &r_ev.x);
    sincospif(2.0f * (float)(k_od + N) / (float)N, &r_od.y, &r_od.x);
    const c2 *const zrd = Zw + e16;                                   // + (cw * 7 + t) * ZP

    const int c_lo = DUMP ? p.dump_ctf : 0, c_hi = DUMP ? p.dump_ctf + 1 : p.n_ctf, ncf = c_hi - c_lo;
    const int S = (o_end - o_begin) * ncf;                            // steps = (orientation, CTF) pairs of this work item
    PkLse st = {LSE_EMPTY, 0.f, -CUDART_INF_F};

    if (warp < NW1) {
        // =========================================================================================== pass-1 warps
        const int nt = warp < 4 ? 3 : 2;                              // tasks of this warp per CTF: warp, warp + 12 (, warp + 24)
        const int slot = warp >> 2;                                   // 0: 192 TMEM columns from 0; 1, 2: 128 columns from 192, 320
        const uint32_t qaddr0 = tm_base + ((uint32_t)(32 * (warp & 3)) << 16) + (uint32_t)(slot == 0 ? 0 : 64 + 128 * slot);
        const bool warp_nyq = warp == 0, nyq = warp_nyq && lane < 7;
        const cf *Oimg = p.Ohat + (size_t)img * H;
        const float4 *kt_l = Kt + lane;                               // Kt[c][task 0..27][g 0..7][lane]
        constexpr size_t KSTR = (size_t)TM::NTASK * 8 * 32;           // float4 per CTF
        float4 kq[8];
#pragma unroll
        for (int g = 0; g < 8; ++g) kq[g] = __ldg(kt_l + (size_t)c_lo * KSTR + ((size_t)warp * 8 + g) * 32);
        int o = o_begin, c = c_lo, s = 0, i = 0;                      // step s = (o, c); i = index of the warp's task within the step
        int pb = 0, pcol = 0;                                         // buffer and first column of the task whose odd-k outputs are still to be formed
        const int total = nt * S;
        for (int n = 0; n <= total; ++n) {
            const bool live = n < total;
            const int b = s & 1;
            const int task = warp + 12 * i, col0 = 4 * task;          // this task: packed columns col0 .. col0 + 3
            if (live && i == 0 && c == c_lo) {
                // ---- Q = conj(Ohat) F0 for this thread's bins (Eq. 12), new orientation -> TMEM
                const cf *F0 = p.F0 + ((size_t)model * p.n_orient + o) * H;
                for (int ii = 0; ii < nt; ++ii) {
                    const size_t qbase = (size_t)(4 * (warp + 12 * ii) + colw) * N + t;
#pragma unroll
                    for (int g = 0; g < 8; ++g) {
                        uint32_t r[8];
#pragma unroll
                        for (int e = 0; e < 4; ++e) {
                            cf pr = {0.f, 0.f};
                            if (has_col) pr = cmulc(Oimg[qbase + 7 * (4 * g + e)], F0[qbase + 7 * (4 * g + e)]);
                            r[2 * e] = __float_as_uint(pr.x); r[2 * e + 1] = __float_as_uint(pr.y);
                        }
                        tm_st8(qaddr0 + 64 * ii + 8 * g, r);
                    }
                }
                if (nyq) {
                    for (int j = 0; j < 32; ++j) {
                        const size_t e = (size_t)(N / 2) * N + 7 * j + t;
                        const cf pr = cmulc(Oimg[e], F0[e]);
                        qn[7 * j + t] = make_float2(pr.x, pr.y);
                    }
                }
                tm_wait_st();
                __syncwarp();
            }
            // ================= slot E: even outputs of this task  ||  odd-k rows of the previous task -> G_T
            c2 a[16];
            if (live) {
                if (warp_nyq && i == 0) tm_p1_radix<false, true>(a, qaddr0, kq, nyq, qn + t, KtN + (size_t)c * N + t);
                else tm_p1_radix<false, false>(a, qaddr0 + 64 * i, kq, false, nullptr, nullptr);
            } else {
#pragma unroll
                for (int j = 0; j < 16; ++j) a[j] = make_float2(0.f, 0.f);
            }
            if (n > 0) {
                c2 *gc = G + (size_t)pb * GSZ + (size_t)pcol * RP + row_od;
#pragma unroll
                for (int cw = 0; cw < 4; ++cw) {
                    const c2 y = tm_horner7(zrd + cw * 7 * ZP, r_od);
                    if (v_od) gc[cw * RP] = y;
                }
            }
            pk_fft16(a);
            __syncwarp();                                             // every lane has read the tile; its G_T stores are done
            if (n > 0 && i == 0 && lane == 0) pk_mbar_arrive(&bar_full[pb]);     // this warp's share of step s - 1 is complete
            if (!live) break;
            if (has_col) pk_spill16(zrow, a);
            __syncwarp();
            // ================= slot O: odd outputs  ||  even-k rows of this task -> G_T
            if (warp_nyq && i == 0) tm_p1_radix<true, true>(a, qaddr0, kq, nyq, qn + t, KtN + (size_t)c * N + t);
            else tm_p1_radix<true, false>(a, qaddr0 + 64 * i, kq, false, nullptr, nullptr);
            const bool last = i + 1 == nt;
            {
                // K of the next task: the next task of this CTF, or task `warp` of the next CTF (wrapping to c_lo with the next orientation)
                const int cn = last ? (c + 1 < c_hi ? c + 1 : c_lo) : c, tn = last ? warp : task + 12;
                const float4 *kp = kt_l + (size_t)cn * KSTR + (size_t)tn * 8 * 32;
#pragma unroll
                for (int g = 0; g < 8; ++g) kq[g] = __ldg(kp + g * 32);
            }
            if (i == 0 && s >= 2) tm_mbar_wait(&bar_empty[b], ((unsigned)(s >> 1) & 1u) ^ 1u);   // pass 2 has read buffer b (step s - 2)
            {
                c2 *gc = G + (size_t)b * GSZ + (size_t)col0 * RP + row_ev;
#pragma unroll
                for (int cw = 0; cw < 4; ++cw) {
                    const c2 y = tm_horner7(zrd + cw * 7 * ZP, r_ev);
                    if (v_ev) gc[cw * RP] = y;
                }
            }
            pk_fft16(a);
            __syncwarp();
            if (has_col) pk_spill16(zrow, a);
            __syncwarp();
            pb = b; pcol = col0;
            if (last) {
                i = 0; ++s;
                if (++c >= c_hi) { c = c_lo; ++o; }
            } else ++i;
        }
    } else {
        // =========================================================================================== pass-2 warps
        const int w2 = warp - NW1;
        const float beta = p.beta[img];
        TopEntry *mylist = tops + w2 * BIOEM_TOPK;
        const int ntask = (NP + 3) / 4;                               // tasks of 4 row pairs; this warp takes tasks w2 and w2 + NW2
        int o = o_begin, c = c_lo;
        // parameters of the task whose odd-dx outputs are still to be scored
        bool have_prev = false;
        int ppair0 = 0;
        float pab = 0.f, ph = 0.f;
        uint32_t ppairidx = 0;
        for (int s = 0; s <= S; ++s) {
            const bool live = s < S;
            const int b = s & 1;
            float ab = 0.f, hterm = 0.f;
            uint32_t pairidx = 0;
            if (live) {
                const size_t moc = ((size_t)model * p.n_orient + o) * p.n_ctf + c;
                ab = p.alpha[moc] * beta; hterm = p.hterm[moc];
                pairidx = (uint32_t)(o * p.n_ctf + c);
                tm_mbar_wait(&bar_full[b], (unsigned)(s >> 1) & 1u);  // all pass-1 warps have stored their part of step s
            }
            const c2 *Gb = G + (size_t)b * GSZ;
#pragma unroll 1
            for (int qi = 0; qi < 2; ++qi) {
                const int q = w2 + NW2 * qi;                          // task: row pairs 4 q .. 4 q + 3
                const bool tact = live && q < ntask;
                const int pl = 4 * q + colw;                          // this thread's row pair (F')
                const bool pv = has_col && tact && pl < NP;
                const int prf = pv ? pl : 0;
                const float bsel = 2 * prf + 1 < KK ? 1.f : 0.f;
                // ================= slot E': even dx of this task  ||  odd dx of the previous task -> a5, a6
                c2 a[16], d[16];
                if (tact) tm_p2_radix(a, d, Gb + 2 * prf, t, bsel);
                else {
#pragma unroll
                    for (int j = 0; j < 16; ++j) { a[j] = make_float2(0.f, 0.f); d[j] = a[j]; }
                }
                __syncwarp();                                         // every lane's loads of G_T[b] are done before the arrival below
                if (qi == 1 && live && lane == 0) pk_mbar_arrive(&bar_empty[b]);
                if (have_prev) {
#pragma unroll
                    for (int cp = 0; cp < 2; ++cp) {
                        c2 y[2];
                        y[0] = tm_horner7(zrd + (2 * cp) * 7 * ZP, r_od);
                        y[1] = tm_horner7(zrd + (2 * cp + 1) * 7 * ZP, r_od);
                        bool v[4];
                        uint32_t sh[4];
#pragma unroll
                        for (int ii = 0; ii < 4; ++ii) {
                            const int row = 2 * (ppair0 + 2 * cp + (ii >> 1)) + (ii & 1);       // row' of value ii
                            const int ky = row < n_even ? 2 * row - 2 * De : 2 * (row - n_even) - (2 * Do - 1);
                            v[ii] = v_od && row < KK;
                            sh[ii] = (uint32_t)((ky + D) * KK + (k_od + D));
                        }
                        pk_score<DUMP, 4>(p, st, mylist, y, v, sh, pab, ph, ppairidx);
                    }
                }
                pk_fft16(a);
                __syncwarp();
                if (!live && qi == 0) break;                          // drained
                if (has_col) pk_spill16(zrow, a);
                __syncwarp();
                // ================= slot O': odd dx  ||  even dx of this task -> a5, a6
#pragma unroll
                for (int j = 0; j < 16; ++j) a[j] = pk_twid(d[j], j);
                if (tact) {
#pragma unroll
                    for (int cp = 0; cp < 2; ++cp) {
                        c2 y[2];
                        y[0] = tm_horner7(zrd + (2 * cp) * 7 * ZP, r_ev);
                        y[1] = tm_horner7(zrd + (2 * cp + 1) * 7 * ZP, r_ev);
                        bool v[4];
                        uint32_t sh[4];
#pragma unroll
                        for (int ii = 0; ii < 4; ++ii) {
                            const int row = 2 * (4 * q + 2 * cp + (ii >> 1)) + (ii & 1);
                            const int ky = row < n_even ? 2 * row - 2 * De : 2 * (row - n_even) - (2 * Do - 1);
                            v[ii] = v_ev && row < KK;
                            sh[ii] = (uint32_t)((ky + D) * KK + (k_ev + D));
                        }
                        pk_score<DUMP, 4>(p, st, mylist, y, v, sh, ab, hterm, pairidx);
                    }
                }
                pk_fft16(a);
                __syncwarp();
                if (has_col) pk_spill16(zrow, a);
                __syncwarp();
                have_prev = tact; ppair0 = 4 * q; pab = ab; ph = hterm; ppairidx = pairidx;
            }
            if (++c >= c_hi) { c = c_lo; ++o; }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tm_base) : "memory");
    if (DUMP) return;

    // ---- block reduction over the pass-2 warps, fixed order
    if (warp >= NW1) {
        float lse_m = st.m, lse_s = st.s;
#pragma unroll
        for (int off = 16; off >= 1; off >>= 1) {
            const float m2 = __shfl_xor_sync(FULLP, lse_m, off), s2 = __shfl_xor_sync(FULLP, lse_s, off);
            const float M = fmaxf(lse_m, m2);
            lse_s = lse_s * pk_ex2(lse_m - M) + s2 * pk_ex2(m2 - M);
            lse_m = M;
        }
        if (lane == 0) { red[2 * (warp - NW1)] = lse_m; red[2 * (warp - NW1) + 1] = lse_s; }
    }
    __syncthreads();
    if (warp == 0) {
        float m = LSE_EMPTY, s = 0.f;
        for (int w = 0; w < NW2; ++w) {
            const float m2 = red[2 * w], s2 = red[2 * w + 1];
            const float M = fmaxf(m, m2);
            s = s * pk_ex2(m - M) + s2 * pk_ex2(m2 - M);
            m = M;
        }
        if (!(s > 0.f)) m = -CUDART_INF_F;                            // the merge kernel's "empty partial"
        float th0 = tops[BIOEM_TOPK - 1].g;
        for (int w = 1; w < NW2; ++w)
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
// Kt[c][task][g][lane] (float4; task = 0..27, g = 0..7): K_c(l = 4 task + lane / 7, m = 7 (4 g + e) + lane % 7), e = 0..3;
// lanes 28..31 have no column: zeros.  KtN[c][7 j + t] = K_c(l = 112, m = 7 j + t).
__global__ void k_relayout_K_tm(const float *K32, float4 *Kt, float *KtN, int n_ctf)
{
    constexpr int N = TM::N, PER = TM::NTASK * 8 * 32;
    const int c = blockIdx.y, i = blockIdx.x * blockDim.x + threadIdx.x;       // i = (task * 8 + g) * 32 + lane
    if (i >= PER) return;
    const int lane = i & 31, g = (i >> 5) & 7, task = i >> 8;
    const float *Kc = K32 + (size_t)c * (N / 2 + 1) * N;
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    if (lane < 28) {
        const int l = 4 * task + lane / 7, t = lane % 7;
        for (int e = 0; e < 4; ++e) v[e] = Kc[(size_t)l * N + 7 * (4 * g + e) + t];
    }
    Kt[(size_t)c * PER + i] = make_float4(v[0], v[1], v[2], v[3]);
    if (i < N) KtN[(size_t)c * N + i] = Kc[(size_t)(N / 2) * N + i];
}

bool tm_supported(int N, int D) { return N == 224 && D <= 31; }
size_t tm_kt_bytes(int n_ctf) { return (size_t)n_ctf * TM::NTASK * 8 * 32 * 16 + (size_t)n_ctf * TM::N * 4; }
static const float *tm_ktn(const float *Kt, int n_ctf) { return Kt + (size_t)n_ctf * TM::NTASK * 8 * 32 * 4; }

cudaError_t launch_relayout_K_tm(const float *K32, float *Kt, int n_ctf, cudaStream_t st)
{
    dim3 g((TM::NTASK * 8 * 32 + 255) / 256, n_ctf);
    k_relayout_K_tm<<<g, 256, 0, st>>>(K32, reinterpret_cast<float4 *>(Kt), const_cast<float *>(tm_ktn(Kt, n_ctf)), n_ctf);
    return cudaGetLastError();
}

// Work items: one CTA per (image, model, chunk); one partial per work item.
cudaError_t launch_fused_tm(const FusedParams &p, const float *Kt, bool dump, cudaStream_t st)
{
    const size_t bytes = ((size_t)TM::NW * TM::ZW + 2 * TM::GSZ + 224) * 8 + (size_t)TM::NW2 * BIOEM_TOPK * sizeof(TopEntry) + 2 * TM::NW2 * 4 + 64;
    const float4 *kt = reinterpret_cast<const float4 *>(Kt);
    const float *ktn = tm_ktn(Kt, p.n_ctf);
    cudaError_t e;
    if (dump) {
        e = cudaFuncSetAttribute(k_fused_tm<true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        k_fused_tm<true><<<1, TM::NT, bytes, st>>>(p, kt, ktn);
    } else {
        e = cudaFuncSetAttribute(k_fused_tm<false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        const int items = p.n_img * p.n_model * p.chunks_per_model;
        k_fused_tm<false><<<items, TM::NT, bytes, st>>>(p, kt, ktn);
    }
    return cudaGetLastError();
}

}  // namespace bioem
