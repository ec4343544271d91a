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
// Pass 2 runs one CTF behind on the other G_T buffer, as HALF-TASKS: thread = (row pair, residue), the radix stage along l (two
// real rows per complex transform, Hermitian completion on load) for the even or the odd dx, one 16-point transform, Horner
// sums -> B(dx, dy), scored at once (a5: form C2; a6: running log-sum-exp + K best).
//
// Warp plan: 16 warps x 128 registers = the whole register file, 4 warps on each of the SM's 4 schedulers (the register
// file is per scheduler: a 5th warp on one of them would cap every thread at 96 registers).  Every warp does both passes;
// what a CTF step costs is set by its busiest warp, so the 28 pass-1 tasks (4 columns x 7 residues = 28 lanes) and the 16
// pass-2 half-tasks (4 row pairs, one dx parity) are dealt as evenly as whole tasks allow.  Scheduler k = warp % 4 carries
//   warp k      (A): pass-1 tasks k, 4 + k                                        2.0  (units of one pass-1 task)
//   warp 4 + k  (B): pass-1 tasks 8 + k, 12 + k;  pass-2 task 4 + k, even dx      2.7
//   warp 8 + k  (C): pass-1 tasks 16 + k, 20 + k; pass-2 task 4 + k, odd dx       2.7
//   warp 12 + k (D): pass-1 task 24 + k;          pass-2 task k, both parities    2.6
// (round 2 measured dedicated pass-1 / pass-2 warps first: 12 x {3, 2, 2} tasks + 4 x 2 whole pass-2 tasks -- the step then
// runs at the pace of a 3.1-unit warp while eight 2-unit warps sleep a third of the time; an earlier capture of this round, not kept.)
// TMEM columns per quadrant: 128 + 128 + 128 + 64 of 512.  Hand-over of G_T: a "full" mbarrier per buffer (16 arrivals: every
// warp after its last pass-1 store of the step) and an "empty" one (12 arrivals: the warps with pass-2 work after their last
// G_T load).  No CTA barrier in the loop, no float atomics, fixed reduction orders: bit-reproducible.
#include "pk_math.cuh"

namespace bioem {

struct TM {
    static constexpr int N = 224, NCOLP = 112, NTASK = 28;        // packed columns (column 0 carries the Nyquist column l = 112); tasks of 4 columns
    static constexpr int NW = 16, NT = NW * 32, NCONS = 12;       // warps; warps that consume G_T (B, C, D)
    static constexpr int ZP = 18, ZW = 32 * ZP;                   // Z tile: one row of 16 outputs per lane (pitch even: 16-byte rows; lanes 28..31 carry zeros)
    static constexpr int RP = 66, GSZ = (NCOLP + 1) * RP;               // G_T [column][row'] pitch (even: 16-byte row pairs; 8 RP = 16 mod 128: the mirrored loads of pass 2 are conflict-free)
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
// The wait names the registers the loads fill, so that their uses depend on it; without a "memory" clobber the compiler may move
// shared-memory loads and stores across it (a slot's Horner sums overlap the TMEM latency of its radix stage).
__device__ __forceinline__ void tm_wait_ld(uint32_t (&a)[8], uint32_t (&b)[8])
{
    asm volatile("tcgen05.wait::ld.sync.aligned;"
                 : "+r"(a[0]), "+r"(a[1]), "+r"(a[2]), "+r"(a[3]), "+r"(a[4]), "+r"(a[5]), "+r"(a[6]), "+r"(a[7]), "+r"(b[0]), "+r"(b[1]), "+r"(b[2]),
                   "+r"(b[3]), "+r"(b[4]), "+r"(b[5]), "+r"(b[6]), "+r"(b[7]));
}
__device__ __forceinline__ void tm_wait_st() { asm volatile("tcgen05.wait::st.sync.aligned;" ::: "memory"); }

// Usually the phase is already complete.  A warp that is early sleeps between probes: mbarrier.try_wait, with or without a
// suspend-time hint, compiles to a probe loop that returns every ~25 cycles and took 20 % of the issue slots (an earlier capture of this round, not kept).
__device__ __forceinline__ void tm_mbar_wait(uint64_t *bar, unsigned parity)
{
    const unsigned b = (unsigned)__cvta_generic_to_shared(bar);
    if (pk_mbar_test(b, parity)) return;
    do { __nanosleep(200); } while (!pk_mbar_test(b, parity));
}

// H-phase of a tile (rows 8 cw + t, 16 outputs k1' each): lane = (e, c2) forms, for the TWO columns (or row pairs) 2 c2 and
// 2 c2 + 1, the two outputs that share k1' = e: k_lo = k1 - 32 and k_hi = k1.  y[2 i + 0 | 1] = sum_t r_lo^t | r_hi^t z[2 c2 + i][t].
// Horner from t = 6, four chains interleaved (a chain alone is 12 dependent FFMA2); the two chains of a column share its loads,
// and the two half-warps read different columns, so every shared-memory wavefront is used once (with lane = output and 4 columns
// per lane both half-warps fetched the same 128 bytes: twice the wavefronts (an earlier capture of this round, not kept)).
__device__ __forceinline__ void tm_horner7x4(c2 (&y)[4], const c2 *zc, c2 r_lo, c2 r_hi)
{
#pragma unroll
    for (int i = 0; i < 2; ++i) { const c2 z = zc[(8 * i + 6) * TM::ZP]; y[2 * i] = z; y[2 * i + 1] = z; }
#pragma unroll
    for (int t = 5; t >= 0; --t)
#pragma unroll
        for (int i = 0; i < 2; ++i) {
            const c2 z = zc[(8 * i + t) * TM::ZP];
            y[2 * i] = pk_cmadd(y[2 * i], r_lo, z);
            y[2 * i + 1] = pk_cmadd(y[2 * i + 1], r_hi, z);
        }
}

// The four pass-1 outputs of a lane -> rows of G_T.  Lanes whose output index lies outside |k| <= D do not store (predicated
// stores: a dummy address for them put a second wavefront on every store, profiles/r2_tm_v8_fused_paper_stride16_full.csv).
// `unpack` (the lanes of warp 0 that hold packed column 0): y = G(., 0) + i G(., 112), both parts real -> two real columns
// (0 and 112 of G_T), so that pass 2 reads column 0 and the Nyquist column like any other: no special case in its load loop.
__device__ __forceinline__ void tm_store_rows(c2 *g_lo, c2 *g_hi, bool v_lo, bool v_hi, const c2 (&y)[4], bool unpack = false)
{
    if (unpack) {
        if (v_lo) { g_lo[0] = make_float2(y[0].x, 0.f); g_lo[112 * TM::RP] = make_float2(y[0].y, 0.f); g_lo[TM::RP] = y[2]; }
        if (v_hi) { g_hi[0] = make_float2(y[1].x, 0.f); g_hi[112 * TM::RP] = make_float2(y[1].y, 0.f); g_hi[TM::RP] = y[3]; }
        return;
    }
    if (v_lo) { g_lo[0] = y[0]; g_lo[TM::RP] = y[2]; }
    if (v_hi) { g_hi[0] = y[1]; g_hi[TM::RP] = y[3]; }
}

// a5 + a6 for the 8 correlations a lane holds after the H-phase of a pass-2 tile: y[2 i + u] = (B(dx_u, row' 2 p), B(dx_u, row' 2 p + 1))
// of row pair p = pA + i, at dx_0 = k_lo, dx_1 = k_hi.  rho^2 = B^2 alpha^2 beta^2; g = cA log1p(-rho^2) + h (form C2, base-2 units);
// log1p(-x) = -x (1 + x/2 + x^2/3 + x^3/4 + x^4/5) for x < 2^-6 (truncation < 2e-10 relative).
// The running sum is s 2^m with m a REFERENCE exponent, not the maximum: the common path is branch-free (8 ex2, no rescaling)
// and one warp vote sends the warp to the careful path when some lane is near the posterior peak (accurate log1pf), holds a
// candidate for the K best, or exceeds the reference by more than 2^64 (re-reference; keeps s far from overflow).
// A dx outside the range passes ok_lo / ok_hi = false; rows' beyond 2 D are masked per value.  Fixed order: bit-reproducible.
struct TmGeom { int D, KK, De, Do, n_even; };
struct TmScore { c2 x2[4], g2[4], h2[4]; bool careful; };
// the arithmetic: straight-line
__device__ __forceinline__ void tm_score_math(TmScore &sc, const FusedParams &p, const PkLse &st, const c2 (&y)[4], int pA, bool ok_lo, bool ok_hi,
                                              const TmGeom &gm, float ab, float hterm)
{
    const float hlo = ok_lo ? hterm : -CUDART_INF_F, hhi = ok_hi ? hterm : -CUDART_INF_F;
#pragma unroll
    for (int c = 0; c < 4; ++c) {
        const int r0 = 2 * (pA + (c >> 1));
        const float hl = (c & 1) ? hhi : hlo;
        sc.h2[c] = make_float2(r0 < gm.KK ? hl : -CUDART_INF_F, r0 + 1 < gm.KK ? hl : -CUDART_INF_F);
        const c2 r = __fmul2_rn(y[c], pk_bc(ab));
        sc.x2[c] = __fmul2_rn(r, r);                                  // rho^2
        c2 q = __ffma2_rn(sc.x2[c], pk_bc(0.2f), pk_bc(0.25f));
        q = __ffma2_rn(sc.x2[c], q, pk_bc(0.33333334f));
        q = __ffma2_rn(sc.x2[c], q, pk_bc(0.5f));
        q = __ffma2_rn(sc.x2[c], q, pk_bc(1.0f));
        sc.g2[c] = __ffma2_rn(__fmul2_rn(sc.x2[c], q), pk_bc(-p.cA), sc.h2[c]);
    }
    const c2 (&x2)[4] = sc.x2, (&g2)[4] = sc.g2;
    const float xmax = fmaxf(fmaxf(fmaxf(x2[0].x, x2[0].y), fmaxf(x2[1].x, x2[1].y)), fmaxf(fmaxf(x2[2].x, x2[2].y), fmaxf(x2[3].x, x2[3].y)));
    const float gmax = fmaxf(fmaxf(fmaxf(g2[0].x, g2[0].y), fmaxf(g2[1].x, g2[1].y)), fmaxf(fmaxf(g2[2].x, g2[2].y), fmaxf(g2[3].x, g2[3].y)));
    sc.careful = xmax >= 0.015625f || gmax >= st.thr || gmax > st.m + 64.0f;
}
// the careful path: out of line, so that the loop body stays small (instruction cache); scalar arguments and a by-value result
// travel in registers (a struct by reference would live in local memory and be stored before every vote)
template <bool DUMP>
__device__ __noinline__ PkLse tm_score_careful(float cA, float *dump, PkLse st, TopEntry *mylist, float y0, float y1, float y2, float y3, float y4, float y5,
                                               float y6, float y7, float hlo, float hhi, float ab, int pA, int k_lo, int k_hi, int D, int De, int Do,
                                               uint32_t pair)
{
    const int KK = 2 * D + 1, n_even = 2 * De + 1;
    const float yv[8] = {y0, y1, y2, y3, y4, y5, y6, y7};             // value i = 2 c + comp: chain c = 2 (pair index) + (hi ? 1 : 0), comp = row of the pair
    float g[8];
    uint32_t sh[8];
    bool v[8];
#pragma unroll
    for (int i = 0; i < 8; ++i) {
        const int c = i >> 1;
        const int row = 2 * (pA + (c >> 1)) + (i & 1);
        const float h = row < KK ? ((c & 1) ? hhi : hlo) : -CUDART_INF_F;
        const float r = yv[i] * ab;
        const float x = fminf(r * r, 0.99999994f);                    // rho^2, R14 clamp
        float q = fmaf(x, 0.2f, 0.25f);
        q = fmaf(x, q, 0.33333334f);
        q = fmaf(x, q, 0.5f);
        q = fmaf(x, q, 1.0f);
        g[i] = x >= 0.015625f ? fmaf(cA, log1pf(-x), h) : fmaf(x * q, -cA, h);
        v[i] = h > -CUDART_INF_F;
        const int ky = row < n_even ? 2 * row - 2 * De : 2 * (row - n_even) - (2 * Do - 1);
        sh[i] = (uint32_t)((ky + D) * KK + (((c & 1) ? k_hi : k_lo) + D));
        if (DUMP && v[i]) dump[sh[i]] = g[i];
    }
    float gm2 = -CUDART_INF_F;
#pragma unroll
    for (int i = 0; i < 8; ++i) gm2 = fmaxf(gm2, g[i]);
    const float mn = fmaxf(st.m, gm2);                                // finite: st.m starts at LSE_EMPTY
    float acc = 0.f;
#pragma unroll
    for (int i = 0; i < 8; ++i) acc += pk_ex2(g[i] - mn);
    st.s = fmaf(st.s, pk_ex2(st.m - mn), acc);
    st.m = mn;
    if (__any_sync(FULLP, gm2 >= st.thr)) {
#pragma unroll
        for (int i = 0; i < 8; ++i) pk_topk_insert(g[i], pair, sh[i], v[i], st.thr, mylist);
    }
    return st;
}
// the vote and the accumulation
template <bool DUMP>
__device__ __forceinline__ void tm_score_commit(const TmScore &sc, const FusedParams &p, PkLse &st, TopEntry *mylist, const c2 (&y)[4], int pA, int k_lo,
                                                int k_hi, bool ok_lo, bool ok_hi, const TmGeom &gm, float ab, float hterm, uint32_t pair)
{
    if (!DUMP && !__any_sync(FULLP, sc.careful)) {
        const c2 nm = pk_bc(-st.m);
        float acc = 0.f;
#pragma unroll
        for (int c = 0; c < 4; ++c) {
            const c2 e = pk_add(sc.g2[c], nm);
            acc += pk_ex2(e.x) + pk_ex2(e.y);
        }
        st.s += acc;
        return;
    }
    st = tm_score_careful<DUMP>(p.cA, p.dump, st, mylist, y[0].x, y[0].y, y[1].x, y[1].y, y[2].x, y[2].y, y[3].x, y[3].y, ok_lo ? hterm : -CUDART_INF_F,
                                ok_hi ? hterm : -CUDART_INF_F, ab, pA, k_lo, k_hi, gm.D, gm.De, gm.Do, pair);
}

// One pass-1 slot = one basic block: (BACK) the Horner sums over the tile of the PREVIOUS slot (-> rows of G_T at g_lo / g_hi) under
// the TMEM latency of the radix-2 stage of this slot's (CTF, task), then the 16-point transform.
// Radix stage: x_j = Q_j K_j re-read from TMEM; ODD = false: a_j = x_j + x_(j+16); ODD = true: a_j = (x_j - x_(j+16)) w32^j.  The
// next 8-word chunk of Q is in flight under the arithmetic of the current one.
// NYQ: the threads of packed column 0 add i Q(112, m) K(112, m) (both columns are Hermitian in m, so the transform of the sum
// is G(., 0) + i G(., 112) with both parts real).
template <bool ODD, bool NYQ, bool BACK>
__device__ __forceinline__ void tm_p1_slot(c2 (&a)[16], uint32_t qaddr, const float4 (&kq)[8], bool nyq, const c2 *qn, const float *__restrict__ kn,
                                           const c2 *zrd, c2 r_lo, c2 r_hi, c2 *g_lo, c2 *g_hi, bool v_lo, bool v_hi, bool unpack = false)
{
    uint32_t qa[2][8], qb[2][8];
    tm_ld8(qaddr, qa[0]);
    tm_ld8(qaddr + 32, qb[0]);
    if (BACK) {
        c2 y[4];
        tm_horner7x4(y, zrd, r_lo, r_hi);
        tm_store_rows(g_lo, g_hi, v_lo, v_hi, y, unpack);
    }
#pragma unroll
    for (int g = 0; g < 4; ++g) {
        tm_wait_ld(qa[g & 1], qb[g & 1]);
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
            c2 v = __ffma2_rn(B, pk_bc(ODD ? -kb[e] : kb[e]), x);
            if (NYQ && nyq) {
                v = __ffma2_rn(pk_rot90(qn[j * 7]), pk_bc(kn[j * 7]), v);
                v = __ffma2_rn(pk_rot90(qn[(j + 16) * 7]), pk_bc(ODD ? -kn[(j + 16) * 7] : kn[(j + 16) * 7]), v);
            }
            a[j] = ODD ? pk_twid(v, j) : v;
        }
    }
    pk_fft16(a);
}

// Radix-2 stage + 16-point transform of a pass-2 half-task for one row pair: the 224-point transform along l of A + i B (rows'
// 2p, 2p+1 of G_T, one 128-bit word per column; a row' that does not exist is all zero), thread = (pair, residue t),
// l = 7 j + t.  Columns l = 1..111 are stored, l = 113..223 are their conjugates (Hermitian half); columns 0 and 112 are real (pass 1
// unpacks them from packed column 0 on store): both formulas below then give (A.x, B.x).  ODD = false: a_j = x_j + x_(j+16) (even dx); ODD = true: a_j = (x_j - x_(j+16)) w32^j (odd dx).
// (Lane = 8 pair + t and 8 RP = 16 mod 128: the eight lanes of a quarter-warp read eight different 16-byte slots, direct and
// mirrored.)  A warp that does both parities loads twice: keeping the other half in registers spills, and parking it in tensor memory or fetching K after pass 2 instead were both slower (DESIGN 7).
template <bool ODD>
__device__ __forceinline__ void tm_p2_front(c2 (&a)[16], const c2 *gt, int t)
{
    const c2 *gl = gt + t * TM::RP, *gh = gt + (112 - t) * TM::RP;    // low half: l = 7 j + t (direct); high half: l = 112 + 7 j + t -> mirrored column 112 - 7 j - t
#pragma unroll
    for (int j = 0; j < 16; ++j) {
        const float4 vl = *reinterpret_cast<const float4 *>(gl + 7 * j * TM::RP);
        const float4 vh = *reinterpret_cast<const float4 *>(gh - 7 * j * TM::RP);
        // direct: A + i B = (A.x - B.y, A.y + B.x); mirrored: conj(A) + i conj(B) = (A.x + B.y, -A.y + B.x)
        c2 xl = pk_add(make_float2(vl.x, vl.y), make_float2(-vl.w, vl.z));
        c2 xh = pk_add(make_float2(vh.x, -vh.y), make_float2(vh.w, vh.z));
        a[j] = ODD ? pk_twid(pk_sub(xl, xh), j) : pk_add(xl, xh);
    }
    pk_fft16(a);
}

// ORIENT = true (bioem_set_orientation_posterior): the running sums are also closed at the end of every orientation of the work
// item -- each warp reduces its (m, s) over its lanes into otab[orientation][warp] and starts again -- and the epilogue combines
// warps -> orientation (written to p.orient_m / p.orient_s) -> work item, in fixed order.  A template parameter, not a run-time
// flag: the flag in the step loop cost the default path 7 % (DESIGN 7).
template <bool DUMP, bool ORIENT>
__global__ void __launch_bounds__(TM::NT, 1) k_fused_tm(FusedParams p, const float4 *__restrict__ Kt, const float *__restrict__ KtN)
{
    constexpr int N = TM::N, NW = TM::NW, ZP = TM::ZP, ZW = TM::ZW, RP = TM::RP, GSZ = TM::GSZ;
    constexpr size_t H = (size_t)(N / 2 + 1) * N;
    const int D = p.D, KK = 2 * D + 1, NP = D + 1;                    // host guarantees D <= 31; NP row pairs (the last one is a single row)
    const int De = D / 2, Do = (D + 1) / 2, n_even = 2 * De + 1;      // rows' 0..n_even-1: k = -2 De, .., 2 De; then the odd k = -(2 Do - 1), .., 2 Do - 1
    const int tid = threadIdx.x, lane = tid & 31, warp = tid >> 5;

    extern __shared__ __align__(16) unsigned char smem_raw[];
    c2 *Z = reinterpret_cast<c2 *>(smem_raw);                         // [NW][32][ZP]   warp-private tiles
    c2 *G = Z + (size_t)NW * ZW;                                      // [2][112][RP]   G_T: pass-1 outputs of one CTF, all columns, double-buffered
    c2 *qn = G + (size_t)2 * GSZ;                                     // [32][7]        Q of the Nyquist column (warp 0)
    TopEntry *tops = reinterpret_cast<TopEntry *>(qn + 224);    // [NW][TOPK]
    float *red = reinterpret_cast<float *>(tops + NW * BIOEM_TOPK);   // [2 NW]
    float2 *otab = reinterpret_cast<float2 *>(red + 2 * NW);          // [32][NW]       ORIENT only: (m, s) per orientation of the item and warp
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
    for (int i = tid; i < (NW * ZW + 2 * GSZ + 224) * 2; i += TM::NT) reinterpret_cast<float *>(Z)[i] = 0.f;
    if (tid < NW * BIOEM_TOPK) { TopEntry e0 = {-CUDART_INF_F, 0xffffffffu, 0xffffffffu}; tops[tid] = e0; }
    if (tid == 0) {
        for (int i = 0; i < 2; ++i) { pk_mbar_init(&bar_full[i], NW); pk_mbar_init(&bar_empty[i], TM::NCONS); }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    asm volatile("tcgen05.fence::after_thread_sync;" ::: "memory");
    const uint32_t tm_base = tm_base_s;

    // ---- lane roles
    // F-phase: lane = 8 cw + t -> (column or row pair cw of the task, residue t); lanes with t = 7 carry zeros
    const int colw = lane >> 3, t7 = lane & 7;
    const bool has_col = t7 < 7;
    const int t = has_col ? t7 : 0;
    c2 *const Zw = Z + (size_t)warp * ZW, *const zrow = Zw + lane * ZP;
    // H-phase: lane = (e, c2) -> columns (row pairs) 2 c2, 2 c2 + 1 of the tile; outputs k_lo = k1 - 32 and k_hi = k1, k1 = 2 e (+ 1)
    const int e16 = lane & 15, c2h = lane >> 4;
    const int kl_ev = 2 * e16 - 32, kh_ev = 2 * e16, kl_od = kl_ev + 1, kh_od = kh_ev + 1;
    const bool vl_ev = -kl_ev <= D, vh_ev = kh_ev <= D, vl_od = -kl_od <= D, vh_od = kh_od <= D;
    const int rl_ev = (kl_ev + 2 * De) / 2, rh_ev = (kh_ev + 2 * De) / 2;                       // rows' (valid outputs only)
    const int rl_od = n_even + (kl_od + 2 * Do - 1) / 2, rh_od = n_even + (kh_od + 2 * Do - 1) / 2;
    c2 wl_ev, wh_ev, wl_od, wh_od;                                    // exp(2 pi i k / N)
    sincospif(2.0f * (float)(kl_ev + N) / (float)N, &wl_ev.y, &wl_ev.x);
    sincospif(2.0f * (float)kh_ev / (float)N, &wh_ev.y, &wh_ev.x);
    sincospif(2.0f * (float)(kl_od + N) / (float)N, &wl_od.y, &wl_od.x);
    sincospif(2.0f * (float)kh_od / (float)N, &wh_od.y, &wh_od.x);
    const c2 *const zrd = Zw + (16 * c2h) * ZP + e16;                 // + (8 i + t) * ZP: residue t of column 2 c2 + i
    // offsets into a G_T buffer of this lane's four pass-1 outputs of a task whose first column is col0: + col0 * RP
    const int gcol = (2 * c2h) * RP;

    const int c_lo = DUMP ? p.dump_ctf : 0, c_hi = DUMP ? p.dump_ctf + 1 : p.n_ctf, ncf = c_hi - c_lo;
    const int S = (o_end - o_begin) * ncf;                            // steps = (orientation, CTF) pairs of this work item
    PkLse st = {LSE_EMPTY, 0.f, -CUDART_INF_F};
    TopEntry *mylist = tops + warp * BIOEM_TOPK;
    const TmGeom gm = {D, KK, De, Do, n_even};

    // ---- this warp's share (see the plan above)
    const int sk = warp & 3, role = warp >> 2;                        // scheduler / TMEM quadrant; 0 A, 1 B, 2 C, 3 D
    const int nt = role == 3 ? 1 : 2;                                 // pass-1 tasks per step: task0, task0 + 4
    const int task0 = 8 * role + sk;
    const int ntask2 = (NP + 3) / 4;                                  // pass-2 tasks of 4 row pairs
    const int q2 = role == 3 ? sk : 4 + sk;                           // the pass-2 task this warp works on (roles B, C, D)
    const bool do_ev = role == 1 || role == 3, do_od = role == 2 || role == 3, cons = role != 0;
    const uint32_t qaddr0 = tm_base + ((uint32_t)(32 * sk) << 16) + (uint32_t)(128 * role);
    const bool warp_nyq = warp == 0, nyq = warp_nyq && lane < 7;
    const bool unpack0 = warp_nyq && c2h == 0;                        // the H-phase lanes whose first column is packed column 0
    const cf *Oimg = p.Ohat + (size_t)img * H;
    const float beta = p.beta[img];
    const float4 *kt_l = Kt + lane;                                   // Kt[c][task 0..27][g 0..7][lane]
    constexpr size_t KSTR = (size_t)TM::NTASK * 8 * 32;               // float4 per CTF
    // pass 2: this thread's row pair (F') of task q2; the pairs this lane scores are pA2, pA2 + 1
    const bool t2act = cons && q2 < ntask2;
    const int pl2 = 4 * q2 + colw, prf2 = (t2act && pl2 < NP) ? pl2 : 0;      // lanes with t7 = 7 read what lane t = 0 of their quarter-warp reads: a broadcast
    const int pA2 = 4 * q2 + 2 * c2h;

    float4 kq[8];
#pragma unroll
    for (int g = 0; g < 8; ++g) kq[g] = __ldg(kt_l + (size_t)c_lo * KSTR + ((size_t)task0 * 8 + g) * 32);
    int o = o_begin, c = c_lo;
    float pab = 0.f, ph = 0.f;                                        // (alpha beta, h, pair index) of the previous step: what pass 2 scores
    uint32_t ppair = 0;
    for (int s = 0; s <= S; ++s) {
        const bool live = s < S;
        const int b = s & 1;
        if (live) {
            // =========================================================================================== pass 1 of step s
            if (c == c_lo) {
                // ---- Q = conj(Ohat) F0 for this thread's bins (Eq. 12), new orientation -> TMEM
                const cf *F0 = p.F0 + ((size_t)model * p.n_orient + o) * H;
                for (int ii = 0; ii < nt; ++ii) {
                    const size_t qbase = (size_t)(4 * (task0 + 4 * ii) + colw) * N + t;
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
                if (warp_nyq) {
                    // the Nyquist column, qn[m] = Q(112, m): all 32 lanes, 7 coalesced loads per array in flight at once (as a loop
                    // of 32 dependent round trips to L2 on 7 lanes it made warp 0 late by ~20 k cycles at every new orientation and
                    // the other 15 warps wait for it: 3 % of the run)
                    cf ov[7], fv[7];
#pragma unroll
                    for (int i = 0; i < 7; ++i) { ov[i] = Oimg[(size_t)(N / 2) * N + lane + 32 * i]; fv[i] = F0[(size_t)(N / 2) * N + lane + 32 * i]; }
#pragma unroll
                    for (int i = 0; i < 7; ++i) { const cf pr = cmulc(ov[i], fv[i]); qn[lane + 32 * i] = make_float2(pr.x, pr.y); }
                }
                tm_wait_st();
                __syncwarp();
            }
            c2 *const Gw = G + (size_t)b * GSZ + gcol;
            for (int i = 0; i < nt; ++i) {
                const int task = task0 + 4 * i, col0 = 4 * task;      // this task: packed columns col0 .. col0 + 3
                // ================= slot E: even outputs of this task  ||  odd-k rows of the warp's previous task of this step -> G_T
                c2 a[16];
                {
                    c2 *gp = Gw + (size_t)(col0 - 16) * RP;
                    c2 *g_lo = gp + rl_od, *g_hi = gp + rh_od;
                    if (i == 0) {
                        if (warp_nyq) tm_p1_slot<false, true, false>(a, qaddr0, kq, nyq, qn + t, KtN + (size_t)c * N + t, zrd, wl_od, wh_od, g_lo, g_hi, vl_od, vh_od);
                        else tm_p1_slot<false, false, false>(a, qaddr0, kq, false, nullptr, nullptr, zrd, wl_od, wh_od, g_lo, g_hi, vl_od, vh_od);
                    } else tm_p1_slot<false, false, true>(a, qaddr0 + 64, kq, false, nullptr, nullptr, zrd, wl_od, wh_od, g_lo, g_hi, vl_od, vh_od, unpack0);
                }
                __syncwarp();                                         // every lane has read the tile
                pk_spill16(zrow, a);
                __syncwarp();
                // ================= slot O: odd outputs  ||  even-k rows of this task -> G_T
                if (i == 0 && s >= 2) tm_mbar_wait(&bar_empty[b], ((unsigned)(s >> 1) & 1u) ^ 1u);   // every consumer has read buffer b (step s - 2)
                {
                    c2 *gp = Gw + (size_t)col0 * RP;
                    c2 *g_lo = gp + rl_ev, *g_hi = gp + rh_ev;
                    if (warp_nyq && i == 0) tm_p1_slot<true, true, true>(a, qaddr0, kq, nyq, qn + t, KtN + (size_t)c * N + t, zrd, wl_ev, wh_ev, g_lo, g_hi, vl_ev, vh_ev, unpack0);
                    else tm_p1_slot<true, false, true>(a, qaddr0 + 64 * i, kq, false, nullptr, nullptr, zrd, wl_ev, wh_ev, g_lo, g_hi, vl_ev, vh_ev);
                }
                {
                    // K of the next task: the next task of this CTF, or the first task of the next CTF (wrapping to c_lo with the next orientation)
                    const bool last = i + 1 == nt;
                    const int cn = last ? (c + 1 < c_hi ? c + 1 : c_lo) : c, tn = last ? task0 : task + 4;
                    const float4 *kp = kt_l + (size_t)cn * KSTR + (size_t)tn * 8 * 32;
#pragma unroll
                    for (int g = 0; g < 8; ++g) kq[g] = __ldg(kp + g * 32);
                }
                __syncwarp();
                pk_spill16(zrow, a);
                __syncwarp();
            }
            {
                // ================= flush: odd-k rows of the last task -> G_T; this warp's share of step s is complete
                c2 *gp = Gw + (size_t)(4 * (task0 + 4 * (nt - 1))) * RP;
                c2 y[4];
                tm_horner7x4(y, zrd, wl_od, wh_od);
                tm_store_rows(gp + rl_od, gp + rh_od, vl_od, vh_od, y);
                __syncwarp();
                if (lane == 0) pk_mbar_arrive(&bar_full[b]);
            }
        }
        // =========================================================================================== pass 2 of step s - 1
        if (s >= 1 && cons) {
            const int b1 = b ^ 1;
            tm_mbar_wait(&bar_full[b1], (unsigned)((s - 1) >> 1) & 1u);    // every warp has stored its part of step s - 1
            const c2 *gt = G + (size_t)b1 * GSZ + 2 * prf2;
#pragma unroll 1
            for (int par = 0; par < 2; ++par) {
                if (!(par ? do_od : do_ev)) continue;
                c2 a[16];
                if (par) tm_p2_front<true>(a, gt, t);
                else tm_p2_front<false>(a, gt, t);
                __syncwarp();                                         // every lane's loads of G_T are done; the tile is free (the flush / the other parity has read it)
                if ((par || !do_od) && lane == 0) pk_mbar_arrive(&bar_empty[b1]);
                pk_spill16(zrow, a);
                __syncwarp();
                c2 y[4];
                tm_horner7x4(y, zrd, par ? wl_od : wl_ev, par ? wh_od : wh_ev);
                TmScore sc;
                tm_score_math(sc, p, st, y, pA2, t2act && (par ? vl_od : vl_ev), t2act && (par ? vh_od : vh_ev), gm, pab, ph);
                tm_score_commit<DUMP>(sc, p, st, mylist, y, pA2, par ? kl_od : kl_ev, par ? kh_od : kh_ev, t2act && (par ? vl_od : vl_ev),
                                      t2act && (par ? vh_od : vh_ev), gm, pab, ph, ppair);
            }
        }
        if (!DUMP && ORIENT && s >= 1 && c == c_lo) {
            // step s - 1 was the last CTF of its orientation: close this warp's sums for it
            float lse_m = st.m, lse_s = st.s;
#pragma unroll
            for (int off = 16; off >= 1; off >>= 1) {
                const float m2 = __shfl_xor_sync(FULLP, lse_m, off), s2 = __shfl_xor_sync(FULLP, lse_s, off);
                const float M = fmaxf(lse_m, m2);
                lse_s = lse_s * pk_ex2(lse_m - M) + s2 * pk_ex2(m2 - M);
                lse_m = M;
            }
            if (lane == 0) otab[(o - 1 - o_begin) * NW + warp] = make_float2(lse_m, lse_s);
            st.m = LSE_EMPTY; st.s = 0.f;
        }
        if (live) {
            const size_t moc = ((size_t)model * p.n_orient + o) * p.n_ctf + c;
            pab = p.alpha[moc] * beta; ph = p.hterm[moc];
            ppair = (uint32_t)((o + p.o_first) * p.n_ctf + c);
            if (++c >= c_hi) { c = c_lo; ++o; }
        }
    }
    asm volatile("tcgen05.fence::before_thread_sync;" ::: "memory");
    __syncthreads();
    if (warp == 0) asm volatile("tcgen05.dealloc.cta_group::1.sync.aligned.b32 %0, 512;" ::"r"(tm_base) : "memory");
    if (DUMP) return;

    // ---- block reduction, fixed order
    if (ORIENT) {
        // warps -> orientation: thread i of warp 0 combines the NW entries of orientation i in warp order and writes its (m, s);
        // (m, s), kept in otab[i * NW]: the work item's partial below is then the combination of its orientations, in order
        const int n_or = o_end - o_begin;
        if (warp == 0 && lane < n_or) {
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
// Kt[c][task][g][lane] (float4; task = 0..27, g = 0..7): K_c(l = 4 task + lane / 8, m = 7 (4 g + e) + lane % 8), e = 0..3;
// lanes with lane % 8 = 7 have no column: zeros.  KtN[c][7 j + t] = K_c(l = 112, m = 7 j + t).
__global__ void k_relayout_K_tm(const float *K32, float4 *Kt, float *KtN, int n_ctf)
{
    constexpr int N = TM::N, PER = TM::NTASK * 8 * 32;
    const int c = blockIdx.y, i = blockIdx.x * blockDim.x + threadIdx.x;       // i = (task * 8 + g) * 32 + lane
    if (i >= PER) return;
    const int lane = i & 31, g = (i >> 5) & 7, task = i >> 8;
    const float *Kc = K32 + (size_t)c * (N / 2 + 1) * N;
    float v[4] = {0.f, 0.f, 0.f, 0.f};
    if ((lane & 7) < 7) {
        const int l = 4 * task + (lane >> 3), t = lane & 7;
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
    const bool orient = p.orient_m != nullptr && !dump;
    const size_t bytes = ((size_t)TM::NW * TM::ZW + 2 * TM::GSZ + 224) * 8 + (size_t)TM::NW * BIOEM_TOPK * sizeof(TopEntry) + 2 * TM::NW * 4 + 64 +
                         (orient ? (size_t)32 * TM::NW * sizeof(float2) : 0);
    if (orient && p.oc > 32) return cudaErrorInvalidValue;            // otab holds 32 orientations per work item
    const float4 *kt = reinterpret_cast<const float4 *>(Kt);
    const float *ktn = tm_ktn(Kt, p.n_ctf);
    cudaError_t e;
    if (dump) {
        e = cudaFuncSetAttribute(k_fused_tm<true, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        k_fused_tm<true, false><<<1, TM::NT, bytes, st>>>(p, kt, ktn);
    } else if (orient) {
        e = cudaFuncSetAttribute(k_fused_tm<false, true>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        const int items = p.n_img * p.n_model * p.chunks_per_model;
        k_fused_tm<false, true><<<items, TM::NT, bytes, st>>>(p, kt, ktn);
    } else {
        e = cudaFuncSetAttribute(k_fused_tm<false, false>, cudaFuncAttributeMaxDynamicSharedMemorySize, (int)bytes);
        if (e != cudaSuccess) return e;
        const int items = p.n_img * p.n_model * p.chunks_per_model;
        k_fused_tm<false, false><<<items, TM::NT, bytes, st>>>(p, kt, ktn);
    }
    return cudaGetLastError();
}

}  // namespace bioem
