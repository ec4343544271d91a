// pk_math.cuh -- packed f32x2 complex arithmetic, the 16-point register transform, the a5/a6 scoring step and the
// shared-memory mbarrier helpers shared by the fused kernels (fused_pk.cu: N = 64, 128; fused_c2.cu: N = 224).
#pragma once
#include "common.cuh"
#include <math_constants.h>

namespace bioem {

typedef float2 c2;
static constexpr unsigned FULLP = 0xffffffffu;
static constexpr float LSE_EMPTY = -3.0e38f;          // "no term yet": finite, so the running log-sum-exp needs no branch


// ---- packed complex helpers (each maps to ONE sm_100a instruction; swizzles / negations fold into the operands)
__device__ __forceinline__ c2 pk_add(c2 a, c2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ c2 pk_sub(c2 a, c2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
__device__ __forceinline__ c2 pk_bc(float s) { return make_float2(s, s); }
__device__ __forceinline__ c2 pk_rot90(c2 a) { return make_float2(-a.y, a.x); }                                   // i a
__device__ __forceinline__ c2 pk_cmul(c2 a, c2 w) { return __ffma2_rn(pk_rot90(a), pk_bc(w.y), __fmul2_rn(a, pk_bc(w.x))); }       // a w
__device__ __forceinline__ c2 pk_cmadd(c2 a, c2 w, c2 z) { return __ffma2_rn(pk_rot90(a), pk_bc(w.y), __ffma2_rn(a, pk_bc(w.x), z)); }   // a w + z

// a * exp(+2 pi i K32 / 32), K32 a compile-time constant after unrolling
__device__ __forceinline__ c2 pk_twid(c2 a, int K32)
{
    if (K32 == 0) return a;
    if (K32 == 8) return pk_rot90(a);
    float c, s;
    if (K32 < 8) { c = (float)cos32(K32); s = (float)cos32(8 - K32); }
    else         { c = -(float)cos32(16 - K32); s = (float)cos32(K32 - 8); }
    return __ffma2_rn(pk_rot90(a), pk_bc(s), __fmul2_rn(a, pk_bc(c)));
}

// in-place 16-point DIF, y[k] = sum_j a[j] exp(+2 pi i j k / 16); on return a[r] = y[bitrev4(r)]
__device__ __forceinline__ void pk_fft16(c2 (&a)[16])
{
#pragma unroll
    for (int half = 8; half >= 1; half /= 2)
#pragma unroll
        for (int base = 0; base < 16; base += 2 * half)
#pragma unroll
            for (int j = 0; j < half; ++j) {
                const c2 u = a[base + j], v = a[base + j + half];
                a[base + j] = pk_add(u, v);
                a[base + j + half] = pk_twid(pk_sub(u, v), j * (16 / half));
            }
}

// spill the bit-reversed FFT output as 8 16-byte stores: (a[r], a[r+8]) = (y[2b], y[2b+1]), b = bitrev3(r)
__device__ __forceinline__ void pk_spill16(c2 *zst, const c2 (&a)[16])
{
#pragma unroll
    for (int r = 0; r < 8; ++r) {
        const int b = bitrev(r, 3);
        *reinterpret_cast<float4 *>(zst + 2 * b) = make_float4(a[r].x, a[r].y, a[r + 8].x, a[r + 8].y);
    }
}


__device__ __forceinline__ float pk_ex2(float x)
{
    float y;
    asm("ex2.approx.ftz.f32 %0, %1;" : "=f"(y) : "f"(x));
    return y;
}

__device__ __forceinline__ bool pk_entry_before(float ga, uint32_t pa, uint32_t sa, float gb, uint32_t pb, uint32_t sb)
{   // ranking: larger g first; ties -> lower flat index (pair, shift) first (R15)
    return ga > gb || (ga == gb && (pa < pb || (pa == pb && sa < sb)));
}

// Insert the candidates of the lanes with `valid && g >= thr` into this warp's sorted K-list (shared memory).
__device__ __forceinline__ void pk_topk_insert(float g, uint32_t pair, uint32_t sh, bool valid, float &thr, TopEntry *list)
{
    unsigned m = __ballot_sync(FULLP, valid && g >= thr);
    const int lane = threadIdx.x & 31;
    while (m) {
        const int src = __ffs(m) - 1;
        m &= m - 1;
        const float gv = __shfl_sync(FULLP, g, src);
        const uint32_t pv = __shfl_sync(FULLP, pair, src), sv = __shfl_sync(FULLP, sh, src);
        TopEntry e = {0.f, 0u, 0u};
        if (lane < BIOEM_TOPK) e = list[lane];
        const bool before = lane < BIOEM_TOPK && pk_entry_before(e.g, e.pair, e.shift, gv, pv, sv);
        const int pos = __popc(__ballot_sync(FULLP, before));          // sorted list: the entries ranked before form a prefix
        if (pos < BIOEM_TOPK) {
            __syncwarp();
            if (lane >= pos && lane < BIOEM_TOPK - 1) list[lane + 1] = e;
            if (lane == pos) { TopEntry n = {gv, pv, sv}; list[pos] = n; }
            __syncwarp();
            thr = list[BIOEM_TOPK - 1].g;
        }
    }
}

struct PkLse { float m, s, thr; };


// a5 + a6 for the NV (2 or 4) correlations a lane holds: b[i] = (B(dx_i, dy_A), B(dx_i, dy_B)).
// log1p(-x) = -x (1 + x/2 + x^2/3 + x^3/4 + x^4/5) for x < 2^-6 (truncation < 2e-10 relative); the accurate routine runs
// only when some lane of the warp is near the posterior peak.
template <bool DUMP, int NV>
__device__ __forceinline__ void pk_score(const FusedParams &p, PkLse &st, TopEntry *mylist, const c2 (&b)[NV / 2], const bool (&v)[NV],
                                         const uint32_t (&sh)[NV], float ab, float hterm, uint32_t pair)
{
    c2 x2[NV / 2], g2[NV / 2];
    float xmax = 0.f;
#pragma unroll
    for (int i = 0; i < NV / 2; ++i) {
        const c2 r = __fmul2_rn(b[i], pk_bc(ab));
        x2[i] = __fmul2_rn(r, r);                                               // rho^2
        xmax = fmaxf(xmax, fmaxf(x2[i].x, x2[i].y));
        c2 q = __ffma2_rn(x2[i], pk_bc(0.2f), pk_bc(0.25f));
        q = __ffma2_rn(x2[i], q, pk_bc(0.33333334f));
        q = __ffma2_rn(x2[i], q, pk_bc(0.5f));
        q = __ffma2_rn(x2[i], q, pk_bc(1.0f));
        g2[i] = __ffma2_rn(__fmul2_rn(x2[i], q), pk_bc(-p.cA), pk_bc(hterm));   // form C2, base-2 units
    }
    float g[NV];
#pragma unroll
    for (int i = 0; i < NV / 2; ++i) { g[2 * i] = g2[i].x; g[2 * i + 1] = g2[i].y; }
    if (__any_sync(FULLP, xmax >= 0.015625f)) {
#pragma unroll
        for (int i = 0; i < NV; ++i) {
            const float x = fminf((i & 1) ? x2[i / 2].y : x2[i / 2].x, 0.99999994f);      // R14 clamp
            if (x >= 0.015625f) g[i] = fmaf(p.cA, log1pf(-x), hterm);
        }
    }
    float gmax = -CUDART_INF_F;
#pragma unroll
    for (int i = 0; i < NV; ++i) {
        if (DUMP && v[i]) p.dump[sh[i]] = g[i];
        g[i] = v[i] ? g[i] : -CUDART_INF_F;
        gmax = fmaxf(gmax, g[i]);
    }
    const float mn = fmaxf(st.m, gmax);                                         // finite: st.m starts at LSE_EMPTY
    float acc = pk_ex2(g[0] - mn) + pk_ex2(g[1] - mn);
    if (NV == 4) acc += pk_ex2(g[2] - mn) + pk_ex2(g[3] - mn);
    st.s = fmaf(st.s, pk_ex2(st.m - mn), acc);
    st.m = mn;
    if (__any_sync(FULLP, gmax >= st.thr)) {
#pragma unroll
        for (int i = 0; i < NV; ++i) pk_topk_insert(g[i], pair, sh[i], v[i], st.thr, mylist);
    }
}

// 16-byte asynchronous global -> shared copy (LDGSTS); completion is awaited by the issuing thread itself
__device__ __forceinline__ void pk_cp_async16(void *smem_dst, const void *gsrc)
{
    const unsigned d = (unsigned)__cvta_generic_to_shared(smem_dst);
    asm volatile("cp.async.cg.shared.global [%0], [%1], 16;" ::"r"(d), "l"(gsrc) : "memory");
}
__device__ __forceinline__ void pk_cp_async_commit() { asm volatile("cp.async.commit_group;" ::: "memory"); }
__device__ __forceinline__ void pk_cp_async_wait_all() { asm volatile("cp.async.wait_group 0;" ::: "memory"); }

// ---- split-phase CTA synchronisation on shared-memory mbarriers (one arrival per warp): a warp ARRIVES when its part of a
// hand-over is done and WAITS only where it needs the other warps' part, so warps drift by up to a slot instead of meeting
// at a CTA barrier once per group.
__device__ __forceinline__ void pk_mbar_init(uint64_t *bar, int count)
{
    asm volatile("mbarrier.init.shared::cta.b64 [%0], %1;" ::"r"((unsigned)__cvta_generic_to_shared(bar)), "r"(count) : "memory");
}
__device__ __forceinline__ void pk_mbar_arrive(uint64_t *bar)
{
    asm volatile("mbarrier.arrive.shared::cta.b64 _, [%0];" ::"r"((unsigned)__cvta_generic_to_shared(bar)) : "memory");
}
__device__ __forceinline__ bool pk_mbar_test(unsigned bar, unsigned parity)
{
    unsigned ok;
    asm volatile(
        "{\n"
        ".reg .pred P1;\n"
        "mbarrier.test_wait.parity.shared::cta.b64 P1, [%1], %2;\n"
        "selp.u32 %0, 1, 0, P1;\n"
        "}" : "=r"(ok) : "r"(bar), "r"(parity) : "memory");
    return ok != 0;
}
// Usually the phase is already complete (the wait sits about a slot after the last arrival).  A warp that is early -- the
// warps without a pass-2 task are -- sleeps between probes instead of spinning in the issue slots of its scheduler.
__device__ __forceinline__ void pk_mbar_wait(uint64_t *bar, unsigned parity)
{
    const unsigned b = (unsigned)__cvta_generic_to_shared(bar);
    while (!pk_mbar_test(b, parity)) __nanosleep(200);
}

}  // namespace bioem
