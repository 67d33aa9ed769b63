// pairs.cuh -- the pair arithmetic shared by the force kernels (walk.cu, hard.cuh): softened monopole
// (Eq. 2), K-weighted pair (Eq. 7-10), and the evaluation of an interaction
// buffer staged in shared memory by a warp that holds S sinks per lane in P copies.
#pragma once
#include "common.cuh"

namespace hyb {

constexpr int WK_SMAX = 4;          // most sinks per lane
constexpr int WK_PAD_SLACK = 64;    // spare buffer entries for padding to a multiple of P U (<= 16 * 4)
constexpr u32 FULL = 0xFFFFFFFFu;

// sink layout by group size (1..64): x = S sinks per lane, y = A lanes per copy, z = P copies,
// w = ceil(32768 / A) for the division of a lane index by A
__constant__ ushort4 c_layout[65];

static void sink_layout(ushort4 *t)
{
    for (int n = 0; n <= 64; n++) {
        if (n == 0) { t[0] = make_ushort4(2, 1, 1, 32768); continue; }
        // maximise n P / (32 S) over S in {2,3,4}; ties go to the larger S
        int S = 2, A = (n + 1) >> 1, P = 32 / A;
        const int A3 = (n + 2) / 3, P3 = 32 / A3, A4 = (n + 3) >> 2, P4 = 32 / A4;
        int best = 6 * P;
        if (4 * P3 >= best) { best = 4 * P3; S = 3; A = A3; P = P3; }
        if (3 * P4 >= best) { S = 4; A = A4; P = P4; }
        if (P > 16) P = 16;               // groups of one or two sinks: keeps the padding step P U <= 64
        t[n] = make_ushort4((unsigned short)S, (unsigned short)A, (unsigned short)P,
                            (unsigned short)((32768 + A - 1) / A));
    }
}

// ---- pair kernels ---------------------------------------------------------------------------
__device__ __forceinline__ float rsqrt_approx(float x)
{
    float r;
    asm("rsqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}
__device__ __forceinline__ float sqrt_approx(float x)
{
    float r;
    asm("sqrt.approx.ftz.f32 %0, %1;" : "=f"(r) : "f"(x));
    return r;
}

// ---- packed FP32 (Blackwell FADD2 / FMUL2 / FFMA2: two IEEE fp32 operations per lane per
// instruction at the same per-flop pipe rate, i.e. half the issue slots).  A "pair" holds the same
// quantity for two sinks of a lane in one 64-bit register pair.
typedef unsigned long long f2;
__device__ __forceinline__ f2 pk(float lo, float hi)
{
    f2 r;
    asm("mov.b64 %0, {%1, %2};" : "=l"(r) : "f"(lo), "f"(hi));
    return r;
}
__device__ __forceinline__ void upk(f2 p, float &lo, float &hi)
{
    asm("mov.b64 {%0, %1}, %2;" : "=f"(lo), "=f"(hi) : "l"(p));
}
__device__ __forceinline__ f2 fma2(f2 a, f2 b, f2 c)
{
    f2 r;
    asm("fma.rn.f32x2 %0, %1, %2, %3;" : "=l"(r) : "l"(a), "l"(b), "l"(c));
    return r;
}
__device__ __forceinline__ f2 add2(f2 a, f2 b)
{
    f2 r;
    asm("add.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}
__device__ __forceinline__ f2 mul2(f2 a, f2 b)
{
    f2 r;
    asm("mul.rn.f32x2 %0, %1, %2;" : "=l"(r) : "l"(a), "l"(b));
    return r;
}

// Sinks of one lane: pair p holds sink slots 2p and 2p+1.  Positions are stored negated so that
// r_j - r_i is one packed add.
struct Sinks {
    f2 nx[2], ny[2], nz[2];       // -x_i
    f2 sx[2], sy[2], sz[2];       // soft (or normal-tree) accumulators
    f2 hx[2], hy[2], hz[2];       // hard accumulators
};

// monopole (Eq. 2) for two sinks: 3 add2 + 3 fma2 + 2 rsqrt + 3 mul2 + 3 fma2
//   = 12 FP32-pipe instructions (24 pipe cycles) + 2 MUFU per pair of interactions
__device__ __forceinline__ void mono2(const float4 s, f2 nx, f2 ny, f2 nz, float eps2, f2 &ax, f2 &ay, f2 &az)
{
    const f2 dx = add2(pk(s.x, s.x), nx), dy = add2(pk(s.y, s.y), ny), dz = add2(pk(s.z, s.z), nz);
    f2 r2 = fma2(dx, dx, pk(eps2, eps2));
    r2 = fma2(dy, dy, r2);
    r2 = fma2(dz, dz, r2);
    float r2a, r2b;
    upk(r2, r2a, r2b);
    const f2 ri = pk(rsqrt_approx(r2a), rsqrt_approx(r2b));
    const f2 ri2 = mul2(ri, ri);
    const f2 mr = mul2(pk(s.w, s.w), ri);
    const f2 mr3 = mul2(mr, ri2);
    ax = fma2(mr3, dx, ax);
    ay = fma2(mr3, dy, ay);
    az = fma2(mr3, dz, az);
}

// the same for the single sink held in the low half of a pair (S = 3)
__device__ __forceinline__ void mono1(const float4 s, f2 nx, f2 ny, f2 nz, float eps2, f2 &ax, f2 &ay, f2 &az)
{
    float x, y, z, a0, a1, a2, t;
    upk(nx, x, t); upk(ny, y, t); upk(nz, z, t);
    float hx, hy, hz;
    upk(ax, a0, hx); upk(ay, a1, hy); upk(az, a2, hz);
    const float dx = s.x + x, dy = s.y + y, dz = s.z + z;
    float r2 = fmaf(dx, dx, eps2);
    r2 = fmaf(dy, dy, r2);
    r2 = fmaf(dz, dz, r2);
    const float ri = rsqrt_approx(r2);
    const float ri2 = ri * ri;
    const float mr = s.w * ri;
    const float mr3 = mr * ri2;
    a0 = fmaf(mr3, dx, a0);
    a1 = fmaf(mr3, dy, a1);
    a2 = fmaf(mr3, dz, a2);
    ax = pk(a0, hx); ay = pk(a1, hy); az = pk(a2, hz);
}

// KF = HYB_K_PAPER: Eq. 10 with Y clamped to [0,1]: K = t^3 (10 - 15 t + 6 t^2), t = Y^2 (T15).
// KF = HYB_K_POLY7 (north_star's alternative, R6): K = 1 - x^4 (35 - 84 x + 70 x^2 - 20 x^3),
// x = (r - r_in)/(r_out - r_in) = 1 - Y on the clamped range.
template <int KF>
__device__ __forceinline__ float kfun(float r, float kc0, float kc1)
{
    const float Y = __saturatef(fmaf(r, kc1, kc0));
    if (KF == HYB_K_POLY7) {
        const float x = 1.0f - Y, x2 = x * x;
        const float poly = fmaf(fmaf(fmaf(-20.0f, x, 70.0f), x, -84.0f), x, 35.0f);
        return fmaf(-(x2 * x2), poly, 1.0f);
    }
    const float t = Y * Y;
    const float poly = fmaf(fmaf(6.0f, t, -15.0f), t, 10.0f);
    return (t * t) * (t * poly);
}

// K-weighted pair (Eq. 8, 9) for two sinks: hard part K F, and (SOFT) the soft part (1 - K) F.
// fused: 25 FP32-pipe instruction equivalents + 4 MUFU per pair of interactions; hard only: 21 + 4.
template <bool SOFT, int KF>
__device__ __forceinline__ void kpair2(const float4 s, f2 nx, f2 ny, f2 nz, float eps2, float kc0, float kc1, f2 &sx,
                                       f2 &sy, f2 &sz, f2 &hx, f2 &hy, f2 &hz)
{
    const f2 dx = add2(pk(s.x, s.x), nx), dy = add2(pk(s.y, s.y), ny), dz = add2(pk(s.z, s.z), nz);
    f2 r2u = mul2(dx, dx);
    r2u = fma2(dy, dy, r2u);
    r2u = fma2(dz, dz, r2u);
    const f2 r2e = add2(r2u, pk(eps2, eps2));
    float ua, ub, ea, eb;
    upk(r2u, ua, ub); upk(r2e, ea, eb);
    const f2 ri = pk(rsqrt_approx(ea), rsqrt_approx(eb));
    const float Ya = __saturatef(fmaf(sqrt_approx(ua), kc1, kc0)), Yb = __saturatef(fmaf(sqrt_approx(ub), kc1, kc0));
    const f2 Y = pk(Ya, Yb);
    f2 K;
    if (KF == HYB_K_POLY7) {
        const f2 x = fma2(Y, pk(-1.0f, -1.0f), pk(1.0f, 1.0f)), x2 = mul2(x, x);
        const f2 poly = fma2(fma2(fma2(pk(-20.0f, -20.0f), x, pk(70.0f, 70.0f)), x, pk(-84.0f, -84.0f)), x, pk(35.0f, 35.0f));
        K = fma2(mul2(mul2(x2, x2), pk(-1.0f, -1.0f)), poly, pk(1.0f, 1.0f));
    } else {
        const f2 t = mul2(Y, Y);
        const f2 poly = fma2(fma2(pk(6.0f, 6.0f), t, pk(-15.0f, -15.0f)), t, pk(10.0f, 10.0f));
        K = mul2(mul2(t, t), mul2(t, poly));
    }
    const f2 ri2 = mul2(ri, ri);
    const f2 mr = mul2(pk(s.w, s.w), ri);
    const f2 mr3 = mul2(mr, ri2);
    const f2 wh = mul2(K, mr3);
    hx = fma2(wh, dx, hx);
    hy = fma2(wh, dy, hy);
    hz = fma2(wh, dz, hz);
    if (SOFT) {
        const f2 ws = fma2(wh, pk(-1.0f, -1.0f), mr3);
        sx = fma2(ws, dx, sx);
        sy = fma2(ws, dy, sy);
        sz = fma2(ws, dz, sz);
    }
}

template <bool SOFT, int KF>
__device__ __forceinline__ void kpair1(const float4 s, f2 nx, f2 ny, f2 nz, float eps2, float kc0, float kc1, f2 &sx,
                                       f2 &sy, f2 &sz, f2 &hx, f2 &hy, f2 &hz)
{
    float x, y, z, t;
    upk(nx, x, t); upk(ny, y, t); upk(nz, z, t);
    const float dx = s.x + x, dy = s.y + y, dz = s.z + z;
    float r2u = dx * dx;
    r2u = fmaf(dy, dy, r2u);
    r2u = fmaf(dz, dz, r2u);
    const float ri = rsqrt_approx(r2u + eps2);
    const float r = sqrt_approx(r2u);
    const float ri2 = ri * ri;
    const float mr = s.w * ri;
    const float mr3 = mr * ri2;
    const float wh = kfun<KF>(r, kc0, kc1) * mr3;
    float a0, a1, a2, b0, b1, b2;
    upk(hx, a0, b0); upk(hy, a1, b1); upk(hz, a2, b2);
    hx = pk(fmaf(wh, dx, a0), b0); hy = pk(fmaf(wh, dy, a1), b1); hz = pk(fmaf(wh, dz, a2), b2);
    if (SOFT) {
        const float ws = mr3 - wh;
        upk(sx, a0, b0); upk(sy, a1, b1); upk(sz, a2, b2);
        sx = pk(fmaf(ws, dx, a0), b0); sy = pk(fmaf(ws, dy, a1), b1); sz = pk(fmaf(ws, dz, a2), b2);
    }
}

// Buffer evaluation.  The caller pads the buffer with zero-mass entries to a multiple of P U, so every
// part runs the same number of iterations and an iteration is U S independent pair chains.
// The U sources x (S/2 pairs [+ 1 single]) chains of an iteration are written stage by stage
// (differences, r^2, rsqrt, products, accumulation) so that independent chains are interleaved and
// the FMA pipe is not left waiting on one chain's latency.
template <int S, int U>
__device__ __forceinline__ void eval_mono(const float4 *buf, int cnt, int part, int P, Sinks &k, float eps2)
{
    constexpr int NP = S / 2;
    constexpr bool ODD = (S & 1) != 0;
    if (part >= P) return;
    const float4 *p = buf + part;
    const int step = P * U;
    const f2 EPS = pk(eps2, eps2);
    float ox = 0, oy = 0, oz = 0, oax = 0, oay = 0, oaz = 0, keepx = 0, keepy = 0, keepz = 0;
    if (ODD) {                      // the single sink lives in the low half of pair NP
        float t;
        upk(k.nx[NP], ox, t); upk(k.ny[NP], oy, t); upk(k.nz[NP], oz, t);
        upk(k.sx[NP], oax, keepx); upk(k.sy[NP], oay, keepy); upk(k.sz[NP], oaz, keepz);
    }
    for (int j = 0; j < cnt; j += step, p += step) {
        float4 s[U];
#pragma unroll
        for (int u = 0; u < U; u++) s[u] = p[u * P];
        f2 dx[U][NP > 0 ? NP : 1], dy[U][NP > 0 ? NP : 1], dz[U][NP > 0 ? NP : 1], w[U][NP > 0 ? NP : 1];
        float ex[U], ey[U], ez[U], ew[U];
#pragma unroll
        for (int u = 0; u < U; u++) {
#pragma unroll
            for (int q = 0; q < NP; q++) {
                dx[u][q] = add2(pk(s[u].x, s[u].x), k.nx[q]);
                dy[u][q] = add2(pk(s[u].y, s[u].y), k.ny[q]);
                dz[u][q] = add2(pk(s[u].z, s[u].z), k.nz[q]);
            }
            if (ODD) { ex[u] = s[u].x + ox; ey[u] = s[u].y + oy; ez[u] = s[u].z + oz; }
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
#pragma unroll
            for (int q = 0; q < NP; q++) w[u][q] = fma2(dx[u][q], dx[u][q], EPS);
            if (ODD) ew[u] = fmaf(ex[u], ex[u], eps2);
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
#pragma unroll
            for (int q = 0; q < NP; q++) w[u][q] = fma2(dy[u][q], dy[u][q], w[u][q]);
            if (ODD) ew[u] = fmaf(ey[u], ey[u], ew[u]);
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
#pragma unroll
            for (int q = 0; q < NP; q++) w[u][q] = fma2(dz[u][q], dz[u][q], w[u][q]);
            if (ODD) ew[u] = fmaf(ez[u], ez[u], ew[u]);
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
#pragma unroll
            for (int q = 0; q < NP; q++) {
                float a, b;
                upk(w[u][q], a, b);
                w[u][q] = pk(rsqrt_approx(a), rsqrt_approx(b));
            }
            if (ODD) ew[u] = rsqrt_approx(ew[u]);
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
#pragma unroll
            for (int q = 0; q < NP; q++) {
                const f2 ri2 = mul2(w[u][q], w[u][q]);
                const f2 mr = mul2(pk(s[u].w, s[u].w), w[u][q]);
                w[u][q] = mul2(mr, ri2);
            }
            if (ODD) { const float ri2 = ew[u] * ew[u]; const float mr = s[u].w * ew[u]; ew[u] = mr * ri2; }
        }
#pragma unroll
        for (int u = 0; u < U; u++) {
#pragma unroll
            for (int q = 0; q < NP; q++) {
                k.sx[q] = fma2(w[u][q], dx[u][q], k.sx[q]);
                k.sy[q] = fma2(w[u][q], dy[u][q], k.sy[q]);
                k.sz[q] = fma2(w[u][q], dz[u][q], k.sz[q]);
            }
            if (ODD) { oax = fmaf(ew[u], ex[u], oax); oay = fmaf(ew[u], ey[u], oay); oaz = fmaf(ew[u], ez[u], oaz); }
        }
    }
    if (ODD) { k.sx[NP] = pk(oax, keepx); k.sy[NP] = pk(oay, keepy); k.sz[NP] = pk(oaz, keepz); }
}

template <int S, int U, bool SOFT, int KF>
__device__ __forceinline__ void eval_near(const float4 *buf, int cnt, int part, int P, Sinks &k, float eps2, float kc0,
                                          float kc1)
{
    if (part >= P) return;
    const float4 *p = buf + part;
    const int step = P * U;
    for (int j = 0; j < cnt; j += step, p += step) {
        float4 s[U];
#pragma unroll
        for (int u = 0; u < U; u++) s[u] = p[u * P];
#pragma unroll
        for (int u = 0; u < U; u++) {
#pragma unroll
            for (int q = 0; q < S / 2; q++)
                kpair2<SOFT, KF>(s[u], k.nx[q], k.ny[q], k.nz[q], eps2, kc0, kc1, k.sx[q], k.sy[q], k.sz[q], k.hx[q], k.hy[q],
                             k.hz[q]);
            if (S & 1)
                kpair1<SOFT, KF>(s[u], k.nx[S / 2], k.ny[S / 2], k.nz[S / 2], eps2, kc0, kc1, k.sx[S / 2], k.sy[S / 2],
                             k.sz[S / 2], k.hx[S / 2], k.hy[S / 2], k.hz[S / 2]);
        }
    }
}

// zero-mass entries up to the next multiple of `step` (the buffers have WK_PAD_SLACK spare entries)
__device__ __forceinline__ int pad_buffer(float4 *buf, int cnt, int step, float4 dummy, int lane)
{
    const int padded = ((cnt + step - 1) / step) * step;
    for (int i = cnt + lane; i < padded; i += 32) buf[i] = dummy;
    return padded;
}

__device__ __forceinline__ u32 warp_excl_scan(u32 v, int lane, u32 &total)
{
    u32 incl = v;
#pragma unroll
    for (int off = 1; off < 32; off <<= 1) {
        u32 t = __shfl_up_sync(FULL, incl, off);
        if (lane >= off) incl += t;
    }
    total = __shfl_sync(FULL, incl, 31);
    return incl - v;
}

}  // namespace hyb
