// fft_pk.cuh -- two-way packed complex64 line FFT for sm_100a (FADD2 / FMUL2 / FFMA2).
//
// Blackwell's packed fp32 instructions do two fp32 operations per issue slot (same lane throughput as
// the scalar forms, half the instructions).  A line of N points is split by one radix-2 step into two
// independent half-length transforms with identical structure and twiddles (even / odd outputs for
// decimation in frequency, even / odd inputs for decimation in time); the two halves travel through
// the radix-32 register butterflies as the two lanes of every packed operation:
//
//   C2 { x = (re_a, re_b), y = (im_a, im_b) }         a, b = the two half-length transforms
//
// so one instruction stream of a half-length FFT transforms the whole line, and each exchange through
// shared memory moves a 16-byte (a, b) pair per access.  A line is held by T = N / 64 threads with 64
// points each: 32 packed pairs in the half transforms, 64 scalar complex values at the radix-2 step.
//
//   layout L1 ("natural"): v[e]  = x[t + T e],               e  < 64  (8-byte coalesced access)
//   layout L2 ("paired") : p[e]  = (x[2 j], x[2 j + 1]), j = t + T e, e < 32
//
//   forward DIF : L1 in  -> L2 out        forward DIT : L2 in -> L1 out
//   inverse     : the forward transform on (im, re)-swapped data (a register renaming)
//
// The half-length transform is H = N / 2 = 32 x R2 points (R2 = 4 .. 32): one radix-32 butterfly per
// thread, ONE exchange, NB2 = 32 / R2 radix-R2 butterflies.  Twiddles are fp64-built table values.
//
// Implements the transforms of PAPER.md:80 (Eq. 2: FFT / inverse FFT around the propagator).
#pragma once
#include <cuda_runtime.h>

namespace prism {
namespace pk {

struct C2 { float2 x, y; };      // x: real parts of (a, b); y: imaginary parts of (a, b)

__device__ __forceinline__ float2 neg2(float2 a) { return make_float2(-a.x, -a.y); }
__device__ __forceinline__ float2 add2(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 sub2(float2 a, float2 b) { return __fadd2_rn(a, neg2(b)); }
__device__ __forceinline__ float2 mul2(float2 a, float2 b) { return __fmul2_rn(a, b); }
__device__ __forceinline__ float2 fma2(float2 a, float2 b, float2 c) { return __ffma2_rn(a, b, c); }
__device__ __forceinline__ float2 bc(float c) { return make_float2(c, c); }

__device__ __forceinline__ C2 cadd(C2 a, C2 b) { return { add2(a.x, b.x), add2(a.y, b.y) }; }
__device__ __forceinline__ C2 csub(C2 a, C2 b) { return { sub2(a.x, b.x), sub2(a.y, b.y) }; }
__device__ __forceinline__ C2 cadd_mi(C2 a, C2 b) { return { add2(a.x, b.y), sub2(a.y, b.x) }; }   // a + (-i) b
__device__ __forceinline__ C2 csub_mi(C2 a, C2 b) { return { sub2(a.x, b.y), add2(a.y, b.x) }; }   // a - (-i) b
__device__ __forceinline__ C2 cswap(C2 a) { return { a.y, a.x }; }
// a * (wr + i wi), the same factor for both lanes
__device__ __forceinline__ C2 cmulc(C2 a, float wr, float wi)
{
    return { fma2(a.x, bc(wr), mul2(a.y, bc(-wi))), fma2(a.x, bc(wi), mul2(a.y, bc(wr))) };
}
// a * w with separate factors for the two lanes: wr = (wr_a, wr_b), wi = (wi_a, wi_b)
__device__ __forceinline__ C2 cmul2(C2 a, float2 wr, float2 wi)
{
    return { fma2(a.x, wr, neg2(mul2(a.y, wi))), fma2(a.x, wi, mul2(a.y, wr)) };
}
// conj(a) * w
__device__ __forceinline__ C2 cmul2_conj(C2 a, float2 wr, float2 wi)
{
    return { fma2(a.x, wr, mul2(a.y, wi)), fma2(a.x, wi, neg2(mul2(a.y, wr))) };
}

template <int R> struct Dft;

template <> struct Dft<1> { __device__ __forceinline__ static void run(C2*) {} };

template <> struct Dft<2> {
    __device__ __forceinline__ static void run(C2* a)
    { C2 t = a[0]; a[0] = cadd(t, a[1]); a[1] = csub(t, a[1]); }
};

template <> struct Dft<4> {
    __device__ __forceinline__ static void run(C2* a)
    {
        const C2 t0 = cadd(a[0], a[2]), t1 = csub(a[0], a[2]);
        const C2 t2 = cadd(a[1], a[3]), d = csub(a[1], a[3]);
        a[0] = cadd(t0, t2); a[2] = csub(t0, t2);
        a[1] = cadd_mi(t1, d); a[3] = csub_mi(t1, d);
    }
};

template <> struct Dft<8> {
    __device__ __forceinline__ static void run(C2* a)
    {
        const float h = 0.70710678118654752440f;
        C2 e[4] = { a[0], a[2], a[4], a[6] };
        C2 o[4] = { a[1], a[3], a[5], a[7] };
        Dft<4>::run(e); Dft<4>::run(o);
        a[0] = cadd(e[0], o[0]); a[4] = csub(e[0], o[0]);
        {   // o1 * w8, w8 = (1 - i) / sqrt2 :  (h (x + y), h (y - x))
            const float2 p = add2(o[1].x, o[1].y), q = sub2(o[1].y, o[1].x);
            a[1] = { fma2(p, bc(h), e[1].x), fma2(q, bc(h), e[1].y) };
            a[5] = { fma2(p, bc(-h), e[1].x), fma2(q, bc(-h), e[1].y) };
        }
        a[2] = cadd_mi(e[2], o[2]); a[6] = csub_mi(e[2], o[2]);
        {   // o3 * w8^3 = (-1 - i) / sqrt2 :  (h (y - x), -h (x + y))
            const float2 p = add2(o[3].x, o[3].y), q = sub2(o[3].y, o[3].x);
            a[3] = { fma2(q, bc(h), e[3].x), fma2(p, bc(-h), e[3].y) };
            a[7] = { fma2(q, bc(-h), e[3].x), fma2(p, bc(h), e[3].y) };
        }
    }
};

// ---- radix-4 butterfly over twiddled inputs, scaled-twiddle form (both lanes) ---------------------------------
// out = DFT4(z0, y1 w^k1, y2 w^(2 k1), y3 w^(3 k1)), w = exp(-2 pi i / R), R = 16 or 32.  Each twiddle is written
// w^m = (-i)^q cos(t) (1 - i tan(t)) with q the nearest quarter turn and |t| <= pi/4: u = (-i)^q y (1 - i tan) costs two
// FFMA2 -- the quarter turn is a renaming -- and the cosines ride on the adds of the butterfly, which become FFMA2 at
// the same cost:  z1 + z3 = c1 (u1 + (c3 / c1) u3),  z0 + z2 = z0 + c2 u2,  out = t0 + c1 S ...
// 22 packed instructions instead of 28 (three complex multiplies + 16 adds).
template <int R> __device__ __forceinline__ constexpr int tw_q(int m)
{ return (m % (R / 4) == R / 8) ? m / (R / 4) : (m + R / 8) / (R / 4); }
// a * (-i)^q
__device__ __forceinline__ C2 rotq(C2 a, int q)
{
    switch (q & 3) {
        case 1: return { a.y, neg2(a.x) };
        case 2: return { neg2(a.x), neg2(a.y) };
        case 3: return { neg2(a.y), a.x };
        default: return a;
    }
}
template <int R>
__device__ __forceinline__ void twiddled_dft4(C2 z0, C2 y1, C2 y2, C2 y3, int k1, C2& o0, C2& o1, C2& o2, C2& o3)
{
    static_assert(R == 16 || R == 32, "tables");
    // cos and tan of 2 pi j / R for j = -R/8 .. R/8
    constexpr float C16[5] = { 0.70710678118654752440f, 0.92387953251128675613f, 1.f, 0.92387953251128675613f,
                               0.70710678118654752440f };
    constexpr float T16[5] = { -1.f, -0.41421356237309504880f, 0.f, 0.41421356237309504880f, 1.f };
    constexpr float C32[9] = { 0.70710678118654752440f, 0.83146961230254523708f, 0.92387953251128675613f,
                               0.98078528040323044913f, 1.f, 0.98078528040323044913f, 0.92387953251128675613f,
                               0.83146961230254523708f, 0.70710678118654752440f };
    constexpr float T32[9] = { -1.f, -0.66817863791929891999f, -0.41421356237309504880f, -0.19891236737965800691f, 0.f,
                               0.19891236737965800691f, 0.41421356237309504880f, 0.66817863791929891999f, 1.f };
    const C2 y[4] = { z0, y1, y2, y3 };
    C2 u[4];
    float c[4] = { 1.f, 1.f, 1.f, 1.f };
#pragma unroll
    for (int n2 = 1; n2 < 4; ++n2) {
        const int m = n2 * k1, q = tw_q<R>(m), j = m - q * (R / 4);
        const float tau = R == 16 ? T16[j + 2] : T32[j + 4];
        c[n2] = R == 16 ? C16[j + 2] : C32[j + 4];
        const C2 v = y[n2];
        const C2 w = (j == 0) ? v : C2{ fma2(v.y, bc(tau), v.x), fma2(v.x, bc(-tau), v.y) };   // v (1 - i tan)
        u[n2] = rotq(w, q);
    }
    const C2 t0 = { fma2(u[2].x, bc(c[2]), z0.x), fma2(u[2].y, bc(c[2]), z0.y) };
    const C2 t1 = { fma2(u[2].x, bc(-c[2]), z0.x), fma2(u[2].y, bc(-c[2]), z0.y) };
    const float r = c[3] / c[1];
    const C2 sp = { fma2(u[3].x, bc(r), u[1].x), fma2(u[3].y, bc(r), u[1].y) };      // (z1 + z3) / c1
    const C2 dm = { fma2(u[3].x, bc(-r), u[1].x), fma2(u[3].y, bc(-r), u[1].y) };    // (z1 - z3) / c1
    o0 = { fma2(sp.x, bc(c[1]), t0.x), fma2(sp.y, bc(c[1]), t0.y) };
    o2 = { fma2(sp.x, bc(-c[1]), t0.x), fma2(sp.y, bc(-c[1]), t0.y) };
    o1 = { fma2(dm.y, bc(c[1]), t1.x), fma2(dm.x, bc(-c[1]), t1.y) };                // t1 + (-i) c1 dm
    o3 = { fma2(dm.y, bc(-c[1]), t1.x), fma2(dm.x, bc(c[1]), t1.y) };
}

template <> struct Dft<16> {
    __device__ __forceinline__ static void run(C2* a)
    {
        // n = 4 n1 + n2 ; k = k1 + 4 k2.  Y[n2][k1] = DFT4 over n1, then twiddle w16^(n2 k1), DFT4 over n2.
        C2 y[4][4];
#pragma unroll
        for (int n2 = 0; n2 < 4; ++n2) {
            y[n2][0] = a[n2]; y[n2][1] = a[n2 + 4]; y[n2][2] = a[n2 + 8]; y[n2][3] = a[n2 + 12];
            Dft<4>::run(y[n2]);
        }
        {
            C2 z[4] = { y[0][0], y[1][0], y[2][0], y[3][0] };
            Dft<4>::run(z);
            a[0] = z[0]; a[4] = z[1]; a[8] = z[2]; a[12] = z[3];
        }
#pragma unroll
        for (int k1 = 1; k1 < 4; ++k1)
            twiddled_dft4<16>(y[0][k1], y[1][k1], y[2][k1], y[3][k1], k1, a[k1], a[k1 + 4], a[k1 + 8], a[k1 + 12]);
    }
};

template <> struct Dft<32> {
    __device__ __forceinline__ static void run(C2* a)
    {
        // n = 4 n1 + n2 (n1 < 8, n2 < 4); k = k1 + 8 k2.  Y[n2][k1] = DFT8 over n1, twiddle w32^(n2 k1), DFT4 over n2.
        C2 y[4][8];
#pragma unroll
        for (int n2 = 0; n2 < 4; ++n2) {
#pragma unroll
            for (int n1 = 0; n1 < 8; ++n1) y[n2][n1] = a[4 * n1 + n2];
            Dft<8>::run(y[n2]);
        }
        {
            C2 z[4] = { y[0][0], y[1][0], y[2][0], y[3][0] };
            Dft<4>::run(z);
            a[0] = z[0]; a[8] = z[1]; a[16] = z[2]; a[24] = z[3];
        }
#pragma unroll
        for (int k1 = 1; k1 < 8; ++k1)
            twiddled_dft4<32>(y[0][k1], y[1][k1], y[2][k1], y[3][k1], k1, a[k1], a[k1 + 8], a[k1 + 16], a[k1 + 24]);
    }
};

// ---- half-length transform: H = 32 x R2 points by T = H / 32 threads, 32 packed pairs per thread ------
template <int N_>
struct PkPlan {
    static constexpr int N = N_, H = N_ / 2, T = N_ / 64, R1 = 32, R2 = H / 32, NB2 = 32 / R2;
    static_assert(N_ >= 256 && N_ <= 2048 && (N_ & (N_ - 1)) == 0, "line length");
    static constexpr int XPAD = H + H / 32;                 // exchange space of one line, in C2 (16-byte) units
    static constexpr int TW2 = (R2 - 1) * 32;               // stage-2 twiddles w_H^(r k), float2 each
    static constexpr int TWN = H;                           // radix-2 twiddles w_N^n, n < N / 2
    static constexpr int TW_BYTES = (TW2 + TWN) * 8;
};

// tables in shared memory: t2[(r - 1) * 32 + k] = w_H^(r k) (k < 32, r < R2), tn[n] = w_N^n (n < N / 2);
// tw_n is the caller's table exp(-2 pi i m / N), m < N.  Every thread of the CTA calls fill().
template <class P>
__device__ __forceinline__ void fill_tables(float2* table, const float2* __restrict__ tw_n, int tid, int nthreads)
{
    for (int i = tid; i < P::TW2; i += nthreads) {
        const int r = i / 32 + 1, k = i % 32;
        table[i] = __ldg(tw_n + ((2 * r * k) & (P::N - 1)));          // w_H^(r k) = w_N^(2 r k)
    }
    for (int i = tid; i < P::TWN; i += nthreads) table[P::TW2 + i] = __ldg(tw_n + i);
}

// Exchange space views.  Element idx is an (a, b) pair of complex values.
// Xchg16: one 16-byte word (re_a, re_b, im_a, im_b) at base[(idx + idx / 32) * stride].
struct Xchg16 {
    static constexpr bool TWO_PHASE = false;
    float4* base;
    int stride;
    __device__ __forceinline__ void st(int idx, C2 v) const
    { base[(idx + (idx >> 5)) * stride] = make_float4(v.x.x, v.x.y, v.y.x, v.y.y); }
    __device__ __forceinline__ C2 ld(int idx) const
    { const float4 q = base[(idx + (idx >> 5)) * stride]; return { make_float2(q.x, q.y), make_float2(q.z, q.w) }; }
};
// Xchg8: two 8-byte words, the real parts at base[(idx + idx / 32) * stride] and the imaginary parts `plane`
// words further on (keeps the packed register pairs free of 16-byte alignment constraints: fewer MOVs, twice
// the shared-memory instructions).
struct Xchg8 {
    static constexpr bool TWO_PHASE = false;
    float2* base;
    int stride, plane;
    __device__ __forceinline__ void st(int idx, C2 v) const
    { float2* q = base + (idx + (idx >> 5)) * stride; q[0] = v.x; q[plane] = v.y; }
    __device__ __forceinline__ C2 ld(int idx) const
    { const float2* q = base + (idx + (idx >> 5)) * stride; return { q[0], q[plane] }; }
};

// XchgPhase: one 8-byte plane used twice -- real parts first, imaginary parts after a barrier (half the space,
// two more barriers per transform; the row pass uses it to fit one more warp per SM).
struct XchgPhase {
    static constexpr bool TWO_PHASE = true;
    float2* base;
    int stride;
    __device__ __forceinline__ void st(int idx, float2 v) const { base[(idx + (idx >> 5)) * stride] = v; }
    __device__ __forceinline__ float2 ld(int idx) const { return base[(idx + (idx >> 5)) * stride]; }
};

// Forward half-length transforms of both lanes: p[e] holds element t + T e (layout in = layout out).
// SYNC() is a barrier among (at least) the threads of the line; the function begins with one, so the
// exchange space may alias storage those threads have just read.
// LEAD_SYNC = false: the caller guarantees that barrier already (nothing has touched the exchange space since).
template <class P, bool LEAD_SYNC = true, class SM, class SYNC>
__device__ __forceinline__ void fft_half(C2 (&p)[32], const float2* __restrict__ t2, int t, const SM& sm, SYNC sync)
{
    constexpr int T = P::T;
    if (LEAD_SYNC) sync();
    Dft<32>::run(p);
    if constexpr (SM::TWO_PHASE) {
#pragma unroll
        for (int r = 0; r < 32; ++r) sm.st(t * 32 + r, p[r].x);
        sync();
#pragma unroll
        for (int e = 0; e < 32; ++e) p[e].x = sm.ld(t + T * e);
        sync();
#pragma unroll
        for (int r = 0; r < 32; ++r) sm.st(t * 32 + r, p[r].y);
        sync();
#pragma unroll
        for (int e = 0; e < 32; ++e) p[e].y = sm.ld(t + T * e);
    } else {
#pragma unroll
        for (int r = 0; r < 32; ++r) sm.st(t * 32 + r, p[r]);
        sync();
#pragma unroll
        for (int e = 0; e < 32; ++e) p[e] = sm.ld(t + T * e);
    }
#pragma unroll
    for (int m = 0; m < P::NB2; ++m) {
        C2 a[P::R2];
        const int k = (t + T * m) & 31;
        a[0] = p[m];
#pragma unroll
        for (int r = 1; r < P::R2; ++r) {
            const float2 w = t2[(r - 1) * 32 + k];
            a[r] = cmulc(p[m + P::NB2 * r], w.x, w.y);
        }
        Dft<P::R2>::run(a);
#pragma unroll
        for (int r = 0; r < P::R2; ++r) p[m + P::NB2 * r] = a[r];
    }
}

// Band description of a length-N axis in layout L1: slot e (element t + T e) is kept iff e < XBE or e >= 64 - XBE.
// XBE = 32 keeps everything.
template <int XBE> __device__ __forceinline__ constexpr bool kept(int e) { return e < XBE || e >= 64 - XBE; }

// Radix-2 step of the DIF form: v (L1; slots not kept<IN>() are taken as exact zeros) -> p (pairs (a, b) whose
// half-length transforms are the even and the odd outputs).  CONJ: the step runs on conj(v) (an inverse transform is
// the conjugate of the forward transform of the conjugate; the signs fold into the adds).
template <class P, int IN, bool CONJ = false>
__device__ __forceinline__ void dif_pre(const float2 (&v)[64], C2 (&p)[32], const float2* __restrict__ tab, int t)
{
    const float2* tn = tab + P::TW2;
    constexpr float S = CONJ ? -1.f : 1.f;
#pragma unroll
    for (int e = 0; e < 32; ++e) {
        const float2 w = tn[t + P::T * e];                       // w_N^n, n = t + T e
        float2 a, d;
        if (kept<IN>(e) && kept<IN>(e + 32)) {
            a = make_float2(v[e].x + v[e + 32].x, S * v[e].y + S * v[e + 32].y);
            d = make_float2(v[e].x - v[e + 32].x, S * v[e].y - S * v[e + 32].y);
        } else if (kept<IN>(e)) { a = make_float2(v[e].x, S * v[e].y); d = a; }
        else if (kept<IN>(e + 32)) { a = make_float2(v[e + 32].x, S * v[e + 32].y); d = make_float2(-a.x, -a.y); }
        else { a = make_float2(0.f, 0.f); d = a; }
        const float2 b = make_float2(fmaf(d.x, w.x, -d.y * w.y), fmaf(d.x, w.y, d.y * w.x));
        p[e] = { make_float2(a.x, b.x), make_float2(a.y, b.y) };
    }
}

// Radix-2 step of the DIT form: p (half-length transforms of the even and odd inputs) -> v (L1); only slots
// kept<OUT>() are computed.
template <class P, int OUT>
__device__ __forceinline__ void dit_post(const C2 (&p)[32], float2 (&v)[64], const float2* __restrict__ tab, int t)
{
    const float2* tn = tab + P::TW2;
#pragma unroll
    for (int e = 0; e < 32; ++e) {
        if (!kept<OUT>(e) && !kept<OUT>(e + 32)) continue;
        const float2 w = tn[t + P::T * e];                       // w_N^k, k = t + T e
        const float2 a = make_float2(p[e].x.x, p[e].y.x), b = make_float2(p[e].x.y, p[e].y.y);
        const float2 bw = make_float2(fmaf(b.x, w.x, -b.y * w.y), fmaf(b.x, w.y, b.y * w.x));
        if (kept<OUT>(e)) v[e] = make_float2(a.x + bw.x, a.y + bw.y);
        if (kept<OUT>(e + 32)) v[e + 32] = make_float2(a.x - bw.x, a.y - bw.y);
    }
}

// Forward DIF: v (L1) -> p (L2 pairs).
template <class P, int IN, class SM, class SYNC>
__device__ __forceinline__ void fft_dif(const float2 (&v)[64], C2 (&p)[32], const float2* __restrict__ tab, int t,
                                        const SM& sm, SYNC sync)
{
    dif_pre<P, IN>(v, p, tab, t);
    fft_half<P>(p, tab, t, sm, sync);
}

// Forward DIT: p (L2 pairs) -> v (L1).
template <class P, int OUT, class SM, class SYNC>
__device__ __forceinline__ void fft_dit(C2 (&p)[32], float2 (&v)[64], const float2* __restrict__ tab, int t,
                                        const SM& sm, SYNC sync)
{
    fft_half<P>(p, tab, t, sm, sync);
    dit_post<P, OUT>(p, v, tab, t);
}

}  // namespace pk
}  // namespace prism
