// fft_core.cuh -- register-resident complex64 line FFT for sm_100a.
//
// One line of N points is transformed by T = N/E threads holding E points each
// in registers (thread t holds x[t + T*e], e = 0..E-1, so global loads and stores
// of a contiguous line are coalesced 8-byte accesses).  The transform is a
// Stockham autosort FFT in up to three radix stages (N = R1*R2*R3); between
// stages the threads of the line exchange data through shared memory, whose
// index space is padded (idx + idx/16) so that both the strided writes and the
// contiguous reads are bank-conflict free for 8-byte words.  Output is in
// natural order and lands in the same register layout as the input, so an
// inverse transform can follow a forward one with no extra exchange.
//
// Inter-stage twiddles are exact table values (fp64-built w_N^m, rounded once to
// fp32) that each thread loads ONCE into registers: they depend on the thread's
// position in the line, not on the line.
//
// The inverse transform is the forward one on (im, re)-swapped data.
//
// Implements the transforms of PAPER.md:80 (Eq. 2 needs FFT / inverse FFT around
// the propagator) and PAPER.md:128 ("the modulus squared of its FFT").
#pragma once
#include <cuda_runtime.h>

namespace prism {

#ifndef PRISM_PACKED_ADDS
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return make_float2(a.x + b.x, a.y + b.y); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return make_float2(a.x - b.x, a.y - b.y); }
#else
// sm_100a packed fp32: one FADD2 per complex add (same rounding as two FADDs, half the issue slots)
__device__ __forceinline__ float2 cadd(float2 a, float2 b) { return __fadd2_rn(a, b); }
__device__ __forceinline__ float2 csub(float2 a, float2 b) { return __fadd2_rn(a, make_float2(-b.x, -b.y)); }
#endif
__device__ __forceinline__ float2 cmul(float2 a, float2 b)
{ return make_float2(fmaf(a.x, b.x, -a.y * b.y), fmaf(a.x, b.y, a.y * b.x)); }
__device__ __forceinline__ float2 cmul_conj(float2 a, float2 b)   // a * conj(b)
{ return make_float2(fmaf(a.x, b.x, a.y * b.y), fmaf(a.y, b.x, -a.x * b.y)); }
__device__ __forceinline__ float2 mul_mi(float2 a) { return make_float2(a.y, -a.x); }   // a * (-i)
__device__ __forceinline__ float2 cswap(float2 a) { return make_float2(a.y, a.x); }

// ---- forward DFT_R on R registers, natural order in and out ------------------
template <int R> struct Dft;

template <> struct Dft<1> { __device__ __forceinline__ static void run(float2*) {} };

template <> struct Dft<2> {
    __device__ __forceinline__ static void run(float2* a)
    { float2 t = a[0]; a[0] = cadd(t, a[1]); a[1] = csub(t, a[1]); }
};

template <> struct Dft<4> {
    __device__ __forceinline__ static void run(float2* a)
    {
        float2 t0 = cadd(a[0], a[2]), t1 = csub(a[0], a[2]);
        float2 t2 = cadd(a[1], a[3]), t3 = mul_mi(csub(a[1], a[3]));
        a[0] = cadd(t0, t2); a[2] = csub(t0, t2);
        a[1] = cadd(t1, t3); a[3] = csub(t1, t3);
    }
};

template <> struct Dft<8> {
    __device__ __forceinline__ static void run(float2* a)
    {
        const float h = 0.70710678118654752440f;
        float2 e[4] = { a[0], a[2], a[4], a[6] };
        float2 o[4] = { a[1], a[3], a[5], a[7] };
        Dft<4>::run(e); Dft<4>::run(o);
        // o[k] *= w8^k : w8 = (1-i)/sqrt2, w8^2 = -i, w8^3 = (-1-i)/sqrt2
        o[1] = make_float2(h * (o[1].x + o[1].y), h * (o[1].y - o[1].x));
        o[2] = mul_mi(o[2]);
        o[3] = make_float2(h * (o[3].y - o[3].x), -h * (o[3].x + o[3].y));
#pragma unroll
        for (int k = 0; k < 4; ++k) { a[k] = cadd(e[k], o[k]); a[k + 4] = csub(e[k], o[k]); }
    }
};

// ---- radix-4 butterfly over twiddled inputs, scaled-twiddle form --------------------------------------------
// out = DFT4(z0, y1 w^k1, y2 w^(2 k1), y3 w^(3 k1)), w = exp(-2 pi i / R).  Each twiddle is written
// w^m = (-i)^q cos(t) (1 - i tan(t)), q the nearest quarter turn, |t| <= pi/4: u = (-i)^q y (1 - i tan) costs two
// FMAs (the quarter turn is a renaming with signs), and the cosines ride on the adds of the butterfly, which become
// FMAs at the same cost: z1 + z3 = c1 (u1 + (c3 / c1) u3), z0 + z2 = z0 + c2 u2, out0 = t0 + c1 S, ...
// 22 FMA-pipe operations instead of 28 (three complex multiplies and sixteen adds).  Measured: column passes 1.41 ->
// 1.35 ms (1024 points), 0.377 -> 0.368 ms (512); resident multislice 16.8 -> 16.65 ms.  Translation units that run
// their adds as packed FADD2 (PRISM_PACKED_ADDS: the row passes, window_out) keep the plain form: there a packed
// version of this butterfly (11 FFMA2) cut the instruction count by 10 % and was not faster (1.50 ms at 1024 points,
// 0.44 against 0.38 ms at 512).
#ifndef PRISM_TAN_TWIDDLES
#ifdef PRISM_PACKED_ADDS
#define PRISM_TAN_TWIDDLES 0
#else
#define PRISM_TAN_TWIDDLES 1
#endif
#endif
template <int R> __device__ __forceinline__ constexpr int tw_quarter(int m)
{ return (m % (R / 4) == R / 8) ? m / (R / 4) : (m + R / 8) / (R / 4); }
__device__ __forceinline__ float2 rot_quarter(float2 a, int q)      // a * (-i)^q
{
    switch (q & 3) {
        case 1: return make_float2(a.y, -a.x);
        case 2: return make_float2(-a.x, -a.y);
        case 3: return make_float2(-a.y, a.x);
        default: return a;
    }
}
template <int R>
__device__ __forceinline__ void twiddled_dft4(float2 z0, float2 y1, float2 y2, float2 y3, int k1,
                                              float2& o0, float2& o1, float2& o2, float2& o3)
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
    const float2 y[4] = { z0, y1, y2, y3 };
    float2 u[4];
    float c[4] = { 1.f, 1.f, 1.f, 1.f };
#pragma unroll
    for (int n2 = 1; n2 < 4; ++n2) {
        const int m = n2 * k1, q = tw_quarter<R>(m), j = m - q * (R / 4);
        const float tau = R == 16 ? T16[j + 2] : T32[j + 4];
        c[n2] = R == 16 ? C16[j + 2] : C32[j + 4];
        const float2 v = y[n2];
        const float2 w = (j == 0) ? v : make_float2(fmaf(v.y, tau, v.x), fmaf(v.x, -tau, v.y));     // v (1 - i tan)
        u[n2] = rot_quarter(w, q);
    }
    const float2 t0 = make_float2(fmaf(u[2].x, c[2], z0.x), fmaf(u[2].y, c[2], z0.y));
    const float2 t1 = make_float2(fmaf(u[2].x, -c[2], z0.x), fmaf(u[2].y, -c[2], z0.y));
    const float r = c[3] / c[1];
    const float2 sp = make_float2(fmaf(u[3].x, r, u[1].x), fmaf(u[3].y, r, u[1].y));            // (z1 + z3) / c1
    const float2 dm = make_float2(fmaf(u[3].x, -r, u[1].x), fmaf(u[3].y, -r, u[1].y));          // (z1 - z3) / c1
    o0 = make_float2(fmaf(sp.x, c[1], t0.x), fmaf(sp.y, c[1], t0.y));
    o2 = make_float2(fmaf(sp.x, -c[1], t0.x), fmaf(sp.y, -c[1], t0.y));
    o1 = make_float2(fmaf(dm.y, c[1], t1.x), fmaf(dm.x, -c[1], t1.y));                          // t1 + (-i) c1 dm
    o3 = make_float2(fmaf(dm.y, -c[1], t1.x), fmaf(dm.x, c[1], t1.y));
}

template <> struct Dft<16> {
    __device__ __forceinline__ static void run(float2* a)
    {
        // n = 4 n1 + n2 ; k = k1 + 4 k2.  Y[n2][k1] = DFT4 over n1, then twiddle w16^(n2 k1), DFT4 over n2.
        float2 y[4][4];
#pragma unroll
        for (int n2 = 0; n2 < 4; ++n2) {
            y[n2][0] = a[n2]; y[n2][1] = a[n2 + 4]; y[n2][2] = a[n2 + 8]; y[n2][3] = a[n2 + 12];
            Dft<4>::run(y[n2]);
        }
#if PRISM_TAN_TWIDDLES
        {
            float2 z[4] = { y[0][0], y[1][0], y[2][0], y[3][0] };
            Dft<4>::run(z);
            a[0] = z[0]; a[4] = z[1]; a[8] = z[2]; a[12] = z[3];
        }
#pragma unroll
        for (int k1 = 1; k1 < 4; ++k1)
            twiddled_dft4<16>(y[0][k1], y[1][k1], y[2][k1], y[3][k1], k1, a[k1], a[k1 + 4], a[k1 + 8], a[k1 + 12]);
#else
        const float c1 = 0.92387953251128675613f, s1 = 0.38268343236508977173f;   // cos, sin(pi/8)
        const float h  = 0.70710678118654752440f;
        // w16^m = exp(-2 pi i m / 16): m=1 (c1,-s1) m=2 (h,-h) m=3 (s1,-c1) m=4 (0,-1) m=6 (-h,-h) m=9 (-c1, s1)
        y[1][1] = cmul(y[1][1], make_float2(c1, -s1));
        y[1][2] = cmul(y[1][2], make_float2(h, -h));
        y[1][3] = cmul(y[1][3], make_float2(s1, -c1));
        y[2][1] = cmul(y[2][1], make_float2(h, -h));
        y[2][2] = mul_mi(y[2][2]);
        y[2][3] = cmul(y[2][3], make_float2(-h, -h));
        y[3][1] = cmul(y[3][1], make_float2(s1, -c1));
        y[3][2] = cmul(y[3][2], make_float2(-h, -h));
        y[3][3] = cmul(y[3][3], make_float2(-c1, s1));
#pragma unroll
        for (int k1 = 0; k1 < 4; ++k1) {
            float2 z[4] = { y[0][k1], y[1][k1], y[2][k1], y[3][k1] };
            Dft<4>::run(z);
            a[k1] = z[0]; a[k1 + 4] = z[1]; a[k1 + 8] = z[2]; a[k1 + 12] = z[3];
        }
#endif
    }
};

template <> struct Dft<32> {
    __device__ __forceinline__ static void run(float2* a)
    {
        // n = 4 n1 + n2 (n1 < 8, n2 < 4); k = k1 + 8 k2.  Y[n2][k1] = DFT8 over n1, twiddle w32^(n2 k1), DFT4 over n2.
        float2 y[4][8];
#pragma unroll
        for (int n2 = 0; n2 < 4; ++n2) {
#pragma unroll
            for (int n1 = 0; n1 < 8; ++n1) y[n2][n1] = a[4 * n1 + n2];
            Dft<8>::run(y[n2]);
        }
#if PRISM_TAN_TWIDDLES
        {
            float2 z[4] = { y[0][0], y[1][0], y[2][0], y[3][0] };
            Dft<4>::run(z);
            a[0] = z[0]; a[8] = z[1]; a[16] = z[2]; a[24] = z[3];
        }
#pragma unroll
        for (int k1 = 1; k1 < 8; ++k1)
            twiddled_dft4<32>(y[0][k1], y[1][k1], y[2][k1], y[3][k1], k1, a[k1], a[k1 + 8], a[k1 + 16], a[k1 + 24]);
#else
        // w32^m = exp(-2 pi i m / 32) = (WC[m], -WS[m]) for m <= 21
        constexpr float WC[22] = { 1.f, 0.98078528040323044913f, 0.92387953251128675613f, 0.83146961230254523708f,
                                   0.70710678118654752440f, 0.55557023301960222474f, 0.38268343236508977173f,
                                   0.19509032201612826785f, 0.f, -0.19509032201612826785f, -0.38268343236508977173f,
                                   -0.55557023301960222474f, -0.70710678118654752440f, -0.83146961230254523708f,
                                   -0.92387953251128675613f, -0.98078528040323044913f, -1.f, -0.98078528040323044913f,
                                   -0.92387953251128675613f, -0.83146961230254523708f, -0.70710678118654752440f,
                                   -0.55557023301960222474f };
        constexpr float WS[22] = { 0.f, 0.19509032201612826785f, 0.38268343236508977173f, 0.55557023301960222474f,
                                   0.70710678118654752440f, 0.83146961230254523708f, 0.92387953251128675613f,
                                   0.98078528040323044913f, 1.f, 0.98078528040323044913f, 0.92387953251128675613f,
                                   0.83146961230254523708f, 0.70710678118654752440f, 0.55557023301960222474f,
                                   0.38268343236508977173f, 0.19509032201612826785f, 0.f, -0.19509032201612826785f,
                                   -0.38268343236508977173f, -0.55557023301960222474f, -0.70710678118654752440f,
                                   -0.83146961230254523708f };
#pragma unroll
        for (int n2 = 1; n2 < 4; ++n2)
#pragma unroll
            for (int k1 = 1; k1 < 8; ++k1)
                y[n2][k1] = cmul(y[n2][k1], make_float2(WC[n2 * k1], -WS[n2 * k1]));
#pragma unroll
        for (int k1 = 0; k1 < 8; ++k1) {
            float2 z[4] = { y[0][k1], y[1][k1], y[2][k1], y[3][k1] };
            Dft<4>::run(z);
            a[k1] = z[0]; a[k1 + 8] = z[1]; a[k1 + 16] = z[2]; a[k1 + 24] = z[3];
        }
#endif
    }
};

// ---- plan ---------------------------------------------------------------------
template <int N_, int E_, int R1_, int R2_, int R3_>
struct Plan {
    static constexpr int N = N_, E = E_, T = N_ / E_, R1 = R1_, R2 = R2_, R3 = R3_;
    static_assert(R1_ * R2_ * R3_ == N_, "radices must multiply to N");
    static_assert(E_ % R1_ == 0 && E_ % R2_ == 0 && E_ % R3_ == 0, "each radix must divide E");
    static constexpr int NB1 = E_ / R1_, NB2 = E_ / R2_, NB3 = (R3_ > 1 ? E_ / R3_ : 1);
    // stage-2 twiddles depend on (t + T m) mod R1: shared by all m when R1 divides T
    static constexpr bool S2_SHARED = (T % R1_ == 0);
    static constexpr int  S2_SETS = S2_SHARED ? 1 : NB2;
    static constexpr int  PADDED = N_ + N_ / 16;      // padded exchange index space
};

template <int N> struct PlanFor;
template <> struct PlanFor<16>   { using type = Plan<16, 4, 4, 4, 1>; };
template <> struct PlanFor<32>   { using type = Plan<32, 8, 8, 4, 1>; };
template <> struct PlanFor<64>   { using type = Plan<64, 8, 8, 8, 1>; };
template <> struct PlanFor<128>  { using type = Plan<128, 16, 16, 8, 1>; };
template <> struct PlanFor<256>  { using type = Plan<256, 16, 16, 16, 1>; };
template <> struct PlanFor<512>  { using type = Plan<512, 16, 16, 16, 2>; };
template <> struct PlanFor<1024> { using type = Plan<1024, 16, 16, 16, 4>; };
template <> struct PlanFor<2048> { using type = Plan<2048, 16, 16, 16, 8>; };

__device__ __forceinline__ int pad16(int i) { return i + (i >> 4); }

// Per-thread twiddles, loaded once from the table tw[m] = exp(-2 pi i m / N) and kept in registers.
template <class P>
struct Twiddles {
    float2 s2[P::S2_SETS][P::R2 > 1 ? P::R2 - 1 : 1];
    float2 s3[P::NB3][P::R3 > 1 ? P::R3 - 1 : 1];

    __device__ __forceinline__ void load(const float2* __restrict__ tw, int t)
    {
#pragma unroll
        for (int m = 0; m < P::S2_SETS; ++m) {
            int k = (t + P::T * m) % P::R1;
#pragma unroll
            for (int r = 1; r < P::R2; ++r)
                s2[m][r - 1] = __ldg(tw + ((r * k * (P::N / (P::R1 * P::R2))) & (P::N - 1)));
        }
        if (P::R3 > 1) {
#pragma unroll
            for (int m = 0; m < P::NB3; ++m) {
                int k = (t + P::T * m) % (P::R1 * P::R2);
#pragma unroll
                for (int r = 1; r < P::R3; ++r)
                    s3[m][r - 1] = __ldg(tw + ((r * k) & (P::N - 1)));
            }
        }
    }
    __device__ __forceinline__ float2 get2(int m, int r) const { return s2[P::S2_SHARED ? 0 : m][r - 1]; }
    __device__ __forceinline__ float2 get3(int m, int r) const { return s3[m][r - 1]; }
};

// The same twiddles kept in shared memory, transposed so that the threads of a line read consecutive
// words:  t2[(r-1) * R1 + k] = w_N^(r k N / (R1 R2)),  t3[(r-1) * R1 R2 + k] = w_N^(r k).
// Costs one LDS.64 per use instead of 2 (R2 - 1 + NB3 (R3 - 1)) registers per thread.
template <class P>
struct SmemTwiddles {
    static constexpr int N2 = (P::R2 > 1 ? P::R2 - 1 : 0) * P::R1;
    static constexpr int N3 = (P::R3 > 1 ? (P::R3 - 1) * P::R1 * P::R2 : 0);
    static constexpr int COUNT = N2 + N3;            // float2 entries
    const float2* t2;
    const float2* t3;
    int k2[P::NB2];                                   // (t + T m) mod R1
    int k3[P::NB3];                                   // (t + T m) mod R1 R2

    // every thread of the CTA calls fill(); the caller synchronises before the first transform
    __device__ __forceinline__ static void fill(float2* table, const float2* __restrict__ tw, int tid, int nthreads)
    {
        for (int i = tid; i < N2; i += nthreads) {
            const int r = i / P::R1 + 1, k = i % P::R1;
            table[i] = __ldg(tw + ((r * k * (P::N / (P::R1 * P::R2))) & (P::N - 1)));
        }
        for (int i = tid; i < N3; i += nthreads) {
            const int r = i / (P::R1 * P::R2) + 1, k = i % (P::R1 * P::R2);
            table[N2 + i] = __ldg(tw + ((r * k) & (P::N - 1)));
        }
    }
    __device__ __forceinline__ void bind(const float2* table, int t)
    {
        t2 = table; t3 = table + N2;
#pragma unroll
        for (int m = 0; m < P::NB2; ++m) k2[m] = (t + P::T * m) % P::R1;
#pragma unroll
        for (int m = 0; m < P::NB3; ++m) k3[m] = (t + P::T * m) % (P::R1 * P::R2);
    }
    __device__ __forceinline__ float2 get2(int m, int r) const { return t2[(r - 1) * P::R1 + k2[m]]; }
    __device__ __forceinline__ float2 get3(int m, int r) const { return t3[(r - 1) * P::R1 * P::R2 + k3[m]]; }
};

// Shared-memory view of one line's exchange space: element idx lives at
// base[pad16(idx) * stride].  stride = 1 for a row buffer, (W+1) for a column of
// a padded [rows][W+1] tile.  sync() is a barrier among the threads of one line (or more): the
// whole warp if the line fits in one, else the whole CTA (every thread of the CTA runs the same sequence).
template <class P>
struct LineSmem {
    float2* base;
    int stride;
    __device__ __forceinline__ void  st(int idx, float2 v) const { base[pad16(idx) * stride] = v; }
    __device__ __forceinline__ void  st2(int idx, float2 v0, float2 v1) const { st(idx, v0); st(idx + 1, v1); }
    __device__ __forceinline__ float2 ld(int idx) const { return base[pad16(idx) * stride]; }
    __device__ __forceinline__ void sync() const { if (P::T <= 32) __syncwarp(); else __syncthreads(); }
};

// Forward transform of the line held as v[e] = x[t + T e].  Begins with a
// sm.sync(), so `sm` may alias storage the line's threads have just read.
// TW supplies get2(m, r) / get3(m, r); SM supplies st(idx, v) / st2(even idx, v0, v1) / ld(idx) / sync().
template <class P, class TW, class SM>
__device__ __forceinline__ void fft_forward(float2 (&v)[P::E], const TW& tw, int t, const SM& sm)
{
    constexpr int E = P::E, T = P::T;
    sm.sync();                               // earlier readers of `sm` (previous transform, tile loads) are done
    // ---- stage 1: radix R1, Ns = 1, no twiddles ----
#pragma unroll
    for (int m = 0; m < P::NB1; ++m) {
        float2 a[P::R1];
#pragma unroll
        for (int r = 0; r < P::R1; ++r) a[r] = v[m + P::NB1 * r];
        Dft<P::R1>::run(a);
        const int j = t + T * m;
#pragma unroll
        for (int r = 0; r < P::R1; r += 2) sm.st2(j * P::R1 + r, a[r], a[r + 1]);   // even idx: may be one 16-byte store
    }
    sm.sync();
#pragma unroll
    for (int e = 0; e < E; ++e) v[e] = sm.ld(t + T * e);
    // ---- stage 2: radix R2, Ns = R1 ----
    if (P::R3 > 1) sm.sync();                // all reads done before the next exchange overwrites
#pragma unroll
    for (int m = 0; m < P::NB2; ++m) {
        float2 a[P::R2];
        a[0] = v[m];
#pragma unroll
        for (int r = 1; r < P::R2; ++r) a[r] = cmul(v[m + P::NB2 * r], tw.get2(m, r));
        Dft<P::R2>::run(a);
        if (P::R3 == 1) {
#pragma unroll
            for (int r = 0; r < P::R2; ++r) v[m + P::NB2 * r] = a[r];
        } else {
            const int j = t + T * m;
            const int k = j % P::R1;
            const int idx = (j / P::R1) * (P::R1 * P::R2) + k;
#pragma unroll
            for (int r = 0; r < P::R2; ++r) sm.st(idx + r * P::R1, a[r]);
        }
    }
    if (P::R3 > 1) {
        sm.sync();
#pragma unroll
        for (int e = 0; e < E; ++e) v[e] = sm.ld(t + T * e);
        // ---- stage 3: radix R3, Ns = R1 R2, in place ----
#pragma unroll
        for (int m = 0; m < P::NB3; ++m) {
            float2 a[P::R3 > 1 ? P::R3 : 1];
            a[0] = v[m];
#pragma unroll
            for (int r = 1; r < P::R3; ++r) a[r] = cmul(v[m + P::NB3 * r], tw.get3(m, r));
            Dft<P::R3>::run(a);
#pragma unroll
            for (int r = 0; r < P::R3; ++r) v[m + P::NB3 * r] = a[r];
        }
    }
}

// Unscaled inverse transform: forward transform of the (im, re)-swapped data.
template <class P, class TW, class SM>
__device__ __forceinline__ void fft_inverse(float2 (&v)[P::E], const TW& tw, int t, const SM& sm)
{
#pragma unroll
    for (int e = 0; e < P::E; ++e) v[e] = cswap(v[e]);
    fft_forward<P>(v, tw, t, sm);
#pragma unroll
    for (int e = 0; e < P::E; ++e) v[e] = cswap(v[e]);
}

}  // namespace prism
