// slice_pipe_row.cu -- software-pipelined row pass of the slice step (lines of 256 .. 1024 points).
//
// PAPER.md:44 Eq. (1)  psi <- psi * exp(i sigma V)          (transmission)
// PAPER.md:80 Eq. (2)  Psi <- Psi * exp(-i pi lambda q^2 t)  (propagation), "done in Fourier space"
//
// Same arithmetic and the same two-pass structure as slice_pass.cu (row pass IFFT_x . t . FFT_x,
// column pass FFT_y . P . IFFT_y, wave kept in mixed space A[w][y][kx] between them), organised so
// that HBM transfers, shared-memory exchanges and butterflies of different lines overlap:
//
//  * every thread holds E = 32 points, so lines up to 1024 points need ONE shared-memory exchange
//    per transform, and inter-stage twiddles come from a transposed shared table;
//  * a team is one warp.  It owns a landing buffer that the TMA engine fills with 1-D bulk copies
//    (cp.async.bulk + mbarrier transaction counts) and a separate exchange space; the next line is
//    requested as soon as the current one is in registers; results go straight from registers to
//    HBM.  There is no CTA-wide barrier in the loop, and 15 teams fit an SM at 128 registers;
//  * band-limit: after the column pass everything with |kx| > kx_max is exactly zero (2/3 rule,
//    BASELINE.json), so mixed space is only ever read and written for kx in [0, xband) and
//    [nx - xband, nx): the row pass moves 2 xband of the nx points of a line.
//
// 2048-point lines run on the packed kernels of slice_pk.cu.
// complex adds of the register butterflies as packed FADD2 (measured: 3-7 % faster row pass, slower column pass)
#define PRISM_PACKED_ADDS 1
#include "fft_core.cuh"
#include "pipe_plan.cuh"
#include "prism_internal.h"
#include "pipe_ptx.cuh"

namespace prism {

constexpr int ROW_MAX_TEAMS = 16;

// =============================================================================
// Row pass
// =============================================================================
// A team is one warp holding LPT = 32 / T lines.  Per team: one landing buffer the TMA engine fills with the
// in-band points of the next line group (compact: [0, xb) then [N - xb, N)) and one exchange space.  The
// landing buffer is refilled as soon as the group is in registers, so the copy of group i + 1 overlaps the
// whole computation of group i.  XBE > 0: the band is xband = XBE * T columns, known at compile time (then
// "in band" depends on the register index e only and out-of-band elements cost no instruction); XBE = 0: any
// xband, tested per element.
template <class P, int XBE>
struct RowCfg {
    static constexpr int T = P::T;
    static_assert(T <= 32, "one warp per line group");
    static constexpr int LPT = 32 / T;                           // lines per team
    static constexpr int LINE = P::N + 2 * (P::N / P::R1);       // padded exchange space of one line (float2)
    static constexpr int LANDW = XBE > 0 ? 2 * XBE * T : P::N;   // points of a line that are moved
    static constexpr int PER_TEAM = LPT * (LINE + LANDW) * 8;
    static constexpr int TWB = round_up_c(SmemTwiddles<P>::COUNT * 8, 128);
    static constexpr int TEAMS_BY_SMEM = (PIPE_SMEM_MAX - PIPE_HEADER - TWB) / PER_TEAM;
    static constexpr int TEAMS = TEAMS_BY_SMEM < ROW_MAX_TEAMS ? TEAMS_BY_SMEM : ROW_MAX_TEAMS;
    static constexpr int THREADS = TEAMS * 32;
    static constexpr size_t SMEM = PIPE_HEADER + TWB + (size_t)TEAMS * PER_TEAM;
};

// exchange space of one line: element idx at base[idx + 2 (idx / R1)].  Two pad words per group of R1 keep
// pairs (even idx, idx + 1) 16-byte aligned, so the radix-R1 outputs of a thread go out as 16-byte stores, and
// a quarter warp of such stores (stride R1 + 2 words) covers all banks once.
template <class P>
struct RowSm {
    float2* base;
    __device__ __forceinline__ static int phys(int idx) { return idx + 2 * (idx / P::R1); }
    __device__ __forceinline__ void  st(int idx, float2 v) const { base[phys(idx)] = v; }
    __device__ __forceinline__ void  st2(int idx, float2 v0, float2 v1) const
    { *reinterpret_cast<float4*>(base + phys(idx)) = make_float4(v0.x, v0.y, v1.x, v1.y); }
    __device__ __forceinline__ float2 ld(int idx) const { return base[phys(idx)]; }
    __device__ __forceinline__ void sync() const { __syncwarp(); }
};

template <class P, int MODE, int XBE>
__global__ void __launch_bounds__(RowCfg<P, XBE>::THREADS, 1) row_pipe_kernel(RowArgs g)
{
    using C = RowCfg<P, XBE>;
    constexpr int E = P::E, T = P::T, N = P::N;
    auto in_band = [&](int e, int kx, int xb) { return XBE > 0 ? (e < XBE || e >= E - XBE) : (kx < xb || kx >= N - xb); };
    extern __shared__ __align__(128) unsigned char smem_raw[];
    uint64_t* bars = reinterpret_cast<uint64_t*>(smem_raw);                    // [TEAMS]
    float2* twtab = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER);
    const int tid = threadIdx.x, team = tid >> 5, tt = tid & 31;
    const int ll = tt / T, t = tt % T;
    float2* land = reinterpret_cast<float2*>(smem_raw + PIPE_HEADER + C::TWB + (size_t)team * C::PER_TEAM);   // [LPT][LANDW]
    float2* xch = land + C::LPT * C::LANDW;                                                                    // [LPT][LINE]

    SmemTwiddles<P>::fill(twtab, g.tw_x, tid, C::THREADS);
    if (MODE != ROW_INIT && tt == 0) { mbar_init(&bars[team], 1); mbar_fence_init(); }
    __syncthreads();
    SmemTwiddles<P> tw;
    tw.bind(twtab, t);
    griddep_wait();                          // the previous kernel of the slice loop has completed (pipe_ptx.cuh)

    const long long n_lines = (long long)g.n_waves * g.ny;
    const long long n_groups = (n_lines + C::LPT - 1) / C::LPT;
    const long long gteam = (long long)blockIdx.x * C::TEAMS + team, gstride = (long long)gridDim.x * C::TEAMS;
    const int xb = XBE > 0 ? XBE * T : g.xband;              // in-band columns: [0, xb) and [N - xb, N)

    // one thread of the team: start the bulk copies of line group `grp` into the landing buffer
    auto issue = [&](long long grp) {
        uint64_t* bar = &bars[team];
        int n_act = 0;
#pragma unroll
        for (int l = 0; l < C::LPT; ++l) n_act += (grp * C::LPT + l < n_lines);
        mbar_expect_tx(bar, (unsigned)(n_act * 2 * xb * (int)sizeof(float2)));
#pragma unroll
        for (int l = 0; l < C::LPT; ++l) {
            const long long line = grp * C::LPT + l;
            if (line < n_lines) {
                const int y = (int)(line / g.n_waves), w = (int)(line % g.n_waves);
                const float2* row = g.a + ((size_t)w * g.ny + y) * N;
                float2* dst = land + l * C::LANDW;
                bulk_g2s(dst, row, (unsigned)(xb * sizeof(float2)), bar);
                bulk_g2s(dst + xb, row + (N - xb), (unsigned)(xb * sizeof(float2)), bar);
            }
        }
    };
    if (MODE != ROW_INIT && tt == 0 && gteam < n_groups) issue(gteam);

    const RowSm<P> sm{ xch + ll * C::LINE };
    int it = 0;
    for (long long grp = gteam; grp < n_groups; grp += gstride, ++it) {
        long long line = grp * C::LPT + ll;
        const bool active = line < n_lines;
        if (!active) line = n_lines - 1;                 // keep every thread in the barriers
        const int y = (int)(line / g.n_waves), w = (int)(line % g.n_waves);
        float2* row = g.a + ((size_t)w * g.ny + y) * N;
        float2 v[E];

        if (MODE == ROW_INIT) {
            // plane wave exp(+2 pi i (kx x / nx + ky y / ny)) * amplitude
            const int2 b = g.beams[w];
            const float2 wy = __ldg(g.tw_y + ((b.y * y) & (g.ny - 1)));
            const float2 base = make_float2(wy.x * g.scale, -wy.y * g.scale);
            // exp(+2 pi i kx (t + T e) / N) = conj(w^(kx t)) conj(w^(kx T e)): one gathered table value per thread and
            // one warp-uniform value per slot instead of E gathered loads
            const float2 bt = cmul_conj(base, __ldg(g.tw_x + ((b.x * t) & (N - 1))));
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const float2 we = __ldg(g.tw_x + ((b.x * T * e) & (N - 1)));
                v[e] = cmul_conj(bt, we);
            }
        } else {
            mbar_wait(&bars[team], (unsigned)(it & 1));
            const float2* lbase = land + ll * C::LANDW;
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int kx = t + T * e;
                int pos;                                    // compact landing: [0, xb) then [N - xb, N)
                if (XBE > 0) pos = e < XBE ? kx : kx - (N - 2 * xb);
                else pos = kx < xb ? kx : (kx >= N - xb ? kx - (N - 2 * xb) : 0);
                if (XBE > 0 && !in_band(e, kx, xb)) { v[e] = make_float2(0.f, 0.f); continue; }
                const float2 q = lbase[pos];
                v[e] = in_band(e, kx, xb) ? q : make_float2(0.f, 0.f);            // out of band: exact zeros
            }
            // the landing buffer is free once every lane has read its points
            __syncwarp();
            if (tt == 0 && grp + gstride < n_groups) { fence_proxy_async(); issue(grp + gstride); }
        }

        if (MODE == ROW_STEP || MODE == ROW_FINAL) fft_inverse<P>(v, tw, t, sm);

        if (MODE == ROW_INIT || MODE == ROW_STEP) {
            const float2* trow = g.t + (size_t)y * N;
#pragma unroll
            for (int e = 0; e < E; ++e) v[e] = cmul(v[e], __ldg(trow + t + T * e));
        }
        if (MODE != ROW_FINAL) fft_forward<P>(v, tw, t, sm);

        if (MODE == ROW_FINAL) {
            float2* dst = g.out + ((size_t)w * g.ny + y) * N;
            if (active) {
#pragma unroll
                for (int e = 0; e < E; ++e) dst[t + T * e] = make_float2(v[e].x * g.scale, v[e].y * g.scale);
            }
        } else if (active) {
#pragma unroll
            for (int e = 0; e < E; ++e) {
                const int kx = t + T * e;
                if (in_band(e, kx, xb)) row[kx] = v[e];
            }
        }
    }
}

template <class P, int MODE, int XBE>
static cudaError_t launch_row_pipe_x(const RowArgs& g, cudaStream_t stream)
{
    using C = RowCfg<P, XBE>;
    auto kern = row_pipe_kernel<P, MODE, XBE>;
    static PerDevice once{};
    if (cudaError_t e = opt_in_smem(kern, C::SMEM, once); e != cudaSuccess) return e;
    const long long n_lines = (long long)g.n_waves * g.ny;
    const long long n_groups = (n_lines + C::LPT - 1) / C::LPT;
    if (n_groups == 0) return cudaSuccess;
    long long grid = (n_groups + C::TEAMS - 1) / C::TEAMS;
    if (grid > num_sms()) grid = num_sms();
    return launch_pdl(kern, (unsigned)grid, C::THREADS, C::SMEM, stream, g);
}


template <class P, int MODE>
static cudaError_t launch_row_pipe_t(const RowArgs& g, cudaStream_t stream)
{
    constexpr int XB = DefaultBand<P::N>::XB;
    static_assert(XB % P::T == 0, "default band must be a whole number of register slots");
    if (g.xband == XB) return launch_row_pipe_x<P, MODE, XB / P::T>(g, stream);
    return launch_row_pipe_x<P, MODE, 0>(g, stream);
}

template <int N>
static cudaError_t launch_row_pipe_n(RowMode mode, const RowArgs& g, cudaStream_t stream)
{
    using P = typename PipePlan<N>::type;
    switch (mode) {
        case ROW_INIT:  return launch_row_pipe_t<P, ROW_INIT>(g, stream);
        case ROW_STEP:  return launch_row_pipe_t<P, ROW_STEP>(g, stream);
        case ROW_FINAL: return launch_row_pipe_t<P, ROW_FINAL>(g, stream);
        default: break;
    }
    return cudaErrorInvalidValue;
}

cudaError_t launch_row_pipe(RowMode mode, const RowArgs& g, cudaStream_t stream)
{
    if (g.xband < 4 || g.xband % 4 || 2 * g.xband > g.nx) return cudaErrorInvalidValue;
    switch (g.nx) {
        case 256:  return launch_row_pipe_n<256>(mode, g, stream);
        case 512:  return launch_row_pipe_n<512>(mode, g, stream);
        case 1024: return launch_row_pipe_n<1024>(mode, g, stream);
    }
    return cudaErrorInvalidValue;
}

}  // namespace prism
